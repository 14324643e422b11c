"""Differential fuzz of the kernel dispatch: seeded random (dim, L, tile, k, n, replicas, layout, couplings, jit mode, series
or not) through whatever kernel family the library chooses, against a launch per coarse colour / per half-sweep of the same
call (ising_force_path 2 — the families pinned to the oracle element by element in test_gpu_parity.py).  Integer work: spins
compared on the device, E, M and the series exactly.  It found the one geometry (an odd number of tiles of a colour per tile
row) on which the strip mapping of k_grid_planes hung; lattices whose tile counts are 2 x odd are therefore drawn on purpose.
Every run is a subprocess with a time limit, so that a kernel that waits for ever fails the test instead of the session."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

CODE = r'''
import os, random, numpy as np, torch
import paper_1006_3865_b200 as P
import ising_workloads as W
P.use_torch()
rnd = random.Random(int(os.environ["FSEED"]))
bad, paths = 0, {}
for it in range(int(os.environ["NCASE"])):
    T = rnd.choice([32, 64])
    B = rnd.choice(list(range(10, 66, 2)))
    L = min(B * T, T * (4096 // T))
    R = rnd.choice([1, 1, 1, 2, 3])
    k = rnd.choice([1, 1, 2, 3, 4])
    n = rnd.randint(2, 10)
    mode = rnd.choice(["dc", "dc", "dc", "plain", "masked"])
    tile = T if mode == "dc" else (0 if mode == "plain" else rnd.choice([4, 8, 16, 128]))
    if tile and (L % tile or (L // tile) % 2): tile = 16
    bits = rnd.random() < 0.4
    jseed = rnd.choice([None, None, 5, 9])
    beta = rnd.choice([0.3, 0.4406868, 0.6, 1.0])
    dim = 2
    if rnd.random() < 0.2:
        dim, L, R = 3, 16 * rnd.randint(4, 10), rnd.choice([1, 2])
        tile = rnd.choice([8, 8, 8, 0, 4, 16])
        if tile and (L % tile or (L // tile) % 2): tile = 8
    if R * L ** dim > (1 << 25): R = 1
    seeds = [rnd.getrandbits(64) for _ in range(R)]
    jit = rnd.choice(["auto", "on", "off"])
    series = rnd.random() < 0.3
    J = W.couplings(dim, L, jseed) if jseed is not None else None
    a = P.Ising(dim, L, coupling=J, seeds=seeds); b = P.Ising(dim, L, coupling=J, seeds=seeds)
    if bits: a.set_layout(P.ISING_LAYOUT_BITS); b.set_layout(P.ISING_LAYOUT_BITS)
    a.set_jit(jit); b.force_path(2)
    ok = True
    if series:
        Ea, Ma = a.sweep_series(beta, n, tile, k); Eb, Mb = b.sweep_series(beta, n, tile, k)
        ok = np.array_equal(Ea, Eb) and np.array_equal(Ma, Mb)
    else:
        a.sweep(beta, n, tile, k); b.sweep(beta, n, tile, k)
    pa = a.sweep_path()
    sa = torch.empty(R * L ** dim, dtype=torch.int8, device="cuda"); sb = torch.empty_like(sa)
    a.copy_spins(sa); b.copy_spins(sb)
    ok = ok and bool(torch.equal(sa, sb))
    Ea, Ma = a.observables(); Eb, Mb = b.observables()
    ok = ok and list(Ea) == list(Eb) and list(Ma) == list(Mb)
    paths[pa] = paths.get(pa, 0) + 1
    if not ok:
        bad += 1
        print("MISMATCH", dict(dim=dim, L=L, tile=tile, k=k, n=n, R=R, bits=bits, jseed=jseed, beta=beta, jit=jit, series=series, path=pa, other=b.sweep_path()), flush=True)
    a.destroy(); b.destroy()
print("fuzz done: bad", bad, "families", len(paths), sorted(paths), flush=True)
'''


@pytest.mark.parametrize("seed,cases,env", [
    (101, 70, {}),                                                   # the launch configurations the library chooses
    (102, 50, {"ISING_GRID_WARPS": "64", "ISING_G2_PARK": "0"}),     # few resident warps: several jobs per warp, strips, unparked constants
    (103, 50, {"ISING_GRID_WARPS": "200"}),
])
def test_dispatch_against_per_colour_launches(seed, cases, env):
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", CODE], cwd=root, capture_output=True, text=True, timeout=900,
                         env=dict(os.environ, FSEED=str(seed), NCASE=str(cases), PYTHONPATH=root, **env))
    assert out.returncode == 0, out.stderr[-3000:]
    assert "fuzz done: bad 0 " in out.stdout, out.stdout[-3000:]
    families = int(out.stdout.split("families")[1].split()[0])
    assert families >= 8, out.stdout[-2000:]                          # the draw reaches many kernel families
