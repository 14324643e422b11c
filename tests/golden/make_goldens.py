"""Writes tests/golden/oracle_goldens.json by running ONLY the CPU oracle (oracle/).

Expected values for the full-size parity tests of BASELINE.json configs 2-5, where running the
oracle inside the test would take too long.  Nothing here touches the CUDA path.  Each job is
one oracle trajectory; checkpoints are [pass, E, M, FNV-1a-64 of the canonical spins]; for jobs
with `series` the FNV-1a-64 of the little-endian int64 E series and M series (one value per
outer pass) up to each checkpoint is stored too.  All jobs use the default RNG mapping "planes"
(DESIGN.md §3.4); the words mapping is pinned by survey_appendix_a.json on the same configs.

    python tests/golden/make_goldens.py [--only SUBSTR] [--procs 8]

Takes ~20-30 min on 8 cores for everything.  Existing entries are kept unless re-run.
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
OUT = os.path.join(HERE, "oracle_goldens.json")

BC = 0.4406868


def jobs():
    J = []
    # config 2: L=1024, tile 32, k=4, five temperatures, full 10^4 passes, E/M series
    for b in (0.30, 0.40, BC, 0.50, 0.60):
        J.append(dict(name=f"c2_beta{b}", dim=2, L=1024, seeds=[2], beta=b, tile=32, k=4,
                      checkpoints=[1, 10, 100, 1000, 10000], series=True))
    # config 3: L=16384, two passes of each of the six trajectories
    for T in (32, 64):
        for k in (1, 4, 16):
            J.append(dict(name=f"c3_L16384_t{T}_k{k}", dim=2, L=16384, seeds=[3], beta=BC, tile=T, k=k,
                          checkpoints=[1, 2]))
            J.append(dict(name=f"c3_L2048_t{T}_k{k}", dim=2, L=2048, seeds=[3], beta=BC, tile=T, k=k,
                          checkpoints=[1, 2, 50, 200]))
    # row a8 at the bench size: plain checkerboard (tile == L) on the config-3 and config-4 lattices, two sweeps
    J.append(dict(name="c3_L16384_plain", dim=2, L=16384, seeds=[3], beta=BC, tile=16384, k=1, checkpoints=[1, 2]))
    J.append(dict(name="c4_plain", dim=3, L=256, seeds=[4], beta=0.2216546, tile=256, k=1, checkpoints=[1, 2]))
    # config 4: 3D L=256, tile 8
    for k in (1, 4):
        J.append(dict(name=f"c4_k{k}", dim=3, L=256, seeds=[4], beta=0.2216546, tile=8, k=k,
                      checkpoints=[1, 10, 100, 500]))
    # config 5: ±J glass L=4096 at the depth SURVEY §8(d) lists: all 16 replicas (with the 120 overlaps) to 100 passes,
    # two replicas in full (1000 passes), two more to 100
    J.append(dict(name="c5_all16", dim=2, L=4096, seeds=list(range(100, 116)), jseed=5, beta=1.0, tile=32, k=4,
                  checkpoints=[1, 10, 100], overlaps=True))
    for sd in (100, 101):
        J.append(dict(name=f"c5_seed{sd}", dim=2, L=4096, seeds=[sd], jseed=5, beta=1.0, tile=32, k=4,
                      checkpoints=[1, 10, 100, 1000]))
    for sd in (114, 115):
        J.append(dict(name=f"c5_seed{sd}", dim=2, L=4096, seeds=[sd], jseed=5, beta=1.0, tile=32, k=4,
                      checkpoints=[1, 10, 100]))
    return J


def run(job):
    from oracle import oracle as O
    import ising_workloads as W
    t0 = time.time()
    Jarr = W.couplings(job["dim"], job["L"], job["jseed"]) if "jseed" in job else None
    o = O.Oracle(job["dim"], job["L"], seeds=job["seeds"], J=Jarr, rng=job.get("rng", "planes"))
    R = len(job["seeds"])
    res = dict(job)
    res["rng"] = job.get("rng", "planes")
    cps = []
    E0, M0 = o.observables()
    cps.append([0, [int(v) for v in E0], [int(v) for v in M0], ["%016x" % o.hash(r) for r in range(R)]])
    done = 0
    Es, Ms = [], []
    for p in job["checkpoints"]:
        if job.get("series"):
            E, M = o.sweep_series(job["beta"], p - done, job["tile"], job["k"])
            Es.append(E); Ms.append(M)
        else:
            o.sweep(job["beta"], p - done, job["tile"], job["k"])
        done = p
        E1, M1 = o.observables()
        cp = [p, [int(v) for v in E1], [int(v) for v in M1], ["%016x" % o.hash(r) for r in range(R)]]
        if job.get("series"):
            cp.append("%016x" % O.hash_bytes(np.ascontiguousarray(np.concatenate(Es)).astype("<i8")))
            cp.append("%016x" % O.hash_bytes(np.ascontiguousarray(np.concatenate(Ms)).astype("<i8")))
        if job.get("overlaps"):
            cp.append({f"{a},{b}": o.overlap(a, b) for a in range(R) for b in range(a + 1, R)})
        cps.append(cp)
    res["checkpoints"] = cps
    res["oracle_seconds"] = round(time.time() - t0, 1)
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="")
    ap.add_argument("--procs", type=int, default=8)
    a = ap.parse_args()
    from oracle import oracle as O
    O.build()
    todo = [j for j in jobs() if a.only in j["name"]]
    # longest first
    todo.sort(key=lambda j: -(j["L"] ** j["dim"]) * j["k"] * max(j["checkpoints"]) * len(j["seeds"]))
    data = {}
    if os.path.exists(OUT):
        data = json.load(open(OUT))
    with mp.Pool(a.procs) as pool:
        for res in pool.imap_unordered(run, todo):
            data[res["name"]] = res
            print(res["name"], res["oracle_seconds"], "s", flush=True)
            with open(OUT + ".tmp", "w") as f:
                json.dump(dict(sorted(data.items())), f, indent=1)
            os.replace(OUT + ".tmp", OUT)


if __name__ == "__main__":
    main()
