"""Writes tests/golden/fullsize_run_<config>.txt: the ORACLE's own free run (oracle.Oracle.solve, fp64, eps = 1e-9) of
the whole column-generation loop of PAPER.md:111-117 on a full-size seeded phantom (BASELINE.json configs[1] "prostate",
configs[2] "hn", configs[4] "stress"; seed 0; 102 s, 271 s and 2508 s on 8 cores), one line per iteration: the beam chosen, its price, F, G, F + gamma G after the master solve,
and the leaf pairs of the committed aperture.

    python tests/golden/make_fullsize_runs.py [prostate] [hn] [stress]     (default: prostate hn)

It imports only `oracle` and `vmat_inputs` (never the CUDA package): the stored values are the oracle's.  The GPU test
tests/test_gpu_fullsize.py::test_whole_plan_matches_the_stored_oracle_run compares the device's whole run with them,
which the oracle is too slow to produce inside the test suite for configs[2] (minutes on 16 host threads).
"""
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))

import vmat_inputs  # noqa: E402
from oracle import Oracle  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
EPS = 1e-9


def write_run(name: str) -> str:
    ph = vmat_inputs.make_phantom(name, seed=0)
    o = Oracle.from_phantom(ph)
    t0 = time.time()
    occ, left, right, y, z, tr = o.solve(o.N, eps=EPS)
    dt = time.time() - t0
    assert tr.iters == o.N and occ.all()
    path = os.path.join(HERE, f"fullsize_run_{name}.txt")
    with open(path, "w") as f:
        f.write(f"# oracle free run, vmat_inputs.make_phantom({name!r}, seed=0), Oracle.solve(N, eps={EPS:g}); "
                f"written by tests/golden/make_fullsize_runs.py\n")
        f.write(f"# N {o.N} R {o.R} C {o.C} V {o.V} nnz {len(o.val)} gamma {o.gamma!r} delta {o.delta}\n")
        f.write("# it beam price F G cost | left[R] | right[R]   (leaf pairs of the aperture committed at this iteration)\n")
        for it in range(tr.iters):
            l = " ".join(str(int(v)) for v in tr.left[it])
            r = " ".join(str(int(v)) for v in tr.right[it])
            f.write(f"{it} {int(tr.beam[it])} {float(tr.price[it])!r} {float(tr.F[it])!r} {float(tr.G[it])!r} "
                    f"{float(tr.cost[it])!r} | {l} | {r}\n")
        f.write("# final y\n")
        f.write("y " + " ".join(repr(float(v)) for v in y) + "\n")
    print(f"{name}: {tr.iters} iterations in {dt:.1f} s, final cost {float(tr.cost[-1])!r} -> {path}")
    return path


if __name__ == "__main__":
    for name in (sys.argv[1:] or ["prostate", "hn"]):
        write_run(name)
