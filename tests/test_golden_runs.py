"""The stored full-size oracle runs (tests/golden/fullsize_run_*.txt, written by tests/golden/make_fullsize_runs.py from
oracle/ alone) checked on what PAPER.md fixes for any run of the loop, without a GPU and without re-running the oracle:
one aperture per beam, deliverable leaf pairs inside the leaf-travel limit of their neighbours
(PAPER.md:111), cost = F + gamma G (Eq. 3) and never increasing from one iteration to the next (the
new aperture enters at y = 0 and the master problem is solved to optimality: DESIGN.md S2)."""
import os
import re

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    path = os.path.join(GOLDEN, f"fullsize_run_{name}.txt")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated")
    meta, rows, y = {}, [], None
    for line in open(path):
        if line.startswith("# N "):
            tok = line[2:].split()
            meta = {tok[i]: float(tok[i + 1]) for i in range(0, len(tok), 2)}
        elif line.startswith("#"):
            continue
        elif line.startswith("y "):
            y = np.array([float(v) for v in line.split()[1:]])
        else:
            head, l, r = line.split("|")
            h = head.split()
            rows.append((int(h[0]), int(h[1]), float(h[2]), float(h[3]), float(h[4]), float(h[5]),
                         np.array(l.split(), int), np.array(r.split(), int)))
    return meta, rows, y


@pytest.mark.parametrize("name", ["prostate", "hn", "stress"])
def test_stored_run_is_a_run_of_the_loop(name):
    meta, rows, y = load(name)
    N, R, C, gamma, delta = int(meta["N"]), int(meta["R"]), int(meta["C"]), meta["gamma"], int(meta["delta"])
    assert len(rows) == N and [r[0] for r in rows] == list(range(N))
    beams = np.array([r[1] for r in rows])
    assert sorted(beams.tolist()) == list(range(N))                       # every beam exactly once
    left = np.zeros((N, R), int)
    right = np.zeros((N, R), int)
    occ = np.zeros(N, bool)
    prev = np.inf
    for it, k, price, F, G, cost, l, r in rows:
        assert l.shape == (R,) and r.shape == (R,)
        assert np.all(0 <= l) and np.all(l <= r) and np.all(r <= C)       # a leaf pair, possibly closed
        # inside the leaf-travel box of the nearest occupied beam on either side at the time it was chosen
        for kk in (max([j for j in np.flatnonzero(occ) if j < k], default=None),
                   min([j for j in np.flatnonzero(occ) if j > k], default=None)):
            if kk is not None:
                b = delta * abs(k - kk)
                assert np.all(np.abs(l - left[kk]) <= b) and np.all(np.abs(r - right[kk]) <= b), (it, k, kk)
        left[k], right[k], occ[k] = l, r, True
        assert abs(cost - (F + gamma * G)) <= 1e-12 * abs(cost)
        assert cost <= prev * (1 + 1e-12), (it, cost, prev)
        assert price < 0.0 or it > 0                                       # the first aperture always pays
        prev = cost
    assert y is not None and y.shape == (N,) and np.all(y >= 0)
    # the smoothing term of the final dose rates is the stored G (Eq. 2 over all N angles: every beam is occupied)
    theta = np.arange(N) * (360.0 / N)
    G_end = float(np.sum((y[1:] - y[:-1]) ** 2 / (theta[1:] - theta[:-1])))
    assert abs(G_end - rows[-1][4]) <= 1e-9 * max(1.0, abs(G_end))
