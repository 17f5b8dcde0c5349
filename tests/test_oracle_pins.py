"""Pins for the CPU oracle (oracle/vmat_oracle.c) against things other than itself:
closed forms, finite differences, brute force, library routines, invariants.
All CPU (-m "not gpu").  Citations: PAPER.md lines / SURVEY.md 8c readings.
"""
import itertools

import numpy as np
import pytest
import scipy.optimize
import scipy.sparse as sp

import oracle as orc
from oracle import Oracle


# ------------------------------------------------------------------------------------------------
# helpers: a small random problem with a dense D we can multiply by hand
# ------------------------------------------------------------------------------------------------
def small_problem(seed=0, V=37, N=5, R=3, C=6, density=0.4, gamma=0.3, delta=1, nonuniform_theta=False):
    rng = np.random.default_rng(seed)
    B = N * R * C
    dense = rng.random((B, V)).astype(np.float32) * (rng.random((B, V)) < density)
    dense[rng.integers(0, B, 3)] = 0.0                      # some empty rows
    csr = sp.csr_matrix(dense)
    csr.sort_indices()
    T = rng.uniform(0.2, 1.0, V).astype(np.float32)
    alpha = (rng.random(V) < 0.5) * rng.uniform(0.5, 2.0, V)
    beta = rng.uniform(0.1, 1.5, V)
    theta = np.cumsum(rng.uniform(1.0, 3.0, N)) if nonuniform_theta else np.arange(N) * 2.0
    o = Oracle(csr.indptr.astype(np.int64), csr.indices.astype(np.int32), csr.data.astype(np.float32),
               T, alpha.astype(np.float32), beta.astype(np.float32), theta, R, C, delta, gamma)
    return o, dense.astype(np.float64), rng


def random_plan(o, rng, n_occ):
    occ = np.zeros(o.N, np.uint8)
    occ[rng.choice(o.N, n_occ, replace=False)] = 1
    left = rng.integers(0, o.C + 1, (o.N, o.R)).astype(np.int32)
    right = np.array([[rng.integers(l, o.C + 1) for l in row] for row in left], np.int32)
    y = rng.uniform(0.1, 2.0, o.N) * occ
    return occ, left, right, y


def open_mask(o, occ, left, right):
    """x_i = 1 if beamlet i is exposed in an occupied beam (the set A_k)."""
    m = np.zeros((o.N, o.R, o.C))
    for k in range(o.N):
        if occ[k]:
            for r in range(o.R):
                m[k, r, left[k, r]:right[k, r]] = 1.0
    return m


# ------------------------------------------------------------------------------------------------
# O2 dose / O4 prices: plain (sparse) matrix-vector products
# ------------------------------------------------------------------------------------------------
def test_dose_equals_dense_product():
    # z = D^T x, x_i = y_k [i in A_k]
    o, D, rng = small_problem(1)
    occ, left, right, y = random_plan(o, rng, 3)
    x = (open_mask(o, occ, left, right) * y[:, None, None]).reshape(-1)
    z = o.dose(occ, left, right, y)
    np.testing.assert_allclose(z, D.T @ x, rtol=1e-13, atol=1e-13)


def test_dose_single_entry_by_hand():
    # one beam, one row, two beamlets, two voxels:  z = y * (D_0. + D_1.)
    row_ptr = np.array([0, 2, 3], np.int64)
    col = np.array([0, 1, 1], np.int32)
    val = np.array([0.5, 0.25, 2.0], np.float32)
    o = Oracle(row_ptr, col, val, [1, 1], [1, 1], [1, 1], [0.0], 1, 2, 1, 0.1)
    z = o.dose([1], [[0]], [[2]], [3.0])
    np.testing.assert_allclose(z, [1.5, 3.0 * 2.25])
    z = o.dose([1], [[1]], [[2]], [3.0])          # only beamlet 1 open
    np.testing.assert_allclose(z, [0.0, 6.0])
    z = o.dose([1], [[1]], [[1]], [3.0])          # closed row
    np.testing.assert_allclose(z, [0.0, 0.0])


def test_prices_equal_scipy_spmv(tiny_phantom, tiny_oracle):
    # g = D w against scipy.sparse in fp64
    ph, o = tiny_phantom, tiny_oracle
    rng = np.random.default_rng(3)
    w = rng.standard_normal(o.V)
    A = sp.csr_matrix((ph.val.astype(np.float64), ph.col_idx, ph.row_ptr), shape=(o.B, o.V))
    g = o.prices(w)
    ref = A @ w
    np.testing.assert_allclose(g, ref, rtol=1e-12, atol=1e-12 * np.abs(ref).max())
    # occupied beams are not priced
    occ = np.zeros(o.N, np.uint8)
    occ[[2, 5]] = 1
    g2 = o.prices(w, occ).reshape(o.N, -1)
    assert np.all(g2[[2, 5]] == 0.0)
    np.testing.assert_array_equal(g2[[0, 1, 3]], g.reshape(o.N, -1)[[0, 1, 3]])


def test_dose_is_transpose_of_prices():
    # <D^T x, w> = <x, D w> ties O2 and O4 to the same matrix (catches a transposed operand)
    o, D, rng = small_problem(5)
    occ, left, right, y = random_plan(o, rng, o.N)
    x = (open_mask(o, occ, left, right) * y[:, None, None]).reshape(-1)
    w = rng.standard_normal(o.V)
    assert np.dot(o.dose(occ, left, right, y), w) == pytest.approx(np.dot(x, o.prices(w)), rel=1e-12)


# ------------------------------------------------------------------------------------------------
# O3 penalty (Eq. 1) and smoothing (Eq. 2)
# ------------------------------------------------------------------------------------------------
def test_penalty_closed_form_one_voxel():
    # Eq. 1: T=1, alpha=2, beta=3
    for z, F, w in [(0.4, 2 * 0.36, -2 * 2 * 0.6), (1.5, 3 * 0.25, 2 * 3 * 0.5), (1.0, 0.0, 0.0)]:
        Fo, wo = orc.penalty([z], [1.0], [2.0], [3.0])
        assert Fo == pytest.approx(F, rel=1e-14)
        assert wo[0] == pytest.approx(w, rel=1e-14, abs=0)
    # critical structure: alpha = 0 -> no penalty below threshold
    Fo, wo = orc.penalty([0.1], [0.5], [0.0], [1.0])
    assert Fo == 0.0 and wo[0] == 0.0


def test_penalty_gradient_finite_difference():
    rng = np.random.default_rng(7)
    V = 200
    T = rng.uniform(0.2, 1.0, V).astype(np.float32)
    a = rng.uniform(0, 2, V).astype(np.float32)
    b = rng.uniform(0, 2, V).astype(np.float32)
    z = rng.uniform(0.0, 1.5, V)
    _, w = orc.penalty(z, T, a, b)
    h = 1e-6
    for j in range(V):
        if abs(z[j] - T[j]) < 10 * h:
            continue                                   # F is C1 but not C2 at the kink
        zp, zm = z.copy(), z.copy()
        zp[j] += h
        zm[j] -= h
        fd = (orc.penalty(zp, T, a, b, False)[0] - orc.penalty(zm, T, a, b, False)[0]) / (2 * h)
        assert w[j] == pytest.approx(fd, rel=1e-6, abs=1e-7)


def test_smooth_closed_forms():
    N, dth = 9, 2.0
    th = np.arange(N) * dth
    G, dG = orc.smooth(np.full(N, 3.7), th)
    assert G == 0.0 and np.all(dG == 0.0)              # constant dose rate costs nothing
    G, _ = orc.smooth(np.arange(N, dtype=float), th)   # ramp: (N-1) unit steps / dtheta (Eq. 2)
    assert G == pytest.approx((N - 1) / dth, rel=1e-15)
    # units are degrees as passed (reading S4): halving the spacing doubles G
    G2, _ = orc.smooth(np.arange(N, dtype=float), th / 2)
    assert G2 == pytest.approx(2 * (N - 1) / dth, rel=1e-15)


def test_smooth_is_laplacian_quadratic_form_and_gradient():
    rng = np.random.default_rng(11)
    N = 12
    th = np.cumsum(rng.uniform(0.5, 3.0, N))
    y = rng.uniform(0, 2, N)
    L = np.zeros((N, N))                                # weighted path-graph Laplacian, no wrap-around (S3)
    for k in range(N - 1):
        wgt = 1.0 / (th[k + 1] - th[k])
        L[k, k] += wgt
        L[k + 1, k + 1] += wgt
        L[k, k + 1] -= wgt
        L[k + 1, k] -= wgt
    G, dG = orc.smooth(y, th)
    assert G == pytest.approx(y @ L @ y, rel=1e-13)
    np.testing.assert_allclose(dG, 2 * L @ y, rtol=1e-12, atol=1e-13)
    h = 1e-6
    for k in range(N):
        yp, ym = y.copy(), y.copy()
        yp[k] += h
        ym[k] -= h
        assert dG[k] == pytest.approx((orc.smooth(yp, th)[0] - orc.smooth(ym, th)[0]) / (2 * h), rel=1e-7, abs=1e-8)


# ------------------------------------------------------------------------------------------------
# O5 leaf-row interval search: brute force over every (l, r') in the box
# ------------------------------------------------------------------------------------------------
# ------------------------------------------------------------------------------------------------
# the other reading of S2: Eq. 2 over successive OCCUPIED beams only (option, default off)
# ------------------------------------------------------------------------------------------------
def test_smooth_occupied_only_closed_forms_and_subpath_laplacian():
    rng = np.random.default_rng(12)
    N = 11
    theta = np.cumsum(rng.uniform(1.0, 3.0, N))
    occ = np.zeros(N, np.uint8)
    occ[[1, 2, 5, 6, 9]] = 1
    ks = np.flatnonzero(occ)
    # a constant over the occupied beams costs nothing, whatever sits at the un-occupied ones
    y = np.where(occ, 3.7, 0.0)
    G, dG = orc.smooth_occ(y, theta, occ)
    assert G == 0.0 and np.all(dG[ks] == 0.0)
    # a ramp in the angle over the occupied beams: G = sum (dtheta)^2 / dtheta = theta_last - theta_first
    y = np.where(occ, theta, 0.0)
    G, dG = orc.smooth_occ(y, theta, occ)
    assert G == pytest.approx(theta[9] - theta[1], rel=1e-13)
    np.testing.assert_allclose(dG[ks], [-2.0, 0.0, 0.0, 0.0, 2.0], atol=1e-12)   # interior terms cancel
    # G = y^T L y and dG = 2 L y with the weighted path-graph Laplacian of the occupied SUB-path, built here
    y = rng.uniform(0.0, 2.0, N) * occ
    L = np.zeros((N, N))
    for a, b in zip(ks[:-1], ks[1:]):
        s = 1.0 / (theta[b] - theta[a])
        L[a, a] += s; L[b, b] += s; L[a, b] -= s; L[b, a] -= s
    G, dG = orc.smooth_occ(y, theta, occ)
    assert G == pytest.approx(float(y @ L @ y), rel=1e-13)
    np.testing.assert_allclose(dG[ks], (2.0 * L @ y)[ks], rtol=1e-12, atol=1e-13)
    # at an un-occupied beam: the derivative at y_k = 0 of G with the beam put into the arc (finite difference)
    for k in (0, 3, 7, 10):
        occ2 = occ.copy()
        occ2[k] = 1
        h = 1e-6
        yp, ym = y.copy(), y.copy()
        yp[k], ym[k] = h, -h
        fd = (orc.smooth_occ(yp, theta, occ2)[0] - orc.smooth_occ(ym, theta, occ2)[0]) / (2 * h)
        assert dG[k] == pytest.approx(fd, rel=1e-6, abs=1e-9)
    # every beam occupied: the reading of the paper's Eq. 2 over all N angles
    full = np.ones(N, np.uint8)
    y = rng.uniform(0.0, 2.0, N)
    Ga, dGa = orc.smooth(y, theta)
    Gb, dGb = orc.smooth_occ(y, theta, full)
    assert Ga == Gb and np.array_equal(dGa, dGb)


def test_occupied_only_price_is_the_finite_difference_of_the_cost_and_master_is_nnls():
    """With the option on: (i) price_k is still the reduced cost, the one-sided finite difference of Phi for the
    chosen aperture put into the arc (S10); (ii) the master on alpha = beta problems is the non-negative least squares
    with the difference operator of the occupied sub-path (scipy.optimize.nnls); (iii) the loop runs, ends with every
    beam occupied and agrees with the default reading from then on (all beams occupied: the readings coincide)."""
    base, D, rng = small_problem(31, V=60, N=7, R=2, C=6, gamma=0.6, delta=2, nonuniform_theta=True)
    om = rng.uniform(0.5, 2.0, base.V).astype(np.float32)
    o = Oracle(base.row_ptr, base.col, base.val, base.T, om, om, base.theta, base.R, base.C, base.delta, base.gamma,
               occupied_only_G=True)
    occ, left, right, y = random_plan(o, rng, 3)
    ks = np.flatnonzero(occ)
    for k in ks[1:]:
        left[k], right[k] = left[ks[0]], right[ks[0]]            # mutually deliverable
    # (ii) master = NNLS over the occupied beams
    y_opt, z, info = o.master(occ, left, right, eps=1e-11)
    Dc = np.einsum("krc,krcv->kv", open_mask(o, occ, left, right), D.reshape(o.N, o.R, o.C, o.V))[ks]
    E = np.zeros((len(ks) - 1, len(ks)))
    for i in range(len(ks) - 1):
        s = 1.0 / np.sqrt(o.theta[ks[i + 1]] - o.theta[ks[i]])
        E[i, i], E[i, i + 1] = -s, s
    sq = np.sqrt(om.astype(np.float64))
    A = np.vstack([sq[:, None] * Dc.T, np.sqrt(o.gamma) * E])
    b = np.concatenate([sq * o.T.astype(np.float64), np.zeros(len(ks) - 1)])
    y_ref, rnorm = scipy.optimize.nnls(A, b)
    assert info.cost == pytest.approx(rnorm ** 2, rel=1e-9)
    np.testing.assert_allclose(y_opt[ks], y_ref, rtol=1e-5, atol=1e-7)
    # (i) the price of the chosen aperture at the master's optimum
    zz = o.dose(occ, left, right, y_opt)
    _, w = o.penalty(zz)
    g32 = o.prices(w, occ).astype(np.float32)
    out = o.price_step(g32, occ, left, right, y_opt)
    k = out["beam"]
    occ2, l2, r2 = occ.copy(), left.copy(), right.copy()
    occ2[k] = 1
    l2[k], r2[k] = out["left"], out["right"]
    h = 1e-7
    yh = y_opt.copy()
    yh[k] = h
    fd = (o.cost(occ2, l2, r2, yh)[2] - o.cost(occ2, l2, r2, y_opt)[2]) / h      # both WITH beam k in the arc
    assert out["price"] == pytest.approx(fd, rel=2e-4, abs=1e-6)
    # (iii) the loop
    occ_f, left_f, right_f, y_f, z_f, tr = o.solve(20)
    assert occ_f.all() and tr.iters == o.N
    d = Oracle(base.row_ptr, base.col, base.val, base.T, om, om, base.theta, base.R, base.C, base.delta, base.gamma)
    assert o.cost(occ_f, left_f, right_f, y_f)[2] == pytest.approx(d.cost(occ_f, left_f, right_f, y_f)[2], rel=1e-14)
    assert d.master(occ_f, left_f, right_f, y0=y_f, eps=1e-10)[2].cost == pytest.approx(tr.cost[-1], rel=1e-8)


def brute_force_row(q, Lmin, Lmax, Rmin, Rmax):
    """Enumerate all admissible leaf pairs; key = (sum of open prices, open count, l) (S8, S9)."""
    C = len(q)
    best = None
    for l in range(max(0, Lmin), min(C, Lmax) + 1):
        for r in range(max(l, Rmin), min(C, Rmax) + 1):
            key = (int(sum(int(v) for v in q[l:r])), r - l, l)
            if best is None or key < best[0]:
                best = (key, l, r)
    return None if best is None else (best[1], best[2], best[0][0])


def test_row_search_matches_brute_force():
    rng = np.random.default_rng(2024)
    n_cases = 0
    for trial in range(4000):
        C = int(rng.integers(1, 13))
        kind = trial % 4
        if kind == 0:
            q = rng.integers(-5, 6, C)                  # many exact ties
        elif kind == 1:
            q = rng.integers(-3, 4, C) * (rng.random(C) < 0.5)   # many zero-price beamlets
        elif kind == 2:
            q = rng.integers(-10**12, 10**12, C)
        else:
            q = orc.quantise(rng.standard_normal(C).astype(np.float32) * (rng.random(C) < 0.8))
        if trial % 3 == 0:
            box = (0, C, 0, C)
        else:
            a, b = sorted(rng.integers(0, C + 1, 2))
            c, d = sorted(rng.integers(0, C + 1, 2))
            box = (int(a), int(b), int(c), int(d))
        ref = brute_force_row(q, *box)
        got = orc.row_search(q, *box)
        assert got == ref, (q, box, got, ref)
        n_cases += ref is not None
    assert n_cases > 3000


def test_row_search_exhaustive_tiny_rows():
    # every price vector over {-1,0,1}^C for C<=5 and every box: no sampling gaps
    for C in range(1, 6):
        boxes = [(a, b, c, d) for a in range(C + 1) for b in range(a, C + 1) for c in range(C + 1) for d in range(c, C + 1)]
        for q in itertools.product((-1, 0, 1), repeat=C):
            for box in boxes[:: max(1, len(boxes) // 40)]:
                assert orc.row_search(np.array(q), *box) == brute_force_row(q, *box)


def test_row_search_unboxed_is_minimum_subarray():
    # with no leaf-travel box the row problem is the textbook minimum-sum subarray (empty allowed)
    rng = np.random.default_rng(5)
    for _ in range(300):
        C = int(rng.integers(1, 81))
        q = rng.integers(-1000, 1000, C)
        best = cur = 0
        for v in q:                                     # Kadane on the negated array
            cur = min(0, cur + int(v))
            best = min(best, cur)
        l, r, v = orc.row_search(q, 0, C, 0, C)
        assert v == best == int(q[l:r].sum())


def test_row_search_prefers_closed_and_narrow_on_ties():
    assert orc.row_search(np.array([0, 0, 0]), 0, 3, 0, 3) == (0, 0, 0)       # closed row, parked lowest
    assert orc.row_search(np.array([0, 0, 0]), 2, 3, 0, 3) == (2, 2, 0)       # closed inside the box
    assert orc.row_search(np.array([0, -1, 0]), 0, 3, 0, 3) == (1, 2, -1)     # zero-price beamlets stay shut
    assert orc.row_search(np.array([-1, 2, -1]), 0, 3, 0, 3) == (0, 1, -1)    # lowest index among equals
    assert orc.row_search(np.array([5, 5]), 0, 0, 2, 2) == (0, 2, 10)         # forced open by the box
    assert orc.row_search(np.array([1, 1]), 2, 2, 0, 1) is None               # l > r' everywhere: empty box


def test_quantise_is_exact_fixed_point():
    g = np.array([0.0, 1.0, -1.0, 0.5, 2.0 ** -30, -(2.0 ** -31), 3.0 * 2.0 ** -31, 1e-12, 123.456], np.float32)
    q = orc.quantise(g)
    # round-half-even at the 2^-30 grid
    assert list(q[:8]) == [0, 2 ** 30, -(2 ** 30), 2 ** 29, 1, 0, 2, 0]
    assert q[8] == int(np.rint(np.float64(g[8]) * 2.0 ** 30))


# ------------------------------------------------------------------------------------------------
# O5 leaf box and O6 beam choice
# ------------------------------------------------------------------------------------------------
def test_leaf_box_from_nearest_occupied_neighbours():
    o, _, _ = small_problem(9, N=9, R=2, C=10, delta=2)
    occ = np.zeros(9, np.uint8)
    left = np.zeros((9, 2), np.int32)
    right = np.zeros((9, 2), np.int32)
    assert o.leaf_box(occ, left, right, 4, 0) == (0, 10, 0, 10)           # no neighbour: whole row
    occ[1] = 1
    left[1], right[1] = [3, 0], [7, 10]
    # one neighbour 3 steps away: +-6 around its tips, clipped to [0, C]
    assert o.leaf_box(occ, left, right, 4, 0) == (0, 9, 1, 10)
    occ[5] = 1
    left[5], right[5] = [5, 0], [6, 10]
    # second neighbour 1 step away: +-2 -> intersection
    assert o.leaf_box(occ, left, right, 4, 0) == (3, 7, 4, 8)
    # beam 0 only sees beam 1 (nearest on the right), beam 8 only beam 5
    assert o.leaf_box(occ, left, right, 0, 0) == (1, 5, 5, 9)
    assert o.leaf_box(occ, left, right, 8, 0) == (0, 10, 0, 10)           # 3 steps from beam 5: +-6 around (5, 6), clipped
    assert o.leaf_box(occ, left, right, 8, 1) == (0, 6, 4, 10)            # row 1 of beam 5 is (0, 10)
    assert o.leaf_box(occ, left, right, 7, 0) == (1, 9, 2, 10)


def test_price_step_matches_bruteforce_and_finite_difference():
    """price_k = [Phi(y with y_k = h) - Phi(y)]/h for the chosen aperture (S10): ties dose, penalty,
    smoothing, pricing and search together."""
    o, D, rng = small_problem(21, V=60, N=6, R=3, C=7, gamma=0.4, delta=1, nonuniform_theta=True)
    occ, left, right, y = random_plan(o, rng, 2)
    # make the occupied apertures mutually deliverable (irrelevant for the FD, needed for a non-empty box)
    ks = np.flatnonzero(occ)
    left[ks[1]], right[ks[1]] = left[ks[0]], right[ks[0]]
    z = o.dose(occ, left, right, y)
    _, w = o.penalty(z)
    g = o.prices(w, occ)
    g32 = g.astype(np.float32)
    out = o.price_step(g32, occ, left, right, y)
    q = orc.quantise(g32).reshape(o.N, o.R, o.C)
    _, dG = o.smooth(y)
    prices = np.full(o.N, np.inf)
    for k in range(o.N):
        if occ[k]:
            continue
        tot = 0
        for r in range(o.R):
            box = o.leaf_box(occ, left, right, k, r)
            l, rr, v = brute_force_row(q[k, r], *box)
            assert (out["all_left"][k, r], out["all_right"][k, r]) == (l, rr)
            tot += v
        prices[k] = tot / 2.0 ** 30 + o.gamma * dG[k]
    np.testing.assert_allclose(out["beam_price"], prices, rtol=1e-15)
    assert out["beam"] == int(np.argmin(prices)) and out["price"] == prices.min()
    # finite difference of the whole cost along the new column
    k = out["beam"]
    occ2, left2, right2 = occ.copy(), left.copy(), right.copy()
    occ2[k] = 1
    left2[k], right2[k] = out["left"], out["right"]
    h = 1e-7
    y2 = y.copy()
    y2[k] = h
    fd = (o.cost(occ2, left2, right2, y2)[2] - o.cost(occ, left, right, y)[2]) / h
    exact = sum(g[(k * o.R + r) * o.C + c] for r in range(o.R) for c in range(out["left"][r], out["right"][r])) + o.gamma * dG[k]
    assert fd == pytest.approx(exact, rel=1e-4, abs=1e-5)
    assert out["price"] == pytest.approx(exact, rel=1e-5, abs=1e-5)        # fp32 hand-over + 2^-30 grid


def test_beam_choice_lowest_index_on_ties():
    # identical beams -> identical prices -> beam 0 (S9)
    R, C, V, N = 2, 4, 8, 4
    one = sp.random(R * C, V, density=0.6, random_state=3, format="csr", dtype=np.float32)
    D = sp.vstack([one] * N).tocsr()
    D.sort_indices()
    o = Oracle(D.indptr.astype(np.int64), D.indices, D.data, np.ones(V), np.ones(V), np.ones(V), np.arange(N) * 2.0, R, C, 1, 0.0)
    occ, left, right, y = o.empty_plan()
    _, w = o.penalty(np.zeros(V))
    out = o.price_step(o.prices(w).astype(np.float32), occ, left, right, y)
    assert out["beam"] == 0 and np.all(out["beam_price"] == out["beam_price"][0])


# ------------------------------------------------------------------------------------------------
# O7 master
# ------------------------------------------------------------------------------------------------
def test_price_step_never_chooses_an_undeliverable_beam():
    """Hand-built occupied neighbours whose leaf-travel boxes do not intersect (they break the travel limit between
    themselves, which the loop can never produce): the beam between them has no deliverable aperture (PAPER.md:111,
    "all the deliverability constraints") and must not be chosen however good its prices are."""
    o, _, rng = small_problem(5, N=5, R=2, C=10, delta=1)
    occ = np.array([1, 0, 1, 0, 0], np.uint8)
    left = np.zeros((5, 2), np.int32)
    right = np.zeros((5, 2), np.int32)
    left[0], right[0] = [0, 2], [1, 5]
    left[2], right[2] = [8, 2], [9, 5]                  # row 0: tips 8 apart over 2 steps of 1 beamlet
    assert o.leaf_box(occ, left, right, 1, 0) == (7, 1, 8, 2)             # Lmin > Lmax: empty
    assert orc.row_search(np.zeros(10, np.int64), 7, 1, 8, 2) is None
    g32 = np.zeros(o.B, np.float32)
    g32[1 * 2 * 10:2 * 2 * 10] = -100.0                # beam 1 would win by far
    g32[3 * 2 * 10 + 12] = -1.0                        # beam 3, row 1, column 2
    out = o.price_step(g32, occ, left, right, np.zeros(5))
    assert out["beam"] == 3 and np.isinf(out["beam_price"][1]) and out["beam_price"][3] == -1.0
    assert out["all_left"][1][0] == -1 and out["all_right"][1][0] == -1
    # nothing deliverable at all: no beam
    occ2 = np.array([1, 0, 1, 1, 1], np.uint8)
    left[3:], right[3:] = left[2], right[2]
    assert o.price_step(g32, occ2, left, right, np.zeros(5))["beam"] == -1


# ------------------------------------------------------------------------------------------------
# O7 master problem
# ------------------------------------------------------------------------------------------------
def test_cost_gradient_matches_central_differences():
    """vo_cost_gradient (the gradient the KKT pins read) against central differences of the cost, which is itself
    pinned by the dense dose product, the one-voxel closed form and the Laplacian form of G."""
    for seed in range(3):
        o, D, rng = small_problem(300 + seed, V=70, N=6, R=3, C=5, gamma=0.35, nonuniform_theta=bool(seed % 2))
        occ, left, right, y = random_plan(o, rng, 4)
        grad, c3 = o.cost_gradient(occ, left, right, y)
        assert c3[2] == pytest.approx(o.cost(occ, left, right, y)[2], rel=1e-14)
        h = 1e-6
        for k in range(o.N):
            if not occ[k]:
                assert grad[k] == 0.0
                continue
            e = np.zeros(o.N)
            e[k] = h
            fd = (o.cost(occ, left, right, y + e)[2] - o.cost(occ, left, right, y - e)[2]) / (2 * h)
            assert grad[k] == pytest.approx(fd, rel=2e-6, abs=1e-7), (seed, k)


def plain_projected_descent(Dc, T, al, be, Lap, gamma, lb, ub, iters=20000):
    """TEST-ONLY reference for the master problem ("gradient projection method"; Eq. 3): plain projected
    steepest descent on the box with Armijo back-tracking along the projection arc (the trial step doubles after an
    accepted step, halves until sufficient decrease) — no conjugate directions, no active-set logic, nothing shared
    with the oracle.  Dc: K x V aperture-dose columns.  Stops when a step no longer lowers the cost."""
    y = np.clip(np.zeros(Dc.shape[0]), lb, ub)

    def phi(y):
        z = y @ Dc
        return float(np.sum(al * np.maximum(0, T - z) ** 2 + be * np.maximum(0, z - T) ** 2) + gamma * y @ Lap @ y), z

    f, z = phi(y)
    t = 1.0
    for _ in range(iters):
        w = -2 * al * np.maximum(0, T - z) + 2 * be * np.maximum(0, z - T)
        g = Dc @ w + 2 * gamma * (Lap @ y)
        t *= 2.0
        while True:
            yn = np.clip(y - t * g, lb, ub)
            fn, zn = phi(yn)
            if fn <= f - 1e-4 * float(g @ (y - yn)) or t < 1e-30:
                break
            t *= 0.5
        if not fn < f:
            break
        y, f, z = yn, fn, zn
    return y, f


def test_master_reaches_the_cost_of_plain_projected_steepest_descent():
    """The oracle's master carries conjugate directions and an active-set restart; this pins its optimum to a solver
    that has neither (and shares no code with it), on small random problems with one-sided penalties (alpha = 0 on
    half the voxels), with and without the box on the dose rates."""
    for seed in range(4):
        o, D, rng = small_problem(400 + seed, V=40, N=5, R=2, C=4, gamma=(0.0, 0.3, 1.0, 0.1)[seed],
                                  nonuniform_theta=bool(seed % 2))
        occ, left, right, _ = random_plan(o, rng, o.N)
        Dc = np.einsum("krc,krcv->kv", open_mask(o, occ, left, right), D.reshape(o.N, o.R, o.C, o.V))
        Lap = np.zeros((o.N, o.N))
        for k in range(o.N - 1):
            s = 1.0 / (o.theta[k + 1] - o.theta[k])
            Lap[k, k] += s; Lap[k + 1, k + 1] += s; Lap[k, k + 1] -= s; Lap[k + 1, k] -= s
        T, al, be = (a.astype(np.float64) for a in (o.T, o.alpha, o.beta))
        for lb, ub in ((0.0, np.inf), (0.02, 0.2)):
            y_ref, f_ref = plain_projected_descent(Dc, T, al, be, Lap, o.gamma, lb, ub)
            y, z, info = o.master(occ, left, right, eps=1e-12, y_min=lb, y_max=ub)
            assert info.cost == pytest.approx(f_ref, rel=1e-9), (seed, lb, ub)


def kkt_violation(o, occ, left, right, y):
    grad, _ = o.cost_gradient(occ, left, right, y)
    viol = 0.0
    for k in range(o.N):
        if not occ[k]:
            continue
        viol = max(viol, abs(grad[k]) if y[k] > 0 else max(0.0, -grad[k]))
    return viol, grad


def test_master_one_voxel_closed_form():
    # one aperture, one voxel, alpha=beta: min (T - y d)^2  ->  y = T/d   (gamma = 0)
    o = Oracle(np.array([0, 1], np.int64), [0], [0.25], [0.8], [1.0], [1.0], [0.0], 1, 1, 1, 0.0)
    y, z, info = o.master([1], [[0]], [[1]])
    assert y[0] == pytest.approx(float(np.float32(0.8)) / 0.25, rel=1e-9) and info.cost == pytest.approx(0.0, abs=1e-15)
    # two beams, same voxel, smoothing couples them: minimise (T - d(y0+y1))^2 + g (y1-y0)^2/dth -> y0=y1=T/(2d)
    o = Oracle(np.array([0, 1, 2], np.int64), [0, 0], [0.25, 0.25], [0.8], [1.0], [1.0], [0.0, 2.0], 1, 1, 1, 0.5)
    y, z, info = o.master([1, 1], [[0], [0]], [[1], [1]])
    np.testing.assert_allclose(y, [1.6, 1.6], rtol=1e-6)
    # the bound is active: a beam that can only overdose an organ at risk stays at y = 0
    o = Oracle(np.array([0, 1, 2], np.int64), [0, 1], [1.0, 1.0], [1.0, 0.0], [1.0, 0.0], [1.0, 5.0], [0.0, 2.0], 1, 1, 1, 0.0)
    y, z, info = o.master([1, 1], [[0], [0]], [[1], [1]], y0=[0.3, 0.7])
    np.testing.assert_allclose(y, [1.0, 0.0], atol=1e-8)


def test_master_satisfies_kkt_random():
    for seed in range(6):
        o, D, rng = small_problem(100 + seed, V=80, N=7, R=3, C=6, gamma=0.2 * seed, delta=2, nonuniform_theta=bool(seed % 2))
        occ, left, right, y0 = random_plan(o, rng, 5)
        y, z, info = o.master(occ, left, right, y0=y0)
        assert np.all(y >= 0) and np.all(y[occ == 0] == 0)
        viol, grad = kkt_violation(o, occ, left, right, y)
        assert viol <= 1e-7 * max(1.0, info.pg_entry), (seed, viol, info)
        np.testing.assert_allclose(z, o.dose(occ, left, right, y), rtol=1e-12, atol=1e-12)
        assert info.cost == pytest.approx(o.cost(occ, left, right, y)[2], rel=1e-13)
        # warm start from the optimum does nothing
        y2, _, info2 = o.master(occ, left, right, y0=y)
        assert info2.pg_entry <= 1e-6 * max(1.0, info.pg_entry) and info2.cost <= info.cost * (1 + 1e-12)


def test_master_equals_nnls_when_all_quadratic():
    """alpha=beta=omega everywhere makes F a plain weighted least squares, so (3) with fixed apertures is
    the non-negative least squares  min_{y>=0} || [sqrt(omega) Dc^T ; sqrt(gamma) E] y - [sqrt(omega) T ; 0] ||^2,
    E the scaled difference operator (G = |E y|^2).  Library routine: scipy.optimize.nnls."""
    o, D, rng = small_problem(77, V=50, N=6, R=2, C=5, gamma=0.7, nonuniform_theta=True)
    om = rng.uniform(0.5, 2.0, o.V).astype(np.float32)
    o = Oracle(o.row_ptr, o.col, o.val, o.T, om, om, o.theta, o.R, o.C, o.delta, o.gamma)
    occ, left, right, _ = random_plan(o, rng, o.N)            # all beams occupied
    Dc = np.einsum("krc,krcv->kv", open_mask(o, occ, left, right), D.reshape(o.N, o.R, o.C, o.V))
    E = np.zeros((o.N - 1, o.N))
    for k in range(o.N - 1):
        s = 1.0 / np.sqrt(o.theta[k + 1] - o.theta[k])
        E[k, k], E[k, k + 1] = -s, s
    sq = np.sqrt(om.astype(np.float64))
    A = np.vstack([sq[:, None] * Dc.T, np.sqrt(o.gamma) * E])
    b = np.concatenate([sq * o.T.astype(np.float64), np.zeros(o.N - 1)])
    y_ref, rnorm = scipy.optimize.nnls(A, b)
    y, z, info = o.master(occ, left, right, eps=1e-11)
    assert info.cost == pytest.approx(rnorm ** 2, rel=1e-9)
    np.testing.assert_allclose(y, y_ref, rtol=1e-5, atol=1e-7)


def priced_out_problem(gamma=0.0):
    """Five beams of one row x three beamlets.  Beams 0 and 1 reach the target voxels 0..3 (alpha > 0), beams 2..4
    only organ-at-risk voxels 4..9 (alpha = 0, T = 0): whatever the dose, w_j >= 0 there, so every aperture of
    those beams has a price >= 0 and the closed one (price 0) is the best."""
    N, R, C, V = 5, 1, 3, 10
    rng = np.random.default_rng(11)
    D = np.zeros((N * R * C, V), np.float32)
    for i in range(N * R * C):
        cols = range(0, 4) if i // C < 2 else range(4, 10)
        for j in cols:
            if rng.random() < 0.8:
                D[i, j] = rng.uniform(0.1, 1.0)
    csr = scipy.sparse.csr_matrix(D)
    csr.sort_indices()
    T = np.array([1.0] * 4 + [0.0] * 6, np.float32)
    alpha = np.array([1.0] * 4 + [0.0] * 6, np.float32)
    beta = np.array([1.0] * 4 + [0.7] * 6, np.float32)
    return Oracle(csr.indptr.astype(np.int64), csr.indices.astype(np.int32), csr.data.astype(np.float32), T, alpha, beta,
                  np.arange(N) * 2.0, R, C, 3, gamma)


def test_solve_stop_when_priced_out_option():
    """Option of reading S5 (the textbook column-generation stop): the loop ends as soon as no aperture has a
    negative price.  Default: it goes on until every beam holds an aperture."""
    o = priced_out_problem()
    occ, left, right, y, z, tr = o.solve(10, stop_when_priced_out=True)
    assert tr.iters == 2 and sorted(tr.beam.tolist()) == [0, 1] and np.all(tr.price < 0)
    assert occ.tolist() == [1, 1, 0, 0, 0]
    g = o.prices(o.penalty(z)[1], occ)
    best = o.price_step(g.astype(np.float32), occ, left, right, y)
    assert best["price"] >= 0.0 and np.all(g[6:] >= 0)                     # nothing prices out at the stop
    occ2, left2, right2, y2, z2, tr2 = o.solve(10)
    assert tr2.iters == 5 and occ2.all()                                   # default: an aperture at every angle
    assert np.array_equal(tr2.beam[:2], tr.beam) and np.array_equal(tr2.cost[:2], tr.cost)
    assert np.all(tr2.price[2:] >= 0) and np.all(left2[2:] == right2[2:])  # the late apertures are closed ...
    assert tr2.cost[-1] == pytest.approx(tr.cost[-1], rel=1e-12)           # ... and buy nothing


# ------------------------------------------------------------------------------------------------
# variant: bounds on the dose rates of occupied beams (PAPER.md:159 names "the maximum and minimum dose rate
# constraints" and leaves them out; reading R4)
# ------------------------------------------------------------------------------------------------
def test_master_bounds_one_voxel_closed_form():
    # one aperture, one voxel: min (T - y d)^2 over lb <= y <= ub is the unconstrained y* = T/d clipped to the box
    o = Oracle(np.array([0, 1], np.int64), [0], [0.25], [0.8], [1.0], [1.0], [0.0], 1, 1, 1, 0.0)
    ystar = float(np.float32(0.8)) / 0.25
    for lb, ub in ((0.0, 2.0), (4.0, 9.0), (1.0, 5.0), (0.0, float("inf"))):
        y, z, info = o.master([1], [[0]], [[1]], y_min=lb, y_max=ub)
        want = min(max(ystar, lb), ub)
        assert y[0] == pytest.approx(want, rel=1e-9)
        assert info.cost == pytest.approx((float(np.float32(0.8)) - want * 0.25) ** 2, rel=1e-9, abs=1e-15)
    # an un-occupied beam stays at 0 whatever the lower bound (it has no aperture: reading R4)
    o = Oracle(np.array([0, 1, 2], np.int64), [0, 0], [0.25, 0.25], [0.8], [1.0], [1.0], [0.0, 2.0], 1, 1, 1, 0.0)
    y, z, info = o.master([1, 0], [[0], [0]], [[1], [1]], y_min=0.5, y_max=2.0)
    assert y[1] == 0.0 and y[0] == pytest.approx(2.0)


def test_master_bounds_satisfy_box_kkt_random():
    """KKT of min Phi over the box: lb < y_k < ub => dPhi/dy_k = 0; y_k = lb => >= 0; y_k = ub => <= 0."""
    hit_lo = hit_hi = inside = 0
    for seed in range(6):
        o, D, rng = small_problem(300 + seed, V=80, N=7, R=3, C=6, gamma=0.2 * seed, delta=2, nonuniform_theta=bool(seed % 2))
        occ, left, right, y0 = random_plan(o, rng, 5)
        yfree, _, free = o.master(occ, left, right, y0=y0)
        pos = yfree[occ == 1]
        lb, ub = 0.5 * float(np.median(pos)), 0.9 * float(pos.max())      # both bounds bind somewhere
        y, z, info = o.master(occ, left, right, y0=y0, y_min=lb, y_max=ub)
        grad, (F, G, cost) = o.cost_gradient(occ, left, right, y)
        assert np.all(y[occ == 0] == 0) and np.all(y[occ == 1] >= lb) and np.all(y[occ == 1] <= ub)
        scale = max(1.0, info.pg_entry)
        for k in np.nonzero(occ)[0]:
            if y[k] <= lb:
                assert grad[k] >= -1e-7 * scale
                hit_lo += 1
            elif y[k] >= ub:
                assert grad[k] <= 1e-7 * scale
                hit_hi += 1
            else:
                assert abs(grad[k]) <= 1e-7 * scale
                inside += 1
        assert info.cost == pytest.approx(cost, rel=1e-13) and info.cost >= free.cost * (1 - 1e-12)
        np.testing.assert_allclose(z, o.dose(occ, left, right, y), rtol=1e-12, atol=1e-12)
    assert hit_lo and hit_hi and inside                                   # the test saw all three cases


def test_solve_with_bounds_keeps_every_master_in_the_box(tiny_oracle, tiny_solution):
    """The loop with bounds on the dose rates (reading R4): prices are those of the paper, every master solve is the
    box-constrained one.  Pinned by what must hold whatever the path: y in the box at occupied beams and 0 elsewhere,
    the recorded cost is the cost of the returned plan, a fresh box-constrained master solve on the final aperture
    set (itself pinned by the BVLS / KKT tests above) cannot lower it, and lb = 0, ub = inf is the unbounded loop."""
    o = tiny_oracle
    occ0, left0, right0, y0, z0, tr0 = tiny_solution
    occ, left, right, y, z, tr = o.solve(40, y_min=0.0, y_max=float("inf"))
    assert np.array_equal(tr.beam, tr0.beam) and np.array_equal(left, left0) and np.array_equal(right, right0)
    np.testing.assert_allclose(tr.cost, tr0.cost, rtol=1e-12)       # (OpenMP sums: the last bits depend on the run)
    np.testing.assert_allclose(y, y0, rtol=1e-7, atol=1e-10)
    lb, ub = 0.3 * float(np.median(y0)), 0.7 * float(y0.max())
    for n in (5, 40):
        occ, left, right, y, z, tr = o.solve(n, y_min=lb, y_max=ub)
        on = occ.astype(bool)
        assert np.all(y[on] >= lb) and np.all(y[on] <= ub) and np.all(y[~on] == 0.0)
        assert np.any(y[on] == lb) or np.any(y[on] == ub)                        # the box binds
        assert tr.cost[-1] == pytest.approx(o.cost(occ, left, right, y)[2], rel=1e-12)
        _, _, info = o.master(occ, left, right, y0=y, eps=1e-10, y_min=lb, y_max=ub)
        assert info.cost == pytest.approx(tr.cost[-1], rel=1e-7) and info.cost <= tr.cost[-1] * (1 + 1e-12)
    assert tr.cost[-1] > tr0.cost[-1]                                            # a binding box costs something


def test_master_bounds_equal_bounded_least_squares_when_all_quadratic():
    """alpha = beta everywhere: (3) with fixed apertures and a box on y is a bounded linear least squares.
    Library routine: scipy.optimize.lsq_linear."""
    o, D, rng = small_problem(78, V=50, N=6, R=2, C=5, gamma=0.7, nonuniform_theta=True)
    om = rng.uniform(0.5, 2.0, o.V).astype(np.float32)
    o = Oracle(o.row_ptr, o.col, o.val, o.T, om, om, o.theta, o.R, o.C, o.delta, o.gamma)
    occ, left, right, _ = random_plan(o, rng, o.N)
    Dc = np.einsum("krc,krcv->kv", open_mask(o, occ, left, right), D.reshape(o.N, o.R, o.C, o.V))
    E = np.zeros((o.N - 1, o.N))
    for k in range(o.N - 1):
        s = 1.0 / np.sqrt(o.theta[k + 1] - o.theta[k])
        E[k, k], E[k, k + 1] = -s, s
    sq = np.sqrt(om.astype(np.float64))
    A = np.vstack([sq[:, None] * Dc.T, np.sqrt(o.gamma) * E])
    b = np.concatenate([sq * o.T.astype(np.float64), np.zeros(o.N - 1)])
    yfree, _, _ = o.master(occ, left, right, eps=1e-11)
    lo, hi = float(yfree.min()), float(yfree.max())
    for lb, ub in ((lo + 0.5 * (hi - lo), np.inf), (0.0, hi - 0.35 * (hi - lo)), (lo + 0.2 * (hi - lo), hi - 0.2 * (hi - lo))):
        ref = scipy.optimize.lsq_linear(A, b, bounds=(lb, ub), method="bvls", tol=1e-14)
        y, z, info = o.master(occ, left, right, eps=1e-11, y_min=lb, y_max=ub)
        assert info.cost == pytest.approx(2.0 * ref.cost, rel=1e-9)       # lsq_linear reports half the squared norm
        np.testing.assert_allclose(y, ref.x, rtol=1e-5, atol=1e-7)
        assert np.any(y <= lb * (1 + 1e-12)) or np.any(y >= ub * (1 - 1e-12))   # a bound binds: not the free optimum


# ------------------------------------------------------------------------------------------------
# O8 trajectory invariants on configs[0]
# ------------------------------------------------------------------------------------------------
def test_tiny_run_invariants(tiny_phantom, tiny_oracle, tiny_solution):
    ph, o = tiny_phantom, tiny_oracle
    occ, left, right, y, z, tr = tiny_solution
    # one aperture in each beam direction, a plan at all gantry angles (reading S5)
    assert tr.iters == o.N == 24 and sorted(tr.beam) == list(range(24)) and np.all(occ == 1)
    # convex model + columns entering at y=0 => cost after each master is non-increasing
    assert np.all(np.diff(tr.cost) <= 1e-9 * tr.cost[:-1])
    assert tr.cost[0] < o.penalty(np.zeros(o.V))[0]
    # every generated column had a negative price (it could decrease the cost)
    assert np.all(tr.price < 0)
    # leaf pairs are legal and the arc is deliverable: |dl|,|dr| <= delta*|k-k'| for ALL pairs (S6)
    assert np.all((0 <= left) & (left <= right) & (right <= o.C))
    for k in range(o.N):
        for k2 in range(k + 1, o.N):
            lim = o.delta * (k2 - k)
            assert np.all(np.abs(left[k] - left[k2]) <= lim) and np.all(np.abs(right[k] - right[k2]) <= lim)
    # final plan is a KKT point of the master and z is its dose
    viol, _ = kkt_violation(o, occ, left, right, y)
    assert viol <= 1e-6
    np.testing.assert_allclose(z, o.dose(occ, left, right, y), rtol=1e-12, atol=1e-12)
    assert tr.cost[-1] == pytest.approx(o.cost(occ, left, right, y)[2], rel=1e-12)


def test_first_aperture_is_target_silhouette(tiny_phantom, tiny_oracle, tiny_solution):
    """At the empty plan w_j = -2 alpha_j T_j <= 0, so every first price is <= 0 and the first aperture
    opens exactly the beamlets that can reach an alpha>0 voxel (beam's-eye-view silhouette widened by
    the kernel reach), trimmed only by the (value, width, l) tie-break on zero-price beamlets."""
    ph, o = tiny_phantom, tiny_oracle
    _, w = o.penalty(np.zeros(o.V))
    assert np.all(w <= 0)
    g = o.prices(w)
    assert np.all(g <= 0)
    occ, left, right, y = o.empty_plan()
    out = o.price_step(g.astype(np.float32), occ, left, right, y)
    tr = tiny_solution[5]
    assert out["beam"] == tr.beam[0]
    np.testing.assert_array_equal(out["left"], tr.left[0])
    np.testing.assert_array_equal(out["right"], tr.right[0])
    gk = g.reshape(o.N, o.R, o.C)[out["beam"]]
    for r in range(o.R):
        neg = np.flatnonzero(gk[r] < 0)
        if neg.size:
            assert (out["left"][r], out["right"][r]) == (neg[0], neg[-1] + 1)
        else:
            assert out["left"][r] == out["right"][r]


def test_solve_resumes_from_a_plan(tiny_oracle, tiny_solution):
    # stopping after 5 iterations and resuming gives the same trajectory as the straight run
    o = tiny_oracle
    occ, left, right, y, z, tr5 = o.solve(5)
    occ2, left2, right2, y2, z2, tr_rest = o.solve(40, plan=(occ, left, right, y))
    full = tiny_solution[5]
    np.testing.assert_array_equal(np.concatenate([tr5.beam, tr_rest.beam]), full.beam)
    np.testing.assert_allclose(tr_rest.cost[-1], full.cost[-1], rtol=1e-9)


# ------------------------------------------------------------------------------------------------
# shapes of the synthetic stand-ins vs. the paper's Table 1 (context only)
# ------------------------------------------------------------------------------------------------
def test_mixed_resolution_phantom_conserves_dose_and_penalty(tiny_phantom):
    """Input preprocessing of PAPER.md:131 (unspecified tissue at twice the voxel size): the coarse column of D is the
    mean of its eight fine columns, so every beamlet deposits the same dose x volume; a dose that is constant on every
    coarsened block costs the same on both grids (weights x 8); structures keep their voxels."""
    import vmat_inputs

    ph = tiny_phantom
    pm = vmat_inputs.make_phantom("tiny", seed=0, mixed_resolution=True)
    assert pm.n_voxels < 0.5 * ph.n_voxels and pm.n_beamlets == ph.n_beamlets
    assert set(np.unique(pm.volume)) == {1.0, 8.0}
    D = sp.csr_matrix((ph.val.astype(np.float64), ph.col_idx, ph.row_ptr), shape=(ph.n_beamlets, ph.n_voxels))
    Dm = sp.csr_matrix((pm.val.astype(np.float64), pm.col_idx, pm.row_ptr), shape=(pm.n_beamlets, pm.n_voxels))
    np.testing.assert_allclose(Dm @ pm.volume.astype(np.float64), np.asarray(D.sum(axis=1)).ravel(), rtol=1e-6)
    assert np.all(np.diff(pm.col_idx)[np.diff(np.repeat(np.arange(pm.n_beamlets), np.diff(pm.row_ptr))) == 0] > 0)
    # structures are untouched: as many target / organ-at-risk voxels as before, all of volume 1
    for T, al in ((1.0, 1.0), (0.3, 0.0)):
        fine = (ph.T == np.float32(T)) & (ph.alpha == np.float32(al)) & (ph.beta > 0.1)
        mix = (pm.T == np.float32(T)) & (pm.alpha == np.float32(al)) & (pm.beta > 0.1) & (pm.volume == 1.0)
        assert fine.sum() == mix.sum() > 0
    # the penalty of a uniform dose is the same on both grids
    for zc in (0.2, 0.7):
        Ff, _ = orc.penalty(np.full(ph.n_voxels, zc), ph.T, ph.alpha, ph.beta)
        Fm, _ = orc.penalty(np.full(pm.n_voxels, zc), pm.T, pm.alpha, pm.beta)
        assert Fm == pytest.approx(Ff, rel=1e-6)
    # the loop runs on it and keeps its invariants
    o = Oracle.from_phantom(pm)
    occ, left, right, y, z, tr = o.solve(6)
    assert tr.iters == 6 and np.all(np.diff(tr.cost) <= 1e-9 * tr.cost[:-1])


def test_phantom_shape_is_in_the_range_of_table1():
    import os

    import vmat_inputs

    rows = [ln.split() for ln in open(os.path.join(os.path.dirname(__file__), "golden", "paper_table1.txt")) if ln[0] != "#"]
    per_beamlet = [float(r[3]) * 1e7 / float(r[1]) for r in rows]          # ~365-700 nnz per beamlet
    assert 300 < min(per_beamlet) < max(per_beamlet) < 700
    ph = vmat_inputs.make_phantom(vmat_inputs.scaled_config("prostate", n_beams=6), check_reach=False)
    mine = ph.nnz / ph.n_beamlets
    assert 0.5 * min(per_beamlet) < mine < 2 * max(per_beamlet)


# ------------------------------------------------------------------------------------------------
# hard dose-rate feasibility after the last aperture (raise gamma, re-solve the master)
# ------------------------------------------------------------------------------------------------
def test_rate_ratio_by_hand():
    o, _, _ = small_problem(seed=3, N=4, nonuniform_theta=True)
    y = np.array([0.0, 1.0, 0.5, 2.5])
    dth = np.diff(o.theta)
    by_hand = max(abs(1.0 - 0.0) / (0.25 * dth[0]), abs(0.5 - 1.0) / (0.25 * dth[1]), abs(2.5 - 0.5) / (0.25 * dth[2]))
    assert o.rate_ratio(y, 0.25) == pytest.approx(by_hand, rel=1e-15)
    assert o.rate_ratio(np.full(4, 0.7), 0.25) == 0.0                       # constant dose rate: no variation


def two_beam_problem(gamma):
    # beam 0 reaches only voxel 0 (D = a), beam 1 only voxel 1 (D = b); alpha = beta = 1: everything is quadratic
    a, b, T0, T1, dth = 0.5, 0.25, 1.0, 0.25, 2.0
    o = Oracle(np.array([0, 1, 2], np.int64), [0, 1], [a, b], [T0, T1], [1.0, 1.0], [1.0, 1.0], [0.0, dth], 1, 1, 1, gamma)
    return o, (a, b, T0, T1, dth)


def two_beam_optimum(a, b, T0, T1, dth, gamma):
    # stationarity of (a y0 - T0)^2 + (b y1 - T1)^2 + gamma (y1 - y0)^2 / dth, written out:
    #   (a^2 + g) y0 - g y1 = a T0 ;  -g y0 + (b^2 + g) y1 = b T1 ,  g = gamma / dth ; Cramer's rule
    g = gamma / dth
    det = (a * a + g) * (b * b + g) - g * g
    return np.array([(a * T0 * (b * b + g) + g * b * T1) / det, ((a * a + g) * b * T1 + g * a * T0) / det])


def test_enforce_rate_two_beam_closed_form():
    gamma0, rho, factor = 0.01, 0.05, 2.0
    o, prm = two_beam_problem(gamma0)
    occ, left, right = [1, 1], [[0], [0]], [[1], [1]]
    y0, _, _ = o.master(occ, left, right)
    np.testing.assert_allclose(y0, two_beam_optimum(*prm, gamma0), rtol=1e-8)
    # the closed form tells how often gamma has to double before |y1 - y0| <= rho dtheta
    want = 0
    while abs(np.diff(two_beam_optimum(*prm, gamma0 * factor ** want))[0]) > rho * prm[4]:
        want += 1
    assert want >= 3                                                          # the case is not trivial
    y, z, info = o.enforce_rate(occ, left, right, y0, rho, factor=factor, tol=0.0)
    assert info["rounds"] == want and info["feasible"]
    assert info["gamma"] == gamma0 * factor ** want
    np.testing.assert_allclose(y, two_beam_optimum(*prm, info["gamma"]), rtol=1e-7)
    assert info["ratio"] == pytest.approx(abs(y[1] - y[0]) / (rho * prm[4]), rel=1e-12) and info["ratio"] <= 1.0
    assert info["cost"] == pytest.approx((prm[0] * y[0] - prm[2]) ** 2 + (prm[1] * y[1] - prm[3]) ** 2
                                         + info["gamma"] * (y[1] - y[0]) ** 2 / prm[4], rel=1e-9)


def test_enforce_rate_random_problems():
    for seed in range(4):
        o, dense, rng = small_problem(seed=50 + seed, N=6, gamma=0.05, nonuniform_theta=bool(seed % 2))
        occ, left, right, y_any = random_plan(o, rng, o.N)
        y0, _, _ = o.master(occ, left, right, eps=1e-11)
        r0 = o.rate_ratio(y0, 1.0)
        # a limit far above the plan's variation: nothing to do, the plan comes back untouched
        y, z, info = o.enforce_rate(occ, left, right, y0, rho=10.0 * r0)
        assert info["rounds"] == 0 and info["feasible"] and info["gamma"] == o.gamma and np.array_equal(y, y0)
        # a limit at a third of it: gamma has to rise
        rho = r0 / 3.0
        y, z, info = o.enforce_rate(occ, left, right, y0, rho=rho, factor=2.0, tol=1e-9, eps=1e-11)
        assert info["feasible"] and info["rounds"] >= 1
        assert info["gamma"] == o.gamma * 2.0 ** info["rounds"]
        assert np.max(np.abs(np.diff(y)) / (rho * np.diff(o.theta))) <= 1.0 + 1e-9      # the definition, by hand
        assert np.all(y >= 0)
        np.testing.assert_allclose(z, dense.T @ (open_mask(o, occ, left, right).reshape(-1) * np.repeat(y, o.R * o.C)), rtol=1e-10, atol=1e-12)
        # y is the master optimum for the gamma at exit (KKT on an oracle built with that gamma) ...
        o_exit = Oracle(o.row_ptr, o.col, o.val, o.T, o.alpha, o.beta, o.theta, o.R, o.C, o.delta, info["gamma"])
        viol, _ = kkt_violation(o_exit, occ, left, right, y)
        assert viol <= 1e-7
        # ... and one round earlier the optimum was still infeasible (gamma is not raised further than needed)
        o_prev = Oracle(o.row_ptr, o.col, o.val, o.T, o.alpha, o.beta, o.theta, o.R, o.C, o.delta, info["gamma"] / 2.0)
        y_prev, _, _ = o_prev.master(occ, left, right, y0=y0, eps=1e-11)
        assert o.rate_ratio(y_prev, rho) > 1.0 + 1e-9


def test_enforce_rate_gives_up_at_the_round_cap():
    o, prm = two_beam_problem(0.01)
    occ, left, right = [1, 1], [[0], [0]], [[1], [1]]
    y0, _, _ = o.master(occ, left, right)
    y, z, info = o.enforce_rate(occ, left, right, y0, rho=1e-9, max_rounds=3)
    assert info["rounds"] == 3 and not info["feasible"] and info["gamma"] == 0.01 * 8.0
