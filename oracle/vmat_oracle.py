"""ctypes wrapper around oracle/vmat_oracle.c (argument marshalling only; all arithmetic is in the C file).

TEST INFRASTRUCTURE — see the header of vmat_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vmat_oracle.c")
_LIB = os.path.join(_HERE, "libvmat_oracle.so")
_lib = None

_c = ctypes
_P = ctypes.c_void_p


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"],
                       check=True)
    return _LIB


class _Problem(_c.Structure):
    _fields_ = [("V", _c.c_int64), ("N", _c.c_int64), ("R", _c.c_int64), ("C", _c.c_int64),
                ("row_ptr", _P), ("col", _P), ("val", _P), ("T", _P), ("alpha", _P), ("beta", _P),
                ("theta", _P), ("delta", _c.c_int32), ("gamma", _c.c_double), ("g_occupied_only", _c.c_int32)]


class _MasterInfo(_c.Structure):
    _fields_ = [("eps", _c.c_double), ("max_inner", _c.c_int64), ("lb", _c.c_double), ("ub", _c.c_double),
                ("inner", _c.c_int64),
                ("backtracks", _c.c_int64), ("pg_entry", _c.c_double), ("pg_exit", _c.c_double),
                ("F", _c.c_double), ("G", _c.c_double), ("cost", _c.c_double)]


class _RateInfo(_c.Structure):
    _fields_ = [("rho", _c.c_double), ("factor", _c.c_double), ("tol", _c.c_double), ("max_rounds", _c.c_int64),
                ("eps", _c.c_double), ("max_inner", _c.c_int64), ("rounds", _c.c_int64), ("feasible", _c.c_int64),
                ("gamma", _c.c_double), ("ratio", _c.c_double), ("F", _c.c_double), ("G", _c.c_double),
                ("cost", _c.c_double)]


class _Trace(_c.Structure):
    _fields_ = [("max_iters", _c.c_int64), ("eps", _c.c_double), ("max_inner", _c.c_int64),
                ("stop_when_priced_out", _c.c_int64), ("lb", _c.c_double), ("ub", _c.c_double), ("iters", _c.c_int64), ("beam", _P), ("price", _P), ("F", _P), ("G", _P), ("cost", _P),
                ("inner", _P), ("it_left", _P), ("it_right", _P),
                ("seconds_price", _c.c_double), ("seconds_master", _c.c_double)]


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        PP = _c.POINTER(_Problem)
        L.vo_dose.argtypes = [PP, _P, _P, _P, _P, _P]
        L.vo_dose.restype = None
        L.vo_penalty.argtypes = [_c.c_int64, _P, _P, _P, _P, _P]
        L.vo_penalty.restype = _c.c_double
        L.vo_smooth.argtypes = [_c.c_int64, _P, _P, _P]
        L.vo_smooth.restype = _c.c_double
        L.vo_smooth_occ.argtypes = [_c.c_int64, _P, _P, _P, _P]
        L.vo_smooth_occ.restype = _c.c_double
        L.vo_prices.argtypes = [PP, _P, _P, _P]
        L.vo_prices.restype = None
        L.vo_quantise.argtypes = [_c.c_int64, _P, _P]
        L.vo_quantise.restype = None
        L.vo_leaf_box.argtypes = [PP, _P, _P, _P, _c.c_int64, _c.c_int64, _P]
        L.vo_leaf_box.restype = None
        L.vo_row_search.argtypes = [_c.c_int64, _P, _c.c_int64, _c.c_int64, _c.c_int64, _c.c_int64, _P, _P, _P]
        L.vo_row_search.restype = _c.c_int
        L.vo_price_step.argtypes = [PP, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P]
        L.vo_price_step.restype = _c.c_int64
        L.vo_master.argtypes = [PP, _P, _P, _P, _P, _P, _c.POINTER(_MasterInfo)]
        L.vo_master.restype = None
        L.vo_cost_gradient.argtypes = [PP, _P, _P, _P, _P, _P, _P]
        L.vo_cost_gradient.restype = None
        L.vo_rate_ratio.argtypes = [_c.c_int64, _P, _P, _c.c_double]
        L.vo_rate_ratio.restype = _c.c_double
        L.vo_enforce_rate.argtypes = [PP, _P, _P, _P, _P, _P, _c.POINTER(_RateInfo)]
        L.vo_enforce_rate.restype = None
        L.vo_solve.argtypes = [PP, _P, _P, _P, _P, _P, _c.POINTER(_Trace)]
        L.vo_solve.restype = None
        L.vo_num_threads.restype = _c.c_int
        L.vo_set_num_threads.argtypes = [_c.c_int]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(_load().vo_num_threads())


def set_num_threads(n: int) -> None:
    _load().vo_set_num_threads(int(n))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data


def _as(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


# ---- free functions (no problem needed) -----------------------------------------------------
def penalty(z, T, alpha, beta, want_w: bool = True):
    """O3 (Eq. 1): returns (F, w)."""
    z = _as(z, np.float64)
    T, alpha, beta = _as(T, np.float32), _as(alpha, np.float32), _as(beta, np.float32)
    w = np.empty_like(z) if want_w else None
    F = _load().vo_penalty(z.size, _ptr(z), _ptr(T), _ptr(alpha), _ptr(beta), _ptr(w))
    return float(F), w


def smooth(y, theta_deg):
    """O3 (Eq. 2): returns (G, dG/dy)."""
    y, th = _as(y, np.float64), _as(theta_deg, np.float64)
    dG = np.empty_like(y)
    G = _load().vo_smooth(y.size, _ptr(y), _ptr(th), _ptr(dG))
    return float(G), dG


def smooth_occ(y, theta_deg, occ):
    """The other reading of Eq. 2 (S2): smoothing over successive OCCUPIED beams only.  Returns (G, dG); dG at an
    un-occupied beam is the derivative at y_k = 0 of G with that beam put into the arc."""
    y, th, occ = _as(y, np.float64), _as(theta_deg, np.float64), _as(occ, np.uint8)
    dG = np.empty_like(y)
    G = _load().vo_smooth_occ(y.size, _ptr(y), _ptr(th), _ptr(occ), _ptr(dG))
    return float(G), dG


def quantise(g32):
    g32 = _as(g32, np.float32)
    q = np.empty(g32.size, np.int64)
    _load().vo_quantise(g32.size, _ptr(g32), _ptr(q))
    return q


def row_search(q, Lmin, Lmax, Rmin, Rmax):
    """O5 one-pass search on int64 prices q[C]. Returns (l, r, value) or None if the box is empty."""
    q = _as(q, np.int64)
    l, r, v = _c.c_int32(0), _c.c_int32(0), _c.c_int64(0)
    rc = _load().vo_row_search(q.size, _ptr(q), int(Lmin), int(Lmax), int(Rmin), int(Rmax),
                               _c.addressof(l), _c.addressof(r), _c.addressof(v))
    return None if rc != 0 else (int(l.value), int(r.value), int(v.value))


@dataclass
class MasterInfo:
    inner: int
    backtracks: int
    pg_entry: float
    pg_exit: float
    F: float
    G: float
    cost: float


@dataclass
class Trace:
    iters: int
    beam: np.ndarray
    price: np.ndarray
    F: np.ndarray
    G: np.ndarray
    cost: np.ndarray
    inner: np.ndarray
    left: np.ndarray          # [iters, R] leaf pairs of the aperture chosen at each iteration
    right: np.ndarray
    seconds_price: float
    seconds_master: float


class Oracle:
    """The oracle bound to one problem instance (a vmat_inputs.Phantom or raw arrays)."""

    def __init__(self, row_ptr, col_idx, val, T, alpha, beta, theta_deg, n_rows, n_cols, max_leaf_travel, gamma,
                 occupied_only_G=False):
        self.row_ptr = _as(row_ptr, np.int64)
        self.col = _as(col_idx, np.int32)
        self.val = _as(val, np.float32)
        self.T, self.alpha, self.beta = _as(T, np.float32), _as(alpha, np.float32), _as(beta, np.float32)
        self.theta = _as(theta_deg, np.float64)
        self.V, self.N, self.R, self.C = self.T.size, self.theta.size, int(n_rows), int(n_cols)
        self.B = self.N * self.R * self.C
        assert self.row_ptr.size == self.B + 1
        self.delta, self.gamma = int(max_leaf_travel), float(gamma)
        self.occupied_only_G = bool(occupied_only_G)
        self._p = _Problem(self.V, self.N, self.R, self.C, _ptr(self.row_ptr), _ptr(self.col), _ptr(self.val),
                           _ptr(self.T), _ptr(self.alpha), _ptr(self.beta), _ptr(self.theta), self.delta, self.gamma,
                           int(self.occupied_only_G))
        self._L = _load()

    @classmethod
    def from_phantom(cls, ph, gamma=None, max_leaf_travel=None, occupied_only_G=False):
        c = ph.config
        return cls(ph.row_ptr, ph.col_idx, ph.val, ph.T, ph.alpha, ph.beta, ph.theta_deg, c.n_rows, c.n_cols,
                   c.max_leaf_travel if max_leaf_travel is None else max_leaf_travel,
                   c.gamma if gamma is None else gamma, occupied_only_G=occupied_only_G)

    # plan helpers -----------------------------------------------------------------------------
    def empty_plan(self):
        return (np.zeros(self.N, np.uint8), np.zeros(self.N * self.R, np.int32), np.zeros(self.N * self.R, np.int32),
                np.zeros(self.N, np.float64))

    def _plan(self, occ, left, right):
        return _as(occ, np.uint8), _as(left, np.int32).reshape(-1), _as(right, np.int32).reshape(-1)

    # O2 ----------------------------------------------------------------------------------------
    def dose(self, occ, left, right, y):
        occ, left, right = self._plan(occ, left, right)
        y = _as(y, np.float64)
        z = np.empty(self.V, np.float64)
        self._L.vo_dose(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), _ptr(y), _ptr(z))
        return z

    # O3 ----------------------------------------------------------------------------------------
    def penalty(self, z):
        return penalty(z, self.T, self.alpha, self.beta)

    def smooth(self, y, occ=None):
        """G and dG in the problem's reading of Eq. 2 (occ is needed for the occupied-only reading)."""
        if self.occupied_only_G:
            return smooth_occ(y, self.theta, occ)
        return smooth(y, self.theta)

    def cost(self, occ, left, right, y):
        z = self.dose(occ, left, right, y)
        F, _ = self.penalty(z)
        G, _ = self.smooth(y, occ)
        return F, G, F + self.gamma * G

    # O4 ----------------------------------------------------------------------------------------
    def prices(self, w, occ=None):
        w = _as(w, np.float64)
        occ = None if occ is None else _as(occ, np.uint8)
        g = np.empty(self.B, np.float64)
        self._L.vo_prices(_c.byref(self._p), _ptr(w), _ptr(occ), _ptr(g))
        return g

    # O5 ----------------------------------------------------------------------------------------
    def leaf_box(self, occ, left, right, k, r):
        occ, left, right = self._plan(occ, left, right)
        box = np.empty(4, np.int64)
        self._L.vo_leaf_box(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), int(k), int(r), _ptr(box))
        return tuple(int(b) for b in box)

    # O5 + O6 -----------------------------------------------------------------------------------
    def price_step(self, g32, occ, left, right, y):
        """Returns dict(beam, price, left[R], right[R], beam_price[N], all_left[N,R], all_right[N,R])."""
        occ, left, right = self._plan(occ, left, right)
        g32, y = _as(g32, np.float32), _as(y, np.float64)
        bp = _c.c_double(0.0)
        bl, br = np.zeros(self.R, np.int32), np.zeros(self.R, np.int32)
        beam_price = np.empty(self.N, np.float64)
        al, ar = np.full(self.N * self.R, -1, np.int32), np.full(self.N * self.R, -1, np.int32)
        k = self._L.vo_price_step(_c.byref(self._p), _ptr(g32), _ptr(occ), _ptr(left), _ptr(right), _ptr(y),
                                  _c.addressof(bp), _ptr(bl), _ptr(br), _ptr(beam_price), _ptr(al), _ptr(ar))
        return dict(beam=int(k), price=float(bp.value), left=bl, right=br, beam_price=beam_price,
                    all_left=al.reshape(self.N, self.R), all_right=ar.reshape(self.N, self.R))

    # O7 ----------------------------------------------------------------------------------------
    def master(self, occ, left, right, y0=None, eps=1e-9, max_inner=20000, y_min=0.0, y_max=float("inf")):
        """Returns (y, z, MasterInfo).  y_min, y_max: bounds on the dose rates of the occupied beams (variant of
        PAPER.md:159's "maximum and minimum dose rate constraints"; default none but y >= 0)."""
        occ, left, right = self._plan(occ, left, right)
        y = np.zeros(self.N, np.float64) if y0 is None else _as(y0, np.float64).copy()
        z = np.empty(self.V, np.float64)
        info = _MasterInfo(eps=eps, max_inner=max_inner, lb=float(y_min), ub=float(y_max))
        self._L.vo_master(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), _ptr(y), _ptr(z), _c.byref(info))
        return y, z, MasterInfo(info.inner, info.backtracks, info.pg_entry, info.pg_exit, info.F, info.G, info.cost)

    def cost_gradient(self, occ, left, right, y):
        """dPhi/dy_k at occupied beams (0 elsewhere) and (F, G, Phi)."""
        occ, left, right = self._plan(occ, left, right)
        y = _as(y, np.float64)
        grad, c3 = np.empty(self.N, np.float64), np.empty(3, np.float64)
        self._L.vo_cost_gradient(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), _ptr(y), _ptr(grad), _ptr(c3))
        return grad, tuple(float(c) for c in c3)

    # hard dose-rate feasibility after the last aperture ---------------------------------
    def rate_ratio(self, y, rho):
        """max_k |y_{k+1} - y_k| / (rho (theta_{k+1} - theta_k)); the plan is feasible iff this is <= 1."""
        y = _as(y, np.float64)
        return float(self._L.vo_rate_ratio(self.N, _ptr(y), _ptr(self.theta), float(rho)))

    def enforce_rate(self, occ, left, right, y, rho, factor=2.0, tol=1e-6, max_rounds=60, eps=1e-9, max_inner=20000):
        """Raise gamma by `factor` and re-solve the master until |dy| <= rho dtheta everywhere.
        Returns (y, z, dict(rounds, feasible, gamma, ratio, F, G, cost))."""
        occ, left, right = self._plan(occ, left, right)
        y = _as(y, np.float64).copy()
        z = np.empty(self.V, np.float64)
        info = _RateInfo(rho=rho, factor=factor, tol=tol, max_rounds=max_rounds, eps=eps, max_inner=max_inner)
        self._L.vo_enforce_rate(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), _ptr(y), _ptr(z), _c.byref(info))
        return y, z, dict(rounds=int(info.rounds), feasible=bool(info.feasible), gamma=float(info.gamma),
                          ratio=float(info.ratio), F=float(info.F), G=float(info.G), cost=float(info.cost))

    # O1 + O8 -----------------------------------------------------------------------------------
    def solve(self, max_iters, plan=None, eps=1e-9, max_inner=20000, stop_when_priced_out=False, y_min=0.0,
              y_max=float("inf")):
        """Run the column-generation loop. Returns (occ, left[N,R], right[N,R], y, z, Trace).  y_min, y_max: bounds on
        the dose rates of occupied beams in every master solve (variant of PAPER.md:159; default the paper's y >= 0)."""
        if plan is None:
            occ, left, right, y = self.empty_plan()
        else:
            occ, left, right = (a.copy() for a in self._plan(*plan[:3]))
            y = _as(plan[3], np.float64).copy()
        z = np.zeros(self.V, np.float64)
        M, R = int(max_iters), self.R
        beam, inner = np.full(M, -1, np.int32), np.zeros(M, np.int64)
        price, F, G, cost = (np.zeros(M, np.float64) for _ in range(4))
        il, ir = np.zeros(M * R, np.int32), np.zeros(M * R, np.int32)
        tr = _Trace(max_iters=M, eps=eps, max_inner=max_inner, stop_when_priced_out=int(bool(stop_when_priced_out)), lb=float(y_min), ub=float(y_max), beam=_ptr(beam), price=_ptr(price), F=_ptr(F),
                    G=_ptr(G), cost=_ptr(cost), inner=_ptr(inner), it_left=_ptr(il), it_right=_ptr(ir))
        self._L.vo_solve(_c.byref(self._p), _ptr(occ), _ptr(left), _ptr(right), _ptr(y), _ptr(z), _c.byref(tr))
        n = int(tr.iters)
        trace = Trace(n, beam[:n], price[:n], F[:n], G[:n], cost[:n], inner[:n], il.reshape(M, R)[:n],
                      ir.reshape(M, R)[:n], tr.seconds_price, tr.seconds_master)
        return occ, left.reshape(self.N, R), right.reshape(self.N, R), y, z, trace
