"""paper_1005_4396_b200 — Python binding of libvmat_b200.so (include/vmat.h).

Argument marshalling only: every step of the column-generation VMAT hot path runs in the CUDA
kernels of csrc/.  PyTorch provides device memory and the stream; nothing here computes, and there
is no CPU fallback — a missing library or a missing GPU raises.

    plan = Plan.create(row_ptr, col_idx, val, T, alpha, beta, theta_deg, n_rows, n_cols,
                       max_leaf_travel, gamma)          # numpy (host) or torch.cuda tensors
    stats = plan.solve(180)
    occ, left, right, y = plan.get_plan()
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvmat_b200.so")

VMAT_OK, VMAT_DONE, VMAT_EINVAL, VMAT_ENOMEM, VMAT_ECUDA, VMAT_ESTATE = 0, 1, -1, -2, -3, -4
VMAT_HOST, VMAT_DEVICE = 0, 1

# every symbol include/vmat.h declares
SYMBOLS = (
    "vmat_default_options", "vmat_create", "vmat_destroy", "vmat_get_info", "vmat_dose", "vmat_dose_recompute",
    "vmat_price",
    "vmat_price_spmv", "vmat_leaf_search", "vmat_master", "vmat_enforce_dose_rate", "vmat_solve", "vmat_get_plan", "vmat_set_plan",
    "vmat_launch_count", "vmat_last_error", "vmat_release_memory", "vmat_set_dose_rate_bounds",
    "vmat_engine_dose_matrix", "vmat_engine_free", "vmat_penalty_noalloc",
)

_P = C.c_void_p


class _Problem(C.Structure):
    _fields_ = [("n_voxels", C.c_int64), ("n_beams", C.c_int64), ("n_rows", C.c_int64), ("n_cols", C.c_int64),
                ("row_ptr", _P), ("col_idx", _P), ("val", _P), ("T", _P), ("alpha", _P), ("beta", _P),
                ("theta_deg", _P), ("max_leaf_travel", C.c_int32), ("gamma", C.c_double), ("mem_space", C.c_int32)]


class Options(C.Structure):
    _fields_ = [("validate", C.c_int32), ("d_format", C.c_int32), ("dose_path", C.c_int32),
                ("master_eps", C.c_double), ("master_max_inner", C.c_int32), ("master_stall_rel", C.c_double),
                ("master_stall_count", C.c_int32), ("record_phases", C.c_int32), ("master_mode", C.c_int32), ("stop_when_priced_out", C.c_int32),
                ("master_unstaged_lists", C.c_int32), ("occupied_only_G", C.c_int32),
                ("master_newton_max_beams", C.c_int32)]


class _Aperture(C.Structure):
    _fields_ = [("beam", C.c_int32), ("price", C.c_double), ("left", _P), ("right", _P)]


class _MasterOpts(C.Structure):
    _fields_ = [("eps", C.c_double), ("max_inner", C.c_int32), ("stall_rel", C.c_double), ("stall_count", C.c_int32)]


class _MasterStats(C.Structure):
    _fields_ = [("inner", C.c_int32), ("backtracks", C.c_int32), ("stop_reason", C.c_int32),
                ("passes", C.c_int32), ("pg_entry", C.c_double), ("pg_exit", C.c_double), ("F", C.c_double), ("G", C.c_double),
                ("cost", C.c_double)]


class _SolveStats(C.Structure):
    _fields_ = [("iters", C.c_int32), ("us_total", C.c_double), ("us_price", C.c_double), ("us_search", C.c_double),
                ("us_column", C.c_double), ("us_master", C.c_double), ("F", C.c_double), ("G", C.c_double),
                ("cost", C.c_double), ("beam", _P), ("price", _P), ("trace_F", _P), ("trace_G", _P),
                ("trace_cost", _P), ("inner", _P), ("master_passes", C.c_double), ("master_bytes", C.c_double),
                ("master_cg_steps", C.c_double), ("master_clk_cg", C.c_double), ("master_clk_wait", C.c_double),
                ("master_clk_load", C.c_double)]


class _RateStats(C.Structure):
    _fields_ = [("rounds", C.c_int32), ("feasible", C.c_int32), ("inner_total", C.c_int32), ("gamma", C.c_double),
                ("ratio", C.c_double), ("F", C.c_double), ("G", C.c_double), ("cost", C.c_double)]


class _Info(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_voxels", "n_beams", "n_rows", "n_cols", "n_beamlets", "nnz",
                                         "nnz_padded", "n_support", "device_bytes", "pricing_bytes")]


class EngineGeometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("voxel_mm", C.c_double),
                ("n_beams", C.c_int32), ("n_rows", C.c_int32), ("n_cols", C.c_int32), ("beamlet_mm", C.c_double),
                ("body_radius_mm", C.c_double), ("mu_per_mm", C.c_double), ("sigma_beamlets", C.c_double),
                ("noise", C.c_double), ("cutoff", C.c_double), ("seed", C.c_uint64)]


class VmatError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"vmat error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libvmat_b200.so and declare its prototypes.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1005_4396_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.vmat_default_options.argtypes = [C.POINTER(Options)]
    L.vmat_default_options.restype = None
    L.vmat_create.argtypes = [C.POINTER(_Problem), C.POINTER(Options), _P, C.POINTER(_P)]
    L.vmat_destroy.argtypes = [_P]
    L.vmat_get_info.argtypes = [_P, C.POINTER(_Info)]
    L.vmat_dose.argtypes = [_P, _P, _P, _P]
    L.vmat_dose_recompute.argtypes = [_P, C.c_int]
    L.vmat_price.argtypes = [_P, _P, _P, _P, C.POINTER(_Aperture), C.c_int]
    L.vmat_price_spmv.argtypes = [_P, _P, _P]
    L.vmat_leaf_search.argtypes = [_P, _P, _P, _P, _P]
    L.vmat_master.argtypes = [_P, C.POINTER(_MasterOpts), C.POINTER(_MasterStats)]
    L.vmat_enforce_dose_rate.argtypes = [_P, C.c_double, C.c_double, C.c_double, C.c_int32, C.POINTER(_RateStats)]
    L.vmat_solve.argtypes = [_P, C.c_int32, C.POINTER(_SolveStats)]
    L.vmat_get_plan.argtypes = [_P, _P, _P, _P, _P]
    L.vmat_set_plan.argtypes = [_P, _P, _P, _P, _P]
    L.vmat_launch_count.argtypes = [_P]
    L.vmat_release_memory.argtypes = []
    L.vmat_set_dose_rate_bounds.argtypes = [_P, C.c_double, C.c_double]
    L.vmat_engine_dose_matrix.argtypes = [C.POINTER(EngineGeometry), _P, C.POINTER(_P), C.POINTER(_P), C.POINTER(_P),
                                          C.POINTER(C.c_int64)]
    L.vmat_engine_dose_matrix.restype = C.c_int
    L.vmat_engine_free.argtypes = [_P, _P]
    L.vmat_engine_free.restype = C.c_int
    L.vmat_penalty_noalloc.argtypes = [_P, _P, _P, _P, C.c_int64, _P, _P, _P]
    L.vmat_penalty_noalloc.restype = C.c_int
    L.vmat_launch_count.restype = C.c_int64
    L.vmat_last_error.argtypes = [_P]
    L.vmat_last_error.restype = C.c_char_p
    for name in ("vmat_create", "vmat_destroy", "vmat_get_info", "vmat_dose", "vmat_dose_recompute", "vmat_price",
                 "vmat_price_spmv",
                 "vmat_leaf_search", "vmat_master", "vmat_enforce_dose_rate", "vmat_solve", "vmat_get_plan",
                 "vmat_set_plan"):
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def release_memory() -> None:
    """vmat_release_memory: hand the device memory that destroyed plans left in the library's pools back to the driver."""
    rc = load_library().vmat_release_memory()
    if rc != 0:
        raise RuntimeError(f"vmat_release_memory failed ({rc})")


class EngineMatrix:
    """D as vmat_engine_dose_matrix left it on the device.  row_ptr / col_idx / val are CUDA torch tensors that view
    the library's buffers (no copy); release() hands the buffers back.  Marshalling only."""

    def __init__(self, geometry: EngineGeometry, stream: Optional[int] = None):
        import torch

        L = load_library()
        if stream is None:
            if not torch.cuda.is_available():
                raise VmatError(VMAT_ECUDA, "no CUDA device (there is no CPU fallback)")
            stream = torch.cuda.current_stream().cuda_stream
        self._stream = stream
        rp, ci, va, nnz = _P(), _P(), _P(), C.c_int64(0)
        rc = L.vmat_engine_dose_matrix(C.byref(geometry), _P(stream), C.byref(rp), C.byref(ci), C.byref(va), C.byref(nnz))
        if rc != VMAT_OK:
            raise VmatError(rc, (L.vmat_last_error(None) or b"").decode())
        self._ptrs = (rp.value, ci.value, va.value)
        self.nnz = int(nnz.value)
        B = geometry.n_beams * geometry.n_rows * geometry.n_cols
        self.n_beamlets = B

        def view(ptr, n, dtype, typestr):
            class _Arr:   # __cuda_array_interface__ carrier: torch wraps the memory without copying
                pass
            a = _Arr()
            a.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 3}
            return torch.as_tensor(a, device="cuda")

        self.row_ptr = view(rp.value, B + 1, None, "<i8")
        self.col_idx = view(ci.value, max(self.nnz, 1), None, "<i4")[:self.nnz]
        self.val = view(va.value, max(self.nnz, 1), None, "<f4")[:self.nnz]

    def release(self):
        L = load_library()
        for ptr in self._ptrs:
            L.vmat_engine_free(_P(ptr), _P(self._stream))
        self._ptrs = ()
        self.row_ptr = self.col_idx = self.val = None


def default_options() -> Options:
    o = Options()
    load_library().vmat_default_options(C.byref(o))
    return o


@dataclass
class Aperture:
    beam: int
    price: float
    left: np.ndarray
    right: np.ndarray


@dataclass
class MasterStats:
    inner: int
    backtracks: int
    stop_reason: int
    pg_entry: float
    pg_exit: float
    F: float
    G: float
    cost: float
    passes: int = 0


@dataclass
class SolveStats:
    iters: int
    us_total: float
    us_price: float
    us_search: float
    us_column: float
    us_master: float
    F: float
    G: float
    cost: float
    beam: np.ndarray
    price: np.ndarray
    trace_F: np.ndarray
    trace_G: np.ndarray
    trace_cost: np.ndarray
    inner: np.ndarray
    master_passes: float = 0.0
    master_bytes: float = 0.0
    master_cg_steps: float = 0.0
    master_clk_cg: float = 0.0
    master_clk_wait: float = 0.0
    master_clk_load: float = 0.0


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


def _dev_ptr(t, dtype_name: str, n: Optional[int] = None) -> int:
    """data_ptr of a contiguous CUDA torch tensor of the given dtype (None -> NULL)."""
    if t is None:
        return 0
    import torch

    want = getattr(torch, dtype_name)
    if not (_is_torch(t) and t.is_cuda and t.dtype == want and t.is_contiguous()):
        raise TypeError(f"expected a contiguous CUDA torch tensor of dtype {dtype_name}")
    if n is not None and t.numel() != n:
        raise ValueError(f"expected {n} elements, got {t.numel()}")
    return t.data_ptr()


NOALLOC_MAX_VOXELS = 1 << 24   # VMAT_NOALLOC_MAX_VOXELS of include/vmat.h


def penalty_noalloc(z, T, alpha, beta, w=None, F=None, stream: Optional[int] = None) -> None:
    """vmat_penalty_noalloc: step (b) on a caller's dose, allocating nothing (its scratch is a fixed array in the
    library's device image: at most NOALLOC_MAX_VOXELS voxels, calls that overlap on one GPU race).  z, T, alpha, beta:
    CUDA float32[n]; w: CUDA float32[n] or None; F: CUDA float64[1] or None.  Stream-ordered (default: torch's current
    stream); argument marshalling only."""
    import torch

    n = int(z.numel())
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    L = load_library()
    rc = L.vmat_penalty_noalloc(_dev_ptr(z, "float32", n), _dev_ptr(T, "float32", n), _dev_ptr(alpha, "float32", n),
                                _dev_ptr(beta, "float32", n), n, _dev_ptr(w, "float32", n), _dev_ptr(F, "float64", 1),
                                _P(stream))
    if rc < 0:
        raise VmatError(rc, (L.vmat_last_error(None) or b"").decode())


class Plan:
    """One vmat_plan (include/vmat.h).  Use Plan.create(...)."""

    def __init__(self, handle: int, keep):
        self._h = _P(handle)
        self._L = load_library()
        self._keep = keep
        info = _Info()
        self._check(self._L.vmat_get_info(self._h, C.byref(info)))
        self.V, self.N, self.R, self.Cc, self.B = info.n_voxels, info.n_beams, info.n_rows, info.n_cols, info.n_beamlets
        self.nnz, self.nnz_padded, self.n_support, self.device_bytes = (info.nnz, info.nnz_padded, info.n_support,
                                                                        info.device_bytes)
        self.pricing_bytes = info.pricing_bytes

    # -- life cycle ----------------------------------------------------------------------------
    @classmethod
    def create(cls, row_ptr, col_idx, val, T, alpha, beta, theta_deg, n_rows, n_cols, max_leaf_travel, gamma,
               options: Optional[Options] = None, stream: Optional[int] = None) -> "Plan":
        """vmat_create.  The six big arrays are either all numpy (host) or all CUDA torch tensors."""
        L = load_library()
        arrays = (row_ptr, col_idx, val, T, alpha, beta)
        on_dev = [_is_torch(a) and a.is_cuda for a in arrays]
        theta = np.ascontiguousarray(theta_deg, dtype=np.float64)
        if all(on_dev):
            names = ("int64", "int32", "float32", "float32", "float32", "float32")
            ptrs = [_dev_ptr(a, n) for a, n in zip(arrays, names)]
            keep = arrays
            space = VMAT_DEVICE
            V = T.numel()
        elif not any(on_dev):
            dts = (np.int64, np.int32, np.float32, np.float32, np.float32, np.float32)
            keep = tuple(np.ascontiguousarray(a.numpy() if _is_torch(a) else a, dtype=d) for a, d in zip(arrays, dts))
            ptrs = [a.ctypes.data for a in keep]
            space = VMAT_HOST
            V = keep[3].size
        else:
            raise TypeError("row_ptr, col_idx, val, T, alpha, beta must all be host arrays or all CUDA tensors")
        B = theta.size * int(n_rows) * int(n_cols)
        n_rp = row_ptr.numel() if _is_torch(row_ptr) else keep[0].size
        if n_rp != B + 1:
            raise ValueError(f"row_ptr must have n_beams*n_rows*n_cols+1 = {B + 1} entries, got {n_rp}")
        if stream is None:
            import torch

            if not torch.cuda.is_available():
                raise VmatError(VMAT_ECUDA, "no CUDA device (there is no CPU fallback)")
            stream = torch.cuda.current_stream().cuda_stream
        pb = _Problem(V, theta.size, int(n_rows), int(n_cols), ptrs[0], ptrs[1], ptrs[2], ptrs[3], ptrs[4], ptrs[5],
                      theta.ctypes.data, int(max_leaf_travel), float(gamma), space)
        h = _P()
        rc = L.vmat_create(C.byref(pb), C.byref(options) if options is not None else None, _P(stream), C.byref(h))
        if rc != VMAT_OK:
            raise VmatError(rc, (L.vmat_last_error(None) or b"").decode())
        return cls(h.value, None)

    @classmethod
    def from_phantom(cls, ph, gamma=None, max_leaf_travel=None, options=None, device_arrays=False) -> "Plan":
        c = ph.config
        arrs = [ph.row_ptr, ph.col_idx, ph.val, ph.T, ph.alpha, ph.beta]
        if device_arrays:
            import torch

            arrs = [torch.from_numpy(a).cuda() for a in arrs]
        return cls.create(*arrs, ph.theta_deg, c.n_rows, c.n_cols,
                          c.max_leaf_travel if max_leaf_travel is None else max_leaf_travel,
                          c.gamma if gamma is None else gamma, options=options)

    def destroy(self):
        if self._h:
            self._L.vmat_destroy(self._h)
            self._h = _P()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _check(self, rc: int) -> int:
        if rc < 0:
            raise VmatError(rc, (self._L.vmat_last_error(self._h) or b"").decode())
        return rc

    # -- steps ----------------------------------------------------------------------------------
    def dose(self, z=None, w=None, want_cost: bool = True):
        """vmat_dose: z, w are optional CUDA float32 tensors of V elements (filled in place).
        Returns (F, G, F + gamma G) or None."""
        cost = (C.c_double * 3)()
        self._check(self._L.vmat_dose(self._h, _dev_ptr(z, "float32", self.V), _dev_ptr(w, "float32", self.V),
                                      C.addressof(cost) if want_cost else None))
        return tuple(cost) if want_cost else None

    def dose_recompute(self, dose_path: int = -1):
        """vmat_dose_recompute: run steps (a)+(b) again by the given path (0 columns, 1 from D).  Stream-ordered."""
        self._check(self._L.vmat_dose_recompute(self._h, int(dose_path)))

    def price(self, w_override=None, g_override=None, g_out=None, commit: bool = False) -> Optional[Aperture]:
        """vmat_price.  Returns the chosen Aperture, or None when every beam is occupied."""
        left, right = np.zeros(self.R, np.int32), np.zeros(self.R, np.int32)
        ap = _Aperture(-1, 0.0, left.ctypes.data, right.ctypes.data)
        rc = self._check(self._L.vmat_price(self._h, _dev_ptr(w_override, "float32", self.V),
                                            _dev_ptr(g_override, "float32", self.B),
                                            _dev_ptr(g_out, "float32", self.B), C.byref(ap), 1 if commit else 0))
        if rc == VMAT_DONE:
            return None
        return Aperture(int(ap.beam), float(ap.price), left, right)

    def price_spmv(self, g, w=None):
        """vmat_price_spmv: g (CUDA float32[B]) = D w for un-occupied beams.  Stream-ordered."""
        self._check(self._L.vmat_price_spmv(self._h, _dev_ptr(w, "float32", self.V), _dev_ptr(g, "float32", self.B)))

    def leaf_search(self, g, all_left=None, all_right=None, beam_price=None):
        """vmat_leaf_search on prices g (CUDA float32[B]).  Stream-ordered."""
        self._check(self._L.vmat_leaf_search(self._h, _dev_ptr(g, "float32", self.B),
                                             _dev_ptr(all_left, "int32", self.N * self.R),
                                             _dev_ptr(all_right, "int32", self.N * self.R),
                                             _dev_ptr(beam_price, "float64", self.N)))

    def master(self, eps: float = 0.0, max_inner: int = 0, stall_rel: float = 0.0, stall_count: int = 0) -> MasterStats:
        """vmat_master; the keyword arguments are the per-call overrides of vmat_master_opts (0 = the plan's option)."""
        s = _MasterStats()
        o = _MasterOpts(float(eps), int(max_inner), float(stall_rel), int(stall_count))
        self._check(self._L.vmat_master(self._h, C.byref(o), C.byref(s)))
        return MasterStats(s.inner, s.backtracks, s.stop_reason, s.pg_entry, s.pg_exit, s.F, s.G, s.cost, s.passes)

    def set_dose_rate_bounds(self, y_min: float = 0.0, y_max: float = float("inf")) -> None:
        """vmat_set_dose_rate_bounds: the master solves from now on keep y_min <= y_k <= y_max at occupied beams."""
        self._check(self._L.vmat_set_dose_rate_bounds(self._h, float(y_min), float(y_max)))

    def enforce_dose_rate(self, max_variation_per_deg: float, gamma_factor: float = 2.0, tol: float = 1e-6,
                          max_rounds: int = 60) -> dict:
        """vmat_enforce_dose_rate: raise gamma and re-solve the master until the dose-rate variation
        between neighbouring angles is within the limit.  Returns the stats as a dict."""
        s = _RateStats()
        self._check(self._L.vmat_enforce_dose_rate(self._h, float(max_variation_per_deg), float(gamma_factor),
                                                   float(tol), int(max_rounds), C.byref(s)))
        return dict(rounds=s.rounds, feasible=bool(s.feasible), inner_total=s.inner_total, gamma=s.gamma,
                    ratio=s.ratio, F=s.F, G=s.G, cost=s.cost)

    def solve(self, max_iters: int, trace: bool = True) -> SolveStats:
        M = max(int(max_iters), 1)
        beam, inner = np.full(M, -1, np.int32), np.zeros(M, np.int32)
        price, tF, tG, tC = (np.zeros(M, np.float64) for _ in range(4))
        s = _SolveStats()
        if trace:
            s.beam, s.price, s.trace_F, s.trace_G, s.trace_cost, s.inner = (a.ctypes.data for a in
                                                                           (beam, price, tF, tG, tC, inner))
        self._check(self._L.vmat_solve(self._h, int(max_iters), C.byref(s)))
        n = int(s.iters)
        return SolveStats(n, s.us_total, s.us_price, s.us_search, s.us_column, s.us_master, s.F, s.G, s.cost,
                          beam[:n], price[:n], tF[:n], tG[:n], tC[:n], inner[:n], s.master_passes, s.master_bytes,
                          s.master_cg_steps, s.master_clk_cg, s.master_clk_wait, s.master_clk_load)

    # -- plan state -------------------------------------------------------------------------------
    def get_plan(self):
        occ = np.zeros(self.N, np.uint8)
        left, right = np.zeros(self.N * self.R, np.int32), np.zeros(self.N * self.R, np.int32)
        y = np.zeros(self.N, np.float64)
        self._check(self._L.vmat_get_plan(self._h, occ.ctypes.data, left.ctypes.data, right.ctypes.data, y.ctypes.data))
        return occ, left.reshape(self.N, self.R), right.reshape(self.N, self.R), y

    def set_plan(self, occ, left, right, y):
        occ = np.ascontiguousarray(occ, np.uint8)
        left = np.ascontiguousarray(left, np.int32).reshape(-1)
        right = np.ascontiguousarray(right, np.int32).reshape(-1)
        y = np.ascontiguousarray(y, np.float64)
        if occ.size != self.N or y.size != self.N or left.size != self.N * self.R or right.size != self.N * self.R:
            raise ValueError("plan arrays have the wrong size")
        self._check(self._L.vmat_set_plan(self._h, occ.ctypes.data, left.ctypes.data, right.ctypes.data, y.ctypes.data))

    @property
    def launch_count(self) -> int:
        return int(self._L.vmat_launch_count(self._h))
