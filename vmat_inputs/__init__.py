"""Seeded synthetic inputs for the VMAT hot path (shared by the CPU oracle tests and the CUDA path).

Holds *inputs only*: the phantoms of BASELINE.json:configs[0,1,2,4] (voxel grid, structures
T/alpha/beta, beam/leaf geometry, dose-deposition matrix D as fp32 CSR) and the isolated-kernel
sweep inputs of configs[3].  None of the method's arithmetic lives here.

The clinical prostate / head-and-neck cases of the paper (Table 1) are not
available; these phantoms stand in for their *shapes*.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libvmat_inputs.so")
_SRC_PATH = os.path.join(_HERE, "gen.c")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c -> libvmat_inputs.so (in-tree). Returns the library path."""
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(_SRC_PATH):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", _SRC_PATH, "-o", _LIB_PATH, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB_PATH


class _Geometry(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
        ("voxel_mm", ctypes.c_double),
        ("n_beams", ctypes.c_int32), ("n_rows", ctypes.c_int32), ("n_cols", ctypes.c_int32),
        ("beamlet_mm", ctypes.c_double), ("body_radius_mm", ctypes.c_double),
        ("mu_per_mm", ctypes.c_double), ("sigma_bw", ctypes.c_double),
        ("noise", ctypes.c_double), ("cutoff", ctypes.c_double),
        ("seed", ctypes.c_uint64),
    ]


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        P = ctypes.POINTER
        lib.vin_dose_matrix_count.restype = ctypes.c_int64
        lib.vin_dose_matrix_count.argtypes = [P(_Geometry), ctypes.c_void_p]
        lib.vin_dose_matrix_fill.restype = None
        lib.vin_dose_matrix_fill.argtypes = [P(_Geometry), ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.vin_sweep_row_lengths.restype = None
        lib.vin_sweep_row_lengths.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_uint64,
                                              ctypes.c_void_p]
        lib.vin_sweep_fill.restype = None
        lib.vin_sweep_fill.argtypes = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32,
                                       ctypes.c_int32, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p]
        lib.vin_normal.restype = None
        lib.vin_normal.argtypes = [ctypes.c_int64, ctypes.c_uint64, ctypes.c_void_p]
        lib.vin_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


# --------------------------------------------------------------------------------------------
# structures
# --------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Structure:
    """Ellipsoid (or z-cylinder if half_z is None) in voxel units relative to the grid centre."""
    name: str
    centre: Tuple[float, float, float]
    half: Tuple[float, float, Optional[float]]      # semi-axes (x, y, z); z None -> cylinder along z
    T: float
    alpha: float
    beta: float


@dataclass(frozen=True)
class PhantomConfig:
    name: str
    grid: Tuple[int, int, int]                      # nx, ny, nz
    voxel_mm: float
    n_beams: int
    n_rows: int
    n_cols: int
    beamlet_mm: float
    max_leaf_travel: int
    gamma: float
    iterations: int
    structures: Tuple[Structure, ...]               # painted last-to-first: earlier entries win overlaps
    other: Tuple[float, float, float] = (0.5, 0.0, 0.05)     # (T, alpha, beta) of unlisted in-body voxels
    body_radius_cap_mm: float = 100.0
    random_oars: int = 0                            # stress phantom: seeded random ellipsoids


def _tiny() -> PhantomConfig:
    return PhantomConfig(
        name="tiny", grid=(32, 32, 8), voxel_mm=5.0, n_beams=24, n_rows=8, n_cols=16, beamlet_mm=5.0,
        max_leaf_travel=3, gamma=0.1, iterations=40,
        structures=(
            Structure("target", (0, 0, 0), (6, 6, None), 1.0, 1.0, 1.0),
            Structure("oar", (9, 0, 0), (3, 3, None), 0.3, 0.0, 0.5),
        ))


def _prostate() -> PhantomConfig:
    return PhantomConfig(
        name="prostate", grid=(128, 128, 64), voxel_mm=4.0, n_beams=180, n_rows=40, n_cols=40, beamlet_mm=5.0,
        max_leaf_travel=2, gamma=0.1, iterations=180,
        structures=(
            Structure("target", (0, 0, 0), (12, 10, 10), 1.0, 1.0, 1.0),
            Structure("rectum", (0, -15, 0), (5, 5, 9), 0.4, 0.0, 1.0),
            Structure("bladder", (0, 18, 2), (9, 8, 8), 0.4, 0.0, 1.0),
            Structure("femoral_l", (-21, 0, 0), (5, 5, 5), 0.3, 0.0, 0.3),
            Structure("femoral_r", (21, 0, 0), (5, 5, 5), 0.3, 0.0, 0.3),
        ))


def _hn() -> PhantomConfig:
    return PhantomConfig(
        name="hn", grid=(160, 160, 96), voxel_mm=3.0, n_beams=180, n_rows=40, n_cols=60, beamlet_mm=5.0,
        max_leaf_travel=2, gamma=0.2, iterations=180,
        structures=(
            Structure("ptv1", (-5, 4, 0), (8, 8, 13), 1.0, 1.0, 1.0),
            Structure("ptv2", (-3, 3, 0), (15, 12, 22), 0.85, 1.0, 1.0),
            Structure("spinal_cord", (0, -17, 0), (2.5, 2.5, None), 0.6, 0.0, 1.0),
            Structure("brainstem", (0, -12, 27), (4, 4, 7), 0.6, 0.0, 1.0),
            Structure("parotid_l", (-22, 2, 8), (5, 6, 9), 0.3, 0.0, 1.0),
            Structure("parotid_r", (22, 2, 8), (5, 6, 9), 0.3, 0.0, 1.0),
            Structure("mandible", (0, 22, -8), (14, 4, 6), 0.9, 0.0, 1.0),
        ))


def _stress() -> PhantomConfig:
    return PhantomConfig(
        name="stress", grid=(256, 256, 128), voxel_mm=2.0, n_beams=360, n_rows=60, n_cols=80, beamlet_mm=2.5,
        max_leaf_travel=1, gamma=0.1, iterations=360,
        structures=(Structure("target", (0, 0, 0), (20, 16, 16), 1.0, 1.0, 1.0),),
        random_oars=6)


CONFIGS: Dict[str, PhantomConfig] = {c.name: c for c in (_tiny(), _prostate(), _hn(), _stress())}


def scaled_config(name: str, **overrides) -> PhantomConfig:
    """A named config with fields overridden (used for mid-size parity cases)."""
    return replace(CONFIGS[name], **overrides)


@dataclass
class Phantom:
    config: PhantomConfig
    seed: int
    n_voxels: int
    n_beamlets: int
    row_ptr: np.ndarray        # int64 [B+1]
    col_idx: np.ndarray        # int32 [nnz], strictly ascending within a row
    val: np.ndarray            # float32 [nnz]
    T: np.ndarray              # float32 [V]
    alpha: np.ndarray          # float32 [V]
    beta: np.ndarray           # float32 [V]
    theta_deg: np.ndarray      # float64 [N]
    body: np.ndarray           # bool [V]
    structures: List[Structure] = field(default_factory=list)
    volume: Optional[np.ndarray] = None   # float32 [V]: fine voxels a voxel stands for (mixed resolution), None = all 1

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])


def body_radius_mm(cfg: PhantomConfig) -> float:
    nx, ny, _ = cfg.grid
    return float(min(0.5 * nx * cfg.voxel_mm, 0.5 * ny * cfg.voxel_mm, cfg.body_radius_cap_mm))


def _random_oars(cfg: PhantomConfig, seed: int) -> List[Structure]:
    rng = np.random.default_rng(seed + 7919)
    rb_vox = body_radius_mm(cfg) / cfg.voxel_mm
    out = []
    for q in range(cfg.random_oars):
        ang = rng.uniform(0, 2 * np.pi)
        rad = rng.uniform(0.35, 0.7) * rb_vox
        half = tuple(float(h) for h in rng.uniform(0.08, 0.18, 3) * rb_vox)
        cz = float(rng.uniform(-0.25, 0.25) * cfg.grid[2])
        out.append(Structure(f"oar{q}", (float(rad * np.cos(ang)), float(rad * np.sin(ang)), cz), half,
                             float(rng.uniform(0.2, 0.7)), 0.0, 1.0))
    return out


def paint_structures(cfg: PhantomConfig, seed: int = 0):
    """Voxel parameters T/alpha/beta (float32[V]) and the body mask for a config."""
    nx, ny, nz = cfg.grid
    x = (np.arange(nx) + 0.5 - 0.5 * nx)[None, None, :]
    y = (np.arange(ny) + 0.5 - 0.5 * ny)[None, :, None]
    z = (np.arange(nz) + 0.5 - 0.5 * nz)[:, None, None]
    rb = body_radius_mm(cfg) / cfg.voxel_mm
    body = np.broadcast_to((x * x + y * y) <= rb * rb, (nz, ny, nx))
    T = np.zeros((nz, ny, nx), np.float32)
    alpha = np.zeros_like(T)
    beta = np.zeros_like(T)
    T[body], alpha[body], beta[body] = cfg.other
    structs = list(cfg.structures) + _random_oars(cfg, seed)
    for s in reversed(structs):
        cx, cy, cz = s.centre
        hx, hy, hz = s.half
        m = ((x - cx) / hx) ** 2 + ((y - cy) / hy) ** 2
        if hz is not None:
            m = m + ((z - cz) / hz) ** 2
        m = np.broadcast_to(m <= 1.0, (nz, ny, nx)) & body
        T[m], alpha[m], beta[m] = s.T, s.alpha, s.beta
    return T.reshape(-1), alpha.reshape(-1), beta.reshape(-1), np.ascontiguousarray(body).reshape(-1), structs


def coarsen_unspecified_tissue(ph: "Phantom") -> "Phantom":
    """Mixed voxel resolution ("For unspecified tissue ... we increased the voxel size in each dimension
    by a factor of 2 to reduce the optimization problem size"): every 2 x 2 x 2 block of the grid whose eight voxels all
    carry the config's `other` parameters (or all lie outside the body) becomes ONE voxel.  Its column of D is the mean
    of the eight columns (the dose of the coarse voxel), its penalty weights are 8 x (it stands for eight voxels'
    worth of volume), T is unchanged.  Voxels of blocks that touch a structure or the body contour stay as they are.
    Voxel ids keep the raster order of the fine grid (a coarse voxel sits where its first fine voxel sat).  This is
    input preprocessing only: none of the method's arithmetic."""
    cfg = ph.config
    nx, ny, nz = cfg.grid
    assert nx % 2 == 0 and ny % 2 == 0 and nz % 2 == 0, "mixed resolution needs even grid dimensions"
    V = ph.n_voxels
    To, ao, bo = (np.float32(v) for v in cfg.other)
    tissue = (ph.T == To) & (ph.alpha == ao) & (ph.beta == bo) & ph.body
    outside = (ph.T == 0) & (ph.alpha == 0) & (ph.beta == 0) & ~ph.body

    def blocks(mask):
        return mask.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).all(axis=(1, 3, 5))

    merge = blocks(tissue) | blocks(outside)                         # [nz/2, ny/2, nx/2]
    merge_fine = np.repeat(np.repeat(np.repeat(merge, 2, 0), 2, 1), 2, 2).reshape(-1)
    idx = np.arange(V).reshape(nz, ny, nx)
    first = (idx[0::2, 0::2, 0::2])                                  # first fine voxel of every block
    first_fine = np.repeat(np.repeat(np.repeat(first, 2, 0), 2, 1), 2, 2).reshape(-1)
    rep = np.where(merge_fine, first_fine, np.arange(V))             # representative fine voxel of every voxel
    keep = rep == np.arange(V)
    new_id = np.cumsum(keep) - 1
    col_new = new_id[rep[ph.col_idx]]
    scale = np.where(merge_fine[ph.col_idx], np.float64(0.125), np.float64(1.0))
    rows = np.repeat(np.arange(ph.n_beamlets, dtype=np.int64), np.diff(ph.row_ptr))
    Vn = int(keep.sum())
    key = rows * Vn + col_new
    order = np.argsort(key, kind="stable")
    key_s = key[order]
    val_s = ph.val[order].astype(np.float64) * scale[order]
    start = np.flatnonzero(np.concatenate([[True], key_s[1:] != key_s[:-1]])) if key_s.size else np.zeros(0, np.int64)
    val_n = np.add.reduceat(val_s, start).astype(np.float32) if key_s.size else np.zeros(0, np.float32)
    key_u = key_s[start] if key_s.size else key_s
    row_u, col_u = key_u // Vn, (key_u % Vn).astype(np.int32)
    row_ptr = np.zeros(ph.n_beamlets + 1, np.int64)
    np.add.at(row_ptr, row_u + 1, 1)
    row_ptr = np.cumsum(row_ptr)
    w8 = np.where(merge_fine[keep], np.float32(8.0), np.float32(1.0))
    return Phantom(cfg, ph.seed, Vn, ph.n_beamlets, row_ptr, col_u, val_n, ph.T[keep].copy(),
                   (ph.alpha[keep] * w8).astype(np.float32), (ph.beta[keep] * w8).astype(np.float32), ph.theta_deg,
                   ph.body[keep].copy(), ph.structures, w8)


def make_phantom(config="tiny", seed: int = 0, check_reach: bool = True, mixed_resolution: bool = False) -> Phantom:
    """Build a phantom (structures + D).  `config` is a name in CONFIGS or a PhantomConfig.  mixed_resolution: coarsen
    the unspecified tissue by a factor of 2 per dimension (coarsen_unspecified_tissue)."""
    if mixed_resolution:
        return coarsen_unspecified_tissue(make_phantom(config, seed, check_reach))
    cfg = CONFIGS[config] if isinstance(config, str) else config
    lib = _load()
    nx, ny, nz = cfg.grid
    g = _Geometry(nx, ny, nz, cfg.voxel_mm, cfg.n_beams, cfg.n_rows, cfg.n_cols, cfg.beamlet_mm,
                  body_radius_mm(cfg), 0.05, 0.6, 0.02, 1e-3, seed)
    B = cfg.n_beams * cfg.n_rows * cfg.n_cols
    row_ptr = np.empty(B + 1, np.int64)
    nnz = lib.vin_dose_matrix_count(ctypes.byref(g), row_ptr.ctypes.data)
    col = np.empty(nnz, np.int32)
    val = np.empty(nnz, np.float32)
    lib.vin_dose_matrix_fill(ctypes.byref(g), row_ptr.ctypes.data, col.ctypes.data, val.ctypes.data)
    T, alpha, beta, body, structs = paint_structures(cfg, seed)
    V = nx * ny * nz
    if check_reach:
        # generator self-check: every underdose-penalised voxel is reachable
        hit = np.zeros(V, bool)
        hit[col] = True
        missed = int(np.count_nonzero((alpha > 0) & ~hit))
        if missed:
            raise RuntimeError(f"phantom {cfg.name}: {missed} voxels with alpha>0 receive no dose from any beamlet")
    theta = np.arange(cfg.n_beams, dtype=np.float64) * (360.0 / cfg.n_beams)
    return Phantom(cfg, seed, V, B, row_ptr, col, val, T, alpha, beta, theta, body, structs)


# --------------------------------------------------------------------------------------------
# BASELINE.json:configs[3] — isolated kernel sweep inputs
# --------------------------------------------------------------------------------------------
def make_sweep_matrix(nnz_target: int, n_voxels: int, seed: int = 0, len_range=(200, 800), run_range=(8, 64)):
    """Beamlet-major fp32 CSR with row lengths U[200,800] and voxel indices in contiguous runs of U[8,64]."""
    lib = _load()
    n_rows = max(1, int(round(nnz_target / (0.5 * (len_range[0] + len_range[1])))))
    row_ptr = np.empty(n_rows + 1, np.int64)
    lib.vin_sweep_row_lengths(n_rows, len_range[0], len_range[1], seed, row_ptr.ctypes.data)
    nnz = int(row_ptr[-1])
    col = np.empty(nnz, np.int32)
    val = np.empty(nnz, np.float32)
    lib.vin_sweep_fill(n_rows, row_ptr.ctypes.data, n_voxels, run_range[0], run_range[1], seed,
                       col.ctypes.data, val.ctypes.data)
    return row_ptr, col, val


def make_normal(n: int, seed: int = 0) -> np.ndarray:
    """w ~ N(0,1), float32[n] (counter-based)."""
    lib = _load()
    out = np.empty(n, np.float32)
    lib.vin_normal(n, seed, out.ctypes.data)
    return out


def make_search_rows(n_beams: int, n_rows: int, n_cols: int, seed: int = 0, zero_frac: float = 0.1):
    """Prices for the isolated leaf-search sweep: N(0,1) fp32 with `zero_frac` exact zeros."""
    g = make_normal(n_beams * n_rows * n_cols, seed)
    rng = np.random.default_rng(seed + 1)
    g[rng.random(g.size) < zero_frac] = 0.0
    return g


def num_threads() -> int:
    return int(_load().vin_num_threads())
