"""ctypes binding of the CPU oracle (oracle/sd_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It does not import, and is not
imported by, the CUDA package paper_1205_6333_b200.

The oracle evaluates Eq. (7a) of the paper as a plain double loop in fp64 with
long-double row accumulation; see the header of sd_oracle.c for the readings.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sd_oracle.c")
_LIB = os.path.join(_HERE, "libsd_oracle.so")

TENSOR_RPY = 0      # Eq. (7b) + RPY overlap branch for r < 2a
TENSOR_OSEEN = 1    # Eq. (4)
TENSOR_RP_FAR = 2   # Eq. (7b) as printed for every r (negative control)
INT_EULER = 0
INT_MIDPOINT = 1
IMAGE_DEFINITION = 0  # nearest image from C99 remainder(): the plain definition
IMAGE_F32 = 1         # image index decided as an fp32 evaluation decides it (B2)
IMAGE_F64 = 2         # image index decided as an fp64 evaluation decides it (B2)

_lib = None


def build(force: bool = False) -> str:
    """Compile sd_oracle.c with gcc into oracle/libsd_oracle.so (no-op when up to date)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB)
    dp = ctypes.POINTER(ctypes.c_double)
    lp = ctypes.POINTER(ctypes.c_longlong)
    ll, dbl, ci = ctypes.c_longlong, ctypes.c_double, ctypes.c_int
    lib.sdo_mu0.restype = dbl
    lib.sdo_mu0.argtypes = [dbl, dbl]
    lib.sdo_apply_rows.restype = ci
    lib.sdo_apply_rows.argtypes = [dp, dp, ll, dbl, dbl, ci, lp, ll, dp]
    lib.sdo_apply.restype = ci
    lib.sdo_apply.argtypes = [dp, dp, ll, dbl, dbl, ci, dp]
    lib.sdo_assemble.restype = ci
    lib.sdo_assemble.argtypes = [dp, ll, dbl, dbl, ci, dp]
    lib.sdo_step.restype = ci
    lib.sdo_step.argtypes = [dp, dp, ll, dbl, dbl, ci, dbl, ll, ci, dp, ll, dp]
    lib.sdo_apply_rows_box.restype = ci
    lib.sdo_apply_rows_box.argtypes = [dp, dp, ll, dbl, dbl, ci, dbl, ci, lp, ll, dp]
    lib.sdo_apply_box.restype = ci
    lib.sdo_apply_box.argtypes = [dp, dp, ll, dbl, dbl, ci, dbl, ci, dp]
    lib.sdo_assemble_box.restype = ci
    lib.sdo_assemble_box.argtypes = [dp, ll, dbl, dbl, ci, dbl, ci, dp]
    lib.sdo_step_box.restype = ci
    lib.sdo_step_box.argtypes = [dp, dp, ll, dbl, dbl, ci, dbl, ci, dbl, ll, ci, dp, ll, dp]
    lib.sdo_lubrication.restype = ci
    lib.sdo_lubrication.argtypes = [dp, dp, ll, dbl, dbl, dbl, ci, ci, dp]
    lib.sdo_step_lub.restype = ci
    lib.sdo_step_lub.argtypes = [dp, dp, dp, ll, dbl, dbl, ci, dbl, ci, ci, dbl, ll, ci]
    lib.sdo_num_threads.restype = ci
    lib.sdo_set_num_threads.argtypes = [ci]
    _lib = lib
    return lib


def _as3(x, name):
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if x.ndim != 2 or x.shape[1] != 3:
        raise ValueError(f"{name} must have shape [N, 3], got {x.shape}")
    return x


def _dp(x):
    return x.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"{what} failed with status {rc}")


def mu0(a: float, eta: float) -> float:
    return float(_load().sdo_mu0(a, eta))


def apply(pos, force, a: float, eta: float, tensor: int = TENSOR_RPY, box: float = 0.0,
          image: int = IMAGE_DEFINITION) -> np.ndarray:
    """All rows of Eq. (7a).  pos, force: [N, 3] -> vel [N, 3] (fp64).  box > 0: periodic cube
    of that side, nearest image only."""
    pos, force = _as3(pos, "pos"), _as3(force, "force")
    if pos.shape != force.shape:
        raise ValueError("pos and force must have the same shape")
    vel = np.empty_like(pos)
    _check(_load().sdo_apply_box(_dp(pos), _dp(force), pos.shape[0], a, eta, tensor, float(box),
                                 int(image), _dp(vel)), "sdo_apply_box")
    return vel


def apply_rows(pos, force, rows, a: float, eta: float, tensor: int = TENSOR_RPY,
               box: float = 0.0, image: int = IMAGE_DEFINITION) -> np.ndarray:
    """Rows `rows` of Eq. (7a): returns [len(rows), 3]."""
    pos, force = _as3(pos, "pos"), _as3(force, "force")
    if pos.shape != force.shape:
        raise ValueError("pos and force must have the same shape")
    rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    out = np.empty((rows.shape[0], 3), dtype=np.float64)
    rc = _load().sdo_apply_rows_box(_dp(pos), _dp(force), pos.shape[0], a, eta, tensor,
                                    float(box), int(image),
                                    rows.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)),
                                    rows.shape[0], _dp(out))
    _check(rc, "sdo_apply_rows_box")
    return out


def assemble(pos, a: float, eta: float, tensor: int = TENSOR_RPY, box: float = 0.0,
             image: int = IMAGE_DEFINITION) -> np.ndarray:
    """Dense 3N x 3N mobility matrix (small N only)."""
    pos = _as3(pos, "pos")
    n = pos.shape[0]
    M = np.empty((3 * n, 3 * n), dtype=np.float64)
    _check(_load().sdo_assemble_box(_dp(pos), n, a, eta, tensor, float(box), int(image), _dp(M)),
           "sdo_assemble_box")
    return M


def step(pos, force, a: float, eta: float, dt: float, n_steps: int, integrator: int,
         tensor: int = TENSOR_RPY, rec_stride: int = 0, box: float = 0.0,
         image: int = IMAGE_DEFINITION):
    """Integrate n_steps with constant forces.  Returns (pos_final, vel_last, traj|None);
    traj[k] = positions after (k+1)*rec_stride steps when rec_stride > 0."""
    pos = _as3(pos, "pos").copy()
    force = _as3(force, "force")
    n = pos.shape[0]
    traj = None
    tp = None
    if rec_stride > 0:
        traj = np.empty((n_steps // rec_stride, n, 3), dtype=np.float64)
        tp = _dp(traj)
    vel = np.zeros_like(pos)
    rc = _load().sdo_step_box(_dp(pos), _dp(force), n, a, eta, tensor, float(box), int(image),
                              dt, n_steps, integrator, tp, max(rec_stride, 1), _dp(vel))
    _check(rc, "sdo_step_box")
    return pos, vel, traj


LUB_SMIN = 1.0e-3  # lower clamp of the surface separation s (reading C2)


def lubrication(pos, vel, a: float, eta: float, box: float = 0.0, image: int = IMAGE_DEFINITION,
                decide_f32: bool = False) -> np.ndarray:
    """C_i = sum'_j f_sing(r_ij).(v_i - v_j), Eq. (8) truncated at r = 3a."""
    pos, vel = _as3(pos, "pos"), _as3(vel, "vel")
    if pos.shape != vel.shape:
        raise ValueError("pos and vel must have the same shape")
    out = np.empty_like(pos)
    _check(_load().sdo_lubrication(_dp(pos), _dp(vel), pos.shape[0], a, eta, float(box), int(image),
                                   1 if decide_f32 else 0, _dp(out)), "sdo_lubrication")
    return out


def step_lub(pos, vel, fext, a: float, eta: float, dt: float, n_steps: int, integrator: int,
             tensor: int = TENSOR_RPY, box: float = 0.0, image: int = IMAGE_DEFINITION,
             decide_f32: bool = False):
    """The paper's loop with lubrication-corrected forces.  Returns (pos_final, vel_last)."""
    pos, vel, fext = _as3(pos, "pos").copy(), _as3(vel, "vel").copy(), _as3(fext, "fext")
    rc = _load().sdo_step_lub(_dp(pos), _dp(vel), _dp(fext), pos.shape[0], a, eta, tensor,
                              float(box), int(image), 1 if decide_f32 else 0, dt, n_steps, integrator)
    _check(rc, "sdo_step_lub")
    return pos, vel


def num_threads() -> int:
    return int(_load().sdo_num_threads())


def set_num_threads(n: int) -> None:
    _load().sdo_set_num_threads(int(n))


# ---- Appendix A access kernels (Algorithms 3 and 4) ---------------------------
ACC_LINEAR, ACC_STRIDED, ACC_UNORDERED = 0, 1, 2
ACC_NAIVE, ACC_SMALL_TILING, ACC_TILING, ACC_BULK = 0, 1, 2, 3
_ACC_P, _ACC_M, _ACC_BLOCK = 131, 32, 128


def _acc_map(k, j, n, pattern):
    """The three mappings of PAPER.md:295: k -> k, k -> k p mod N, k -> (k p + j M) mod N."""
    k = np.asarray(k, dtype=np.int64)
    if pattern == ACC_LINEAR:
        return k + 0 * np.asarray(j, dtype=np.int64)
    if pattern == ACC_STRIDED:
        return (k * _ACC_P) % n + 0 * np.asarray(j, dtype=np.int64)
    return (k * _ACC_P + np.asarray(j, dtype=np.int64) * _ACC_M) % n


def access_sums(data, pattern: int, scheme: int) -> np.ndarray:
    """What thread j of the Appendix-A kernels stores: its own element plus the N elements it
    visits, an element counting as the sum of its floats.  data: [N] or [N, 4].  Naive (Alg. 3):
    the elements map(k, j).  Tiled schemes (Alg. 4; W = 32 small-tiling, 128 tiling; blocks of
    128 threads): tile m holds, at place n, the element map(m + n, j_n) with j_n the global id of
    the thread of the SAME block that copied it, and every thread of the block sums the whole
    tile.  Bulk copies: linear pattern, same sums as naive.  Plain numpy, fp64 sums."""
    data = np.asarray(data, dtype=np.float64)
    val = data.sum(axis=1) if data.ndim == 2 else data
    n = val.shape[0]
    j = np.arange(n, dtype=np.int64)
    out = val.copy()
    if scheme in (ACC_NAIVE, ACC_BULK):
        if scheme == ACC_BULK and pattern != ACC_LINEAR:
            raise ValueError("bulk copies exist for the linear pattern only")
        for k in range(n):
            out += val[_acc_map(k, j, n, pattern)]
        return out
    w = 32 if scheme == ACC_SMALL_TILING else 128
    for b0 in range(0, n, _ACC_BLOCK):            # one block of 128 threads
        tile_sum = 0.0
        for m in range(0, n, w):
            nn = np.arange(min(w, n - m), dtype=np.int64)
            tile_sum += val[_acc_map(m + nn, b0 + nn, n, pattern)].sum()
        out[b0:b0 + _ACC_BLOCK] += tile_sum
    return out
