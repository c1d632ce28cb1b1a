"""Thin ctypes binding of libsd_b200.so (include/sd_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; there is no CPU fallback and
the module raises if the library is missing.  PyTorch is used for device memory and streams.

    ctx = sd.Context(N, a, eta)                       # sd_create
    ctx.set_tensor(sd.TENSOR_RPY); ctx.set_precision(sd.PREC_F32_KAHAN)
    ctx.mobility_apply(pos, force, vel)               # sd_mobility_apply   (Eq. 7a)
    ctx.step(pos, dt, n_steps, sd.INT_MIDPOINT, gravity=(0, 0, -1))   # sd_step

pos / force / vel are torch CUDA tensors of shape [N, 4] (xyz + pad lane), float32 for the F32
modes and float64 for PREC_F64.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsd_b200.so")

OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_CUDA, ERR_UNSUPPORTED = 0, 1, 2, 3, 4
TENSOR_RPY, TENSOR_OSEEN = 0, 1
PREC_F32_KAHAN, PREC_F64, PREC_F32_PLAIN = 0, 1, 2
INT_EULER, INT_MIDPOINT = 0, 1
STAGE_BULK, STAGE_NAIVE, STAGE_SYNC = 0, 1, 2

FORCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                            ctypes.c_void_p, ctypes.c_void_p)

# name -> (restype, argtypes); also the list the CPU test checks against include/sd_b200.h
_P, _LL, _D, _I = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_double, ctypes.c_int
SYMBOLS = {
    "sd_create": (_I, [ctypes.POINTER(_P), _LL, _D, _D]),
    "sd_set_tensor": (_I, [_P, _I]),
    "sd_set_precision": (_I, [_P, _I]),
    "sd_schedule_plan": (_I, [_LL, _I, _I, _LL, _I, ctypes.POINTER(_LL), ctypes.POINTER(_I),
                               ctypes.POINTER(_I), ctypes.POINTER(_I), ctypes.POINTER(_I)]),
    "sd_set_dispatch": (_I, [_P, _LL, _I]),
    "sd_set_staging": (_I, [_P, _I]),
    "sd_set_jsplit": (_I, [_P, _I]),
    "sd_set_box": (_I, [_P, _D]),
    "sd_box": (_D, [_P]),
    "sd_mobility_apply": (_I, [_P, _P, _P, _P, _P]),
    "sd_mobility_apply_host": (_I, [_P, _P, _P, _P, _P]),
    "sd_mobility_apply_noalloc": (_I, [_LL, _D, _D, _I, _P, _P, _P, _P]),
    "sd_noalloc_max_particles": (_LL, []),
    "sd_step": (_I, [_P, _P, FORCE_FN, _P, _P, ctypes.POINTER(_D), _D, _LL, _I, _P]),
    "sd_get_velocity": (_I, [_P, _P, _P]),
    "sd_lubrication_apply": (_I, [_P, _P, _P, _P, ctypes.POINTER(_D), _P, _P]),
    "sd_set_lubrication": (_I, [_P, _I]),
    "sd_set_velocity": (_I, [_P, _P, _P]),
    "sd_reset_compensation": (_I, [_P, _P]),
    "sd_set_position_compensation": (_I, [_P, _I]),
    "sd_num_particles": (_LL, [_P]),
    "sd_self_mobility": (_D, [_P]),
    "sd_launch_count": (_LL, [_P]),
    "sd_kernel_name": (ctypes.c_char_p, [_P]),
    "sd_profile_enable": (_I, [_P, _I]),
    "sd_profile_read": (_I, [_P, ctypes.POINTER(_D), ctypes.POINTER(_LL)]),
    "sd_fma_peak_probe": (_I, [_P, _I, ctypes.POINTER(_D), _P]),
    "sd_access_bench": (_I, [_I, _I, _I, _LL, _I, _P, _P, ctypes.POINTER(_D), _P]),
    "sd_last_error": (ctypes.c_char_p, [_P]),
    "sd_destroy": (None, [_P]),
}

_lib = None


class SdError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"sd_b200 status {status}: {message}")
        self.status = status


def load_library() -> ctypes.CDLL:
    """Open libsd_b200.so and declare every symbol of include/sd_b200.h.  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; "
                          "g.build()'` (there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def noalloc_max_particles() -> int:
    return int(load_library().sd_noalloc_max_particles())


def mobility_apply_noalloc(pos, force, vel, a: float, eta: float, tensor: int = TENSOR_RPY, stream=None):
    """sd_mobility_apply_noalloc: v = M(pos) F in fp32 without a context and without any device
    allocation (static 4-MiB scratch array inside the library; N <= noalloc_max_particles();
    calls that overlap on the GPU race on that array).  pos, force, vel: contiguous CUDA float32
    tensors [N, 4] on the current device."""
    import torch
    lib = load_library()
    n = int(pos.shape[0])
    for t, name in ((pos, "pos"), (force, "force"), (vel, "vel")):
        if not t.is_cuda or t.dtype != torch.float32 or tuple(t.shape) != (n, 4) or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous CUDA float32 tensor [{n}, 4], got "
                             f"{tuple(t.shape)} {t.dtype} {t.device}")
    status = lib.sd_mobility_apply_noalloc(n, float(a), float(eta), int(tensor), ctypes.c_void_p(pos.data_ptr()),
                                           ctypes.c_void_p(force.data_ptr()), ctypes.c_void_p(vel.data_ptr()),
                                           _stream_ptr(stream))
    if status != 0:
        raise SdError(status, (lib.sd_last_error(None) or b"").decode())
    return vel


def schedule_plan(n: int, particles_per_block: int, tile_j: int, max_ctas: int, num_sms: int):
    """sd_schedule_plan: the static schedule of the tiled kernels (host only, no GPU).  Returns a
    dict with B, T, G, max_slots and the arrays cta_u0, cta_piece, blk_first, blk_nslots."""
    lib = load_library()
    dims = (ctypes.c_int * 4)()
    null_ll, null_i = ctypes.POINTER(_LL)(), ctypes.POINTER(_I)()
    st = lib.sd_schedule_plan(n, particles_per_block, tile_j, max_ctas, num_sms, null_ll, null_i,
                              null_i, null_i, dims)
    if st != OK:
        raise SdError(st, (lib.sd_last_error(None) or b"").decode())
    B, T, G, ms = (int(x) for x in dims)
    u0, piece = (ctypes.c_longlong * (G + 1))(), (ctypes.c_int * G)()
    first, nslots = (ctypes.c_int * B)(), (ctypes.c_int * B)()
    st = lib.sd_schedule_plan(n, particles_per_block, tile_j, max_ctas, num_sms, u0, piece, first,
                              nslots, dims)
    if st != OK:
        raise SdError(st, (lib.sd_last_error(None) or b"").decode())
    return {"B": B, "T": T, "G": G, "max_slots": ms, "cta_u0": list(u0), "cta_piece": list(piece),
            "blk_first": list(first), "blk_nslots": list(nslots)}


def access_bench(data, out, pattern: int, scheme: int, reps: int = 10, stream=None) -> float:
    """sd_access_bench (Appendix A).  data: CUDA float32 tensor [N] or [N, 4]; out: CUDA
    float32 tensor [N].  Returns the mean milliseconds per launch."""
    lib = load_library()
    elem = 4 if data.dim() == 2 else 1
    ms = ctypes.c_double(0.0)
    st = lib.sd_access_bench(elem, int(pattern), int(scheme), int(data.shape[0]), int(reps),
                             ctypes.c_void_p(data.data_ptr()), ctypes.c_void_p(out.data_ptr()),
                             ctypes.byref(ms), _stream_ptr(stream))
    if st != OK:
        raise SdError(st, (lib.sd_last_error(None) or b"").decode())
    return ms.value


class Context:
    """Owns one sd_ctx.  All methods only enqueue work on the (current or given) CUDA stream."""

    def __init__(self, n: int, a: float, eta: float):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        st = self._lib.sd_create(ctypes.byref(self._h), int(n), float(a), float(eta))
        if st != OK:
            raise SdError(st, (self._lib.sd_last_error(None) or b"").decode())
        self.n = int(n)
        self.precision = PREC_F32_KAHAN
        self._keep = None

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, st: int):
        if st != OK:
            raise SdError(st, (self._lib.sd_last_error(self._h) or b"").decode())

    def _dtype(self):
        import torch
        return torch.float64 if self.precision == PREC_F64 else torch.float32

    def _ptr(self, t, name, allow_none=False):
        if t is None and allow_none:
            return ctypes.c_void_p(0)
        if not t.is_cuda or t.dtype != self._dtype() or tuple(t.shape) != (self.n, 4) \
                or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous CUDA tensor [{self.n}, 4] of "
                             f"{self._dtype()}, got {tuple(t.shape)} {t.dtype} {t.device}")
        return ctypes.c_void_p(t.data_ptr())

    # -- C ABI -----------------------------------------------------------------------------
    def set_tensor(self, tensor: int):
        self._check(self._lib.sd_set_tensor(self._h, int(tensor)))

    def set_precision(self, precision: int):
        self._check(self._lib.sd_set_precision(self._h, int(precision)))
        self.precision = int(precision)

    def set_dispatch(self, small_apply_max: int = -1, particles_per_thread: int = 0):
        """Dispatch knobs of the small-N path (ablations / tests); defaults = measured crossovers."""
        self._check(self._lib.sd_set_dispatch(self._h, int(small_apply_max),
                                              int(particles_per_thread)))

    def set_jsplit(self, mode: int = 0):
        """0 automatic, 1 classic tiled kernels only, 2 warp-split one-launch kernel wherever it exists."""
        self._check(self._lib.sd_set_jsplit(self._h, int(mode)))

    def set_staging(self, mode: int):
        """Memory-access ablation (Appendix A): 0 bulk copies, 1 naive, 2 tiled + barriers."""
        self._check(self._lib.sd_set_staging(self._h, int(mode)))

    def set_box(self, box_side: float):
        """Periodic cube of that side, nearest image only; 0 = free space."""
        self._check(self._lib.sd_set_box(self._h, float(box_side)))

    @property
    def box(self) -> float:
        return float(self._lib.sd_box(self._h))

    def mobility_apply(self, pos, force, vel, stream=None):
        self._check(self._lib.sd_mobility_apply(self._h, self._ptr(pos, "pos"),
                                                self._ptr(force, "force"), self._ptr(vel, "vel"),
                                                _stream_ptr(stream)))

    def mobility_apply_host(self, pos, force, vel, stream=None):
        """pos/force/vel: CPU tensors [N, 4] (pinned for async copies); returns when vel landed."""
        for t, name in ((pos, "pos"), (force, "force"), (vel, "vel")):
            if t.is_cuda or t.dtype != self._dtype() or tuple(t.shape) != (self.n, 4) \
                    or not t.is_contiguous():
                raise ValueError(f"{name} must be a contiguous CPU tensor [{self.n}, 4]")
        self._check(self._lib.sd_mobility_apply_host(
            self._h, ctypes.c_void_p(pos.data_ptr()), ctypes.c_void_p(force.data_ptr()),
            ctypes.c_void_p(vel.data_ptr()), _stream_ptr(stream)))

    def step(self, pos, dt: float, n_steps: int, integrator: int, gravity=None, force=None,
             force_fn=None, user=None, stream=None):
        g = None
        if gravity is not None:
            g = (ctypes.c_double * 3)(*[float(x) for x in gravity])
        cb = FORCE_FN(force_fn) if force_fn is not None else ctypes.cast(None, FORCE_FN)
        self._keep = cb
        self._check(self._lib.sd_step(self._h, self._ptr(pos, "pos"), cb,
                                      ctypes.c_void_p(user or 0),
                                      self._ptr(force, "force", allow_none=True), g, float(dt),
                                      int(n_steps), int(integrator), _stream_ptr(stream)))

    def lubrication_apply(self, pos, vel, force_out, f_ext=None, gravity=None, stream=None):
        """force_out = F_ext - sum' f_sing.(v_i - v_j), Eq. (8) truncated at 3a."""
        g = (ctypes.c_double * 3)(*[float(x) for x in gravity]) if gravity is not None else None
        self._check(self._lib.sd_lubrication_apply(
            self._h, self._ptr(pos, "pos"), self._ptr(vel, "vel"),
            self._ptr(f_ext, "f_ext", allow_none=True), g, self._ptr(force_out, "force_out"),
            _stream_ptr(stream)))

    def set_lubrication(self, on: bool):
        self._check(self._lib.sd_set_lubrication(self._h, 1 if on else 0))

    def set_velocity(self, vel=None, stream=None):
        self._check(self._lib.sd_set_velocity(self._h, self._ptr(vel, "vel", allow_none=True),
                                              _stream_ptr(stream)))

    def get_velocity(self, vel, stream=None):
        self._check(self._lib.sd_get_velocity(self._h, self._ptr(vel, "vel"), _stream_ptr(stream)))

    def set_position_compensation(self, on: bool):
        """False: plain fp32 positions in sd_step (ablation of PAPER.md:253-263)."""
        self._check(self._lib.sd_set_position_compensation(self._h, 1 if on else 0))

    def reset_compensation(self, stream=None):
        self._check(self._lib.sd_reset_compensation(self._h, _stream_ptr(stream)))

    def fma_peak_probe(self, precision: int, stream=None) -> float:
        out = ctypes.c_double(0.0)
        self._check(self._lib.sd_fma_peak_probe(self._h, int(precision), ctypes.byref(out),
                                                _stream_ptr(stream)))
        return out.value

    def profile_enable(self, on: bool = True):
        self._check(self._lib.sd_profile_enable(self._h, 1 if on else 0))

    def profile_read(self):
        """(summed pair-kernel ms, launches) since the last read; waits for those launches."""
        ms, cnt = ctypes.c_double(0.0), ctypes.c_longlong(0)
        self._check(self._lib.sd_profile_read(self._h, ctypes.byref(ms), ctypes.byref(cnt)))
        return ms.value, cnt.value

    @property
    def self_mobility(self) -> float:
        return float(self._lib.sd_self_mobility(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._lib.sd_launch_count(self._h))

    @property
    def kernel_name(self) -> str:
        return (self._lib.sd_kernel_name(self._h) or b"").decode()

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.sd_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
