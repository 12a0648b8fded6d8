"""Thin Python binding of libdebye's C ABI (include/debye.h): argument marshalling only.

Every step of the path (type sort, pair kernel, FP64 reduction, epilogue) runs in the CUDA library; torch is
used for device memory and streams.  There is NO CPU fallback: if libdebye.so is missing or cannot be loaded
the first call raises LibdebyeError."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# LIBDEBYE_PATH: load another build of the same library (e.g. one compiled with different tuning macros)
LIB_PATH = os.environ.get("LIBDEBYE_PATH") or os.path.join(HERE, "libdebye.so")

FLAGS = {"fp64": 1 << 0, "mufu": 1 << 2, "recur": 1 << 3, "accurate": 1 << 4, "centred": 1 << 5, "auto": 0}
QHINT_PIECES = 1 << 12

EXPORTS = ("debye_profile", "debye_profile_batch", "debye_profile_host", "debye_profile_batch_host",
           "debye_profile_weighted", "debye_profile_batch_weighted", "debye_profile_weighted_host", "debye_partials",
           "debye_partials_shard", "debye_profile_from_partials", "debye_profile_peratom", "debye_profile_peratom_host", "debye_workspace_bytes", "debye_set_workspace", "debye_shutdown",
           "debye_launch_info", "debye_set_pairs_events", "debye_q_hint", "debye_plan_create", "debye_plan_execute",
           "debye_plan_destroy", "debye_strerror", "debye_last_cuda_error", "debye_version", "debye_pipe_bench_count",
           "debye_pipe_bench_name", "debye_pipe_bench", "debye_mufu_sin_error", "debye_mufu_rsq_error",
           "debye_profile_static", "debye_profile_static_error", "debye_profile_static_limits", "debye_q_hint_pieces", "debye_profile_peratom_batch")


# status codes of include/debye.h (debye_status)
DEBYE_OK, DEBYE_EINVAL, DEBYE_EUNSUPPORTED, DEBYE_ENOMEM, DEBYE_ECUDA = 0, 1, 2, 3, 4


class LibdebyeError(RuntimeError):
    """code: the library's status (DEBYE_E*), or None for an error raised by the binding's own argument checks."""
    code = None


_lib = None


def lib():
    """Load libdebye.so (built by `python -m paper_1306_2258_b200.build`); raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LibdebyeError(f"{LIB_PATH} not found: build it with `python -m paper_1306_2258_b200.build` "
                            "(there is no CPU fallback)")
    try:
        L = C.CDLL(LIB_PATH)
    except OSError as e:  # pragma: no cover
        raise LibdebyeError(f"cannot load {LIB_PATH}: {e}") from e
    vp, i32, u32, sz = C.c_void_p, C.c_int32, C.c_uint32, C.c_size_t
    L.debye_profile.argtypes = [vp, vp, i32, vp, i32, vp, i32, vp, u32, vp]
    L.debye_profile_host.argtypes = L.debye_profile.argtypes
    L.debye_profile_batch.argtypes = [vp, vp, i32, i32, vp, i32, vp, i32, vp, u32, vp]
    L.debye_profile_batch_host.argtypes = L.debye_profile_batch.argtypes
    L.debye_partials.argtypes = [vp, vp, i32, i32, vp, i32, i32, vp, vp, u32, vp]
    L.debye_partials_shard.argtypes = [vp, vp, i32, i32, vp, i32, i32, vp, vp, u32, i32, i32, vp]
    L.debye_profile_from_partials.argtypes = [vp, i32, vp, vp, i32, i32, i32, vp, vp]
    L.debye_profile_peratom.argtypes = [vp, vp, i32, vp, i32, vp, u32, vp]
    L.debye_profile_peratom.restype = C.c_int
    L.debye_profile_peratom_host.argtypes = L.debye_profile_peratom.argtypes
    L.debye_profile_peratom_batch.argtypes = [vp, vp, i32, i32, vp, i32, vp, u32, vp]
    L.debye_profile_peratom_batch.restype = C.c_int
    L.debye_profile_peratom_host.restype = C.c_int
    L.debye_profile_weighted.argtypes = [vp, vp, vp, i32, vp, i32, vp, i32, vp, u32, vp]
    L.debye_profile_weighted_host.argtypes = L.debye_profile_weighted.argtypes
    L.debye_profile_batch_weighted.argtypes = [vp, vp, vp, i32, i32, vp, i32, vp, i32, vp, u32, vp]
    for n in ("debye_profile", "debye_profile_host", "debye_profile_batch", "debye_profile_batch_host",
              "debye_profile_weighted", "debye_profile_batch_weighted", "debye_profile_weighted_host", "debye_partials",
              "debye_partials_shard", "debye_profile_from_partials"):
        getattr(L, n).restype = C.c_int
    L.debye_workspace_bytes.argtypes = [i32, i32, i32, i32, u32]
    L.debye_workspace_bytes.restype = sz
    L.debye_set_workspace.argtypes = [vp, sz]
    L.debye_set_workspace.restype = C.c_int
    L.debye_shutdown.argtypes = []
    L.debye_shutdown.restype = None
    L.debye_launch_info.argtypes = [i32, i32, i32, i32, u32] + [C.POINTER(i32)] * 4
    L.debye_launch_info.restype = C.c_int
    L.debye_set_pairs_events.argtypes = [vp, vp]
    L.debye_set_pairs_events.restype = C.c_int
    L.debye_plan_create.argtypes = [C.POINTER(vp), vp, i32, i32, i32, vp, i32, vp, u32, vp]
    L.debye_plan_create.restype = C.c_int
    L.debye_plan_execute.argtypes = [vp, vp, vp, vp, vp]
    L.debye_plan_execute.restype = C.c_int
    L.debye_plan_destroy.argtypes = [vp]
    L.debye_plan_destroy.restype = None
    L.debye_q_hint.argtypes = [vp, i32]
    L.debye_q_hint.restype = u32
    L.debye_q_hint_pieces.argtypes = [vp, i32]
    L.debye_q_hint_pieces.restype = u32
    L.debye_strerror.argtypes = [C.c_int]
    L.debye_strerror.restype = C.c_char_p
    L.debye_last_cuda_error.restype = C.c_int
    L.debye_version.restype = C.c_int
    L.debye_pipe_bench_count.restype = C.c_int
    L.debye_pipe_bench_name.argtypes = [C.c_int]
    L.debye_pipe_bench_name.restype = C.c_char_p
    L.debye_pipe_bench.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
    L.debye_pipe_bench.restype = C.c_int
    L.debye_mufu_sin_error.argtypes = [C.c_int] + [C.POINTER(C.c_double)] * 3 + [vp]
    L.debye_mufu_sin_error.restype = C.c_int
    L.debye_mufu_rsq_error.argtypes = L.debye_mufu_sin_error.argtypes
    L.debye_mufu_rsq_error.restype = C.c_int
    L.debye_profile_static.argtypes = L.debye_profile.argtypes
    L.debye_profile_static.restype = C.c_int
    L.debye_profile_static_error.argtypes = []
    L.debye_profile_static_error.restype = C.c_char_p
    L.debye_profile_static_limits.argtypes = [C.POINTER(i32)] * 3 + [C.POINTER(sz)]
    L.debye_profile_static_limits.restype = None
    _lib = L
    return L


def _check(st: int):
    if st != 0:
        L = lib()
        e = LibdebyeError(f"libdebye status {st}: {L.debye_strerror(st).decode()} "
                          f"(cuda error {L.debye_last_cuda_error()})")
        e.code = int(st)
        raise e


def _flags(variant, hint: int = 0) -> int:
    return (variant if isinstance(variant, int) else FLAGS[variant]) | int(hint)


def q_hint(q_host) -> int:
    """Grid hint flags (DEBYE_QHINT_*) for a HOST copy of the q grid (numpy float32): pass as `hint=` to the profile calls
    so that only the pairs instantiation this grid needs is launched.  A wrong hint gives NaN, never a wrong number."""
    q_host = np.ascontiguousarray(q_host, dtype=np.float32)
    return int(lib().debye_q_hint(C.c_void_p(q_host.ctypes.data), q_host.shape[0]))


def q_hint_pieces(q_host) -> int:
    """The piecewise-uniform hint (centred product form) for ANY grid made of at most 32 uniform pieces, 0 if q is not one;
    q_hint() returns it by itself for grids that are not uniform as a whole.  (pieces, K) = pieces_of(hint)."""
    q_host = np.ascontiguousarray(q_host, dtype=np.float32)
    return int(lib().debye_q_hint_pieces(C.c_void_p(q_host.ctypes.data), q_host.shape[0]))


def pieces_of(hint: int):
    """(number of uniform pieces, accumulators per thread) a piecewise-uniform hint carries; (0, 0) for any other hint."""
    if not hint & QHINT_PIECES:
        return 0, 0
    return ((hint >> 16) & 31) + 1, 8 * (((hint >> 21) & 31) + 1)


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev(t, dtype, name, shape=None):
    """Device pointer of a contiguous CUDA tensor of the given dtype on the CURRENT device (the library keys its scratch on
    cudaGetDevice); shape: expected shape, None entries are free."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise LibdebyeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    if t.device.index != torch.cuda.current_device():
        raise LibdebyeError(f"{name}: tensor on cuda:{t.device.index}, current device is cuda:{torch.cuda.current_device()}")
    if shape is not None and (t.dim() != len(shape) or any(e is not None and int(d) != int(e) for d, e in zip(t.shape, shape))):
        raise LibdebyeError(f"{name}: shape {tuple(t.shape)}, expected {tuple('*' if e is None else e for e in shape)}")
    return C.c_void_p(t.data_ptr())


def debye_profile(xyz, type, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    """I_out[M] (float64, CUDA) for xyz[N,3] f32, type[N] i32, fftab[T,M] f32, q[M] f32 (CUDA tensors).
    Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    N, T, M = xyz.shape[0], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = torch.empty(M, dtype=torch.float64, device=xyz.device)
    _check(lib().debye_profile(_dev(xyz, torch.float32, "xyz", (N, 3)), _dev(type, torch.int32, "type", (N,)), N,
                               _dev(fftab, torch.float32, "fftab", (T, M)), T, _dev(q, torch.float32, "q", (M,)), M,
                               _dev(I_out, torch.float64, "I_out", (M,)), _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def static_limits():
    """(max atoms, max types, max non-zero q values, bytes of the static scratch) of debye_profile_static."""
    a, t, m, b = C.c_int32(), C.c_int32(), C.c_int32(), C.c_size_t()
    lib().debye_profile_static_limits(C.byref(a), C.byref(t), C.byref(m), C.byref(b))
    return a.value, t.value, m.value, b.value


def debye_profile_static(xyz, type, fftab, q, I_out, hint, stream=None):
    """debye_profile for one small structure with NO allocation anywhere (include/debye.h debye_profile_static): the scratch
    is a fixed __device__ array of the library.  I_out is the caller's (this wrapper does not allocate it either); `hint` must
    be q_hint() of a uniform grid starting at 0 or dq.  Beyond static_limits() the library refuses (DEBYE_EUNSUPPORTED) and
    the error names the limit.  Calls that overlap on the GPU (different streams, no event between them) race."""
    import torch
    N, T, M = xyz.shape[0], fftab.shape[0], q.shape[0]
    L = lib()
    st = L.debye_profile_static(_dev(xyz, torch.float32, "xyz", (N, 3)), _dev(type, torch.int32, "type", (N,)), N,
                                _dev(fftab, torch.float32, "fftab", (T, M)), T, _dev(q, torch.float32, "q", (M,)), M,
                                _dev(I_out, torch.float64, "I_out", (M,)), int(hint), _stream_ptr(stream))
    if st != 0:
        e = LibdebyeError(f"libdebye status {st}: {L.debye_profile_static_error().decode() or L.debye_strerror(st).decode()}")
        e.code = int(st)
        raise e
    return I_out


def debye_profile_batch(xyz, type, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    """I_out[B,M] for B conformers xyz[B,N,3] sharing type / fftab / q."""
    import torch
    B, N, T, M = xyz.shape[0], xyz.shape[1], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = torch.empty((B, M), dtype=torch.float64, device=xyz.device)
    _check(lib().debye_profile_batch(_dev(xyz, torch.float32, "xyz", (B, N, 3)), _dev(type, torch.int32, "type", (N,)), N, B,
                                     _dev(fftab, torch.float32, "fftab", (T, M)), T, _dev(q, torch.float32, "q", (M,)), M,
                                     _dev(I_out, torch.float64, "I_out", (B, M)), _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def debye_profile_weighted(xyz, type, weight, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    """As debye_profile with per-atom weights: f_j(q) = weight[j] * fftab[type[j]] (weight[N] f32 CUDA tensor).
    xyz[N,3] gives I_out[M]; xyz[B,N,3] gives I_out[B,M] (weights shared by the conformers)."""
    import torch
    batch = xyz.dim() == 3
    N, T, M = xyz.shape[-2], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = torch.empty((xyz.shape[0], M) if batch else M, dtype=torch.float64, device=xyz.device)
    a = (_dev(xyz, torch.float32, "xyz", (xyz.shape[0], N, 3) if batch else (N, 3)), _dev(type, torch.int32, "type", (N,)),
         _dev(weight, torch.float32, "weight", (N,)), N)
    b = (_dev(fftab, torch.float32, "fftab", (T, M)), T, _dev(q, torch.float32, "q", (M,)), M,
         _dev(I_out, torch.float64, "I_out", (xyz.shape[0], M) if batch else (M,)), _flags(variant, hint), _stream_ptr(stream))
    if batch:
        _check(lib().debye_profile_batch_weighted(*a, xyz.shape[0], *b))
    else:
        _check(lib().debye_profile_weighted(*a, *b))
    return I_out


def debye_profile_weighted_host(xyz, type, weight, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    N, T, M = xyz.shape[0], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = np.empty(M, dtype=np.float64)
    _check(lib().debye_profile_weighted_host(_host(xyz, np.float32, "xyz"), _host(type, np.int32, "type"),
                                             _host(weight, np.float32, "weight"), N, _host(fftab, np.float32, "fftab"), T,
                                             _host(q, np.float32, "q"), M, _host(I_out, np.float64, "I_out"),
                                             _flags(variant, hint), _stream_ptr(stream)))
    return I_out


class Plan:
    """debye_plan_*: setup once for one molecule (type, q, optional weights, batch size), then execute(xyz, fftab) per
    set of coordinates.  Creation synchronises the stream once; execute never does."""

    def __init__(self, type, q, T, B=1, weight=None, variant="auto", stream=None):
        import torch
        self.N, self.M, self.T, self.B = type.shape[0], q.shape[0], T, B
        self._h = C.c_void_p()
        _check(lib().debye_plan_create(C.byref(self._h), _dev(type, torch.int32, "type", (self.N,)), self.N, B, T,
                                       _dev(q, torch.float32, "q", (self.M,)), self.M,
                                       _dev(weight, torch.float32, "weight", (self.N,)) if weight is not None else None,
                                       _flags(variant), _stream_ptr(stream)))

    def execute(self, xyz, fftab, I_out=None, stream=None):
        import torch
        batch = xyz.dim() == 3
        if (batch and xyz.shape[0] != self.B) or (not batch and self.B != 1):
            raise LibdebyeError(f"xyz: the plan was created for B = {self.B} conformers")
        if I_out is None:
            I_out = torch.empty((self.B, self.M) if batch else self.M, dtype=torch.float64, device=xyz.device)
        _check(lib().debye_plan_execute(self._h, _dev(xyz, torch.float32, "xyz", (self.B, self.N, 3) if batch else (self.N, 3)),
                                        _dev(fftab, torch.float32, "fftab", (self.T, self.M)),
                                        _dev(I_out, torch.float64, "I_out", (self.B, self.M) if batch else (self.M,)), _stream_ptr(stream)))
        return I_out

    def destroy(self):
        if self._h:
            lib().debye_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def debye_partials(xyz, type, q, T, variant="auto", stream=None, hint=0):
    """(S[B,T(T+1)/2,M] float64, n[T] int32): per-type-pair sums of sinc(q r) over pairs i<j, atoms per type."""
    import torch
    x3 = xyz if xyz.dim() == 3 else xyz[None]
    B, N, M = x3.shape[0], x3.shape[1], q.shape[0]
    S = torch.empty((B, T * (T + 1) // 2, M), dtype=torch.float64, device=xyz.device)
    n = torch.empty(T, dtype=torch.int32, device=xyz.device)
    _check(lib().debye_partials(_dev(x3, torch.float32, "xyz", (B, N, 3)), _dev(type, torch.int32, "type", (N,)), N, B,
                                _dev(q, torch.float32, "q", (M,)), T, M, _dev(S, torch.float64, "S_out"),
                                _dev(n, torch.int32, "n_out"), _flags(variant, hint), _stream_ptr(stream)))
    return S, n


def debye_profile_peratom(xyz, ff, q, I_out=None, variant="auto", stream=None, hint=0):
    """I_out[M] for per-ATOM form factors ff[N,M] f32 (the paper's general case).  variant: "auto" (with a
    grid hint that promises q_k = (k + koff) dq, koff in {0, 1}, and at most 256 chain indices: the recurrence, 2 FP32 lane-ops per
    term; otherwise one MUFU.SIN per term), "mufu", "recur" or "fp64".  hint: q_hint(q_host)."""
    import torch
    N, M = xyz.shape[0], q.shape[0]
    if tuple(ff.shape) != (N, M):
        raise LibdebyeError("ff: expected shape [N, M]")
    if I_out is None:
        I_out = torch.empty(M, dtype=torch.float64, device=xyz.device)
    _check(lib().debye_profile_peratom(_dev(xyz, torch.float32, "xyz", (N, 3)), _dev(ff, torch.float32, "ff", (N, M)), N,
                                       _dev(q, torch.float32, "q", (M,)), M, _dev(I_out, torch.float64, "I_out", (M,)),
                                       _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def debye_profile_peratom_batch(xyz, ff, q, I_out=None, variant="auto", stream=None, hint=0):
    """I_out[B,M] for B conformers xyz[B,N,3] sharing the per-atom table ff[N,M]; with the hint of a grid q_k = (k + koff) dq all
    conformers run in one launch sequence."""
    import torch
    B, N, M = xyz.shape[0], xyz.shape[1], q.shape[0]
    if I_out is None:
        I_out = torch.empty((B, M), dtype=torch.float64, device=xyz.device)
    _check(lib().debye_profile_peratom_batch(_dev(xyz, torch.float32, "xyz", (B, N, 3)), _dev(ff, torch.float32, "ff", (N, M)), N, B,
                                             _dev(q, torch.float32, "q", (M,)), M, _dev(I_out, torch.float64, "I_out", (B, M)),
                                             _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def debye_partials_shard(xyz, type, q, T, shard_rank, shard_world, variant="auto", stream=None, hint=0):
    """This rank's part of debye_partials when ONE structure is split over `shard_world` GPUs by tiles (pairs CTA c works
    iff c % shard_world == shard_rank): (S_part[B,T(T+1)/2,M] float64, n[T] int32).  The parts of all ranks sum to S."""
    import torch
    x3 = xyz if xyz.dim() == 3 else xyz[None]
    B, N, M = x3.shape[0], x3.shape[1], q.shape[0]
    S = torch.empty((B, T * (T + 1) // 2, M), dtype=torch.float64, device=xyz.device)
    n = torch.empty(T, dtype=torch.int32, device=xyz.device)
    _check(lib().debye_partials_shard(_dev(x3, torch.float32, "xyz", (B, N, 3)), _dev(type, torch.int32, "type", (N,)), N, B,
                                      _dev(q, torch.float32, "q", (M,)), T, M, _dev(S, torch.float64, "S_out"),
                                      _dev(n, torch.int32, "n_out"), _flags(variant, hint), int(shard_rank), int(shard_world),
                                      _stream_ptr(stream)))
    return S, n


def debye_profile_from_partials(S_parts, n, fftab, I_out=None, stream=None):
    """I_out[B,M] from gathered parts S_parts[n_parts,B,T(T+1)/2,M] (summed in part order on the device), n[T], fftab[T,M]."""
    import torch
    n_parts, B, n_tp, M = S_parts.shape
    T = fftab.shape[0]
    if n_tp != T * (T + 1) // 2 or fftab.shape[1] != M or n.shape[0] != T:
        raise LibdebyeError("S_parts / n / fftab shapes do not agree")
    if I_out is None:
        I_out = torch.empty((B, M), dtype=torch.float64, device=S_parts.device)
    _check(lib().debye_profile_from_partials(_dev(S_parts, torch.float64, "S_parts"), n_parts, _dev(n, torch.int32, "n"),
                                             _dev(fftab, torch.float32, "fftab"), B, T, M,
                                             _dev(I_out, torch.float64, "I_out"), _stream_ptr(stream)))
    return I_out


def _host(a, dtype, name):
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous):
        raise LibdebyeError(f"{name}: expected a C-contiguous numpy array of dtype {dtype}")
    return C.c_void_p(a.ctypes.data)


def debye_profile_host(xyz, type, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    """Host-buffer entry (numpy arrays, ideally pinned): H2D copies + device path + D2H copy + stream sync
    all happen inside the C call."""
    N, T, M = xyz.shape[0], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = np.empty(M, dtype=np.float64)
    _check(lib().debye_profile_host(_host(xyz, np.float32, "xyz"), _host(type, np.int32, "type"), N,
                                    _host(fftab, np.float32, "fftab"), T, _host(q, np.float32, "q"), M,
                                    _host(I_out, np.float64, "I_out"), _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def debye_profile_batch_host(xyz, type, fftab, q, I_out=None, variant="auto", stream=None, hint=0):
    B, N, T, M = xyz.shape[0], xyz.shape[1], fftab.shape[0], q.shape[0]
    if I_out is None:
        I_out = np.empty((B, M), dtype=np.float64)
    _check(lib().debye_profile_batch_host(_host(xyz, np.float32, "xyz"), _host(type, np.int32, "type"), N, B,
                                          _host(fftab, np.float32, "fftab"), T, _host(q, np.float32, "q"), M,
                                          _host(I_out, np.float64, "I_out"), _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def debye_profile_peratom_host(xyz, ff, q, I_out=None, variant="auto", stream=None, hint=0):
    N, M = xyz.shape[0], q.shape[0]
    if I_out is None:
        I_out = np.empty(M, dtype=np.float64)
    _check(lib().debye_profile_peratom_host(_host(xyz, np.float32, "xyz"), _host(ff, np.float32, "ff"), N,
                                            _host(q, np.float32, "q"), M, _host(I_out, np.float64, "I_out"),
                                            _flags(variant, hint), _stream_ptr(stream)))
    return I_out


def set_pairs_events(start=None, stop=None):
    """Record torch.cuda.Event `start` / `stop` (created with enable_timing=True and already recorded once, so the
    handles exist) around the pairs kernel of every following call; None, None switches the hook off."""
    a = C.c_void_p(start.cuda_event) if start is not None else None
    b = C.c_void_p(stop.cuda_event) if stop is not None else None
    _check(lib().debye_set_pairs_events(a, b))


def launch_info(N, B, T, M, variant="auto", with_grid=False, hint=0):
    """dict(n_launches, q_chunk, n_chunks[, pairs_grid]) for a call with these sizes (host-side query)."""
    L = lib()
    a, g, k, c = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
    _check(L.debye_launch_info(N, B, T, M, _flags(variant, hint), C.byref(a), C.byref(g) if with_grid else None,
                               C.byref(k), C.byref(c)))
    out = {"n_launches": a.value, "q_chunk": k.value, "n_chunks": c.value}
    if with_grid:
        out["pairs_grid"] = g.value
    return out


def pipe_bench(test: int, ctas_per_sm: int, iters: int = 2000, stream=None):
    """(name, FP32-pipe lane-operations per clock and SM, scheduler cycles per warp instruction) of one micro-kernel
    (include/debye.h, debye_pipe_bench); None if ctas_per_sm CTAs of that test do not fit on an SM."""
    L = lib()
    rate, cpi = C.c_double(), C.c_double()
    st = L.debye_pipe_bench(test, ctas_per_sm, iters, C.byref(rate), C.byref(cpi), _stream_ptr(stream))
    if st == 2:
        return None
    _check(st)
    return L.debye_pipe_bench_name(test).decode(), rate.value, cpi.value


def mufu_sin_error(n: int = 1 << 24, stream=None):
    """max |e|, rms, mean of MUFU.SIN against double sin on n points of (0, 1/2] turns (debye_mufu_sin_error)."""
    mx, rms, mean = C.c_double(), C.c_double(), C.c_double()
    _check(lib().debye_mufu_sin_error(n, C.byref(mx), C.byref(rms), C.byref(mean), _stream_ptr(stream)))
    return mx.value, rms.value, mean.value


def mufu_rsq_error(n: int = 1 << 24, stream=None):
    """max, rms, mean RELATIVE error of MUFU.RSQ on n log-uniform points of [1, 4) (debye_mufu_rsq_error)."""
    mx, rms, mean = C.c_double(), C.c_double(), C.c_double()
    _check(lib().debye_mufu_rsq_error(n, C.byref(mx), C.byref(rms), C.byref(mean), _stream_ptr(stream)))
    return mx.value, rms.value, mean.value
