"""Thin Python binding of the C ABI in include/rosen.h (argument marshalling only).

Same names as the C entry points. PyTorch is used for device memory (output tensors) and for the
current CUDA stream; every step of the path runs inside librosen.so's kernels. There is no CPU
fallback: if the library is missing or no CUDA device is present the calls raise RosenError.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Iterable, Optional, Tuple

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librosen.so")

ROSEN_OK, ROSEN_EINVAL, ROSEN_ERANGE, ROSEN_ECUDA, ROSEN_ENOMEM = 0, -1, -2, -3, -4
ROSEN_MEM_DEVICE, ROSEN_MEM_HOST = 0, 1

PER_CHAIN = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")


class RosenError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"librosen error {code}: {message}")
        self.code = code


class rosen_summary(C.Structure):
    _fields_ = [
        ("n_chains", C.c_uint64), ("n_dead", C.c_uint64), ("n_steps_attempted", C.c_uint64),
        ("ln_shift", C.c_double),
        ("sum_w", C.c_double), ("sum_w_ree2", C.c_double), ("sum_w_rg2", C.c_double), ("sum_w2", C.c_double),
        ("mean_ree2", C.c_double), ("mean_rg2", C.c_double), ("attrition", C.c_double), ("ln_mean_W", C.c_double),
        ("digest_xor", C.c_uint64), ("digest_sum", C.c_uint64),
    ]

    def as_dict(self) -> Dict[str, float]:
        return {name: getattr(self, name) for name, _ in self._fields_}

    @classmethod
    def from_dict(cls, d: Dict[str, float]) -> "rosen_summary":
        return cls(**{name: d[name] for name, _ in cls._fields_})


class rosen_outputs(C.Structure):
    _fields_ = [
        ("lnW", C.c_void_p), ("alive", C.c_void_p), ("m_seq", C.c_void_p), ("digest", C.c_void_p),
        ("conf", C.c_void_p), ("ree2", C.c_void_p), ("rg2", C.c_void_p),
        ("memory", C.c_int32), ("reserved", C.c_int32),
    ]


_lib: Optional[C.CDLL] = None


def load_library() -> C.CDLL:
    """dlopen librosen.so and declare every symbol of include/rosen.h. Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RosenError(ROSEN_ECUDA, f"{LIB_PATH} not built -- run `python -m paper_1704_04381_b200.build` "
                                      "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    u64, i32, vp = C.c_uint64, C.c_int32, C.c_void_p
    L.rosen_lattice_generate.argtypes = [i32, u64, u64, u64, C.POINTER(rosen_outputs), C.POINTER(rosen_summary), vp]
    L.rosen_lattice_generate.restype = C.c_int
    L.rosen_realspace_generate.argtypes = [i32, u64, i32, C.c_float, C.c_float, u64, u64,
                                           C.POINTER(rosen_outputs), C.POINTER(rosen_summary), vp]
    L.rosen_realspace_generate.restype = C.c_int
    L.rosen_lattice_generate_async.argtypes = [i32, u64, u64, u64, C.POINTER(rosen_outputs), vp, vp]
    L.rosen_lattice_generate_async.restype = C.c_int
    L.rosen_realspace_generate_async.argtypes = [i32, u64, i32, C.c_float, C.c_float, u64, u64,
                                                 C.POINTER(rosen_outputs), vp, vp]
    L.rosen_realspace_generate_async.restype = C.c_int
    L.rosen_lattice_generate_noalloc.argtypes = [i32, u64, u64, u64, C.POINTER(rosen_outputs), vp, vp]
    L.rosen_lattice_generate_noalloc.restype = C.c_int
    L.rosen_lattice_dump.argtypes = [i32, u64, u64, u64, vp, vp, i32, C.POINTER(rosen_summary), vp]
    L.rosen_lattice_dump.restype = C.c_int
    L.rosen_realspace_dump.argtypes = [i32, u64, i32, C.c_float, C.c_float, u64, u64, vp, vp, i32,
                                       C.POINTER(rosen_summary), vp]
    L.rosen_realspace_dump.restype = C.c_int
    L.rosen_summary_merge.argtypes = [C.POINTER(rosen_summary), i32, C.POINTER(rosen_summary)]
    L.rosen_summary_merge.restype = C.c_int
    L.rosen_fit_exponents.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_double), C.POINTER(C.c_double), i32, i32,
                                      C.POINTER(rosen_fit)]
    L.rosen_fit_exponents.restype = C.c_int
    L.rosen_lattice_generate_model.argtypes = [i32, u64, u64, u64, i32, C.c_double, C.POINTER(rosen_outputs),
                                               C.POINTER(rosen_summary), vp]
    L.rosen_lattice_generate_model.restype = C.c_int
    L.rosen_realspace_generate_model.argtypes = [i32, u64, i32, C.c_float, C.c_float, C.c_float, C.c_double, u64, u64,
                                                 C.POINTER(rosen_outputs), C.POINTER(rosen_summary), vp]
    L.rosen_realspace_generate_model.restype = C.c_int
    L.rosen_lattice_perm.argtypes = [i32, u64, u64, u64, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double, C.c_uint32,
                                     C.POINTER(rosen_outputs), C.POINTER(rosen_summary), vp]
    L.rosen_lattice_perm.restype = C.c_int
    L.rosen_realspace_dump_probe.argtypes = [i32, u64, vp, vp, vp]
    L.rosen_realspace_dump_probe.restype = C.c_int
    L.rosen_direction_eval.argtypes = [vp, vp, u64, vp, i32, vp]
    L.rosen_direction_eval.restype = C.c_int
    L.rosen_workspace_bytes.argtypes = []
    L.rosen_workspace_bytes.restype = C.c_size_t
    L.rosen_workspace_release.argtypes = []
    L.rosen_workspace_release.restype = C.c_int
    L.rosen_debug_set.argtypes = [C.c_char_p, C.c_int64]
    L.rosen_debug_set.restype = C.c_int
    L.rosen_last_launch_count.argtypes = []
    L.rosen_last_launch_count.restype = i32
    for name in ("rosen_last_kernel_name", "rosen_last_error", "rosen_version"):
        getattr(L, name).argtypes = []
        getattr(L, name).restype = C.c_char_p
    L.rosen_strerror.argtypes = [C.c_int]
    L.rosen_strerror.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int) -> None:
    if rc != ROSEN_OK:
        L = load_library()
        detail = L.rosen_last_error().decode()
        raise RosenError(rc, L.rosen_strerror(rc).decode() + (f" ({detail})" if detail else ""))


def _torch():
    import torch
    return torch


def _alloc_outputs(N: int, n_chains: int, conf_dtype: str, outputs: Iterable[str], device, host: bool,
                   cache: Optional[dict] = None):
    """Allocate the requested per-chain buffers: torch CUDA tensors, or pinned host tensors.
    `cache` (a dict the caller keeps) lets repeated calls reuse buffers of the same shape."""
    torch = _torch()
    want = set(outputs)
    unknown = want - set(PER_CHAIN)
    if unknown:
        raise ValueError(f"unknown outputs {sorted(unknown)}; choose from {PER_CHAIN}")
    kw = dict(device="cpu", pin_memory=True) if host else dict(device=device)
    shapes = {
        "lnW": ((n_chains,), torch.float64), "alive": ((n_chains,), torch.uint8),
        "m_seq": ((n_chains, N - 1), torch.uint8), "digest": ((n_chains,), torch.int64),
        "conf": ((n_chains, N, 3), torch.int32 if conf_dtype == "int32" else torch.float32),
        "ree2": ((n_chains,), torch.float64), "rg2": ((n_chains,), torch.float64),
    }
    tensors = {}
    for k in PER_CHAIN:
        if k not in want:
            continue
        t = cache.get(k) if cache is not None else None
        if t is None or tuple(t.shape) != shapes[k][0] or t.dtype != shapes[k][1] or t.is_cuda == host:
            t = torch.empty(shapes[k][0], dtype=shapes[k][1], **kw)
            if cache is not None:
                cache[k] = t
        tensors[k] = t
    st = rosen_outputs(*[tensors[k].data_ptr() if k in tensors else None for k in PER_CHAIN],
                       ROSEN_MEM_HOST if host else ROSEN_MEM_DEVICE, 0)
    return tensors, st


def _stream_ptr(stream) -> int:
    torch = _torch()
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def rosen_lattice_generate(N: int, n_chains: int, seed: int, chain_offset: int = 0, outputs: Iterable[str] = (),
                           summary: bool = True, stream=None, host_outputs: bool = False, device=None,
                           host_buffers: Optional[dict] = None) -> Tuple[Optional[Dict[str, float]], Dict[str, "object"]]:
    """rosen_lattice_generate of include/rosen.h. Returns (summary dict or None, {name: tensor})."""
    L = load_library()
    torch = _torch()
    device = device if device is not None else torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else None
    if device is None:
        raise RosenError(ROSEN_ECUDA, "no CUDA device (there is no CPU fallback)")
    tensors, st = _alloc_outputs(N, n_chains, "int32", outputs, device, host_outputs, host_buffers)
    s = rosen_summary()
    _check(L.rosen_lattice_generate(N, n_chains, seed, chain_offset, C.byref(st),
                                    C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), tensors


def rosen_realspace_generate(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, seed: int,
                             chain_offset: int = 0, outputs: Iterable[str] = (), summary: bool = True, stream=None,
                             host_outputs: bool = False, device=None, host_buffers: Optional[dict] = None
                             ) -> Tuple[Optional[Dict[str, float]], Dict[str, "object"]]:
    """rosen_realspace_generate of include/rosen.h. Returns (summary dict or None, {name: tensor})."""
    L = load_library()
    torch = _torch()
    device = device if device is not None else torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else None
    if device is None:
        raise RosenError(ROSEN_ECUDA, "no CUDA device (there is no CPU fallback)")
    tensors, st = _alloc_outputs(N, n_chains, "float32", outputs, device, host_outputs, host_buffers)
    s = rosen_summary()
    _check(L.rosen_realspace_generate(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, C.byref(st),
                                      C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), tensors


def rosen_lattice_generate_model(N: int, n_chains: int, seed: int, z: int = 6, beta_eps: float = 0.0, chain_offset: int = 0,
                                 outputs: Iterable[str] = (), stream=None, host_outputs: bool = False, summary: bool = True):
    """rosen_lattice_generate_model of include/rosen.h (z = 6 / 26 trial set, contact energy). Returns (summary, tensors)."""
    L = load_library()
    torch = _torch()
    if not torch.cuda.is_available():
        raise RosenError(ROSEN_ECUDA, "no CUDA device (there is no CPU fallback)")
    tensors, st = _alloc_outputs(N, n_chains, "int32", outputs, torch.device("cuda", torch.cuda.current_device()), host_outputs)
    s = rosen_summary()
    _check(L.rosen_lattice_generate_model(N, n_chains, seed, chain_offset, z, beta_eps, C.byref(st),
                                          C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), tensors


def rosen_realspace_generate_model(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, lam: float,
                                   beta_eps: float, seed: int, chain_offset: int = 0, outputs: Iterable[str] = (),
                                   stream=None, host_outputs: bool = False, summary: bool = True):
    """rosen_realspace_generate_model of include/rosen.h (square well of range lam * sigma). Returns (summary, tensors)."""
    L = load_library()
    torch = _torch()
    if not torch.cuda.is_available():
        raise RosenError(ROSEN_ECUDA, "no CUDA device (there is no CPU fallback)")
    tensors, st = _alloc_outputs(N, n_chains, "float32", outputs, torch.device("cuda", torch.cuda.current_device()), host_outputs)
    s = rosen_summary()
    _check(L.rosen_realspace_generate_model(N, n_chains, k_trials, bond_len, sigma, lam, beta_eps, seed, chain_offset,
                                            C.byref(st), C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), tensors


def rosen_lattice_perm(N: int, n_tours: int, seed: int, ln_lo, ln_hi, ln_ref: float, max_nodes: int = 1 << 20,
                       tour_offset: int = 0, outputs: Iterable[str] = (), stream=None, host_outputs: bool = False,
                       summary: bool = True):
    """rosen_lattice_perm of include/rosen.h: ln_lo, ln_hi = sequences of N+1 floats. Returns (summary, tensors)."""
    L = load_library()
    torch = _torch()
    if not torch.cuda.is_available():
        raise RosenError(ROSEN_ECUDA, "no CUDA device (there is no CPU fallback)")
    if len(ln_lo) != N + 1 or len(ln_hi) != N + 1:
        raise ValueError("ln_lo, ln_hi need N + 1 entries")
    lo = (C.c_double * (N + 1))(*[float(v) for v in ln_lo]); hi = (C.c_double * (N + 1))(*[float(v) for v in ln_hi])
    tensors, st = _alloc_outputs(N, n_tours, "int32", outputs, torch.device("cuda", torch.cuda.current_device()), host_outputs)
    s = rosen_summary()
    _check(L.rosen_lattice_perm(N, n_tours, seed, tour_offset, lo, hi, ln_ref, max_nodes, C.byref(st),
                                C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), tensors


SUMMARY_BYTES = C.sizeof(rosen_summary)


def _outputs_struct(tensors: Optional[Dict[str, "object"]]) -> rosen_outputs:
    tensors = tensors or {}
    return rosen_outputs(*[tensors[k].data_ptr() if k in tensors else None for k in PER_CHAIN], ROSEN_MEM_DEVICE, 0)


def summary_from_device(summary_device) -> Dict[str, float]:
    """Decode a uint8 CUDA tensor of SUMMARY_BYTES written by an _async call (synchronises via .cpu())."""
    raw = bytes(summary_device.cpu().numpy().tobytes())
    return rosen_summary.from_buffer_copy(raw).as_dict()


def rosen_lattice_generate_async(N: int, n_chains: int, seed: int, chain_offset: int = 0, outputs=None,
                                 summary_device=None, stream=None) -> None:
    """rosen_lattice_generate_async: enqueue only. outputs = {name: CUDA tensor}; summary_device = uint8 CUDA
    tensor of SUMMARY_BYTES (8-byte aligned) or None."""
    L = load_library()
    st = _outputs_struct(outputs)
    _check(L.rosen_lattice_generate_async(N, n_chains, seed, chain_offset, C.byref(st),
                                          summary_device.data_ptr() if summary_device is not None else None,
                                          _stream_ptr(stream)))


ROSEN_NOALLOC_MAX_N, ROSEN_NOALLOC_MAX_CHAINS, ROSEN_NOALLOC_SCRATCH_BYTES = 512, 1 << 24, 8192 * 64 + 256


def rosen_lattice_generate_noalloc(N: int, n_chains: int, seed: int, chain_offset: int = 0, outputs=None,
                                   summary_device=None, stream=None) -> None:
    """rosen_lattice_generate_noalloc of include/rosen.h: the lattice call for programs that cannot let a library
    allocate GPU memory (their own allocator owns the device, or their footprint is fixed, or they cannot afford the
    device-wide stall of cudaMalloc). Enqueue only, and this wrapper allocates nothing either: outputs = {name: CUDA
    tensor the caller made}, summary_device = a uint8 CUDA tensor of SUMMARY_BYTES (8-byte aligned) the caller made, or
    None. N <= ROSEN_NOALLOC_MAX_N and n_chains <= ROSEN_NOALLOC_MAX_CHAINS, else RosenError(ROSEN_ERANGE). Calls
    on one device share one static scratch array: do not let two of them overlap on the GPU."""
    L = load_library()
    st = _outputs_struct(outputs)
    _check(L.rosen_lattice_generate_noalloc(N, n_chains, seed, chain_offset, C.byref(st),
                                            summary_device.data_ptr() if summary_device is not None else None,
                                            _stream_ptr(stream)))


def rosen_realspace_generate_async(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, seed: int,
                                   chain_offset: int = 0, outputs=None, summary_device=None, stream=None) -> None:
    """rosen_realspace_generate_async: enqueue only (see rosen_lattice_generate_async)."""
    L = load_library()
    st = _outputs_struct(outputs)
    _check(L.rosen_realspace_generate_async(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, C.byref(st),
                                            summary_device.data_ptr() if summary_device is not None else None,
                                            _stream_ptr(stream)))


def rosen_lattice_dump(N: int, n_chains: int, seed: int, chain_offset: int = 0, conf=None, lnW=None,
                       summary: bool = True, stream=None):
    """rosen_lattice_dump: conf int32 [n_chains, N, 3] and lnW float64 [n_chains] CUDA tensors (allocated if None)."""
    L = load_library()
    torch = _torch()
    conf = conf if conf is not None else torch.empty((n_chains, N, 3), dtype=torch.int32, device="cuda")
    lnW = lnW if lnW is not None else torch.empty((n_chains,), dtype=torch.float64, device="cuda")
    s = rosen_summary()
    _check(L.rosen_lattice_dump(N, n_chains, seed, chain_offset, conf.data_ptr(), lnW.data_ptr(), ROSEN_MEM_DEVICE,
                                C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), conf, lnW


def rosen_realspace_dump(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, seed: int,
                         chain_offset: int = 0, conf=None, lnW=None, summary: bool = True, stream=None):
    """rosen_realspace_dump: conf float32 [n_chains, N, 3] and lnW float64 [n_chains] CUDA tensors."""
    L = load_library()
    torch = _torch()
    conf = conf if conf is not None else torch.empty((n_chains, N, 3), dtype=torch.float32, device="cuda")
    lnW = lnW if lnW is not None else torch.empty((n_chains,), dtype=torch.float64, device="cuda")
    s = rosen_summary()
    _check(L.rosen_realspace_dump(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset, conf.data_ptr(),
                                  lnW.data_ptr(), ROSEN_MEM_DEVICE, C.byref(s) if summary else None, _stream_ptr(stream)))
    return (s.as_dict() if summary else None), conf, lnW


def rosen_summary_merge(parts) -> Dict[str, float]:
    """rosen_summary_merge: merge summary dicts of disjoint chain ranges (rank order)."""
    L = load_library()
    arr = (rosen_summary * len(parts))(*[rosen_summary.from_dict(p) for p in parts])
    out = rosen_summary()
    _check(L.rosen_summary_merge(arr, len(parts), C.byref(out)))
    return out.as_dict()


class rosen_fit(C.Structure):
    _fields_ = [("nu", C.c_double), ("ln_a", C.c_double), ("mu", C.c_double), ("gamma", C.c_double), ("c", C.c_double),
                ("rms_ree2", C.c_double), ("rms_lnZ", C.c_double)]


def rosen_fit_exponents(N, mean_ree2, ln_mean_W, use_steps: bool = True) -> Dict[str, float]:
    """rosen_fit_exponents: nu (Eq. 4) and mu, gamma (Eq. 5-7) by least squares over a length sweep."""
    L = load_library()
    n = len(N)
    out = rosen_fit()
    _check(L.rosen_fit_exponents((C.c_int32 * n)(*[int(v) for v in N]), (C.c_double * n)(*[float(v) for v in mean_ree2]),
                                 (C.c_double * n)(*[float(v) for v in ln_mean_W]), n, 1 if use_steps else 0, C.byref(out)))
    return {name: getattr(out, name) for name, _ in out._fields_}


def rosen_realspace_dump_probe(N: int, n_chains: int, conf, lnW=None, stream=None) -> None:
    """rosen_realspace_dump_probe: conf = float32 CUDA tensor [n_chains, N, 3], lnW = float64 CUDA tensor [n_chains] or None."""
    _check(load_library().rosen_realspace_dump_probe(N, n_chains, conf.data_ptr(), lnW.data_ptr() if lnW is not None else None,
                                                     _stream_ptr(stream)))


def rosen_direction_eval(wz, wphi, stream=None):
    """rosen_direction_eval: wz, wphi = int32/uint32 CUDA tensors of n Philox words (bit patterns); returns a float32
    CUDA tensor [n, 3] (enqueue only, on `stream`)."""
    L = load_library()
    torch = _torch()
    n = int(wz.numel())
    if not (wz.is_cuda and wphi.is_cuda and wz.element_size() == 4 and wphi.element_size() == 4 and wphi.numel() == n
            and wz.is_contiguous() and wphi.is_contiguous()):
        raise ValueError("wz, wphi: contiguous 32-bit CUDA tensors of equal length")
    out = torch.empty((n, 3), dtype=torch.float32, device=wz.device)
    _check(L.rosen_direction_eval(wz.data_ptr(), wphi.data_ptr(), n, out.data_ptr(), ROSEN_MEM_DEVICE, _stream_ptr(stream)))
    return out


def rosen_workspace_bytes() -> int:
    return int(load_library().rosen_workspace_bytes())


def rosen_workspace_release() -> int:
    return int(load_library().rosen_workspace_release())


def rosen_debug_set(knob: str, value: int) -> None:
    """rosen_debug_set of include/rosen.h (test / tuning knobs; 0 = default)."""
    _check(load_library().rosen_debug_set(knob.encode(), int(value)))


def rosen_last_launch_count() -> int:
    return int(load_library().rosen_last_launch_count())


def rosen_last_kernel_name() -> str:
    return load_library().rosen_last_kernel_name().decode()


def rosen_strerror(code: int) -> str:
    return load_library().rosen_strerror(code).decode()


def rosen_last_error() -> str:
    return load_library().rosen_last_error().decode()


def rosen_version() -> str:
    return load_library().rosen_version().decode()
