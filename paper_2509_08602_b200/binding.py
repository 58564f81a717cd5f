"""ctypes binding of libadmm_b200.so -- argument marshalling only, same names as include/admm_b200.h.

Every step of the path runs in the CUDA kernels behind the C ABI; there is no Python or CPU
fallback.  If the shared library is missing the import fails loudly (build it with
`python -m paper_2509_08602_b200.build` or `__graft_entry__.build()`).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libadmm_b200.so")

ADMM_OK, ADMM_EINVAL, ADMM_ENOMEM, ADMM_ECUDA, ADMM_ENOTSPD, ADMM_ESTATE = range(6)
STATUS_NAMES = ["ADMM_OK", "ADMM_EINVAL", "ADMM_ENOMEM", "ADMM_ECUDA", "ADMM_ENOTSPD", "ADMM_ESTATE"]
ADMM_STORAGE_FP32_3XTF32, ADMM_STORAGE_FP32_TF32, ADMM_STORAGE_BF16, ADMM_STORAGE_CSR = range(4)
ADMM_PATH_TCGEN05, ADMM_PATH_SIMT = 0, 1

# every symbol include/admm_b200.h declares (tests/test_abi.py checks the library exports them all)
EXPORTS = [
    "admm_default_options", "admm_setup", "admm_solve_batch", "admm_get_state", "admm_get_preconditioner",
    "admm_get_timing", "admm_get_kernel_times", "admm_last_launch_count", "admm_last_error", "admm_destroy",
    "admm_version", "admm_contract_probe", "admm_dose", "admm_lowdose_volumes", "admm_phit_apply_static",
]


class AdmmError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {message}")
        self.status = status


class admm_class(C.Structure):
    _fields_ = [("sense", C.c_int32), ("threshold", C.c_float), ("hard", C.c_int32)]


class admm_options(C.Structure):
    _fields_ = [("storage", C.c_int32), ("kernel_path", C.c_int32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("check_every", C.c_int32), ("eps_abs", C.c_float), ("compaction", C.c_int32),
                ("csr_rel_threshold", C.c_float), ("profile_kernels", C.c_int32), ("drain_kb", C.c_int32),
                ("k1_slab_kb", C.c_int32), ("presolve", C.c_int32), ("accum_debias", C.c_int32), ("dose_only", C.c_int32),
                ("warm_start_ratio", C.c_float), ("bot_rows", C.c_void_p)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: the CUDA extension has not been built and there is no CPU fallback. "
            "Run `python -m paper_2509_08602_b200.build`.")
    lib = C.CDLL(LIB_PATH, mode=C.RTLD_GLOBAL)
    vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
    lib.admm_default_options.argtypes = [C.POINTER(admm_options)]; lib.admm_default_options.restype = None
    lib.admm_setup.argtypes = [C.POINTER(vp), vp, i32, i64, i64, i64, vp, C.POINTER(admm_class), i32, C.POINTER(admm_options)]
    lib.admm_setup.restype = i32
    lib.admm_solve_batch.argtypes = [vp, i32, vp, vp, vp, f32, i32, i32, vp, vp, vp, vp]
    lib.admm_solve_batch.restype = i32
    lib.admm_get_state.argtypes = [vp, i32, vp, vp, vp, vp]; lib.admm_get_state.restype = i32
    lib.admm_get_preconditioner.argtypes = [vp, vp, vp, vp]; lib.admm_get_preconditioner.restype = i32
    lib.admm_get_timing.argtypes = [vp, C.POINTER(C.c_double * 8), C.POINTER(i64)]; lib.admm_get_timing.restype = i32
    lib.admm_get_kernel_times.argtypes = [vp, C.POINTER(C.c_double * 4), C.POINTER(i64 * 4)]; lib.admm_get_kernel_times.restype = i32
    lib.admm_last_launch_count.argtypes = [vp]; lib.admm_last_launch_count.restype = i64
    lib.admm_last_error.argtypes = [vp]; lib.admm_last_error.restype = C.c_char_p
    lib.admm_destroy.argtypes = [vp]; lib.admm_destroy.restype = None
    lib.admm_version.argtypes = []; lib.admm_version.restype = C.c_char_p
    lib.admm_contract_probe.argtypes = [vp, i32, i32, vp, vp]; lib.admm_contract_probe.restype = i32
    lib.admm_dose.argtypes = [vp, i32, vp, i64, vp]; lib.admm_dose.restype = i32
    lib.admm_lowdose_volumes.argtypes = [vp, i32, vp, i64, f32, f32, vp, vp, vp]; lib.admm_lowdose_volumes.restype = i32
    lib.admm_phit_apply_static.argtypes = [vp, i64, i64, i64, vp, i64, i32, vp, i32, vp, C.c_char_p, i32]
    lib.admm_phit_apply_static.restype = i32
    return lib


_lib = _load()


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def _ptr(x) -> Optional[int]:
    """Raw address of a numpy array (host) or a torch tensor (host or device)."""
    if x is None:
        return None
    if _is_torch(x):
        return x.data_ptr()
    return x.ctypes.data


def _check(status: int, handle) -> None:
    if status != ADMM_OK:
        raise AdmmError(status, _lib.admm_last_error(handle).decode())


class Handle:
    def __init__(self, ptr: int, N: int, n: int, n_classes: int):
        self.ptr, self.N, self.n, self.n_classes = ptr, N, n, n_classes

    def close(self) -> None:
        if self.ptr:
            _lib.admm_destroy(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def admm_version() -> str:
    return _lib.admm_version().decode()


def admm_default_options() -> admm_options:
    o = admm_options()
    _lib.admm_default_options(C.byref(o))
    return o


def admm_setup(phi, point_class, classes: Sequence, *, storage: int = ADMM_STORAGE_FP32_3XTF32,
               kernel_path: int = ADMM_PATH_TCGEN05, device: int = 0, stream: Optional[int] = None,
               check_every: int = 10, eps_abs: float = 1e-6, compaction: bool = True,
               profile_kernels: bool = False, drain_kb: int = 0, k1_slab_kb: int = 0,
               csr_rel_threshold: float = 0.0, presolve: bool = True, accum_debias: int = 0,
               dose_only: bool = False, bot_rows=None, warm_start_ratio: float = 0.0) -> Handle:
    """phi: [N, n] float32, numpy (host) or torch CUDA tensor, row-major (last stride 1).
    classes: sequence of objects with .sense, .threshold, .hard (e.g. workloads.ClassSpec)."""
    if _is_torch(phi):
        on_device = int(phi.is_cuda)
        assert phi.dim() == 2 and phi.stride(1) == 1 and str(phi.dtype) == "torch.float32"
        N, n, ld = int(phi.shape[0]), int(phi.shape[1]), int(phi.stride(0))
    else:
        phi = np.ascontiguousarray(phi, dtype=np.float32)
        on_device, (N, n), ld = 0, phi.shape, phi.shape[1]
    pc = np.ascontiguousarray(point_class, dtype=np.uint8)
    assert pc.shape == (N,)
    cls = (admm_class * len(classes))(*[admm_class(int(c.sense), float(c.threshold), int(getattr(c, "hard", 0))) for c in classes])
    o = admm_default_options()
    o.storage, o.kernel_path, o.device = storage, kernel_path, device
    o.stream = stream
    o.check_every, o.eps_abs, o.compaction, o.profile_kernels = check_every, eps_abs, int(compaction), int(profile_kernels)
    o.drain_kb = int(drain_kb)
    o.k1_slab_kb = int(k1_slab_kb)
    o.csr_rel_threshold = float(csr_rel_threshold)
    o.presolve = int(presolve)
    o.accum_debias = int(accum_debias)
    o.dose_only = int(dose_only)
    o.warm_start_ratio = float(warm_start_ratio)
    br = None
    if bot_rows is not None:
        br = np.ascontiguousarray(bot_rows, dtype=np.uint8)
        assert br.shape == (n,)
        o.bot_rows = br.ctypes.data
    out = C.c_void_p()
    st = _lib.admm_setup(C.byref(out), _ptr(phi), on_device, N, n, ld, _ptr(pc), cls, len(classes), C.byref(o))
    _check(st, None)
    return Handle(out.value, int(N), int(n), len(classes))


def admm_solve_batch(h: Handle, weights, rho=None, row_mask=None, *, tol: float = 1e-4, max_iter: int = 3000,
                     fixed_iters: int = 0, out=None) -> dict:
    """weights [B, n_classes+1]; rho [B] or None; row_mask [B, ceil(N/32)] uint32 (numpy or torch CUDA) or None.
    `out`: optional dict of preallocated outputs (numpy or torch, host or device): t, obj, res, iters."""
    w = np.ascontiguousarray(weights, dtype=np.float32)
    B = w.shape[0]
    assert w.shape == (B, h.n_classes + 1)
    r = None if rho is None else np.ascontiguousarray(rho, dtype=np.float32)
    if row_mask is not None and not _is_torch(row_mask):
        row_mask = np.ascontiguousarray(row_mask, dtype=np.uint32)
        assert row_mask.shape == (B, (h.N + 31) // 32)
    out = dict(out or {})
    out.setdefault("t", np.empty((B, h.n), dtype=np.float32))
    out.setdefault("obj", np.empty(B, dtype=np.float64))
    out.setdefault("res", np.empty((B, 2), dtype=np.float32))
    out.setdefault("iters", np.empty(B, dtype=np.int32))
    st = _lib.admm_solve_batch(h.ptr, B, _ptr(w), _ptr(r), _ptr(row_mask), float(tol), int(max_iter), int(fixed_iters),
                               _ptr(out["t"]), _ptr(out["obj"]), _ptr(out["res"]), _ptr(out["iters"]))
    _check(st, h.ptr)
    return out


def admm_get_state(h: Handle, plan: int):
    z1 = np.empty(h.N, np.float32); y1 = np.empty(h.N, np.float32)
    z2 = np.empty(h.n, np.float64); y2 = np.empty(h.n, np.float64)
    _check(_lib.admm_get_state(h.ptr, int(plan), _ptr(z1), _ptr(y1), _ptr(z2), _ptr(y2)), h.ptr)
    return z1, y1, z2, y2


def admm_contract_probe(h: Handle, which: int, small) -> np.ndarray:
    small = np.ascontiguousarray(small, dtype=np.float32)
    B = small.shape[0]
    rows = h.n if which == 0 else h.N
    assert small.shape[1] == (h.N if which == 0 else h.n)
    out = np.empty((B, rows), dtype=np.float64)
    _check(_lib.admm_contract_probe(h.ptr, int(which), B, _ptr(small), _ptr(out)), h.ptr)
    return out


def admm_dose(h: Handle, t, out=None):
    """dose [B, N] = t [B, n] . Phi^T on the handle's resident Phi (include/admm_b200.h admm_dose).  t: numpy or torch (host or CUDA),
    float32, last stride 1; out: optional preallocated [B, N] float32 (numpy or torch CUDA)."""
    if _is_torch(t):
        assert t.dim() == 2 and t.stride(1) == 1 and str(t.dtype) == "torch.float32"
        B, ld = int(t.shape[0]), int(t.stride(0))
        assert int(t.shape[1]) == h.n
    else:
        t = np.ascontiguousarray(t, dtype=np.float32)
        B, ld = t.shape[0], t.shape[1]
        assert t.shape[1] == h.n
    if out is None:
        out = np.empty((B, h.N), dtype=np.float32)
    _check(_lib.admm_dose(h.ptr, B, _ptr(t), ld, _ptr(out)), h.ptr)
    return out


def admm_lowdose_volumes(h: Handle, t, d_lo: float, d_hi: float, want_dose: bool = False):
    """(in_volume [B, ceil(N/32)] uint32, any_volume [ceil(N/32)] uint32[, dose [B, N] float32]) -- include/admm_b200.h."""
    t = np.ascontiguousarray(t, dtype=np.float32)
    B = t.shape[0]
    assert t.shape[1] == h.n
    words = (h.N + 31) // 32
    inv = np.empty((B, words), dtype=np.uint32); anyv = np.empty(words, dtype=np.uint32)
    dose = np.empty((B, h.N), dtype=np.float32) if want_dose else None
    _check(_lib.admm_lowdose_volumes(h.ptr, B, _ptr(t), t.shape[1], float(d_lo), float(d_hi), _ptr(inv), _ptr(anyv), _ptr(dose)), h.ptr)
    return (inv, anyv, dose) if want_dose else (inv, anyv)


ADMM_STATIC_SCRATCH_BYTES = 8 * 1024 * 1024


def admm_phit_apply_static(phi, g, w_out, *, stream=None) -> None:
    """w_out [B, n] float64 = g [B, N] . phi [N, n], all three torch CUDA tensors of one device (include/admm_b200.h
    admm_phit_apply_static): allocates nothing, enqueues on `stream` (a cudaStream_t as int; default: torch's current stream) and
    does not synchronise.  phi / g: float32, last stride 1; w_out: float64, contiguous.  B * n <= 2093056."""
    import torch
    for x, dt in ((phi, torch.float32), (g, torch.float32), (w_out, torch.float64)):
        assert _is_torch(x) and x.is_cuda and x.dim() == 2 and x.dtype == dt and x.stride(1) == 1
    N, n = int(phi.shape[0]), int(phi.shape[1])
    B = int(g.shape[0])
    assert int(g.shape[1]) == N and tuple(w_out.shape) == (B, n) and w_out.is_contiguous()
    dev = phi.device.index
    assert g.device.index == dev and w_out.device.index == dev
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    err = C.create_string_buffer(512)
    st = _lib.admm_phit_apply_static(phi.data_ptr(), N, n, int(phi.stride(0)), g.data_ptr(), int(g.stride(0)), B, w_out.data_ptr(),
                                     int(dev), C.c_void_p(stream), err, 512)
    if st != ADMM_OK:
        raise AdmmError(st, err.value.decode())


def admm_get_preconditioner(h: Handle, want_sinv: bool = True):
    D = np.empty(h.N, np.float64); R = np.empty(h.n, np.float64)
    S = np.empty((h.n, h.n), np.float64) if want_sinv else None
    _check(_lib.admm_get_preconditioner(h.ptr, _ptr(D), _ptr(R), _ptr(S)), h.ptr)
    return D, R, S


def admm_get_timing(h: Handle) -> dict:
    ms = (C.c_double * 8)(); it = C.c_int64()
    _check(_lib.admm_get_timing(h.ptr, C.byref(ms), C.byref(it)), h.ptr)
    keys = ["upload_ms", "syrk_ms", "factor_ms", "setup_ms", "iterate_ms", "finalise_ms", "solve_wall_ms", "csr_density"]
    d = {k: ms[i] for i, k in enumerate(keys)}
    d["plan_iters"] = it.value
    return d


def admm_get_kernel_times(h: Handle) -> dict:
    ms = (C.c_double * 4)(); n = (C.c_int64 * 4)()
    _check(_lib.admm_get_kernel_times(h.ptr, C.byref(ms), C.byref(n)), h.ptr)
    names = ["k1_phiT_g", "k2_sinv", "k3_phi_v", "convergence"]
    return {nm: dict(total_ms=ms[i], launches=n[i]) for i, nm in enumerate(names)}


def admm_last_launch_count(h: Handle) -> int:
    return int(_lib.admm_last_launch_count(h.ptr))


def admm_last_error(h: Optional[Handle] = None) -> str:
    return _lib.admm_last_error(h.ptr if h else None).decode()


def admm_destroy(h: Handle) -> None:
    h.close()
