"""ctypes binding of libls_b200.so — the same names as include/ls.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; nothing here computes.  There is
no CPU fallback: if the shared library is missing (not built) or no CUDA device is usable the
calls raise.  PyTorch is used by callers for device memory and streams only; this module accepts
anything exposing `.data_ptr()` (torch tensors), raw integer device addresses, or — for
`ls_execute_host` — C-contiguous numpy arrays / pinned torch CPU tensors.
"""
from __future__ import annotations

import ctypes as C
import os

__all__ = [
    "LS_F32", "LS_F64", "LS_OK", "STAGES", "LsError", "ls_opts", "lib_path", "load",
    "ls_plan", "ls_execute", "ls_execute_host", "ls_destroy", "ls_get_info", "ls_workspace_bytes", "ls_set_workspace",
    "ls_get_stage_ms", "ls_get_launch_counts", "ls_debug_modes", "ls_debug_stats", "ls_debug_points", "ls_debug_bins", "ls_debug_grid", "ls_debug_dinv",
    "ls_debug_assemble", "ls_debug_guards", "ls_strerror", "ls_direct_power", "ls_direct_sums", "ls_direct_power_noalloc",
    "exported_symbols", "Plan",
]

LS_F32, LS_F64 = 0, 1
LS_OK = 0
LS_NORM_STANDARD, LS_NORM_MODEL, LS_NORM_LOG, LS_NORM_PSD = 0, 1, 2, 3
STAGES = ("stats", "sort", "premul", "spread", "fft", "assemble", "total", "fft_pass1", "fft_pass2", "fft_pass3")

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libls_b200.so")


class ls_opts(C.Structure):
    _fields_ = [
        ("dy_per_series", C.c_int),
        ("upsampfac", C.c_double),
        ("kernel_width", C.c_int),
        ("timing", C.c_int),
        ("device", C.c_int),
        ("tile_cells", C.c_int),
        ("batch_chunk", C.c_int),
        ("no_autotune", C.c_int),
        ("graph", C.c_int),
        ("fft_impl", C.c_int),
        ("no_floating_mean", C.c_int),
        ("normalization", C.c_int),
        ("t_is_dtype", C.c_int),
        ("reserved", C.c_int * 2),
    ]


class LsError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = int(code)
        super().__init__(f"{where}: {ls_strerror(code)} (code {code})")


_lib = None

# every symbol include/ls.h declares: (name, restype, argtypes)
_SIGNATURES = {
    "ls_plan": (C.c_int, [C.POINTER(C.c_void_p), C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double,
                          C.c_int, C.c_int, C.POINTER(ls_opts)]),
    "ls_execute": (C.c_int, [C.c_void_p] * 6),
    "ls_execute_host": (C.c_int, [C.c_void_p] * 6),
    "ls_get_info": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_double),
                              C.POINTER(C.c_int64), C.POINTER(C.c_int), C.POINTER(C.c_double)]),
    "ls_workspace_bytes": (C.c_size_t, [C.c_void_p]),
    "ls_set_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "ls_get_stage_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_float), C.c_int]),
    "ls_get_launch_counts": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "ls_debug_modes": (C.c_int, [C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_double)]),
    "ls_debug_stats": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "ls_debug_points": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_double)]),
    "ls_debug_bins": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int)]),
    "ls_debug_grid": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double)]),
    "ls_debug_dinv": (C.c_int, [C.c_void_p, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_double)]),
    "ls_debug_guards": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "ls_debug_assemble": (C.c_int, [C.c_int64, C.POINTER(C.c_double), C.c_double, C.c_double, C.c_int, C.c_int,
                                    C.POINTER(C.c_double)]),
    "ls_direct_power": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64] + [C.c_void_p] * 5),
    "ls_direct_sums": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64] + [C.c_void_p] * 5),
    "ls_direct_power_noalloc": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64] + [C.c_void_p] * 5),
    "ls_strerror": (C.c_char_p, [C.c_int]),
    "ls_destroy": (C.c_int, [C.c_void_p]),
}


def lib_path() -> str:
    return _LIB


def load():
    """dlopen the in-tree library (fails loudly when it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB):
            raise ImportError(f"{_LIB} is missing: run `python -m paper_2409_08090_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(_LIB)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def exported_symbols():
    return tuple(_SIGNATURES)


def _ptr(a) -> int:
    """Address of a buffer: torch tensor (.data_ptr), numpy array (.ctypes.data) or int."""
    if a is None:
        return 0
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return int(a.data_ptr())
    if hasattr(a, "ctypes"):
        return int(a.ctypes.data)
    raise TypeError(f"cannot take the address of {type(a)!r}")


def ls_strerror(code: int) -> str:
    return load().ls_strerror(int(code)).decode()


def ls_plan(Nd, Nf, f0, df, eps, dtype, batch=1, opts: ls_opts | None = None) -> int:
    h = C.c_void_p()
    rc = load().ls_plan(C.byref(h), int(Nd), int(Nf), float(f0), float(df), float(eps), int(dtype), int(batch),
                        C.byref(opts) if opts is not None else None)
    if rc != LS_OK:
        raise LsError(rc, "ls_plan")
    return h.value


def ls_execute(plan, t, y, dy, power, stream=0) -> None:
    rc = load().ls_execute(plan, _ptr(t), _ptr(y), _ptr(dy), _ptr(power), _ptr(stream))
    if rc != LS_OK:
        raise LsError(rc, "ls_execute")


def ls_execute_host(plan, t, y, dy, power, stream=0) -> None:
    rc = load().ls_execute_host(plan, _ptr(t), _ptr(y), _ptr(dy), _ptr(power), _ptr(stream))
    if rc != LS_OK:
        raise LsError(rc, "ls_execute_host")


def ls_destroy(plan) -> None:
    rc = load().ls_destroy(plan)
    if rc != LS_OK:
        raise LsError(rc, "ls_destroy")


def ls_get_info(plan) -> dict:
    sigma, beta, mb = C.c_double(), C.c_double(), C.c_double()
    w, M = C.c_int(), C.c_int()
    n = C.c_int64()
    rc = load().ls_get_info(plan, C.byref(sigma), C.byref(w), C.byref(beta), C.byref(n), C.byref(M), C.byref(mb))
    if rc != LS_OK:
        raise LsError(rc, "ls_get_info")
    return {"sigma": sigma.value, "w": w.value, "beta": beta.value, "n": n.value, "M": M.value,
            "model_bytes": mb.value}


def ls_workspace_bytes(plan) -> int:
    return int(load().ls_workspace_bytes(plan))


def ls_set_workspace(plan, buf, nbytes: int) -> None:
    rc = load().ls_set_workspace(plan, C.c_void_p(_ptr(buf)), C.c_size_t(int(nbytes)))
    if rc != LS_OK:
        raise LsError(rc, "ls_set_workspace")


def ls_direct_power(Nd, f0, df, k0, K, t, y, dy, power, stream=0) -> None:
    """Brute-force power of frequencies f0 + (k0 .. k0+K-1) df of one fp64 series (device buffers)."""
    rc = load().ls_direct_power(int(Nd), float(f0), float(df), int(k0), int(K), C.c_void_p(_ptr(t)), C.c_void_p(_ptr(y)),
                                C.c_void_p(_ptr(dy)), C.c_void_p(_ptr(power)), C.c_void_p(int(stream)))
    if rc != LS_OK:
        raise LsError(rc, "ls_direct_power")


def ls_direct_sums(Nd, f0, df, k0, K, t, y, dy, sums, stream=0) -> None:
    """The six brute-force sums (Sh, Ch, S, C, S2, C2) of frequencies f0 + (k0 .. k0+K-1) df into sums[K][6] (device)."""
    rc = load().ls_direct_sums(int(Nd), float(f0), float(df), int(k0), int(K), C.c_void_p(_ptr(t)), C.c_void_p(_ptr(y)),
                               C.c_void_p(_ptr(dy)), C.c_void_p(_ptr(sums)), C.c_void_p(int(stream)))
    if rc != LS_OK:
        raise LsError(rc, "ls_direct_sums")


LS_NOALLOC_MAX_ND = 65536
LS_ERR_TOO_LARGE = 7


def ls_direct_power_noalloc(Nd, f0, df, k0, K, t, y, dy, power, stream=0) -> None:
    """ls_direct_power without any allocation (fixed scratch inside the library, Nd <= LS_NOALLOC_MAX_ND); asynchronous:
    the caller synchronises the stream.  Calls that overlap on the GPU race on the shared scratch (ls.h)."""
    rc = load().ls_direct_power_noalloc(int(Nd), float(f0), float(df), int(k0), int(K), C.c_void_p(_ptr(t)),
                                        C.c_void_p(_ptr(y)), C.c_void_p(_ptr(dy)), C.c_void_p(_ptr(power)),
                                        C.c_void_p(int(stream)))
    if rc != LS_OK:
        raise LsError(rc, "ls_direct_power_noalloc")


def ls_get_stage_ms(plan) -> dict:
    ms = (C.c_float * len(STAGES))()
    rc = load().ls_get_stage_ms(plan, ms, len(STAGES))
    if rc != LS_OK:
        raise LsError(rc, "ls_get_stage_ms")
    return {k: float(ms[i]) for i, k in enumerate(STAGES)}


def ls_get_launch_counts(plan) -> tuple[int, int]:
    a, b = C.c_int(), C.c_int()
    rc = load().ls_get_launch_counts(plan, C.byref(a), C.byref(b))
    if rc != LS_OK:
        raise LsError(rc, "ls_get_launch_counts")
    return a.value, b.value


def ls_debug_modes(plan, series, kidx):
    import numpy as np
    k = np.ascontiguousarray(kidx, dtype=np.int64)
    out = np.empty((k.size, 6), dtype=np.float64)
    rc = load().ls_debug_modes(plan, int(series), k.size, k.ctypes.data_as(C.POINTER(C.c_int64)),
                               out.ctypes.data_as(C.POINTER(C.c_double)))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_modes")
    return out


def ls_debug_stats(plan, batch):
    import numpy as np
    out = np.empty((int(batch), 3), dtype=np.float64)
    rc = load().ls_debug_stats(plan, out.ctypes.data_as(C.POINTER(C.c_double)))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_stats")
    return out


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def ls_debug_points(plan, Nd, point_set):
    """Bin-sorted point records of the last execute: [Nd, 4] = (eta, l0, q_re, q_im); point_set 0 = x1, 1 = x2."""
    import numpy as np
    out = np.empty((int(Nd), 4), dtype=np.float64)
    rc = load().ls_debug_points(plan, int(point_set), _dp(out))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_points")
    return out


def ls_debug_bins(plan, nbins, point_set):
    import numpy as np
    out = np.empty(int(nbins) + 1, dtype=np.int32)
    rc = load().ls_debug_bins(plan, int(point_set), out.ctypes.data_as(C.POINTER(C.c_int)))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_bins")
    return out


def ls_debug_grid(plan, n, t, y, dy, slot):
    """Fine grid `slot` ([n] complex128) after K1..K4 on the device buffers t, y, dy."""
    import numpy as np
    out = np.empty((int(n), 2), dtype=np.float64)
    rc = load().ls_debug_grid(plan, C.c_void_p(_ptr(t)), C.c_void_p(_ptr(y)), C.c_void_p(_ptr(dy)), int(slot), _dp(out))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_grid")
    return out[:, 0] + 1j * out[:, 1]


def ls_debug_dinv(plan, kabs):
    import numpy as np
    k = np.ascontiguousarray(kabs, dtype=np.int64)
    out = np.empty(k.size, dtype=np.float64)
    rc = load().ls_debug_dinv(plan, k.size, k.ctypes.data_as(C.POINTER(C.c_int64)), _dp(out))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_dinv")
    return out


def ls_debug_guards(plan) -> int:
    """Guard-zone bytes overwritten by any kernel since the plan was made (needs LS_B200_GUARD in the environment)."""
    n = C.c_int64()
    rc = load().ls_debug_guards(plan, C.byref(n))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_guards")
    return int(n.value)


def ls_debug_assemble(sums, YY, W=1.0, no_floating_mean=0, normalization=0):
    import numpy as np
    s = np.ascontiguousarray(sums, dtype=np.float64).reshape(-1, 6)
    out = np.empty(s.shape[0], dtype=np.float64)
    rc = load().ls_debug_assemble(s.shape[0], _dp(s), float(YY), float(W), int(no_floating_mean), int(normalization), _dp(out))
    if rc != LS_OK:
        raise LsError(rc, "ls_debug_assemble")
    return out


class Plan:
    """Owning handle around ls_plan / ls_destroy (context manager)."""

    def __init__(self, Nd, Nf, f0, df, eps=1e-9, dtype=LS_F64, batch=1, **opts):
        o = ls_opts()
        for k, v in opts.items():
            if not hasattr(o, k):
                raise TypeError(f"unknown ls_opts field {k!r}")
            setattr(o, k, v)
        self.Nd, self.Nf, self.batch, self.dtype = int(Nd), int(Nf), int(batch), int(dtype)
        self.handle = ls_plan(Nd, Nf, f0, df, eps, dtype, batch, o)

    def execute(self, t, y, dy, power, stream=0):
        ls_execute(self.handle, t, y, dy, power, stream)

    def execute_host(self, t, y, dy, power, stream=0):
        ls_execute_host(self.handle, t, y, dy, power, stream)

    @property
    def info(self):
        return ls_get_info(self.handle)

    def stage_ms(self):
        return ls_get_stage_ms(self.handle)

    def launch_counts(self):
        return ls_get_launch_counts(self.handle)

    def workspace_bytes(self):
        return ls_workspace_bytes(self.handle)

    def set_workspace(self, buf, nbytes):
        """Move the plan's large buffers into caller-owned device memory (keep `buf` alive)."""
        ls_set_workspace(self.handle, buf, nbytes)
        self._workspace = buf

    def close(self):
        if self.handle:
            ls_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
