"""ctypes binding of libs2b200.so -- same names as include/s2b200.h, argument marshalling only.

Host arrays are numpy (fp64 / int32, C-contiguous); device arrays are torch CUDA tensors
(passed as raw pointers).  PyTorch supplies device memory (its caching allocator, through the
s2_allocator callbacks) and the stream (torch.cuda.current_stream()); every step of the hot
path runs in the library's CUDA kernels.  There is no CPU fallback: if the library cannot be
loaded, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libs2b200.so")
HEADER_PATH = os.path.join(os.path.dirname(_PKG), "include", "s2b200.h")
TEST_HEADER_PATH = os.path.join(os.path.dirname(_PKG), "include", "s2b200_test.h")   # tuning overrides, microbenchmarks

S2_FP64, S2_DS, S2_FP32 = 0, 1, 2
S2_WANT_NN, S2_WANT_NGB = 1, 2
S2_OK, S2_EINVAL, S2_ERANGE, S2_ENOMEM, S2_ECUDA, S2_ESTATE, S2_EOVERFLOW = 0, -1, -2, -3, -4, -5, -6

_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class s2_allocator(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


class S2Error(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: {s2_strerror(code)} ({code}){' -- ' + detail if detail else ''}")


_lib = None


def header_symbols(which: str = "all") -> list[str]:
    """Every function include/s2b200.h (the product ABI) and include/s2b200_test.h (test hooks) declare;
    which = "product" | "test" | "all"."""
    paths = {"product": [HEADER_PATH], "test": [TEST_HEADER_PATH], "all": [HEADER_PATH, TEST_HEADER_PATH]}[which]
    names = set()
    for path in paths:
        src = re.sub(r"/\*.*?\*/", "", open(path).read(), flags=re.S)
        names.update(re.findall(r"\b(s2_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def lib() -> C.CDLL:
    """Loads libs2b200.so (building it in-tree with nvcc if it is absent).  Raises if it cannot."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from .build import build
        build()
    L = C.CDLL(LIB_PATH)
    vp, ip, dp = C.c_void_p, C.c_void_p, C.c_void_p
    sig = {
        "s2_open": (C.c_int, [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(s2_allocator), vp]),
        "s2_close": (C.c_int, [vp]),
        "s2_set_stream": (C.c_int, [vp, vp]),
        "s2_synchronize": (C.c_int, [vp]),
        "s2_set_j": (C.c_int, [vp, C.c_int, ip, ip] + [dp] * 8),
        "s2_commit_j": (C.c_int, [vp]),
        "s2_commit_j_device": (C.c_int, [vp, C.c_int, ip, ip] + [dp] * 8),
        "s2_predict": (C.c_int, [vp, C.c_double, C.c_int]),
        "s2_set_j_range": (C.c_int, [vp, C.c_int, C.c_int]),
        "s2_calc_ilist": (C.c_int, [vp, C.c_int, ip, dp, C.c_double, C.c_uint]),
        "s2_calc_ilist_device": (C.c_int, [vp, C.c_int, ip, dp, C.c_double, C.c_uint]),
        "s2_calc_ilist_batch": (C.c_int, [vp, C.c_int, ip, ip, dp, C.c_double, C.c_uint]),
        "s2_calc_explicit": (C.c_int, [vp, C.c_int, ip, dp, dp, dp, dp, C.c_double, C.c_uint]),
        "s2_get_results": (C.c_int, [vp, C.c_int, dp, dp, dp, dp, ip, dp, ip]),
        "s2_get_results_device": (C.c_int, [vp, C.c_int, dp, dp, dp, dp, ip, dp, ip]),
        "s2_get_neighbours": (C.c_int, [vp, C.c_int, C.c_int, C.POINTER(C.c_int), ip]),
        "s2_get_neighbours_csr": (C.c_int, [vp, C.c_int, vp, ip, C.c_longlong]),
        "s2_get_neighbours_csr_device": (C.c_int, [vp, C.c_int, C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_longlong)]),
        "s2_get_csr_timing": (C.c_int, [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]),
        "s2_get_predicted_j": (C.c_int, [vp, C.c_int, C.c_int, dp, dp, dp]),
        "s2_get_j": (C.c_int, [vp, C.c_int, C.c_int, ip, dp, dp, dp]),
        "s2_set_tuning": (C.c_int, [vp, C.c_int, C.c_int]),
        "s2_last_launch_info": (C.c_int, [vp, C.POINTER(C.c_int * 10)]),
        "s2_test_ds_ops": (C.c_int, [vp, C.c_int, dp, dp, dp]),
        "s2_kernel_launches": (C.c_longlong, [vp]),
        "s2_enable_timing": (C.c_int, [vp, C.c_int]),
        "s2_get_timing": (C.c_int, [vp, C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_float)]),
        "s2_fp32_fixup_count": (C.c_int, [vp, C.POINTER(C.c_int)]),
        "s2_bts_small_stats": (C.c_int, [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_double)]),
        "s2_bts_small_profile": (C.c_int, [vp, C.c_int, C.POINTER(C.c_longlong)]),
        "s2_peak_fma": (C.c_int, [vp, C.c_int, C.c_int, C.POINTER(C.c_double)]),
        "s2_hop_latency": (C.c_int, [vp, C.c_int, C.c_int, C.POINTER(C.c_double)]),
        "s2_time_host_roundtrip": (C.c_int, [vp, C.c_int, C.POINTER(C.c_int), C.c_double, C.c_uint, C.c_int, C.POINTER(C.c_double)]),
        "s2_bts_open": (C.c_int, [C.POINTER(vp), vp, C.c_int] + [C.c_double] * 5 + [C.c_int, C.c_double]),
        "s2_bts_close": (C.c_int, [vp]),
        "s2_bts_init": (C.c_int, [vp, dp, dp, dp]),
        "s2_bts_run": (C.c_int, [vp, C.c_double, C.c_longlong, C.c_int, C.POINTER(C.c_longlong)]),
        "s2_bts_get_state": (C.c_int, [vp, C.POINTER(C.c_double)] + [dp] * 7),
        "s2_bts_stats": (C.c_int, [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong),
                                   C.POINTER(C.c_longlong), C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_longlong)]),
        "s2_bts_get_history": (C.c_int, [vp, C.c_longlong, C.c_int, ip]),
        "s2_forces_noalloc": (C.c_int, [C.c_int, vp, C.c_int, dp, dp, dp, ip, C.c_int, ip, C.c_double, dp, dp, dp]),
        "s2_noalloc_limits": (C.c_int, [C.POINTER(C.c_int), C.POINTER(C.c_longlong)]),
        "s2_strerror": (C.c_char_p, [C.c_int]),
        "s2_last_cuda_error": (C.c_char_p, [vp]),
        "s2_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


# ---- marshalling helpers ------------------------------------------------------------------

def _h(a, dtype, shape_tail=None, n=None, name="array"):
    """host numpy array -> pointer (None passes NULL)."""
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=dtype)
    if n is not None:
        want = (n,) + (shape_tail or ())
        if a.shape != want:
            raise ValueError(f"{name}: expected shape {want}, got {a.shape}")
    return a.ctypes.data_as(C.c_void_p), a


def _d(t, dtype_name, numel=None, name="tensor"):
    """torch CUDA tensor -> raw device pointer (None passes NULL)."""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise ValueError(f"{name}: need a contiguous CUDA tensor")
    if str(t.dtype) != "torch." + dtype_name:
        raise ValueError(f"{name}: need dtype {dtype_name}, got {t.dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _check(rc: int, where: str, ctx=None, ok=(S2_OK,)):
    if rc in ok:
        return rc
    detail = ""
    if rc == S2_ECUDA and ctx is not None:
        detail = (lib().s2_last_cuda_error(ctx) or b"").decode()
    raise S2Error(rc, where, detail)


class _TorchAllocator:
    """s2_allocator backed by torch's CUDA caching allocator (uint8 tensors kept alive by pointer)."""

    def __init__(self, device: int):
        import torch
        self._torch = torch
        self._device = torch.device("cuda", device)
        self._live: dict[int, object] = {}
        self._alloc_cb = _ALLOC_FN(self._alloc)
        self._free_cb = _FREE_FN(self._free)
        self.struct = s2_allocator(self._alloc_cb, self._free_cb, None)
        self.bytes_live = 0

    def _alloc(self, nbytes, _user):
        try:
            t = self._torch.empty(int(nbytes), dtype=self._torch.uint8, device=self._device)
        except Exception:
            return None
        self._live[t.data_ptr()] = t
        self.bytes_live += int(nbytes)
        return t.data_ptr()

    def _free(self, ptr, _user):
        t = self._live.pop(ptr, None)
        if t is not None:
            self.bytes_live -= t.numel()


# ---- the calls, one per header entry --------------------------------------------------------

class s2_ctx:
    """Opaque context handle plus the Python objects that must outlive it."""

    def __init__(self, handle, allocator, order, precision, device):
        self.handle, self.allocator = handle, allocator
        self.order, self.precision, self.device = order, precision, device
        self._keep = []          # device tensors referenced by the last ASYNC call


def s2_version() -> str:
    return lib().s2_version().decode()


def s2_strerror(code: int) -> str:
    return lib().s2_strerror(int(code)).decode()


def s2_open(device: int = 0, order: int = 4, precision: int = S2_FP64, nj_capacity: int = 1, ngb_cap: int = 256,
            use_torch_allocator: bool = True, stream=None) -> s2_ctx:
    L = lib()
    import torch
    if not torch.cuda.is_available():
        raise S2Error(S2_ECUDA, "s2_open", "no CUDA device visible; this library has no CPU fallback")
    alloc = _TorchAllocator(device) if use_torch_allocator else None
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    h = C.c_void_p()
    rc = L.s2_open(C.byref(h), device, order, precision, nj_capacity, ngb_cap,
                   C.byref(alloc.struct) if alloc else None, C.c_void_p(stream))
    _check(rc, "s2_open")
    return s2_ctx(h, alloc, order, precision, device)


def s2_close(ctx: s2_ctx):
    if ctx.handle:
        _check(lib().s2_close(ctx.handle), "s2_close")
        ctx.handle = None
        ctx._keep = []


def s2_set_stream(ctx, stream):
    _check(lib().s2_set_stream(ctx.handle, C.c_void_p(stream)), "s2_set_stream", ctx.handle)


def s2_synchronize(ctx):
    _check(lib().s2_synchronize(ctx.handle), "s2_synchronize", ctx.handle)
    ctx._keep = []


def s2_set_j(ctx, address, ident, t, mass, pos, vel, acc=None, jerk=None, snap=None, crackle=None):
    n = int(np.asarray(address).shape[0])
    i32, f64 = np.int32, np.float64
    keep = []
    args = []
    for a, dt, tail, nm in ((address, i32, (), "address"), (ident, i32, (), "id"), (t, f64, (), "t"), (mass, f64, (), "mass"),
                            (pos, f64, (3,), "pos"), (vel, f64, (3,), "vel"), (acc, f64, (3,), "acc"),
                            (jerk, f64, (3,), "jerk"), (snap, f64, (3,), "snap"), (crackle, f64, (3,), "crackle")):
        p, arr = _h(a, dt, tail, n, nm)
        args.append(p)
        keep.append(arr)
    _check(lib().s2_set_j(ctx.handle, n, *args), "s2_set_j", ctx.handle)


def s2_commit_j(ctx):
    _check(lib().s2_commit_j(ctx.handle), "s2_commit_j", ctx.handle)


def s2_commit_j_device(ctx, d_address, d_id, d_t, d_mass, d_pos, d_vel, d_acc=None, d_jerk=None, d_snap=None, d_crackle=None):
    n = d_address.numel()
    args = [_d(d_address, "int32", n, "address"), _d(d_id, "int32", n, "id"), _d(d_t, "float64", n, "t"),
            _d(d_mass, "float64", n, "mass")]
    for tns, nm in ((d_pos, "pos"), (d_vel, "vel"), (d_acc, "acc"), (d_jerk, "jerk"), (d_snap, "snap"), (d_crackle, "crackle")):
        args.append(_d(tns, "float64", 3 * n, nm))
    ctx._keep = [d_address, d_id, d_t, d_mass, d_pos, d_vel, d_acc, d_jerk, d_snap, d_crackle]
    _check(lib().s2_commit_j_device(ctx.handle, n, *args), "s2_commit_j_device", ctx.handle)


def s2_predict(ctx, t: float, nj: int):
    _check(lib().s2_predict(ctx.handle, float(t), int(nj)), "s2_predict", ctx.handle)


def s2_set_j_range(ctx, first: int, count: int):
    _check(lib().s2_set_j_range(ctx.handle, int(first), int(count)), "s2_set_j_range", ctx.handle)


def s2_calc_ilist(ctx, i_address, h2=None, eps2: float = 0.0, flags: int = 0):
    ni = int(np.asarray(i_address).shape[0])
    pa, ka = _h(i_address, np.int32, (), ni, "i_address")
    ph, kh = _h(h2, np.float64, (), ni, "h2")
    _check(lib().s2_calc_ilist(ctx.handle, ni, pa, ph, float(eps2), int(flags)), "s2_calc_ilist", ctx.handle)


def s2_calc_ilist_batch(ctx, lists, h2_lists=None, eps2: float = 0.0, flags: int = 0) -> np.ndarray:
    """k i-lists in one launch sequence; returns the offsets (k + 1) of each list's results in the next s2_get_results."""
    ni = np.array([len(x) for x in lists], dtype=np.int32)
    cat = np.ascontiguousarray(np.concatenate([np.asarray(x, dtype=np.int32) for x in lists]))
    h2 = None if h2_lists is None else np.ascontiguousarray(np.concatenate([np.asarray(x, dtype=np.float64) for x in h2_lists]))
    _check(lib().s2_calc_ilist_batch(ctx.handle, len(lists), ni.ctypes.data_as(C.c_void_p), cat.ctypes.data_as(C.c_void_p),
                                     None if h2 is None else h2.ctypes.data_as(C.c_void_p), float(eps2), int(flags)),
           "s2_calc_ilist_batch", ctx.handle)
    return np.concatenate([[0], np.cumsum(ni)])


def s2_calc_ilist_device(ctx, d_i_address, d_h2=None, eps2: float = 0.0, flags: int = 0):
    ni = d_i_address.numel()
    ctx._keep = [d_i_address, d_h2]
    _check(lib().s2_calc_ilist_device(ctx.handle, ni, _d(d_i_address, "int32", ni, "i_address"),
                                      _d(d_h2, "float64", ni, "h2"), float(eps2), int(flags)),
           "s2_calc_ilist_device", ctx.handle)


def s2_calc_explicit(ctx, ident, pos, vel, acc=None, h2=None, eps2: float = 0.0, flags: int = 0):
    ni = int(np.asarray(ident).shape[0])
    f64 = np.float64
    pi, k0 = _h(ident, np.int32, (), ni, "id")
    pp, k1 = _h(pos, f64, (3,), ni, "pos")
    pv, k2 = _h(vel, f64, (3,), ni, "vel")
    pa, k3 = _h(acc, f64, (3,), ni, "acc")
    ph, k4 = _h(h2, f64, (), ni, "h2")
    _check(lib().s2_calc_explicit(ctx.handle, ni, pi, pp, pv, pa, ph, float(eps2), int(flags)),
           "s2_calc_explicit", ctx.handle)


def s2_get_results(ctx, ni: int, allow_overflow: bool = True) -> dict:
    """Returns dict(acc, jerk, snap, pot, nn_id, nn_r2, ngb_count, overflow)."""
    out = dict(acc=np.empty((ni, 3)), jerk=np.empty((ni, 3)), snap=np.empty((ni, 3)) if ctx.order == 6 else None,
               pot=np.empty(ni), nn_id=np.empty(ni, np.int32), nn_r2=np.empty(ni), ngb_count=np.empty(ni, np.int32))
    p = lambda a: None if a is None else a.ctypes.data_as(C.c_void_p)
    rc = lib().s2_get_results(ctx.handle, ni, p(out["acc"]), p(out["jerk"]), p(out["snap"]), p(out["pot"]),
                              p(out["nn_id"]), p(out["nn_r2"]), p(out["ngb_count"]))
    _check(rc, "s2_get_results", ctx.handle, ok=(S2_OK, S2_EOVERFLOW) if allow_overflow else (S2_OK,))
    out["overflow"] = rc == S2_EOVERFLOW
    ctx._keep = []
    return out


def s2_get_results_device(ctx, ni: int, acc=None, jerk=None, snap=None, pot=None, nn_id=None, nn_r2=None, ngb_count=None):
    """Unpacks the results of the last s2_calc_* into the given torch CUDA tensors (any may be None).  ASYNC."""
    args = [_d(acc, "float64", 3 * ni, "acc"), _d(jerk, "float64", 3 * ni, "jerk"), _d(snap, "float64", 3 * ni, "snap"),
            _d(pot, "float64", ni, "pot"), _d(nn_id, "int32", ni, "nn_id"), _d(nn_r2, "float64", ni, "nn_r2"),
            _d(ngb_count, "int32", ni, "ngb_count")]
    ctx._keep = ctx._keep + [acc, jerk, snap, pot, nn_id, nn_r2, ngb_count]
    _check(lib().s2_get_results_device(ctx.handle, int(ni), *args), "s2_get_results_device", ctx.handle)


def s2_get_neighbours(ctx, i: int, cap: int) -> np.ndarray:
    lst = np.empty(max(cap, 1), np.int32)
    n = C.c_int(0)
    rc = lib().s2_get_neighbours(ctx.handle, int(i), int(cap), C.byref(n), lst.ctypes.data_as(C.c_void_p))
    _check(rc, "s2_get_neighbours", ctx.handle, ok=(S2_OK, S2_EOVERFLOW))
    return lst[:n.value].copy()


class _DeviceView:
    """Zero-copy view of library-owned device memory (valid until the next s2_calc_* / s2_close)."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


def s2_get_neighbours_csr_device(ctx, ni: int):
    """(offsets, list, total): torch views of the device-resident CSR (int64 offsets of the whole last call, int32
    addresses); total = offsets[ni].  No list data crosses the host link."""
    import torch
    po, pl, tot = C.c_void_p(), C.c_void_p(), C.c_longlong()
    rc = lib().s2_get_neighbours_csr_device(ctx.handle, int(ni), C.byref(po), C.byref(pl), C.byref(tot))
    _check(rc, "s2_get_neighbours_csr_device", ctx.handle, ok=(S2_OK, S2_EOVERFLOW))
    dev = torch.device("cuda", ctx.device)
    off = torch.as_tensor(_DeviceView(po.value, ni + 1, "<i8"), device=dev)
    lst = torch.as_tensor(_DeviceView(pl.value, max(int(tot.value), 1), "<i4"), device=dev)[:int(tot.value)]
    return off, lst, int(tot.value)


def s2_get_neighbours_csr(ctx, ni: int, list_cap: int | None = None):
    """(offsets, list) on the host.  One read-back: the library compacts the lists on the device once per force call;
    the sizing query below only reads the 8-byte total."""
    off = np.zeros(ni + 1, np.int64)
    if list_cap is None:
        po, pl, tot = C.c_void_p(), C.c_void_p(), C.c_longlong()
        rc = lib().s2_get_neighbours_csr_device(ctx.handle, int(ni), C.byref(po), C.byref(pl), C.byref(tot))
        _check(rc, "s2_get_neighbours_csr", ctx.handle, ok=(S2_OK, S2_EOVERFLOW))
        list_cap = int(tot.value)
    lst = np.empty(max(list_cap, 1), np.int32)
    rc = lib().s2_get_neighbours_csr(ctx.handle, ni, off.ctypes.data_as(C.c_void_p), lst.ctypes.data_as(C.c_void_p), list_cap)
    _check(rc, "s2_get_neighbours_csr", ctx.handle, ok=(S2_OK, S2_EOVERFLOW))
    return off, lst[:off[ni]]


def s2_get_csr_timing(ctx) -> dict:
    a, b = C.c_float(), C.c_float()
    _check(lib().s2_get_csr_timing(ctx.handle, C.byref(a), C.byref(b)), "s2_get_csr_timing", ctx.handle)
    return dict(scan_ms=a.value, fill_ms=b.value)


def s2_get_predicted_j(ctx, first: int, n: int):
    pos, vel = np.empty((n, 3)), np.empty((n, 3))
    acc = np.empty((n, 3)) if ctx.order == 6 else None
    p = lambda a: None if a is None else a.ctypes.data_as(C.c_void_p)
    _check(lib().s2_get_predicted_j(ctx.handle, first, n, p(pos), p(vel), p(acc)), "s2_get_predicted_j", ctx.handle)
    return pos, vel, acc


def s2_get_j(ctx, first: int, n: int):
    ident, t, mass, pos = np.empty(n, np.int32), np.empty(n), np.empty(n), np.empty((n, 3))
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    _check(lib().s2_get_j(ctx.handle, first, n, p(ident), p(t), p(mass), p(pos)), "s2_get_j", ctx.handle)
    return ident, t, mass, pos


def s2_set_tuning(ctx, key: int, value: int):
    _check(lib().s2_set_tuning(ctx.handle, key, value), "s2_set_tuning", ctx.handle)


def s2_last_launch_info(ctx) -> dict:
    arr = (C.c_int * 10)()
    _check(lib().s2_last_launch_info(ctx.handle, C.byref(arr)), "s2_last_launch_info", ctx.handle)
    keys = ("S", "lanes_per_i", "warp_columns", "grid", "threads", "smem", "reduced", "ctas_per_sm", "i_per_thread",
            "cluster")
    return dict(zip(keys, list(arr)))


def s2_kernel_launches(ctx) -> int:
    return int(lib().s2_kernel_launches(ctx.handle))


def s2_enable_timing(ctx, on: bool = True):
    _check(lib().s2_enable_timing(ctx.handle, int(on)), "s2_enable_timing", ctx.handle)


def s2_get_timing(ctx) -> dict:
    a, b, c = C.c_float(), C.c_float(), C.c_float()
    _check(lib().s2_get_timing(ctx.handle, C.byref(a), C.byref(b), C.byref(c)), "s2_get_timing", ctx.handle)
    return dict(predict_ms=a.value, force_ms=b.value, reduce_ms=c.value)


def s2_time_host_roundtrip(ctx, i_address, eps2: float = 0.0, flags: int = 0, reps: int = 1000) -> float:
    """Microseconds per (s2_calc_ilist + s2_get_results) as timed inside the library (no binding in the loop)."""
    ia = np.ascontiguousarray(i_address, dtype=np.int32)
    v = C.c_double()
    _check(lib().s2_time_host_roundtrip(ctx.handle, ia.size, ia.ctypes.data_as(C.POINTER(C.c_int)), float(eps2), int(flags),
                                        int(reps), C.byref(v)), "s2_time_host_roundtrip", ctx.handle)
    return v.value


def s2_fp32_fixup_count(ctx) -> int:
    n = C.c_int()
    _check(lib().s2_fp32_fixup_count(ctx.handle, C.byref(n)), "s2_fp32_fixup_count", ctx.handle)
    return n.value


def s2_hop_latency(ctx, ctas: int, iters: int = 2000) -> float:
    v = C.c_double()
    _check(lib().s2_hop_latency(ctx.handle, int(ctas), int(iters), C.byref(v)), "s2_hop_latency", ctx.handle)
    return v.value


def s2_peak_fma(ctx, kind: int, iters: int = 2000) -> float:
    v = C.c_double()
    _check(lib().s2_peak_fma(ctx.handle, kind, iters, C.byref(v)), "s2_peak_fma", ctx.handle)
    return v.value


def s2_test_ds_ops(ctx, a, b) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    if a.ndim != 1 or a.shape != b.shape:
        raise ValueError("s2_test_ds_ops: a and b must be 1-D arrays of equal length")
    out = np.empty((a.shape[0], 8), np.float64)
    _check(lib().s2_test_ds_ops(ctx.handle, a.shape[0], a.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p),
                                out.ctypes.data_as(C.c_void_p)), "s2_test_ds_ops", ctx.handle)
    return out


# ---- block-time-step integrator (include/s2b200.h, s2_bts_*) ------------------------------------------------

class s2_bts:
    def __init__(self, handle, ctx, n):
        self.handle, self.ctx, self.n = handle, ctx, n


def s2_bts_open(ctx, n: int, eps2: float, eta: float, eta_start: float, dt_max: float = 2.0 ** -3, dt_min: float = 2.0 ** -40,
                averaged: bool = False, eta4: float = 0.01):
    h = C.c_void_p()
    _check(lib().s2_bts_open(C.byref(h), ctx.handle, int(n), float(eps2), float(eta), float(eta_start), float(dt_max),
                             float(dt_min), int(averaged), float(eta4)), "s2_bts_open", ctx.handle)
    return s2_bts(h, ctx, int(n))


def s2_bts_close(b):
    if b.handle:
        _check(lib().s2_bts_close(b.handle), "s2_bts_close")
        b.handle = None


def s2_bts_init(b, mass, pos, vel):
    pm, k0 = _h(mass, np.float64, (), b.n, "mass")
    pp, k1 = _h(pos, np.float64, (3,), b.n, "pos")
    pv, k2 = _h(vel, np.float64, (3,), b.n, "vel")
    _check(lib().s2_bts_init(b.handle, pm, pp, pv), "s2_bts_init", b.ctx.handle)


def s2_bts_run(b, t_end: float, max_block_steps: int = 1 << 62, time_device: bool = False) -> int:
    done = C.c_longlong()
    _check(lib().s2_bts_run(b.handle, float(t_end), int(max_block_steps), int(time_device), C.byref(done)), "s2_bts_run",
           b.ctx.handle)
    return done.value


def s2_bts_get_state(b) -> dict:
    n = b.n
    out = dict(t=np.empty(n), dt=np.empty(n), pos=np.empty((n, 3)), vel=np.empty((n, 3)), acc=np.empty((n, 3)),
               jerk=np.empty((n, 3)), pot=np.empty(n))
    tm = C.c_double()
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    _check(lib().s2_bts_get_state(b.handle, C.byref(tm), p(out["t"]), p(out["dt"]), p(out["pos"]), p(out["vel"]), p(out["acc"]),
                                  p(out["jerk"]), p(out["pot"])), "s2_bts_get_state", b.ctx.handle)
    out["time"] = tm.value
    return out


def s2_bts_stats(b) -> dict:
    tm, tn, wall, dev = C.c_double(), C.c_double(), C.c_double(), C.c_double()
    nn = C.c_int()
    bs, ps, ts = C.c_longlong(), C.c_longlong(), C.c_longlong()
    _check(lib().s2_bts_stats(b.handle, C.byref(tm), C.byref(tn), C.byref(nn), C.byref(bs), C.byref(ps), C.byref(wall), C.byref(dev),
                              C.byref(ts)), "s2_bts_stats")
    return dict(time=tm.value, t_next=tn.value, n_next=nn.value, block_steps=bs.value, particle_steps=ps.value,
                wall_ms=wall.value, device_ms=dev.value, timed_steps=ts.value)


def s2_bts_small_stats(b) -> dict:
    ln, st, ms = C.c_longlong(), C.c_longlong(), C.c_double()
    _check(lib().s2_bts_small_stats(b.handle, C.byref(ln), C.byref(st), C.byref(ms)), "s2_bts_small_stats")
    return dict(launches=ln.value, steps=st.value, device_ms=ms.value)


_SMALL_PARTS = ("headers", "records", "sweep", "rows_out", "rows_in", "corrector", "barrier", "predict", "publish")


def s2_bts_small_profile(b, on: int = 1) -> dict:
    """Switches the in-kernel profile of the small-step kernel on (1 + index of the CTA to watch) or off (0); returns the
    sums so far (SM cycles per part)."""
    out = (C.c_longlong * 10)()
    _check(lib().s2_bts_small_profile(b.handle, int(on), out), "s2_bts_small_profile", b.ctx.handle)
    d = {k: int(out[i]) for i, k in enumerate(_SMALL_PARTS)}
    d["steps"] = int(out[9])
    return d


def s2_bts_get_history(b, first: int = 0, count: int | None = None) -> np.ndarray:
    if count is None:
        count = s2_bts_stats(b)["block_steps"] - first
    out = np.empty(max(count, 1), np.int32)
    _check(lib().s2_bts_get_history(b.handle, int(first), int(count), out.ctypes.data_as(C.c_void_p)), "s2_bts_get_history")
    return out[:count]


# ---- allocation-free entry point (include/s2b200.h, s2_forces_noalloc) -----------------------------------

def s2_noalloc_limits() -> dict:
    n, b = C.c_int(), C.c_longlong()
    _check(lib().s2_noalloc_limits(C.byref(n), C.byref(b)), "s2_noalloc_limits")
    return dict(max_ni=n.value, scratch_bytes=b.value)


def s2_forces_noalloc(d_pos, d_vel, d_mass, d_id, d_i_address, eps2, d_acc, d_jerk, d_pot, device: int = 0, stream=None):
    """acc, jerk, pot (torch CUDA tensors the caller owns) of the listed i-particles; the library allocates nothing."""
    nj, ni = d_mass.numel(), d_i_address.numel()
    if stream is None:
        import torch
        stream = torch.cuda.current_stream(device).cuda_stream
    rc = lib().s2_forces_noalloc(int(device), C.c_void_p(stream), nj, _d(d_pos, "float64", 3 * nj, "pos"),
                                 _d(d_vel, "float64", 3 * nj, "vel"), _d(d_mass, "float64", nj, "mass"), _d(d_id, "int32", nj, "id"),
                                 ni, _d(d_i_address, "int32", ni, "i_address"), float(eps2), _d(d_acc, "float64", 3 * ni, "acc"),
                                 _d(d_jerk, "float64", 3 * ni, "jerk"), _d(d_pot, "float64", ni, "pot"))
    if rc == S2_ERANGE:
        raise S2Error(rc, "s2_forces_noalloc", f"n_i = {ni} exceeds the fixed maximum of {s2_noalloc_limits()['max_ni']} "
                                               f"(static scratch); use s2_calc_ilist for larger i-lists")
    _check(rc, "s2_forces_noalloc")


def s2_last_cuda_error(ctx) -> str:
    return (lib().s2_last_cuda_error(ctx.handle) or b"").decode()
