"""Thin ctypes binding of libgpuann.so (include/gpuann.h): argument marshalling only.

Same names as the C ABI.  Device arrays are passed as integer addresses (e.g. `tensor.data_ptr()`), streams as the
integer `torch.cuda.current_stream().cuda_stream`.  The library has no CPU fallback: if libgpuann.so is missing or
cannot be loaded this module raises, and `gpuann_create` fails without an sm_100 device.
"""
from __future__ import annotations

import ctypes as C
import os
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

# GPUANN_DEBUG_SPIN=1 selects the debug build (python -m paper_2402_18858_b200.build --debug), whose mbarrier waits trap
# after 2 s instead of hanging the GPU; same ABI, same kernels otherwise
_LIB_PATH = Path(__file__).resolve().parent / (
    "libgpuann_debug.so" if os.environ.get("GPUANN_DEBUG_SPIN") == "1" else "libgpuann.so")

GPUANN_OK = 0
GPUANN_ERR_INVALID_ARG = 1
GPUANN_ERR_NOT_READY = 2
GPUANN_ERR_UNSUPPORTED = 3
GPUANN_ERR_ALLOC = 4
GPUANN_ERR_CUDA = 5
GPUANN_PRECISION_FP32 = 0
GPUANN_PRECISION_BF16 = 1
GPUANN_PRECISION_FP16 = 2
GPUANN_STATIC_MAX_SPECIES = 64
GPUANN_STATIC_SCRATCH_BYTES = 271392

# every symbol include/gpuann.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "gpuann_default_params", "gpuann_create", "gpuann_load_net", "gpuann_load_net_ensemble", "gpuann_load_thermo", "gpuann_chem_step",
    "gpuann_chem_step_ex",
    "gpuann_chem_step_host", "gpuann_debug_forward", "gpuann_get_stats", "gpuann_reset_stats", "gpuann_enthalpy",
    "gpuann_input_moments", "gpuann_input_moments_static", "gpuann_launch_count", "gpuann_timing_enable", "gpuann_timing_read",
    "gpuann_timing_num_classes", "gpuann_timing_class_name", "gpuann_describe", "gpuann_last_error", "gpuann_destroy",
]


class gpuann_params(C.Structure):
    _fields_ = [
        ("precision", C.c_int), ("newton_max_iter", C.c_int), ("newton_tol", C.c_double),
        ("T_min", C.c_double), ("T_max", C.c_double), ("T_active", C.c_double),
        ("device", C.c_int), ("chunk_cells", C.c_int64),
    ]


class GpuannError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"gpuann status {status}: {message}")
        self.status = status
        self.message = message


_lib = None


def lib() -> C.CDLL:
    """Loads libgpuann.so (built in-tree by `python -m paper_2402_18858_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2402_18858_b200.build"
                           f"{' --debug' if _LIB_PATH.name.endswith('_debug.so') else ''}` (there is no CPU fallback)")
    L = C.CDLL(str(_LIB_PATH))
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    fpp = C.POINTER(C.POINTER(C.c_float))
    L.gpuann_default_params.restype = None
    L.gpuann_default_params.argtypes = [C.POINTER(gpuann_params)]
    L.gpuann_create.restype = C.c_int
    L.gpuann_create.argtypes = [C.POINTER(gpuann_params), C.POINTER(vp)]
    L.gpuann_load_net.restype = C.c_int
    L.gpuann_load_net.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_int), fpp, fpp, vp, vp, vp, vp, dbl]
    L.gpuann_load_net_ensemble.restype = C.c_int
    L.gpuann_load_net_ensemble.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_int), fpp, fpp, vp, vp, vp, vp, dbl]
    L.gpuann_load_thermo.restype = C.c_int
    L.gpuann_load_thermo.argtypes = [vp, C.c_int, vp, vp, vp, vp]
    L.gpuann_chem_step.restype = C.c_int
    L.gpuann_chem_step.argtypes = [vp, i64, vp, vp, vp, vp, dbl, vp]
    L.gpuann_chem_step_ex.restype = C.c_int
    L.gpuann_chem_step_ex.argtypes = [vp, i64, vp, vp, vp, vp, dbl, vp, vp]
    L.gpuann_chem_step_host.restype = C.c_int
    L.gpuann_chem_step_host.argtypes = [vp, i64, vp, vp, vp, vp, dbl]
    L.gpuann_debug_forward.restype = C.c_int
    L.gpuann_debug_forward.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    L.gpuann_get_stats.restype = C.c_int
    L.gpuann_get_stats.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
    L.gpuann_reset_stats.restype = C.c_int
    L.gpuann_reset_stats.argtypes = [vp]
    L.gpuann_enthalpy.restype = C.c_int
    L.gpuann_enthalpy.argtypes = [vp, i64, vp, vp, vp, vp]
    L.gpuann_input_moments.restype = C.c_int
    L.gpuann_input_moments.argtypes = [vp, i64, C.c_int, vp, vp, vp, dbl, vp, vp, vp]
    L.gpuann_input_moments_static.restype = C.c_int
    L.gpuann_input_moments_static.argtypes = [vp, i64, C.c_int, vp, vp, vp, dbl, vp, vp, vp]
    L.gpuann_launch_count.restype = i64
    L.gpuann_launch_count.argtypes = [vp]
    L.gpuann_timing_enable.restype = C.c_int
    L.gpuann_timing_enable.argtypes = [vp, C.c_int]
    L.gpuann_timing_read.restype = C.c_int
    L.gpuann_timing_read.argtypes = [vp, C.c_int, C.POINTER(dbl), C.POINTER(i64)]
    L.gpuann_timing_num_classes.restype = C.c_int
    L.gpuann_timing_num_classes.argtypes = []
    L.gpuann_timing_class_name.restype = C.c_char_p
    L.gpuann_timing_class_name.argtypes = [C.c_int]
    L.gpuann_describe.restype = C.c_int
    L.gpuann_describe.argtypes = [vp, C.POINTER(i64), C.POINTER(C.c_char_p)]
    L.gpuann_last_error.restype = C.c_char_p
    L.gpuann_last_error.argtypes = [vp]
    L.gpuann_destroy.restype = C.c_int
    L.gpuann_destroy.argtypes = [vp]
    _lib = L
    return L


def gpuann_last_error(ctx: Optional[int]) -> str:
    m = lib().gpuann_last_error(C.c_void_p(ctx) if ctx else None)
    return m.decode() if m else ""


def _check(status: int, ctx: Optional[int]):
    if status != GPUANN_OK:
        raise GpuannError(status, gpuann_last_error(ctx))


def gpuann_default_params() -> gpuann_params:
    p = gpuann_params()
    lib().gpuann_default_params(C.byref(p))
    return p


def gpuann_create(params: Optional[gpuann_params] = None) -> int:
    out = C.c_void_p(0)
    st = lib().gpuann_create(C.byref(params) if params is not None else None, C.byref(out))
    _check(st, None)
    return out.value


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else C.c_void_p(a.ctypes.data)


def gpuann_load_net(ctx: int, n_species: int, sizes: Sequence[int], weights: Sequence[np.ndarray],
                    biases: Sequence[np.ndarray], in_mean, in_std, out_mean, out_std, lam: float) -> None:
    sz = np.ascontiguousarray(sizes, dtype=np.int32)
    Lw = len(sz) - 1
    ws = [_f32(w) for w in weights]
    bs = [_f32(b) for b in biases]
    if len(ws) != Lw or len(bs) != Lw:
        raise ValueError("len(weights) and len(biases) must be len(sizes) - 1")
    for l in range(Lw):
        if ws[l].shape != (sz[l + 1], sz[l]) or bs[l].shape != (sz[l + 1],):
            raise ValueError(f"layer {l}: weights must be [out][in] = {(sz[l + 1], sz[l])}, biases [out]")
    fp = C.POINTER(C.c_float)
    wp = (fp * Lw)(*[w.ctypes.data_as(fp) for w in ws])
    bp = (fp * Lw)(*[b.ctypes.data_as(fp) for b in bs])
    im, isd, om, osd = _f32(in_mean), _f32(in_std), _f32(out_mean), _f32(out_std)
    st = lib().gpuann_load_net(ctx, int(n_species), Lw, sz.ctypes.data_as(C.POINTER(C.c_int)), wp, bp,
                               _ptr(im), _ptr(isd), _ptr(om), _ptr(osd), float(lam))
    _check(st, ctx)


def gpuann_load_net_ensemble(ctx: int, n_species: int, sizes: Sequence[int], weights, biases, in_mean, in_std, out_mean,
                             out_std, lam: float) -> None:
    """weights[k][l], biases[k][l]: layer l of the net of species k (every net has the shape `sizes`, sizes[-1] == 1)."""
    sz = np.ascontiguousarray(sizes, dtype=np.int32)
    Lw = len(sz) - 1
    if len(weights) != n_species or len(biases) != n_species:
        raise ValueError("one list of layers per species")
    ws = [[_f32(w) for w in net] for net in weights]
    bs = [[_f32(b) for b in net] for net in biases]
    for k in range(n_species):
        if len(ws[k]) != Lw or len(bs[k]) != Lw:
            raise ValueError("every net needs len(sizes) - 1 layers")
        for l in range(Lw):
            if ws[k][l].shape != (sz[l + 1], sz[l]) or bs[k][l].shape != (sz[l + 1],):
                raise ValueError(f"net {k} layer {l}: weights must be [out][in] = {(sz[l + 1], sz[l])}, biases [out]")
    fp = C.POINTER(C.c_float)
    wp = (fp * (Lw * n_species))(*[w.ctypes.data_as(fp) for net in ws for w in net])
    bp = (fp * (Lw * n_species))(*[b.ctypes.data_as(fp) for net in bs for b in net])
    im, isd, om, osd = _f32(in_mean), _f32(in_std), _f32(out_mean), _f32(out_std)
    st = lib().gpuann_load_net_ensemble(ctx, int(n_species), Lw, sz.ctypes.data_as(C.POINTER(C.c_int)), wp, bp,
                                        _ptr(im), _ptr(isd), _ptr(om), _ptr(osd), float(lam))
    _check(st, ctx)


def gpuann_load_thermo(ctx: int, n_species: int, nasa_lo, nasa_hi, T_mid, W) -> None:
    lo, hi, tm, w = _f64(nasa_lo), _f64(nasa_hi), _f64(T_mid), _f64(W)
    if lo.shape != (n_species, 7) or w.shape != (n_species,):
        raise ValueError("nasa_lo must be [Ns][7] and W [Ns]")
    st = lib().gpuann_load_thermo(ctx, int(n_species), _ptr(lo), _ptr(hi), _ptr(tm), _ptr(w))
    _check(st, ctx)


def gpuann_chem_step(ctx: int, n_cells: int, T: int, p: int, Y: int, h: int, dt: float, stream: int = 0) -> None:
    _check(lib().gpuann_chem_step(ctx, int(n_cells), T, p, Y, h, float(dt), stream or None), ctx)


class gpuann_step_outputs(C.Structure):
    _fields_ = [("rr", C.c_void_p), ("hrr", C.c_void_p), ("cp", C.c_void_p), ("rho", C.c_void_p), ("psi", C.c_void_p)]


def gpuann_chem_step_ex(ctx: int, n_cells: int, T: int, p: int, Y: int, h: int, dt: float, stream: int = 0, *,
                        rr: int = 0, hrr: int = 0, cp: int = 0, rho: int = 0, psi: int = 0) -> None:
    """gpuann_chem_step plus the optional outputs (device addresses; 0 = not computed)."""
    out = gpuann_step_outputs(rr or None, hrr or None, cp or None, rho or None, psi or None)
    _check(lib().gpuann_chem_step_ex(ctx, int(n_cells), T, p, Y, h, float(dt), C.byref(out), stream or None), ctx)


def gpuann_chem_step_host(ctx: int, n_cells: int, T: int, p: int, Y: int, h: int, dt: float) -> None:
    """T, p, Y, h are HOST addresses (e.g. pinned torch tensors' data_ptr(), numpy arrays' ctypes.data)."""
    _check(lib().gpuann_chem_step_host(ctx, int(n_cells), T, p, Y, h, float(dt)), ctx)


def gpuann_debug_forward(ctx: int, n_cells: int, T: int, p: int, Y: int, o_raw: int, stream: int = 0) -> None:
    _check(lib().gpuann_debug_forward(ctx, int(n_cells), T, p, Y, o_raw, stream or None), ctx)


def gpuann_get_stats(ctx: int):
    """Returns (n_active, n_not_converged, n_degenerate)."""
    a, b, c = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    _check(lib().gpuann_get_stats(ctx, C.byref(a), C.byref(b), C.byref(c)), ctx)
    return a.value, b.value, c.value


def gpuann_reset_stats(ctx: int) -> None:
    _check(lib().gpuann_reset_stats(ctx), ctx)


def gpuann_enthalpy(ctx: int, n_cells: int, T: int, Y: int, h_out: int, stream: int = 0) -> None:
    _check(lib().gpuann_enthalpy(ctx, int(n_cells), T, Y, h_out, stream or None), ctx)


def gpuann_input_moments(ctx: int, n_cells: int, n_species: int, T: int, p: int, Y: int, lam: float, stream: int = 0):
    """Returns (mean, std) as float64 arrays of 2 + Ns entries."""
    mean = np.empty(n_species + 2, dtype=np.float64)
    std = np.empty(n_species + 2, dtype=np.float64)
    st = lib().gpuann_input_moments(ctx, int(n_cells), int(n_species), T, p, Y, float(lam), _ptr(mean), _ptr(std),
                                    stream or None)
    _check(st, ctx)
    return mean, std


def gpuann_input_moments_static(ctx: int, n_cells: int, n_species: int, T: int, p: int, Y: int, lam: float, stream: int = 0):
    """gpuann_input_moments for callers that must not allocate device memory (scratch in a static device array of the
    library; at most GPUANN_STATIC_MAX_SPECIES species).  Returns (mean, std) as float64 arrays of 2 + Ns entries."""
    mean = np.empty(n_species + 2, dtype=np.float64)
    std = np.empty(n_species + 2, dtype=np.float64)
    st = lib().gpuann_input_moments_static(ctx, int(n_cells), int(n_species), T, p, Y, float(lam), _ptr(mean), _ptr(std),
                                           stream or None)
    _check(st, ctx)
    return mean, std


def gpuann_launch_count(ctx: int) -> int:
    return int(lib().gpuann_launch_count(ctx))


def gpuann_timing_enable(ctx: int, enable: bool) -> None:
    _check(lib().gpuann_timing_enable(ctx, 1 if enable else 0), ctx)


def gpuann_timing_read(ctx: int) -> dict:
    """Returns {class name: (summed device ms, launches)} for the classes that launched since the last enable/read."""
    n = lib().gpuann_timing_num_classes()
    ms = (C.c_double * n)()
    cnt = (C.c_int64 * n)()
    _check(lib().gpuann_timing_read(ctx, n, ms, cnt), ctx)
    return {lib().gpuann_timing_class_name(i).decode(): (ms[i], cnt[i]) for i in range(n) if cnt[i] > 0}


def gpuann_describe(ctx: int):
    """Returns (issued_mac_per_cell, variant)."""
    mac = C.c_int64(0)
    name = C.c_char_p()
    st = lib().gpuann_describe(ctx, C.byref(mac), C.byref(name))
    _check(st, ctx)
    return mac.value, (name.value.decode() if name.value else "")


def gpuann_destroy(ctx: Optional[int]) -> None:
    if ctx:
        lib().gpuann_destroy(ctx)
