"""ctypes wrapper around oracle.c (plain C, FP64).  TEST INFRASTRUCTURE, not the product.

Argument marshalling only: every number is computed by oracle.c.  See the header of oracle.c for the
passages of PAPER.md each function follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oracle.c"
_LIB = _HERE / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile oracle.c -> liboracle.so with gcc (-O2, OpenMP over cells, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Model(C.Structure):
    _fields_ = [
        ("n_species", C.c_int), ("n_layers", C.c_int),
        ("sizes", C.POINTER(C.c_int)),
        ("weights", C.POINTER(C.c_float)), ("biases", C.POINTER(C.c_float)),
        ("in_mean", C.POINTER(C.c_float)), ("in_std", C.POINTER(C.c_float)),
        ("out_mean", C.POINTER(C.c_float)), ("out_std", C.POINTER(C.c_float)),
        ("lambda_", C.c_double),
        ("nasa_lo", C.POINTER(C.c_double)), ("nasa_hi", C.POINTER(C.c_double)),
        ("T_mid", C.POINTER(C.c_double)), ("W", C.POINTER(C.c_double)),
        ("T_min", C.c_double), ("T_max", C.c_double), ("newton_tol", C.c_double),
        ("newton_max_iter", C.c_int),
        ("T_active", C.c_double),
        ("n_nets", C.c_int),
    ]


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = C.CDLL(str(_LIB))
    d, dp, fp, ip = C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
    lib.oracle_boxcox.restype = d
    lib.oracle_boxcox.argtypes = [d, d]
    lib.oracle_boxcox_inv.restype = d
    lib.oracle_boxcox_inv.argtypes = [d, d]
    lib.oracle_gelu.restype = d
    lib.oracle_gelu.argtypes = [d]
    lib.oracle_mlp_forward.restype = C.c_int
    lib.oracle_mlp_forward.argtypes = [C.c_int, ip, fp, fp, dp, dp]
    lib.oracle_species_cp.restype = d
    lib.oracle_species_cp.argtypes = [dp, d, d]
    lib.oracle_species_h.restype = d
    lib.oracle_species_h.argtypes = [dp, d, d]
    lib.oracle_mixture_h.restype = d
    lib.oracle_mixture_h.argtypes = [C.c_int, dp, d, dp, dp, dp, dp]
    lib.oracle_mixture_cp.restype = d
    lib.oracle_mixture_cp.argtypes = [C.c_int, dp, d, dp, dp, dp, dp]
    lib.oracle_newton_T.restype = d
    lib.oracle_newton_T.argtypes = [C.c_int, dp, d, d, dp, dp, dp, dp, d, d, d, C.c_int, ip, ip]
    lib.oracle_enthalpy_field.restype = C.c_int
    lib.oracle_enthalpy_field.argtypes = [C.c_int64, C.c_int, fp, fp, dp, dp, dp, dp, dp]
    lib.oracle_input_moments.restype = C.c_int
    lib.oracle_input_moments.argtypes = [C.c_int64, C.c_int, fp, fp, fp, d, dp, dp]
    lib.oracle_chem_step.restype = C.c_int
    lib.oracle_chem_step.argtypes = [C.POINTER(_Model), C.c_int64, fp, fp, fp, fp, d, dp, dp, dp,
                                     C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    lib.oracle_derived_outputs.restype = C.c_int
    lib.oracle_derived_outputs.argtypes = [C.c_int64, C.c_int, fp, fp, fp, d, dp, dp, C.POINTER(C.c_int32), dp, dp, dp, dp,
                                           dp, dp, dp, dp, dp, dp]
    _lib = lib
    return lib


_forced_threads: Optional[int] = None


def set_num_threads(n: int) -> None:
    """Sets the OpenMP thread count of the loop over cells (harness plumbing for the 1-thread timing leg of bench.py;
    no arithmetic of the oracle depends on it)."""
    global _forced_threads
    C.CDLL("libgomp.so.1").omp_set_num_threads(C.c_int(max(1, int(n))))
    _forced_threads = max(1, int(n))


def num_threads() -> int:
    """Threads the OpenMP loop over cells will use (set_num_threads, OMP_NUM_THREADS or all cores)."""
    if _forced_threads is not None:
        return _forced_threads
    v = os.environ.get("OMP_NUM_THREADS")
    if v:
        try:
            return max(1, int(v.split(",")[0]))
        except ValueError:
            pass
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: Optional[np.ndarray], ct):
    if a is None:
        return C.cast(None, C.POINTER(ct))
    return a.ctypes.data_as(C.POINTER(ct))


# ------------------------------------------------------------------ scalar pieces
def boxcox(x: float, lam: float) -> float:
    return _load().oracle_boxcox(float(x), float(lam))


def boxcox_inv(y: float, lam: float) -> float:
    return _load().oracle_boxcox_inv(float(y), float(lam))


def gelu(v: float) -> float:
    return _load().oracle_gelu(float(v))


def mlp_forward(sizes: Sequence[int], weights: Sequence[np.ndarray], biases: Sequence[np.ndarray],
                z: np.ndarray) -> np.ndarray:
    """One input vector through the net.  weights[l] is [out][in] FP32, biases[l] is [out] FP32."""
    lib = _load()
    sz = np.ascontiguousarray(sizes, dtype=np.int32)
    L = len(sz) - 1
    assert len(weights) == L and len(biases) == L
    for l in range(L):
        assert tuple(np.shape(weights[l])) == (sz[l + 1], sz[l]), (l, np.shape(weights[l]))
    w = _f32(np.concatenate([_f32(x).ravel() for x in weights]))
    b = _f32(np.concatenate([_f32(x).ravel() for x in biases]))
    zz = _f64(z)
    assert zz.shape == (sz[0],)
    o = np.empty(sz[-1], dtype=np.float64)
    rc = lib.oracle_mlp_forward(L, _p(sz, C.c_int), _p(w, C.c_float), _p(b, C.c_float), _p(zz, C.c_double),
                                _p(o, C.c_double))
    assert rc == 0
    return o


def species_cp(a7: np.ndarray, W: float, T: float) -> float:
    a = _f64(a7)
    assert a.shape == (7,)
    return _load().oracle_species_cp(_p(a, C.c_double), float(W), float(T))


def species_h(a7: np.ndarray, W: float, T: float) -> float:
    a = _f64(a7)
    assert a.shape == (7,)
    return _load().oracle_species_h(_p(a, C.c_double), float(W), float(T))


def _thermo_args(nasa_lo, nasa_hi, T_mid, W):
    lo = _f64(nasa_lo)
    Ns = lo.shape[0]
    assert lo.shape == (Ns, 7)
    hi = None if nasa_hi is None else _f64(nasa_hi)
    tm = None if T_mid is None else _f64(T_mid)
    w = _f64(W)
    assert w.shape == (Ns,)
    if hi is not None:
        assert hi.shape == (Ns, 7)
    if tm is not None:
        assert tm.shape == (Ns,)
    return Ns, lo, hi, tm, w


def mixture_h(Y, T, nasa_lo, nasa_hi, T_mid, W) -> float:
    Ns, lo, hi, tm, w = _thermo_args(nasa_lo, nasa_hi, T_mid, W)
    y = _f64(Y)
    assert y.shape == (Ns,)
    return _load().oracle_mixture_h(Ns, _p(y, C.c_double), float(T), _p(lo, C.c_double), _p(hi, C.c_double),
                                    _p(tm, C.c_double), _p(w, C.c_double))


def mixture_cp(Y, T, nasa_lo, nasa_hi, T_mid, W) -> float:
    Ns, lo, hi, tm, w = _thermo_args(nasa_lo, nasa_hi, T_mid, W)
    y = _f64(Y)
    assert y.shape == (Ns,)
    return _load().oracle_mixture_cp(Ns, _p(y, C.c_double), float(T), _p(lo, C.c_double), _p(hi, C.c_double),
                                     _p(tm, C.c_double), _p(w, C.c_double))


def newton_T(Y, h, T_start, nasa_lo, nasa_hi, T_mid, W, T_min=200.0, T_max=3500.0, tol=1e-6, max_iter=20):
    """Returns (T, iters, converged)."""
    Ns, lo, hi, tm, w = _thermo_args(nasa_lo, nasa_hi, T_mid, W)
    y = _f64(Y)
    assert y.shape == (Ns,)
    it = C.c_int(0)
    cv = C.c_int(0)
    T = _load().oracle_newton_T(Ns, _p(y, C.c_double), float(h), float(T_start), _p(lo, C.c_double),
                                _p(hi, C.c_double), _p(tm, C.c_double), _p(w, C.c_double), float(T_min),
                                float(T_max), float(tol), int(max_iter), C.byref(it), C.byref(cv))
    return T, it.value, bool(cv.value)


# ------------------------------------------------------------------ input-recipe helpers
def enthalpy_field(T, Y, nasa_lo, nasa_hi, T_mid, W) -> np.ndarray:
    """G5: h_i = sum_k Y[k,i] h_k(T_i), FP64, from the FP32 state.  Y is [Ns][n]."""
    Ns, lo, hi, tm, w = _thermo_args(nasa_lo, nasa_hi, T_mid, W)
    t = _f32(T)
    y = _f32(Y)
    n = t.shape[0]
    assert y.shape == (Ns, n)
    out = np.empty(n, dtype=np.float64)
    rc = _load().oracle_enthalpy_field(n, Ns, _p(t, C.c_float), _p(y, C.c_float), _p(lo, C.c_double),
                                       _p(hi, C.c_double), _p(tm, C.c_double), _p(w, C.c_double),
                                       _p(out, C.c_double))
    assert rc == 0
    return out


def input_moments(T, p, Y, lam):
    """G4: mean and population std of [T, p, F(Y_1..Ns)] over the batch (FP64).  Returns (mean, std)."""
    t, pp, y = _f32(T), _f32(p), _f32(Y)
    n = t.shape[0]
    Ns = y.shape[0]
    assert y.shape == (Ns, n) and pp.shape == (n,)
    mean = np.empty(2 + Ns, dtype=np.float64)
    std = np.empty(2 + Ns, dtype=np.float64)
    rc = _load().oracle_input_moments(n, Ns, _p(t, C.c_float), _p(pp, C.c_float), _p(y, C.c_float), float(lam),
                                      _p(mean, C.c_double), _p(std, C.c_double))
    assert rc == 0
    return mean, std


# ------------------------------------------------------------------ the whole step
@dataclass
class OracleModel:
    sizes: Sequence[int]
    weights: Sequence[np.ndarray]   # [out][in] FP32 per layer
    biases: Sequence[np.ndarray]
    in_mean: np.ndarray
    in_std: np.ndarray
    out_mean: np.ndarray
    out_std: np.ndarray
    lam: float
    nasa_lo: np.ndarray
    W: np.ndarray
    nasa_hi: Optional[np.ndarray] = None
    T_mid: Optional[np.ndarray] = None
    T_min: float = 200.0
    T_max: float = 3500.0
    newton_tol: float = 1e-6
    newton_max_iter: int = 20
    T_active: float = 0.0
    # per-species ensemble (R24): sizes ends in 1 and weights / biases are lists over the Ns nets of the
    # per-layer lists of one net
    ensemble: bool = False


@dataclass
class OracleResult:
    T_new: np.ndarray      # [n] f64
    Y_new: np.ndarray      # [Ns][n] f64
    o_raw: np.ndarray      # [Ns][n] f64
    iters: np.ndarray      # [n] i32
    flags: np.ndarray      # [n] i32: bit0 not converged, bit1 degenerate sum, 4 = skipped


class Oracle:
    """Holds the marshalled model; `chem_step` runs O0..O7 for every cell."""

    def __init__(self, m: OracleModel):
        self._sizes = np.ascontiguousarray(m.sizes, dtype=np.int32)
        L = len(self._sizes) - 1
        if m.ensemble:
            Ns = int(self._sizes[0]) - 2
            assert int(self._sizes[-1]) == 1 and len(m.weights) == Ns and len(m.biases) == Ns
            nets_w, nets_b = m.weights, m.biases
        else:
            Ns = int(self._sizes[-1])
            nets_w, nets_b = [m.weights], [m.biases]
        assert int(self._sizes[0]) == Ns + 2
        for ws, bs in zip(nets_w, nets_b):
            for l in range(L):
                assert tuple(np.shape(ws[l])) == (self._sizes[l + 1], self._sizes[l])
                assert tuple(np.shape(bs[l])) == (self._sizes[l + 1],)
        self._w = _f32(np.concatenate([_f32(x).ravel() for ws in nets_w for x in ws]))
        self._b = _f32(np.concatenate([_f32(x).ravel() for bs in nets_b for x in bs]))
        self._im, self._is = _f32(m.in_mean), _f32(m.in_std)
        self._om, self._os = _f32(m.out_mean), _f32(m.out_std)
        assert self._im.shape == (Ns + 2,) and self._is.shape == (Ns + 2,)
        assert self._om.shape == (Ns,) and self._os.shape == (Ns,)
        _, self._lo, self._hi, self._tm, self._W = _thermo_args(m.nasa_lo, m.nasa_hi, m.T_mid, m.W)
        assert self._lo.shape[0] == Ns
        self.n_species = Ns
        self._c = _Model(
            Ns, L, _p(self._sizes, C.c_int), _p(self._w, C.c_float), _p(self._b, C.c_float),
            _p(self._im, C.c_float), _p(self._is, C.c_float), _p(self._om, C.c_float), _p(self._os, C.c_float),
            float(m.lam), _p(self._lo, C.c_double), _p(self._hi, C.c_double), _p(self._tm, C.c_double),
            _p(self._W, C.c_double), float(m.T_min), float(m.T_max), float(m.newton_tol),
            int(m.newton_max_iter), float(m.T_active), Ns if m.ensemble else 1)

    def chem_step(self, T, p, Y, h, dt: float) -> OracleResult:
        lib = _load()
        t, pp, y, hh = _f32(T), _f32(p), _f32(Y), _f32(h)
        n = t.shape[0]
        Ns = self.n_species
        assert y.shape == (Ns, n) and pp.shape == (n,) and hh.shape == (n,)
        T_new = np.empty(n, dtype=np.float64)
        Y_new = np.empty((Ns, n), dtype=np.float64)
        o_raw = np.empty((Ns, n), dtype=np.float64)
        iters = np.empty(n, dtype=np.int32)
        flags = np.empty(n, dtype=np.int32)
        rc = lib.oracle_chem_step(C.byref(self._c), n, _p(t, C.c_float), _p(pp, C.c_float), _p(y, C.c_float),
                                  _p(hh, C.c_float), float(dt), _p(T_new, C.c_double), _p(Y_new, C.c_double),
                                  _p(o_raw, C.c_double), _p(iters, C.c_int32), _p(flags, C.c_int32))
        if rc != 0:
            raise RuntimeError("oracle_chem_step failed (bad arguments or allocation)")
        return OracleResult(T_new, Y_new, o_raw, iters, flags)

    def derived(self, T, p, Y, dt: float, res: OracleResult) -> "OracleDerived":
        """O8 / O9: reaction rates, heat release rate and thermal properties from the results of `chem_step`."""
        lib = _load()
        t, pp, y = _f32(T), _f32(p), _f32(Y)
        n = t.shape[0]
        Ns = self.n_species
        assert y.shape == (Ns, n) and pp.shape == (n,)
        tn, yn, fl = _f64(res.T_new), _f64(res.Y_new), np.ascontiguousarray(res.flags, dtype=np.int32)
        rr = np.empty((Ns, n), dtype=np.float64)
        out = [np.empty(n, dtype=np.float64) for _ in range(5)]
        rc = lib.oracle_derived_outputs(n, Ns, _p(t, C.c_float), _p(pp, C.c_float), _p(y, C.c_float), float(dt),
                                        _p(tn, C.c_double), _p(yn, C.c_double), _p(fl, C.c_int32),
                                        _p(self._lo, C.c_double), _p(self._hi, C.c_double), _p(self._tm, C.c_double),
                                        _p(self._W, C.c_double), _p(rr, C.c_double), *[_p(o, C.c_double) for o in out])
        if rc != 0:
            raise RuntimeError("oracle_derived_outputs failed (bad arguments)")
        return OracleDerived(rr, *out)


@dataclass
class OracleDerived:
    rr: np.ndarray        # [Ns][n] kg/(m3 s)
    hrr: np.ndarray       # [n] W/m3
    cp: np.ndarray        # [n] J/(kg K)
    rmix: np.ndarray      # [n] J/(kg K)
    rho_new: np.ndarray   # [n] kg/m3
    psi: np.ndarray       # [n] s2/m2
