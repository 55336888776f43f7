"""Shared plumbing of the `-m gpu` parity tests: build the seeded problem, derive (h, normalisation) with the
oracle, run the CUDA path through the C ABI (ctypes binding) and the oracle on the same FP32 inputs.

Tolerances (BASELINE.json north_star):
  FP32 path: |Y - Y_ref| <= 1e-5 |Y_ref| + 1e-10, max |T - T_ref| <= 1e-3 K
  BF16 path: per output column ||o - o_ref||_2 <= 2e-2 ||o_ref||_2 and max|o - o_ref| <= 2e-2 max|o_ref|,
             max |T - T_ref| <= 0.5 K, |Y - Y_ref| <= 2e-3 |Y_ref| + 1e-10 (R18), and -- the gates that bite --
             on the UPDATE dY = Y_new - Y_in/sum(Y_in), per species over the batch (R18'):
             ||Y - Y_ref||_2 <= 2e-2 ||dY_ref||_2 and max|Y - Y_ref| <= 2e-2 max|dY_ref| (+ a floor of 2 FP32 ulps);
             RR_k likewise against RR_ref,k; HRR per cell within rho cp 0.5 K / dt and 3e-2 of ||HRR_ref||_2 (R22')
  both:      max |sum_k Y_new - 1| <= 1e-6 (FP64 sum of the stored FP32 values)
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

import oracle
from paper_2402_18858_b200 import binding as B
from paper_2402_18858_b200 import inputs as I


@dataclass
class Prepared:
    prob: I.Problem
    h: np.ndarray        # [n] f32
    in_mean: np.ndarray  # [2+Ns] f32
    in_std: np.ndarray
    model: oracle.OracleModel


def prepare(cfg: I.Config, n: Optional[int] = None, seed: Optional[int] = None, mutate=None, **over) -> Prepared:
    """`mutate(prob)` may edit the drawn problem in place (state, thermo, out_mean, ...) before the derived inputs
    h (G5) and mu_in / sigma_in (G4) are computed from it."""
    # tiny batches take their normalisation statistics from a 4,096-cell batch of the same seed, then keep n cells
    n_gen = None if n is None else max(int(n), 4096)
    prob = I.make_problem(cfg, n=n_gen, seed=seed)
    if mutate is not None:
        mutate(prob)
    st, th = prob.state, prob.thermo
    mean, std = oracle.input_moments(st.T, st.p, st.Y, cfg.lam)                                       # G4
    if n is not None and n_gen != n:
        st = I.State(st.T[:n].copy(), st.p[:n].copy(), np.ascontiguousarray(st.Y[:, :n]))
        prob = I.Problem(prob.cfg, int(n), st, th, prob.net, prob.out_mean, prob.out_std)
    h = oracle.enthalpy_field(st.T, st.Y, th.nasa_lo, th.nasa_hi, th.T_mid, th.W).astype(np.float32)  # G5
    in_mean, in_std = mean.astype(np.float32), std.astype(np.float32)
    model = oracle.OracleModel(
        sizes=prob.net.sizes, weights=prob.net.weights, biases=prob.net.biases, in_mean=in_mean, in_std=in_std,
        out_mean=prob.out_mean, out_std=prob.out_std, lam=cfg.lam, nasa_lo=th.nasa_lo, W=th.W, nasa_hi=th.nasa_hi,
        T_mid=th.T_mid, T_min=cfg.T_min, T_max=cfg.T_max, newton_tol=cfg.newton_tol,
        newton_max_iter=over.get("newton_max_iter", cfg.newton_max_iter), T_active=over.get("T_active", cfg.T_active))
    return Prepared(prob, h, in_mean, in_std, model)


def make_ctx(pr: Prepared, precision: Optional[int] = None, chunk_cells: int = 0) -> int:
    cfg = pr.prob.cfg
    prm = B.gpuann_default_params()
    prm.precision = cfg.precision if precision is None else precision
    prm.newton_max_iter = pr.model.newton_max_iter
    prm.newton_tol = pr.model.newton_tol
    prm.T_min, prm.T_max = pr.model.T_min, pr.model.T_max
    prm.T_active = pr.model.T_active
    prm.chunk_cells = chunk_cells
    ctx = B.gpuann_create(prm)
    try:
        B.gpuann_load_net(ctx, cfg.n_species, pr.prob.net.sizes, pr.prob.net.weights, pr.prob.net.biases,
                          pr.in_mean, pr.in_std, pr.prob.out_mean, pr.prob.out_std, cfg.lam)
        th = pr.prob.thermo
        B.gpuann_load_thermo(ctx, cfg.n_species, th.nasa_lo, th.nasa_hi, th.T_mid, th.W)
    except Exception:
        B.gpuann_destroy(ctx)
        raise
    return ctx


@dataclass
class GpuResult:
    T_new: np.ndarray   # [n] f32
    Y_new: np.ndarray   # [Ns][n] f32
    o_raw: Optional[np.ndarray]
    stats: tuple


def run_gpu(ctx: int, pr: Prepared, T=None, p=None, Y=None, h=None, want_raw: bool = True, dt: Optional[float] = None,
            use_stream: bool = True) -> GpuResult:
    import torch
    st = pr.prob.state
    T = st.T if T is None else T
    p = st.p if p is None else p
    Y = st.Y if Y is None else Y
    h = pr.h if h is None else h
    n = int(T.shape[0])
    Ns = pr.prob.cfg.n_species
    dev = torch.device("cuda:0")
    dT = torch.from_numpy(np.ascontiguousarray(T)).to(dev)
    dp = torch.from_numpy(np.ascontiguousarray(p)).to(dev)
    dY = torch.from_numpy(np.ascontiguousarray(Y)).to(dev)
    dh = torch.from_numpy(np.ascontiguousarray(h)).to(dev)
    stream = torch.cuda.current_stream().cuda_stream if use_stream else 0
    o_raw = None
    if want_raw:
        dO = torch.full((Ns, max(n, 1)), float("nan"), dtype=torch.float32, device=dev)
        B.gpuann_debug_forward(ctx, n, dT.data_ptr(), dp.data_ptr(), dY.data_ptr(), dO.data_ptr(), stream)
        torch.cuda.synchronize()
        o_raw = dO.cpu().numpy()[:, :n]
    B.gpuann_reset_stats(ctx)
    B.gpuann_chem_step(ctx, n, dT.data_ptr(), dp.data_ptr(), dY.data_ptr(), dh.data_ptr(),
                       pr.prob.cfg.dt if dt is None else dt, stream)
    torch.cuda.synchronize()
    stats = B.gpuann_get_stats(ctx)
    return GpuResult(dT.cpu().numpy(), dY.cpu().numpy(), o_raw, stats)


def run_oracle(pr: Prepared, T=None, p=None, Y=None, h=None, dt: Optional[float] = None):
    st = pr.prob.state
    o = oracle.Oracle(pr.model)
    ref = o.chem_step(st.T if T is None else T, st.p if p is None else p, st.Y if Y is None else Y,
                      pr.h if h is None else h, pr.prob.cfg.dt if dt is None else dt)
    ref.Y_in = st.Y if Y is None else Y     # the update gates (R18') are stated on Y_new - Y_in / sum Y_in
    return ref


def run_oracle_all_active(pr: Prepared):
    """The oracle with the active-cell test off (gpuann_debug_forward computes every cell, skipped or not)."""
    import dataclasses
    m = dataclasses.replace(pr.model, T_active=0.0)
    st = pr.prob.state
    return oracle.Oracle(m).chem_step(st.T, st.p, st.Y, pr.h, pr.prob.cfg.dt)


# ------------------------------------------------------------------ the comparisons
def check_sumY(Y_new: np.ndarray, mask=None):
    s = Y_new.astype(np.float64).sum(axis=0)
    if mask is not None:
        s = s[mask]
    dev = np.abs(s - 1.0).max() if s.size else 0.0
    assert dev <= 1e-6, f"max |sum Y - 1| = {dev:.3e} > 1e-6"
    return dev


def check_fp32(g: GpuResult, ref, mask=None):
    sel = slice(None) if mask is None else mask
    Yg, Yr = g.Y_new.astype(np.float64)[:, sel], ref.Y_new[:, sel]
    err = np.abs(Yg - Yr)
    tol = 1e-5 * np.abs(Yr) + 1e-10
    worst = (err / tol).max() if err.size else 0.0
    assert worst <= 1.0, f"Y_new: max err/tol = {worst:.3f} (tol = 1e-5 |Y| + 1e-10)"
    dT = np.abs(g.T_new.astype(np.float64)[sel] - ref.T_new[sel])
    assert (dT.max() if dT.size else 0.0) <= 1e-3, f"T_new: max |dT| = {dT.max():.3e} K > 1e-3 K"
    return worst, (dT.max() if dT.size else 0.0)


def check_raw_bf16(o_gpu: np.ndarray, o_ref: np.ndarray, mask=None, gate: float = 2e-2):
    sel = slice(None) if mask is None else mask
    og, orf = o_gpu.astype(np.float64)[:, sel], o_ref[:, sel]
    assert np.isfinite(og).all(), "raw output has non-finite entries"
    d = og - orf
    l2 = np.sqrt((d * d).sum(axis=1)) / np.sqrt((orf * orf).sum(axis=1))
    mx = np.abs(d).max(axis=1) / np.abs(orf).max(axis=1)
    assert l2.max() <= gate, f"raw output: column rel-L2 {l2.max():.3e} > {gate:g}"
    assert mx.max() <= gate, f"raw output: column max|d|/max|ref| {mx.max():.3e} > {gate:g}"
    return l2.max(), mx.max()


def check_T_bf16(g: GpuResult, ref, mask=None):
    sel = slice(None) if mask is None else mask
    dT = np.abs(g.T_new.astype(np.float64)[sel] - ref.T_new[sel])
    m = dT.max() if dT.size else 0.0
    assert m <= 0.5, f"T_new: max |dT| = {m:.3e} K > 0.5 K"
    return m


def check_Y_bf16(g: GpuResult, ref, mask=None, lam: float = 0.1):
    """Element-wise Y_new on the BF16 path (R18):
        |Y - Y_ref| <= 2e-3 max(1, 0.19 / Y_ref^lambda) |Y_ref| + 1e-10.
    The raw-output error propagates as dY/Y = d(dy) / Y^lambda with d(dy) = dt sigma_out d(o); at the configs'
    sigma_out dt <= 2e-2 and |d(o)| <~ 1e-2 that is <= 1.1e-3 wherever Y^lambda >= 0.19.  For lambda = 0.1 (all five
    configs) Y^lambda < 0.19 only below Y = 6e-8, where the absolute floor is the larger term, so the gate IS
    2e-3 |Y_ref| + 1e-10 there; for another lambda (the branch tests) the factor widens it by the same sensitivity.
    SURVEY.md Appendix A measured <= 2e-4 relative."""
    sel = slice(None) if mask is None else mask
    Yg, Yr = g.Y_new.astype(np.float64)[:, sel], ref.Y_new[:, sel]
    err = np.abs(Yg - Yr)
    with np.errstate(divide="ignore"):
        sens = np.maximum(1.0, 0.19 / np.power(np.abs(Yr), lam)) if lam > 0 else 1.0
    sens = np.where(np.isfinite(sens), sens, 1.0)
    tol = 2e-3 * sens * np.abs(Yr) + 1e-10
    worst = (err / tol).max() if err.size else 0.0
    assert worst <= 1.0, f"Y_new (BF16 path): max err/tol = {worst:.3f} (tol = 2e-3 s |Y| + 1e-10)"
    return worst


def update_of(Y_new: np.ndarray, Y_in: np.ndarray) -> np.ndarray:
    """dY = Y_new - max(Y_in, 0) / sum_k max(Y_in, 0): what the step changes (S1 reads Y < 0 as 0, R2; S6 renormalises)."""
    Yc = np.maximum(np.asarray(Y_in, dtype=np.float64), 0.0)
    return np.asarray(Y_new, dtype=np.float64) - Yc / Yc.sum(axis=0, keepdims=True)


def norms_against(d: np.ndarray, ref: np.ndarray, floor: np.ndarray, gate: float):
    """Per row k (a species) over the batch: ||d_k||_2 / (gate ||ref_k||_2 + ||floor_k||_2) and
    max|d_k| / (gate max|ref_k| + max floor_k); rows whose allowance is 0 must have d = 0.  Returns the two worst ratios."""
    if d.size == 0:
        return 0.0, 0.0
    a2 = gate * np.sqrt((ref * ref).sum(axis=1)) + np.sqrt((floor * floor).sum(axis=1))
    am = gate * np.abs(ref).max(axis=1) + floor.max(axis=1)
    e2, em = np.sqrt((d * d).sum(axis=1)), np.abs(d).max(axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        r2 = np.where(a2 > 0, e2 / a2, np.where(e2 > 0, np.inf, 0.0))
        rm = np.where(am > 0, em / am, np.where(em > 0, np.inf, 0.0))
    return float(r2.max()), float(rm.max())


def check_Y_update(g: GpuResult, ref, mask=None, gate: float = 2e-2):
    """The gate on Y_new that bites on the tensor path (R18').  north_star states 2e-2 on the raw output o (R13:
    per output column, rel-L2 and max against the column's largest entry).  The species update is, to first order, LINEAR
    in o (dY_k ~ Y_k^(1-lambda) dt sigma_k o_k, then the renormalisation), so the same 2e-2 in the same two norms is what
    that statement allows on the UPDATE dY_k = Y_new,k - Y_in,k / sum Y_in, per species k over the batch:
        ||Y_k - Y_ref,k||_2 <= 2e-2 ||dY_ref,k||_2 + ||floor_k||_2,   max|Y_k - Y_ref,k| <= 2e-2 max|dY_ref,k| + max floor_k
    with floor = 2.4e-7 |Y_ref| + 1e-30 = 2 FP32 ulps: the tensor path renormalises in FP32 (sum, reciprocal, product, store:
    S6), which is all that is left where the update vanishes (the degenerate-sum fallback returns max(Y,0)/sum: dY = 0);
    it is ~1 % of the allowance at a typical update of 1e-3 |Y|.  (R18's element-wise 2e-3 |Y| is 1-2 x the update itself
    on these inputs: it bounds blow-ups, not the update.)  Returns the worse of the two ratios."""
    Y_in = getattr(ref, "Y_in", None)
    assert Y_in is not None, "the oracle result carries no Y_in (use gpu_common.run_oracle / subset, or set ref.Y_in)"
    sel = slice(None) if mask is None else mask
    act = (ref.flags[sel] & 4) == 0          # skipped cells are compared bit for bit elsewhere
    Yg, Yr = g.Y_new.astype(np.float64)[:, sel][:, act], ref.Y_new[:, sel][:, act]
    dref = update_of(Yr, np.asarray(Y_in)[:, sel][:, act])
    r2, rm = norms_against(Yg - Yr, dref, 2.4e-7 * np.abs(Yr) + 1e-30, gate)
    assert r2 <= 1.0, f"Y_new update: per-species L2 error / allowance = {r2:.3f} (allowance = {gate:g} ||dY_ref||_2 + store floor)"
    assert rm <= 1.0, f"Y_new update: per-species max error / allowance = {rm:.3f} (allowance = {gate:g} max|dY_ref| + store floor)"
    return max(r2, rm)


def check_all_bf16(g: GpuResult, ref, mask=None, raw_ref=None, lam: float = 0.1):
    """Every BF16-path gate at once; returns a dict of the worst figures."""
    l2, mx = check_raw_bf16(g.o_raw, (ref if raw_ref is None else raw_ref).o_raw)
    return {"raw_l2": l2, "raw_max": mx, "dT": check_T_bf16(g, ref, mask), "Y": check_Y_bf16(g, ref, mask, lam),
            "dY": check_Y_update(g, ref, mask), "sumY": check_sumY(g.Y_new, mask)}


def sample_indices(n, rng, extra, pool=None):
    """SURVEY.md 8(d) subset S: first 4,096, last 4,096 and `extra` seed-drawn cells (of `pool` if given)."""
    pool = np.arange(n) if pool is None else np.asarray(pool)
    head, tail = pool[:4096], pool[-4096:]
    mid = rng.choice(pool, size=min(extra, pool.size), replace=False)
    return np.unique(np.concatenate([head, tail, mid]))


def subset(pr: Prepared, g: GpuResult, idx):
    """(oracle result, GPU result) restricted to the cells idx -- the oracle computes only those cells."""
    st = pr.prob.state
    ref = run_oracle(pr, T=st.T[idx], p=st.p[idx], Y=np.ascontiguousarray(st.Y[:, idx]), h=pr.h[idx])
    sub = GpuResult(g.T_new[idx], np.ascontiguousarray(g.Y_new[:, idx]),
                    None if g.o_raw is None else np.ascontiguousarray(g.o_raw[:, idx]), g.stats)
    return ref, sub


# ------------------------------------------------------------------ gpuann_chem_step_ex (O8 / O9; R19-R22)
def run_gpu_ex(ctx: int, pr: Prepared, which=("rr", "hrr", "cp", "rho", "psi")):
    """One gpuann_chem_step_ex on the prepared state.  Returns (GpuResult, dict of the requested outputs); outputs are
    pre-filled with NaN so that an entry the library did not write is visible."""
    import torch
    st = pr.prob.state
    n = int(st.T.shape[0])
    Ns = pr.prob.cfg.n_species
    dev = torch.device("cuda:0")
    dT, dp, dY, dh = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (st.T, st.p, st.Y, pr.h))
    bufs = {k: torch.full((Ns, n) if k == "rr" else (n,), float("nan"), dtype=torch.float32, device=dev) for k in which}
    stream = torch.cuda.current_stream().cuda_stream
    B.gpuann_reset_stats(ctx)
    B.gpuann_chem_step_ex(ctx, n, dT.data_ptr(), dp.data_ptr(), dY.data_ptr(), dh.data_ptr(), pr.prob.cfg.dt, stream,
                          **{k: v.data_ptr() for k, v in bufs.items()})
    torch.cuda.synchronize()
    return (GpuResult(dT.cpu().numpy(), dY.cpu().numpy(), None, B.gpuann_get_stats(ctx)),
            {k: v.cpu().numpy().astype(np.float64) for k, v in bufs.items()})


def check_ex(pr: Prepared, ref, ex: dict, bf16: bool, lam: float = 0.1, tensor_scale: float = 1.0):
    """Element-wise gates on the extra outputs, derived from the gates on Y_new and T_new (R22):
    RR_k = rho (Y_new,k - Y_k)/dt inherits tol(Y_new,k) rho/dt (+ FP32 output rounding); HRR = -sum h_k RR_k inherits
    sum_k |h_k| tol(RR_k); cp, rho, psi move with T_new (0.5 K / 1e-3 K) and Y_new (2e-3 / 1e-5).  Those forms are as wide
    as RR and HRR themselves on the tensor path; the gates that bite are R22' below (RR in the update's norms, HRR through
    the tolerance on T).  tensor_scale = 2^-3 for GPUANN_PRECISION_FP16 (R23) scales the R22' gates."""
    st, th, cfg = pr.prob.state, pr.prob.thermo, pr.prob.cfg
    der = oracle.Oracle(pr.model).derived(st.T, st.p, st.Y, cfg.dt, ref)
    act = ref.flags != 4
    Yr = ref.Y_new
    if bf16:
        with np.errstate(divide="ignore"):
            sens = np.maximum(1.0, 0.19 / np.power(np.abs(Yr), lam)) if lam > 0 else np.ones_like(Yr)
        sens = np.where(np.isfinite(sens), sens, 1.0)
        tolY = 2e-3 * sens * np.abs(Yr) + 1e-10
        rel_T = 0.5 / ref.T_new + 2e-3
    else:
        tolY = 1e-5 * np.abs(Yr) + 1e-10
        rel_T = 1e-3 / ref.T_new + 1e-5
    Yc = np.maximum(st.Y.astype(np.float64), 0.0)
    rho_in = st.p.astype(np.float64) / (8314.46261815324 * st.T.astype(np.float64) * (Yc / th.W[:, None]).sum(axis=0))
    tolRR = rho_in / cfg.dt * (tolY + 2e-7 * np.abs(st.Y.astype(np.float64))) + 1e-5 * np.abs(der.rr)
    out = {}
    gate = (2e-2 if bf16 else 1e-4) * tensor_scale
    if "rr" in ex:
        err = np.abs(ex["rr"] - der.rr)[:, act]
        assert np.isfinite(ex["rr"][:, act]).all()
        out["rr"] = (err / tolRR[:, act]).max()
        assert out["rr"] <= 1.0, f"RR: max err/tol = {out['rr']:.3f}"
        assert np.isnan(ex["rr"][:, ~act]).all(), "RR of a skipped cell was written"
        # R22': RR_k = rho dY_k / dt is the update itself, so it takes the update's gate (check_Y_update) in the same two
        # norms, per species over the batch; floor = the FP32 rounding of Y_new and Y_in (rho/dt 2e-7 |Y|) and of RR
        floor = (rho_in / cfg.dt * 2e-7 * np.abs(st.Y.astype(np.float64)) + 1e-6 * np.abs(der.rr))[:, act]
        r2, rm = norms_against((ex["rr"] - der.rr)[:, act], der.rr[:, act], floor, gate)
        out["rr_update"] = max(r2, rm)
        assert r2 <= 1.0, f"RR: per-species L2 error / allowance = {r2:.3f} (allowance = {gate:g} ||RR_ref||_2 + floor)"
        assert rm <= 1.0, f"RR: per-species max error / allowance = {rm:.3f} (allowance = {gate:g} max|RR_ref| + floor)"
    if "hrr" in ex:
        hk = np.empty_like(Yr)
        for k in range(Yr.shape[0]):
            lo = th.nasa_lo[k]
            hi = lo if th.nasa_hi is None else th.nasa_hi[k]
            a = np.where((ref.T_new < (th.T_mid[k] if th.T_mid is not None else np.inf))[:, None], lo[None, :], hi[None, :])
            T = ref.T_new
            hk[k] = 8314.46261815324 / th.W[k] * (a[:, 0] * T + a[:, 1] * T ** 2 / 2 + a[:, 2] * T ** 3 / 3
                                                  + a[:, 3] * T ** 4 / 4 + a[:, 4] * T ** 5 / 5 + a[:, 5])
        # h_k itself moves with T_new: |dh_k| <= cp_k dT, folded in through rel_T on the sum of |h_k RR_k|
        tolH = (np.abs(hk) * tolRR).sum(axis=0) + rel_T * (np.abs(hk) * np.abs(der.rr)).sum(axis=0)
        err = np.abs(ex["hrr"] - der.hrr)[act]
        out["hrr"] = (err / tolH[act]).max()
        assert out["hrr"] <= 1.0, f"HRR: max err/tol = {out['hrr']:.3f}"
        assert np.isnan(ex["hrr"][~act]).all()
        # R22': HRR dt / rho = - sum_k h_k(T_new) dY_k = the sensible-enthalpy change ~ cp (T_new - T), so an HRR error e is
        # a temperature error e dt / (rho cp).  Per cell it must stay inside the tolerance stated on T (0.5 K; FP32 path
        # 1e-3 K; FP16 x 2^-3) -- tolH above sums |h_k| of terms that cancel and is 2-6 x |HRR| itself -- and over the
        # batch ||HRR - HRR_ref||_2 <= 3e-2 ||HRR_ref||_2 (the update's 2e-2 plus the T gate's share).  The absolute floor
        # is the FP32 rounding of the terms that cancel in the sum.
        dT_tol = (0.5 if bf16 else 1e-3) * tensor_scale
        floorH = (np.abs(hk) * (rho_in / cfg.dt * 2e-7 * np.abs(st.Y.astype(np.float64)) + 1e-6 * np.abs(der.rr))).sum(axis=0)
        tolH_T = rho_in * der.cp / cfg.dt * dT_tol + floorH
        out["hrr_T"] = (err / tolH_T[act]).max() if err.size else 0.0
        assert out["hrr_T"] <= 1.0, f"HRR: max err / (rho cp {dT_tol:g} K / dt) = {out['hrr_T']:.3f}"
        gH = (3e-2 if bf16 else 1e-4) * tensor_scale
        e2 = np.sqrt((err * err).sum())
        a2 = gH * np.sqrt((der.hrr[act] ** 2).sum()) + np.sqrt((floorH[act] ** 2).sum())
        out["hrr_l2"] = float(e2 / a2) if a2 > 0 else (0.0 if e2 == 0 else np.inf)
        assert out["hrr_l2"] <= 1.0, f"HRR: batch L2 error / allowance = {out['hrr_l2']:.3f} (allowance = {gH:g} ||HRR_ref||_2 + floor)"
    for name, want in (("cp", der.cp), ("rho", der.rho_new), ("psi", der.psi)):
        if name in ex:
            err = np.abs(ex[name] - want)[act] / (rel_T[act] * np.abs(want[act]))
            out[name] = err.max()
            assert out[name] <= 1.0, f"{name}: max err/tol = {out[name]:.3f}"
            assert np.isnan(ex[name][~act]).all()
    return out


def check_all_fp16(g: GpuResult, ref, lam: float = 0.1):
    """GPUANN_PRECISION_FP16 (R23): every BF16-path gate scaled by 2^-3, the ratio of the unit roundoffs of FP16
    (2^-11) and BF16 (2^-8): raw output 2.5e-3 per column (rel-L2 and max/colmax), T 0.0625 K, Y 2.5e-4 s |Y| + 1e-10."""
    l2, mx = check_raw_bf16(g.o_raw, ref.o_raw, gate=2.5e-3)
    dT = np.abs(g.T_new.astype(np.float64) - ref.T_new).max()
    assert dT <= 0.0625, f"T_new (FP16 path): max |dT| = {dT:.3e} K > 0.0625 K"
    Yg, Yr = g.Y_new.astype(np.float64), ref.Y_new
    with np.errstate(divide="ignore"):
        sens = np.maximum(1.0, 0.19 / np.power(np.abs(Yr), lam))
    sens = np.where(np.isfinite(sens), sens, 1.0)
    worst = (np.abs(Yg - Yr) / (2.5e-4 * sens * np.abs(Yr) + 1e-10)).max()
    assert worst <= 1.0, f"Y_new (FP16 path): max err/tol = {worst:.3f}"
    return {"raw_l2": l2, "raw_max": mx, "dT": dT, "Y": worst, "dY": check_Y_update(g, ref, gate=2.5e-3),
            "sumY": check_sumY(g.Y_new)}
