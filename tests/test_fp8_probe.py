"""`-m "not gpu"`: error-budget probe for the FP8 half of SURVEY.md 8(f) NEXT-4 (PAPER.md:56 half-precision inference, :228 /
:236 "optimizing the inference framework ... future work"; VERDICT r2 task 6: measure first, then build or close).

Question: can layers 2 and 3 of the tensor path (97 % of the MACs) run on `tcgen05.mma kind::f8f6f4` with e4m3 operands
and stay inside north_star's tolerances (2e-2 on the raw output per column, 0.5 K on T)?  This is a numpy emulation of
that path -- NOT the CUDA path and not the oracle: weights of layers 2-3 quantised to e4m3 with one scale per output
channel, their input activations quantised to e4m3 with one scale per 128-cell tile (amax / 448), products accumulated
exactly (FP64 stands in for the FP32 accumulator), layers 1 and 4 and every other activation in BF16 as today.  The same
emulation with BF16 everywhere calibrates it against the GPU's measured figures (profiles/r03_gates.md: raw rel-L2
3.6e-3 .. 6.9e-3, |dT| <= 0.13 K).  The result of each variant goes through S4-S7 written out in numpy FP64 (checked
against the oracle on the oracle's own raw output first) and is compared with the FP64 oracle.

Outcome (asserted below, printed with -s, NEXT-4), c1 at 16,384 cells / c2 at 4,096 cells:
    BF16 emulation        raw rel-L2 4.9e-3 / 5.0e-3   max|dT| 0.09 / 0.04 K   update error / R18' allowance 0.26 / 0.31
    e4m3 in layers 2-3    raw rel-L2 8.7e-2 / 8.8e-2   max|dT| 1.5  / 0.77 K   4.5 / 4.8
    e4m3 in layer 2 only  raw rel-L2 5.4e-2 / 6.6e-2   max|dT| 1.4  / 0.80 K   3.1 / 3.1
e4m3 (3 mantissa bits, unit roundoff 2^-4 against BF16's 2^-9) misses 2e-2 on the raw output by 2.7-4.4 x and the 0.5 K on
T, so no GPUANN_PRECISION_FP8 is built: it could not pass this repository's parity gates.
"""
import numpy as np
import pytest
from scipy.special import erf

from paper_2402_18858_b200 import inputs as I

import gpu_common as G

RU = 8314.46261815324


def q_e4m3(x):
    """Round to the nearest e4m3 value (4 exponent bits, bias 7, 3 mantissa bits, max 448, subnormals of 2^-9), ties to even,
    saturating."""
    a = np.minimum(np.abs(x), 448.0)
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -20)))
    step = 2.0 ** (np.maximum(e, -6.0) - 3.0)
    return np.sign(x) * np.minimum(np.round(a / step) * step, 448.0)


def bf16(x):
    return I.round_to_bf16(np.asarray(x, dtype=np.float32)).astype(np.float64)


def gelu(v):
    return 0.5 * v * (1.0 + erf(v / np.sqrt(2.0)))


def forward(pr, fp8_layers, tile=128):
    """Raw network output [Ns][n] of the emulated tensor path; layers in `fp8_layers` (0-based) take e4m3 operands."""
    st, cfg, net = pr.prob.state, pr.prob.cfg, pr.prob.net
    Yc = np.maximum(st.Y.astype(np.float64), 0.0)
    y = (Yc ** cfg.lam - 1.0) / cfg.lam
    x = np.concatenate([st.T[None, :].astype(np.float64), st.p[None, :].astype(np.float64), y], axis=0)
    a = bf16((x - pr.in_mean[:, None].astype(np.float64)) / pr.in_std[:, None].astype(np.float64)).T     # [n][D]
    L = len(net.weights)
    for l in range(L):
        W, b = net.weights[l].astype(np.float64), net.biases[l].astype(np.float64)
        if l in fp8_layers:
            sw = np.abs(W).max(axis=1, keepdims=True) / 448.0
            sw[sw == 0] = 1.0
            Wq = q_e4m3(W / sw)
            n = a.shape[0]
            pad = (-n) % tile
            at = np.pad(a, ((0, pad), (0, 0))).reshape(-1, tile, a.shape[1])
            sa = np.abs(at).max(axis=(1, 2), keepdims=True) / 448.0
            sa[sa == 0] = 1.0
            aq = (q_e4m3(at / sa) * sa).reshape(-1, a.shape[1])[:n]
            acc = (aq @ Wq.T) * sw.T + b
        else:
            acc = a @ bf16(W).T + b
        a = bf16(gelu(acc)) if l < L - 1 else acc
    return a.T


def post_step(pr, o):
    """S4-S7 in numpy FP64 from a raw output o [Ns][n] (one-range NASA-7 table): returns (T_new, Y_new)."""
    st, cfg, th, m = pr.prob.state, pr.prob.cfg, pr.prob.thermo, pr.model
    lam = cfg.lam
    Yc = np.maximum(st.Y.astype(np.float64), 0.0)
    y = (Yc ** lam - 1.0) / lam
    dy = cfg.dt * (o * pr.prob.out_std[:, None].astype(np.float64) + pr.prob.out_mean[:, None].astype(np.float64))
    Ys = np.maximum(1.0 + lam * (y + dy), 0.0) ** (1.0 / lam)
    Yn = Ys / Ys.sum(axis=0, keepdims=True)
    a = th.nasa_lo
    s = (RU / th.W)[:, None]
    T = np.clip(st.T.astype(np.float64), m.T_min, m.T_max)
    done = np.zeros(T.shape, dtype=bool)
    for _ in range(m.newton_max_iter):
        Tr = T[None, :]
        cpk = s * (a[:, 0:1] + a[:, 1:2] * Tr + a[:, 2:3] * Tr ** 2 + a[:, 3:4] * Tr ** 3 + a[:, 4:5] * Tr ** 4)
        hk = s * (a[:, 0:1] * Tr + a[:, 1:2] * Tr ** 2 / 2 + a[:, 2:3] * Tr ** 3 / 3 + a[:, 3:4] * Tr ** 4 / 4
                  + a[:, 4:5] * Tr ** 5 / 5 + a[:, 5:6])
        dT = -((Yn * hk).sum(axis=0) - pr.h.astype(np.float64)) / (Yn * cpk).sum(axis=0)
        T = np.where(done, T, np.clip(T + dT, m.T_min, m.T_max))
        done |= np.abs(dT) < m.newton_tol
    return T, Yn


def errors(pr, ref, o):
    d = o - ref.o_raw
    l2 = (np.sqrt((d * d).sum(axis=1)) / np.sqrt((ref.o_raw ** 2).sum(axis=1))).max()
    mx = (np.abs(d).max(axis=1) / np.abs(ref.o_raw).max(axis=1)).max()
    T, Yn = post_step(pr, o)
    dref = G.update_of(ref.Y_new, pr.prob.state.Y)
    r2, rm = G.norms_against(Yn - ref.Y_new, dref, 2.4e-7 * np.abs(ref.Y_new) + 1e-30, 2e-2)
    return {"raw_l2": float(l2), "raw_max": float(mx), "dT": float(np.abs(T - ref.T_new).max()), "dY": max(r2, rm)}


@pytest.mark.parametrize("name,n", [("c1", 16384), ("c2", 4096)])
def test_fp8_error_budget(name, n):
    pr = G.prepare(I.get_config(name), n=n, seed=17)
    assert pr.prob.thermo.nasa_hi is None
    ref = G.run_oracle(pr)
    # the numpy S4-S7 reproduces the oracle on the oracle's own raw output
    T, Yn = post_step(pr, ref.o_raw)
    assert np.abs(T - ref.T_new).max() < 1e-6 and np.abs(Yn - ref.Y_new).max() < 1e-12
    e_bf16 = errors(pr, ref, forward(pr, fp8_layers=()))
    e_fp8 = errors(pr, ref, forward(pr, fp8_layers=(1, 2)))
    e_fp8_l2only = errors(pr, ref, forward(pr, fp8_layers=(1,)))
    print(f"\n{name} n={n}: BF16 emulation {e_bf16}\n{name} n={n}: e4m3 layers 2-3 {e_fp8}\n{name} n={n}: e4m3 layer 2 only {e_fp8_l2only}")
    # the emulation is calibrated: its BF16 variant lands where the GPU's BF16 path was measured, inside every gate
    assert 2e-3 < e_bf16["raw_l2"] < 1e-2 and e_bf16["raw_max"] < 2e-2 and e_bf16["dT"] < 0.5 and e_bf16["dY"] < 1.0
    # e4m3 operands in layers 2-3 -- even in layer 2 alone -- miss north_star's 2e-2 on the raw output by more than 2.5 x,
    # the 0.5 K on T, and the update gate R18' by 3-5 x: the FP8 half of NEXT-4 is closed as "does not meet the tolerances"
    for e in (e_fp8, e_fp8_l2only):
        assert e["raw_l2"] > 2.5 * 2e-2 and e["raw_max"] > 2.5 * 2e-2
        assert e["dT"] > 0.5
        assert e["dY"] > 3.0
