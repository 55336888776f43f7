"""`-m "not gpu"`: the parity CHECKERS of tests/gpu_common.py reject wrong results (task 1).

The GPU tests assert `error / allowance <= 1`; that proves something only if the allowance is narrower than the
mistakes it is there to catch.  Here the checkers are fed oracle results with a known slip built in -- no GPU, no CUDA
path: the "result under test" is the FP64 oracle's own, rounded to FP32 the way the library stores it -- and must
(1) accept the unmodified result and (2) reject each slip:
  (a) the species update 5 % too large (dy x 1.05: "variation in mass fractions", R3), which the
      element-wise R18 gate (2e-3 |Y|) lets through -- the reason the update gates R18' exist;
  (b) RR_k computed with the density of the UPDATED state instead of the input state (R19);
  (c) HRR computed with h_k at the OLD temperature instead of T_new (PAPER.md:112-115 Eq. 10, :142; R20).
(b) and (c) differ from the right answer by dT/T and by dT sum_k cp_k dY_k / cp: on the configs' dt = 1e-6 s that is
below the resolution any gate derived from north_star's 2e-2 / 0.5 K can have (0.2 % and < 0.01 K), so they are
exercised on the same problem with dt x 20 (median |dT| 64 K), where they are 5 % and several K.
"""
import dataclasses

import numpy as np
import pytest

from paper_2402_18858_b200 import inputs as I

import gpu_common as G
import oracle

RU = 8314.46261815324


def _as_stored(ref):
    """The oracle's result as the library would store it: FP32."""
    return G.GpuResult(ref.T_new.astype(np.float32), ref.Y_new.astype(np.float32), ref.o_raw.astype(np.float32), (0, 0, 0))


def _ex_as_stored(der):
    return {"rr": der.rr.astype(np.float32).astype(np.float64), "hrr": der.hrr.astype(np.float32).astype(np.float64),
            "cp": der.cp.astype(np.float32).astype(np.float64), "rho": der.rho_new.astype(np.float32).astype(np.float64),
            "psi": der.psi.astype(np.float32).astype(np.float64)}


@pytest.fixture(scope="module")
def c1():
    pr = G.prepare(I.get_config("c1"), n=4096, seed=5)
    return pr, G.run_oracle(pr)


@pytest.fixture(scope="module")
def c1_long_dt():
    cfg = I.get_config("c1")
    pr = G.prepare(dataclasses.replace(cfg, dt=20 * cfg.dt), n=4096, seed=5)
    ref = G.run_oracle(pr)
    st = pr.prob.state
    der = oracle.Oracle(pr.model).derived(st.T, st.p, st.Y, pr.prob.cfg.dt, ref)
    return pr, ref, der


def test_checkers_accept_the_oracle_result_as_stored(c1, c1_long_dt):
    pr, ref = c1
    w = G.check_all_bf16(_as_stored(ref), ref)
    assert w["dY"] < 1e-2 and w["Y"] < 1e-3            # only the FP32 store floor is left
    G.check_all_fp16(_as_stored(ref), ref)
    for prx, refx in ((pr, ref), c1_long_dt[:2]):
        st = prx.prob.state
        der = oracle.Oracle(prx.model).derived(st.T, st.p, st.Y, prx.prob.cfg.dt, refx)
        for bf16, scale in ((True, 1.0), (True, 2.0 ** -3), (False, 1.0)):
            out = G.check_ex(prx, refx, _ex_as_stored(der), bf16=bf16, tensor_scale=scale)
            assert max(out.values()) <= 1.0


def test_update_five_percent_too_large_is_rejected(c1):
    """(a) dy x 1.05 through the whole oracle (sigma_out and mu_out scaled): the old element-wise gate accepts it."""
    pr, ref = c1
    m = dataclasses.replace(pr.model, out_std=(1.05 * pr.model.out_std).astype(np.float32),
                            out_mean=(1.05 * pr.model.out_mean).astype(np.float32))
    st = pr.prob.state
    wrong = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, pr.h, pr.prob.cfg.dt)
    g = _as_stored(wrong)
    assert G.check_Y_bf16(g, ref) <= 1.0                # R18 alone does not see a 5 % error of the update ...
    with pytest.raises(AssertionError, match="Y_new update"):
        G.check_Y_update(g, ref)                         # ... R18' does
    with pytest.raises(AssertionError):
        G.check_all_bf16(g, ref)                         # (here the 0.5 K on T trips first: 1.7 K)
    # and so does its RR form: RR of the wrong update against the right one
    der_w = oracle.Oracle(pr.model).derived(st.T, st.p, st.Y, pr.prob.cfg.dt, wrong)
    with pytest.raises(AssertionError, match="RR: per-species"):
        G.check_ex(pr, ref, {"rr": der_w.rr}, bf16=True)
    # a 1 % error of the update is inside north_star's 2e-2 and must pass
    m1 = dataclasses.replace(pr.model, out_std=(1.01 * pr.model.out_std).astype(np.float32),
                             out_mean=(1.01 * pr.model.out_mean).astype(np.float32))
    ok = oracle.Oracle(m1).chem_step(st.T, st.p, st.Y, pr.h, pr.prob.cfg.dt)
    assert 0.3 < G.check_Y_update(_as_stored(ok), ref) <= 1.0


def test_density_of_the_updated_state_in_RR_is_rejected(c1_long_dt):
    """(b) rho(T_new, Y_new) instead of rho(T, Y) in RR_k = rho (Y_new - Y) / dt."""
    pr, ref, der = c1_long_dt
    st = pr.prob.state
    Yc = np.maximum(st.Y.astype(np.float64), 0.0)
    W = pr.prob.thermo.W[:, None]
    rho_in = st.p / (RU * st.T.astype(np.float64) * (Yc / W).sum(axis=0))
    rr_wrong = der.rr * (der.rho_new / rho_in)[None, :]
    with pytest.raises(AssertionError, match="RR"):
        G.check_ex(pr, ref, {"rr": rr_wrong}, bf16=True)
    # the R22' norms on their own (on this problem the element-wise form trips as well)
    floor = rho_in / pr.prob.cfg.dt * 2e-7 * np.abs(st.Y.astype(np.float64)) + 1e-6 * np.abs(der.rr)
    r2, rm = G.norms_against(rr_wrong - der.rr, der.rr, floor, 2e-2)
    assert r2 > 1.5 and rm > 1.5, (r2, rm)


def test_enthalpies_at_the_old_temperature_in_HRR_are_rejected(c1_long_dt):
    """(c) h_k(T) instead of h_k(T_new) in HRR = - sum_k h_k RR_k (one-range NASA-7 table of the configs)."""
    pr, ref, der = c1_long_dt
    st, th = pr.prob.state, pr.prob.thermo
    assert th.nasa_hi is None
    T = st.T.astype(np.float64)[None, :]
    a = th.nasa_lo
    hk_old = (RU / th.W)[:, None] * (a[:, 0:1] * T + a[:, 1:2] * T ** 2 / 2 + a[:, 2:3] * T ** 3 / 3
                                     + a[:, 3:4] * T ** 4 / 4 + a[:, 4:5] * T ** 5 / 5 + a[:, 5:6])
    hrr_wrong = -(hk_old * der.rr).sum(axis=0)
    with pytest.raises(AssertionError, match="HRR"):
        G.check_ex(pr, ref, {"hrr": hrr_wrong}, bf16=True)
    # the R22' per-cell form on its own: the slip as a temperature error, against the 0.5 K stated on T
    Yc = np.maximum(st.Y.astype(np.float64), 0.0)
    rho_in = st.p / (RU * st.T.astype(np.float64) * (Yc / th.W[:, None]).sum(axis=0))
    as_kelvin = np.abs(hrr_wrong - der.hrr) * pr.prob.cfg.dt / (rho_in * der.cp)
    assert (as_kelvin > 0.5).mean() > 0.3 and as_kelvin.max() > 5.0, ((as_kelvin > 0.5).mean(), as_kelvin.max())
    # the same checker accepts the right HRR
    assert max(G.check_ex(pr, ref, {"hrr": der.hrr.astype(np.float32).astype(np.float64)}, bf16=True).values()) <= 1.0
