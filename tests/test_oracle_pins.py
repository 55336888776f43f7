"""Pins for the FP64 oracle against things OTHER than itself (no GPU needed).

Each test names the passage of PAPER.md (or the DESIGN.md reading) it pins and is chosen so that a plausible
mistake in oracle.c -- a dropped term, a wrong sign or index, a transposed operand -- fails it.
"""
import math

import numpy as np
import pytest
from scipy import optimize, special

import oracle
from conftest import read_golden
from paper_2402_18858_b200 import inputs

RU = 8314.46261815324


# ------------------------------------------------------------------ Box-Cox (O1, O5) -- PAPER.md:98-103, Eq. 7
def test_boxcox_paper_endpoints():
    for lam, x, fx in read_golden("boxcox_eq7.txt"):
        assert oracle.boxcox(float(x), float(lam)) == float(fx)  # exact: pow(0, .1) = 0, pow(1, .1) = 1


def test_boxcox_zero_maps_exactly_to_minus_inverse_lambda_and_back():
    for lam in (0.1, 0.25, 0.5):
        assert oracle.boxcox(0.0, lam) == -1.0 / lam
        assert oracle.boxcox_inv(-1.0 / lam, lam) == 0.0


def test_boxcox_lambda_to_zero_is_log():
    for x in (1e-12, 1e-6, 0.03, 0.5, 1.0):
        assert oracle.boxcox(x, 0.0) == math.log(x)
        assert abs(oracle.boxcox(x, 1e-9) - math.log(x)) <= 1e-7 * max(1.0, abs(math.log(x)) ** 2)
    assert abs(oracle.boxcox_inv(-3.0, 0.0) - math.exp(-3.0)) < 1e-16


def test_boxcox_round_trip_1e12():
    xs = np.concatenate([10.0 ** np.linspace(-20, 0, 401), [0.0, 1.0]])
    for x in xs:
        back = oracle.boxcox_inv(oracle.boxcox(x, 0.1), 0.1)
        assert abs(back - x) <= 1e-12 * x


def test_boxcox_independent_formula_and_monotone():
    xs = 10.0 ** np.linspace(-15, 0, 200)
    got = np.array([oracle.boxcox(x, 0.1) for x in xs])
    want = special.boxcox(xs, 0.1)          # scipy's own implementation of Box & Cox (1964)
    assert np.allclose(got, want, rtol=1e-13, atol=1e-13)
    assert np.all(np.diff(got) > 0)
    assert got.min() >= -10.0 and got.max() <= 0.0
    inv = np.array([oracle.boxcox_inv(y, 0.1) for y in got])
    assert np.allclose(inv, special.inv_boxcox(got, 0.1), rtol=1e-12, atol=0)


def test_boxcox_inverse_clamps_below_zero():
    # R7: 1 + lambda*y < 0 -> species vanishes
    assert oracle.boxcox_inv(-10.5, 0.1) == 0.0
    assert oracle.boxcox_inv(0.5, 0.1) == pytest.approx(1.05 ** 10, rel=1e-15)  # no upper clamp


# ------------------------------------------------------------------ GELU / MLP (O3) -- PAPER.md:103
def test_gelu_textbook_values():
    for v, g in read_golden("gelu_textbook.txt"):
        assert abs(oracle.gelu(float(v)) - float(g)) < 1e-15


def test_gelu_against_scipy_ndtr():
    vs = np.linspace(-6, 6, 241)
    got = np.array([oracle.gelu(v) for v in vs])
    assert np.allclose(got, vs * special.ndtr(vs), rtol=0, atol=2e-16 * 8)


def test_mlp_hand_expanded_3_2_2():
    """3-2-2 net, small integer weights; every output written out as an explicit sum (no loops, no matmul)."""
    W1 = np.array([[1, -2, 3], [0, 2, -1]], dtype=np.float32)   # [out=2][in=3]
    b1 = np.array([0.5, -1.0], dtype=np.float32)
    W2 = np.array([[2, -1], [-3, 4]], dtype=np.float32)
    b2 = np.array([0.25, -0.75], dtype=np.float32)
    z = np.array([0.5, -1.5, 2.0])
    g = lambda v: v * special.ndtr(v)
    h0 = g(1 * 0.5 + (-2) * (-1.5) + 3 * 2.0 + 0.5)     # 10.0
    h1 = g(0 * 0.5 + 2 * (-1.5) + (-1) * 2.0 - 1.0)     # -6.0
    o0 = 2 * h0 + (-1) * h1 + 0.25
    o1 = (-3) * h0 + 4 * h1 - 0.75
    got = oracle.mlp_forward([3, 2, 2], [W1, W2], [b1, b2], z)
    assert np.allclose(got, [o0, o1], rtol=1e-14, atol=1e-14)
    # a transposed W1 ([in][out] read as [out][in]) or swapped biases would change the result:
    assert abs(o0 - (2 * g(10.0) - g(-6.0) + 0.25)) < 1e-14


def test_mlp_non_square_layout_catches_transposition():
    """2-3-1 net: W1 is [3][2]; row r of W1 multiplies the whole input."""
    W1 = np.array([[1, 2], [3, 4], [5, 6]], dtype=np.float32)
    b1 = np.zeros(3, dtype=np.float32)
    W2 = np.array([[1, 10, 100]], dtype=np.float32)
    b2 = np.array([7.0], dtype=np.float32)
    z = np.array([1.0, -1.0])
    g = lambda v: v * special.ndtr(v)
    want = 1 * g(1 - 2) + 10 * g(3 - 4) + 100 * g(5 - 6) + 7.0
    got = oracle.mlp_forward([2, 3, 1], [W1, W2], [b1, b2], z)
    assert abs(got[0] - want) < 1e-13


def test_mlp_matches_numpy_scipy_on_random_net():
    rng = np.random.default_rng(11)
    sizes = [11, 17, 13, 9]
    net = inputs.gen_net(rng, sizes, bf16_weights=False)
    z = rng.normal(size=11)
    a = z.copy()
    for l, (W, b) in enumerate(zip(net.weights, net.biases)):
        a = W.astype(np.float64) @ a + b.astype(np.float64)
        if l < len(sizes) - 2:
            a = 0.5 * a * (1.0 + special.erf(a / math.sqrt(2.0)))
    got = oracle.mlp_forward(sizes, net.weights, net.biases, z)
    assert np.allclose(got, a, rtol=1e-13, atol=1e-13)


def test_mlp_zero_weights_returns_last_bias_and_no_activation_on_output():
    sizes = [4, 5, 3]
    W = [np.zeros((5, 4), np.float32), np.zeros((3, 5), np.float32)]
    b = [np.ones(5, np.float32), np.array([-2.0, 0.0, 3.0], np.float32)]
    got = oracle.mlp_forward(sizes, W, b, np.ones(4))
    assert np.array_equal(got, [-2.0, 0.0, 3.0])   # a GELU on the output would give -0.0455, 0, 2.996


# ------------------------------------------------------------------ NASA-7 and Newton (O7) -- PAPER.md:57
def _thermo(Ns=5, seed=3):
    return inputs.gen_thermo(np.random.default_rng(seed), Ns)


def test_nasa7_h_is_integral_of_cp():
    """dh/dT = cp for the full 5-term polynomial: pins every coefficient's place and divisor."""
    a = np.array([3.1, 1.2e-3, -2.5e-7, 3.0e-11, -1.5e-15, -1.2e4, 4.0])
    W = 28.0
    for T in (300.0, 1000.0, 2500.0):
        d = 1e-3 * T
        num = (oracle.species_h(a, W, T + d) - oracle.species_h(a, W, T - d)) / (2 * d)
        assert abs(num - oracle.species_cp(a, W, T)) < 1e-6 * oracle.species_cp(a, W, T)
    # closed form at T = 1000 K, written out term by term
    T = 1000.0
    cp = (RU / W) * (3.1 + 1.2e-3 * 1e3 - 2.5e-7 * 1e6 + 3.0e-11 * 1e9 - 1.5e-15 * 1e12)
    h = (RU / W) * (3.1 * 1e3 + 1.2e-3 * 1e6 / 2 - 2.5e-7 * 1e9 / 3 + 3.0e-11 * 1e12 / 4 - 1.5e-15 * 1e15 / 5 - 1.2e4)
    assert oracle.species_cp(a, W, T) == pytest.approx(cp, rel=1e-14)
    assert oracle.species_h(a, W, T) == pytest.approx(h, rel=1e-14)


def test_newton_manufactured_root_from_far_starts():
    th = _thermo(9, 5)
    rng = np.random.default_rng(0)
    for _ in range(20):
        Y = rng.dirichlet(0.5 * np.ones(9))
        Tstar = rng.uniform(300, 2500)
        h = oracle.mixture_h(Y, Tstar, th.nasa_lo, None, None, th.W)
        for T0 in (Tstar - 500, Tstar + 500, 200.0, 3500.0):
            T, it, conv = oracle.newton_T(Y, h, T0, th.nasa_lo, None, None, th.W)
            assert conv and abs(T - Tstar) < 1e-6 and it <= 8


def test_newton_quadratic_closed_form():
    """a3 = a4 = a5 = 0  =>  h = A T + B T^2/2 + C, T = (-A + sqrt(A^2 + 2B(h - C)))/B."""
    th = _thermo(6, 7)
    lo = th.nasa_lo.copy()
    lo[:, 2:5] = 0.0
    rng = np.random.default_rng(1)
    Y = rng.dirichlet(np.ones(6))
    A = float(np.sum(Y * (RU / th.W) * lo[:, 0]))
    B = float(np.sum(Y * (RU / th.W) * lo[:, 1]))
    Cc = float(np.sum(Y * (RU / th.W) * lo[:, 5]))
    for Tstar in (350.0, 1234.5, 3000.0):
        h = A * Tstar + B * Tstar ** 2 / 2 + Cc
        want = (-A + math.sqrt(A * A + 2 * B * (h - Cc))) / B
        T, it, conv = oracle.newton_T(Y, h, 1000.0, lo, None, None, th.W)
        assert conv and abs(T - want) < 1e-6 and abs(want - Tstar) < 1e-8


def test_newton_linear_exact_after_one_update_converged_on_second():
    th = _thermo(4, 9)
    lo = th.nasa_lo.copy()
    lo[:, 1:5] = 0.0
    Y = np.array([0.1, 0.2, 0.3, 0.4])
    A = float(np.sum(Y * (RU / th.W) * lo[:, 0]))
    Cc = float(np.sum(Y * (RU / th.W) * lo[:, 5]))
    h = A * 1500.0 + Cc
    T1, it1, conv1 = oracle.newton_T(Y, h, 800.0, lo, None, None, th.W, max_iter=1)
    assert it1 == 1 and not conv1 and abs(T1 - 1500.0) < 1e-9
    T2, it2, conv2 = oracle.newton_T(Y, h, 800.0, lo, None, None, th.W, max_iter=20)
    assert it2 == 2 and conv2 and abs(T2 - 1500.0) < 1e-9


def test_newton_against_brentq():
    th = _thermo(21, 2)
    rng = np.random.default_rng(2)
    for _ in range(10):
        Y = rng.dirichlet(0.5 * np.ones(21))
        h = oracle.mixture_h(Y, rng.uniform(300, 2500), th.nasa_lo, None, None, th.W)

        def f(T):  # independent evaluation of sum_k Y_k h_k(T) - h with numpy
            a = th.nasa_lo
            hk = (RU / th.W) * (a[:, 0] * T + a[:, 1] * T ** 2 / 2 + a[:, 2] * T ** 3 / 3 + a[:, 3] * T ** 4 / 4
                                + a[:, 4] * T ** 5 / 5 + a[:, 5])
            return float(np.dot(Y, hk)) - h

        root = optimize.brentq(f, 200.0, 3500.0, xtol=1e-11, rtol=1e-14)
        T, _, conv = oracle.newton_T(Y, h, 1000.0, th.nasa_lo, None, None, th.W, tol=1e-9)
        assert conv and abs(T - root) < 1e-8


def test_newton_two_ranges_select_and_same_coeffs_ignore_tmid():
    th = _thermo(5, 4)
    Y = np.full(5, 0.2)
    h = oracle.mixture_h(Y, 1700.0, th.nasa_lo, None, None, th.W)
    base = oracle.newton_T(Y, h, 900.0, th.nasa_lo, None, None, th.W)
    for tm in (500.0, 1000.0, 1700.0, 3000.0):
        same = oracle.newton_T(Y, h, 900.0, th.nasa_lo, th.nasa_lo.copy(), np.full(5, tm), th.W)
        assert same == base
    # different high range: below T_mid the low set is used, at/above it the high set
    hi = th.nasa_lo.copy()
    hi[:, 0] += 1.0
    tmid = np.full(5, 1000.0)
    assert oracle.mixture_cp(Y, 999.999, th.nasa_lo, hi, tmid, th.W) == oracle.mixture_cp(Y, 999.999, th.nasa_lo, None, None, th.W)
    assert oracle.mixture_cp(Y, 1000.0, th.nasa_lo, hi, tmid, th.W) == oracle.mixture_cp(Y, 1000.0, hi, None, None, th.W)


def test_newton_clamps_and_reports_non_convergence():
    th = _thermo(3, 8)
    Y = np.array([0.3, 0.3, 0.4])
    h_hot = oracle.mixture_h(Y, 5000.0, th.nasa_lo, None, None, th.W)   # root outside [200, 3500]
    T, it, conv = oracle.newton_T(Y, h_hot, 1000.0, th.nasa_lo, None, None, th.W, max_iter=7)
    assert T == 3500.0 and it == 7 and not conv


# ------------------------------------------------------------------ whole step (O0..O7)
def _small_problem(cfg_name="c0", n=257, seed=123, **over):
    cfg = inputs.get_config(cfg_name)
    pr = inputs.make_problem(cfg, n=n, seed=seed)
    st, th = pr.state, pr.thermo
    h = oracle.enthalpy_field(st.T, st.Y, th.nasa_lo, th.nasa_hi, th.T_mid, th.W).astype(np.float32)
    mean, std = oracle.input_moments(st.T, st.p, st.Y, cfg.lam)
    kw = dict(sizes=pr.net.sizes, weights=pr.net.weights, biases=pr.net.biases,
              in_mean=mean.astype(np.float32), in_std=std.astype(np.float32),
              out_mean=pr.out_mean, out_std=pr.out_std, lam=cfg.lam, nasa_lo=th.nasa_lo, W=th.W,
              T_min=cfg.T_min, T_max=cfg.T_max, newton_tol=cfg.newton_tol,
              newton_max_iter=cfg.newton_max_iter, T_active=cfg.T_active)
    kw.update(over)
    return pr, h, oracle.OracleModel(**kw)


def test_input_moments_against_numpy():
    pr, h, m = _small_problem(n=1000)
    st = pr.state
    x = np.vstack([st.T.astype(np.float64), st.p.astype(np.float64),
                   special.boxcox(np.maximum(st.Y.astype(np.float64), 0.0), 0.1)])
    mean, std = oracle.input_moments(st.T, st.p, st.Y, 0.1)
    assert np.allclose(mean, x.mean(axis=1), rtol=1e-12)
    assert np.allclose(std, x.std(axis=1), rtol=1e-10)          # population std, ddof = 0


def test_enthalpy_field_against_numpy():
    pr, h, m = _small_problem(n=64)
    st, th = pr.state, pr.thermo
    T = st.T.astype(np.float64)
    a = th.nasa_lo
    hk = (RU / th.W)[:, None] * (a[:, 0:1] * T + a[:, 1:2] * T ** 2 / 2 + a[:, 2:3] * T ** 3 / 3 + a[:, 5:6])
    want = (st.Y.astype(np.float64) * hk).sum(axis=0)
    got = oracle.enthalpy_field(st.T, st.Y, th.nasa_lo, None, None, th.W)
    assert np.allclose(got, want, rtol=1e-13)


def test_step_sum_to_one_and_physical_ranges():
    pr, h, m = _small_problem()
    st = pr.state
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    assert np.all(np.abs(r.Y_new.sum(axis=0) - 1.0) < 1e-14)
    assert np.all(r.Y_new >= 0.0) and np.all((r.T_new >= 200.0) & (r.T_new <= 3500.0))
    assert np.all(r.flags == 0) and r.iters.max() <= 6 and r.iters.min() >= 1
    # the step does something: species move by up to ~10 %, T by kelvins (G4)
    assert 1e-3 < np.abs(r.T_new - st.T).max() < 200.0


def test_step_zero_net_is_fixed_point():
    """W_L = 0, b_L = 0, mu_out = 0  =>  Y_new = Y / sum(Y), T_new = T when h = h(T, Y)."""
    pr, h, m = _small_problem(n=200)
    m.weights = [w.copy() for w in m.weights]
    m.biases = [b.copy() for b in m.biases]
    m.weights[-1][:] = 0.0
    m.biases[-1][:] = 0.0
    st = pr.state
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    Y64 = st.Y.astype(np.float64)
    assert np.allclose(r.Y_new, Y64 / Y64.sum(axis=0), rtol=1e-12, atol=1e-300)
    # h was rounded to FP32 (rel 6e-8 of ~1e7 J/kg over cp ~ 1.5e3): T moves by < 1e-3 K, not more
    assert np.abs(r.T_new - st.T).max() < 2e-3
    assert np.all(r.o_raw == 0.0)


def test_step_denormalise_is_linear_in_dt_and_dt_to_zero():
    pr, h, m = _small_problem(n=64)
    st = pr.state
    orc = oracle.Oracle(m)
    r1 = orc.chem_step(st.T, st.p, st.Y, h, 1e-6)
    r2 = orc.chem_step(st.T, st.p, st.Y, h, 2e-6)
    assert np.array_equal(r1.o_raw, r2.o_raw)            # the net does not see dt
    # recover Delta y from the outputs of O5/O6 by an independent route: ratios of Y_new remove the 1/S factor
    lam = 0.1
    Y64 = np.maximum(st.Y.astype(np.float64), 0)
    y = special.boxcox(Y64, lam)
    for r, dt in ((r1, 1e-6), (r2, 2e-6)):
        dy = dt * (r.o_raw * m.out_std[:, None].astype(np.float64) + m.out_mean[:, None])
        Ystar = special.inv_boxcox(y + dy, lam)
        assert np.allclose(r.Y_new, Ystar / Ystar.sum(axis=0), rtol=1e-11, atol=1e-300)
    r0 = orc.chem_step(st.T, st.p, st.Y, h, 1e-30)
    assert np.allclose(r0.Y_new, Y64 / Y64.sum(axis=0), rtol=1e-12, atol=1e-300)


def test_step_residual_of_newton_on_converged_cells():
    pr, h, m = _small_problem(n=300)
    st, th = pr.state, pr.thermo
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    for i in range(0, 300, 7):
        f = oracle.mixture_h(r.Y_new[:, i], r.T_new[i], th.nasa_lo, None, None, th.W) - float(h[i])
        cp = oracle.mixture_cp(r.Y_new[:, i], r.T_new[i], th.nasa_lo, None, None, th.W)
        assert abs(f / cp) < 1e-6


def test_step_permutation_and_batch_independence():
    pr, h, m = _small_problem(n=128)
    st = pr.state
    orc = oracle.Oracle(m)
    r = orc.chem_step(st.T, st.p, st.Y, h, 1e-6)
    perm = np.random.default_rng(5).permutation(128)
    rp = orc.chem_step(st.T[perm], st.p[perm], st.Y[:, perm], h[perm], 1e-6)
    assert np.array_equal(rp.T_new, r.T_new[perm]) and np.array_equal(rp.Y_new, r.Y_new[:, perm])
    rs = orc.chem_step(st.T[:17], st.p[:17], np.ascontiguousarray(st.Y[:, :17]), h[:17], 1e-6)
    assert np.array_equal(rs.T_new, r.T_new[:17]) and np.array_equal(rs.Y_new, r.Y_new[:, :17])


def test_step_negative_and_zero_mass_fractions():
    """R2: Y < 0 is clamped to 0 before the transform; Y = 0 maps to -1/lambda and can grow back."""
    pr, h, m = _small_problem(n=8)
    st = pr.state
    Y = st.Y.copy()
    Y[0, :] = 0.0
    Y[1, :4] = -1e-9
    Y2 = Y.copy()
    Y2[1, :4] = 0.0
    orc = oracle.Oracle(m)
    a = orc.chem_step(st.T, st.p, Y, h, 1e-6)
    b = orc.chem_step(st.T, st.p, Y2, h, 1e-6)
    assert np.array_equal(a.Y_new, b.Y_new) and np.array_equal(a.T_new, b.T_new)
    # species 0 started at exactly zero: Y* = max(lambda * dy, 0)^(1/lambda)
    dy = 1e-6 * (a.o_raw[0] * 2.0e4)
    ystar0 = np.maximum(0.1 * dy, 0.0) ** 10
    ratio = a.Y_new[0] / a.Y_new[2]
    Y64 = np.maximum(Y.astype(np.float64), 0)
    ystar2 = special.inv_boxcox(special.boxcox(Y64[2], 0.1) + 1e-6 * a.o_raw[2] * 2.0e4, 0.1)
    assert np.allclose(ratio, ystar0 / ystar2, rtol=1e-9, atol=1e-300)


def test_step_active_threshold_skips_cold_cells_bit_identically():
    pr, h, m = _small_problem("c4", n=512, seed=77)
    cfg = pr.cfg
    assert cfg.T_active == 600.0 and m.T_active == 600.0
    st = pr.state
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    cold = st.T < np.float32(600.0)
    assert 0.4 < cold.mean() < 0.65 and np.array_equal(r.flags == 4, cold)
    assert np.array_equal(r.T_new[cold], st.T[cold].astype(np.float64))
    assert np.array_equal(r.Y_new[:, cold], st.Y[:, cold].astype(np.float64))
    # active cells equal the result of running only those cells
    act = ~cold
    ra = oracle.Oracle(m).chem_step(st.T[act], st.p[act], np.ascontiguousarray(st.Y[:, act]), h[act], 1e-6)
    assert np.array_equal(ra.T_new, r.T_new[act]) and np.array_equal(ra.Y_new, r.Y_new[:, act])


# ------------------------------------------------------------------ pins added in round 2 ("What's weak" #1)
# Each docstring names the mutation of oracle.c that it catches (all of them passed the round-1 pins).
def _numpy_net(net, z):
    """numpy / scipy MLP on columns of z ([D][m]); exact-erf GELU on hidden layers."""
    a = z
    L = len(net.weights)
    for l, (W, b) in enumerate(zip(net.weights, net.biases)):
        a = W.astype(np.float64) @ a + b.astype(np.float64)[:, None]
        if l < L - 1:
            a = 0.5 * a * (1.0 + special.erf(a / math.sqrt(2.0)))
    return a


def test_step_raw_output_from_independently_built_z():
    """PAPER.md:98 (input = {T, p, F(Y)} in this order), R4 (z = (x - mu)/sigma).  z is built here with numpy / scipy
    alone and pushed through a numpy / scipy MLP; chem_step's o_raw must agree to 1e-12.
    Catches: `* in_std` for `/ in_std` at O2; T and p swapped at O2; y_k fed in the wrong slot."""
    pr, h, m = _small_problem("c0", n=16, seed=41)
    st = pr.state
    # statistics that are NOT symmetric between T, p and the species, and sigma far from 1
    rng = np.random.default_rng(5)
    m.in_mean = (np.asarray(m.in_mean) + rng.normal(size=11).astype(np.float32) * np.asarray(m.in_std)).astype(np.float32)
    m.in_std = (np.asarray(m.in_std) * rng.uniform(0.5, 3.0, 11)).astype(np.float32)
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    x = np.vstack([st.T.astype(np.float64), st.p.astype(np.float64),
                   special.boxcox(np.maximum(st.Y.astype(np.float64), 0.0), 0.1)])
    z = (x - m.in_mean.astype(np.float64)[:, None]) / m.in_std.astype(np.float64)[:, None]
    want = _numpy_net(pr.net, z)
    assert np.allclose(r.o_raw, want, rtol=1e-12, atol=1e-12)
    # the test has teeth: swapping the first two features or multiplying by sigma changes the output
    zs = z.copy()
    zs[[0, 1]] = zs[[1, 0]]
    assert np.abs(_numpy_net(pr.net, zs) - want).max() > 1e-3


def test_step_nonzero_output_mean_enters_with_plus_sign():
    """R3: dy = dt (o sigma_out + mu_out).  mu_out = +-5e3 1/s per species; Y_new recomputed through scipy's
    inv_boxcox from the oracle's own o_raw.  Catches: `- out_mean` at O4, mu_out dropped, mu_out not scaled by dt."""
    pr, h, m = _small_problem("c0", n=48, seed=43)
    st = pr.state
    mu = np.array([5e3 if k % 2 == 0 else -5e3 for k in range(9)], dtype=np.float32) * np.linspace(0.5, 1.5, 9).astype(np.float32)
    m.out_mean = mu
    dt = 1e-6
    r = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, dt)
    y = special.boxcox(np.maximum(st.Y.astype(np.float64), 0.0), 0.1)
    dy = dt * (r.o_raw * m.out_std.astype(np.float64)[:, None] + mu.astype(np.float64)[:, None])
    Ystar = special.inv_boxcox(y + dy, 0.1)
    want = Ystar / Ystar.sum(axis=0)
    assert np.allclose(r.Y_new, want, rtol=1e-11, atol=1e-300)
    wrong = special.inv_boxcox(y + dt * (r.o_raw * m.out_std.astype(np.float64)[:, None] - mu.astype(np.float64)[:, None]), 0.1)
    assert np.abs(wrong / wrong.sum(axis=0) - want).max() > 1e-6     # the sign matters at this size of mu_out


def test_step_threshold_boundary_600_is_active():
    """R12: FP32 `T < 600.0f` means skipped, so T == 600.0f is ACTIVE and nextafter(600, 0) is skipped.
    Catches: `<=` for `<` at O0."""
    pr, h, m = _small_problem("c4", n=64, seed=47)
    st = pr.state
    T = st.T.copy()
    T[0] = np.float32(600.0)
    T[1] = np.nextafter(np.float32(600.0), np.float32(0.0))
    T[2] = np.nextafter(np.float32(600.0), np.float32(1e9))
    th = pr.thermo
    h2 = oracle.enthalpy_field(T, st.Y, th.nasa_lo, th.nasa_hi, th.T_mid, th.W).astype(np.float32)
    r = oracle.Oracle(m).chem_step(T, st.p, st.Y, h2, 1e-6)
    assert r.flags[0] != 4 and r.flags[2] != 4 and r.flags[1] == 4
    assert r.iters[0] >= 1 and np.abs(r.Y_new[:, 0].sum() - 1.0) < 1e-14
    assert np.array_equal(r.Y_new[:, 1], st.Y[:, 1].astype(np.float64)) and r.T_new[1] == float(T[1])
    assert not np.array_equal(r.Y_new[:, 0], st.Y[:, 0].astype(np.float64))     # cell 0 was really stepped


def test_step_vanishing_sum_falls_back_to_clamped_input_over_its_sum():
    """R8: every 1 + lambda (y + dy) <= 0 (mu_out = -1e8 1/s => dy = -100)  =>  Y_new = Yc / sum(Yc), flag bit 1.
    The inputs do NOT sum to one (and hold a negative entry), so the division by sum(Yc) is visible.
    Catches: the fallback without `/ Sc`, Y instead of Yc in the fallback, the flag not set."""
    pr, h, m = _small_problem("c0", n=12, seed=53)
    st = pr.state
    Y = (st.Y * np.float32(0.8)).astype(np.float32)
    Y[3, :] = -1e-4
    m.out_mean = np.full(9, -1e8, dtype=np.float32)
    r = oracle.Oracle(m).chem_step(st.T, st.p, Y, h, 1e-6)
    Yc = np.maximum(Y.astype(np.float64), 0.0)
    assert np.allclose(r.Y_new, Yc / Yc.sum(axis=0), rtol=1e-15, atol=0)
    assert np.all(r.Y_new[3] == 0.0) and np.all((r.flags & 2) == 2)
    assert np.all(np.abs(Yc.sum(axis=0) - 1.0) > 0.1)


def test_newton_stops_at_once_when_cp_is_not_positive():
    """R10: c = sum Y_k cp_k <= 0 at the (clamped) start  =>  no update, 0 iterations, not converged, T = start.
    Catches: the `if (!(c > 0)) break` removed (the iteration would then walk away on a negative slope)."""
    th = _thermo(4, 13)
    lo = th.nasa_lo.copy()
    lo[:, 0] = -np.abs(lo[:, 0])          # a1 < 0 and a2..a5 small: cp < 0 on the whole range
    lo[:, 1:5] = 0.0
    Y = np.array([0.25, 0.25, 0.25, 0.25])
    assert oracle.mixture_cp(Y, 900.0, lo, None, None, th.W) < 0.0
    h = oracle.mixture_h(Y, 1200.0, lo, None, None, th.W)
    T, it, conv = oracle.newton_T(Y, h, 900.0, lo, None, None, th.W)
    assert T == 900.0 and it == 0 and not conv
    # and through the whole step: flag bit 0 set, T_new = the incoming T
    pr, hh, m = _small_problem("c0", n=8, seed=59)
    lo9 = pr.thermo.nasa_lo.copy()
    lo9[:, 0] = -np.abs(lo9[:, 0])
    lo9[:, 1:5] = 0.0
    m.nasa_lo = lo9
    r = oracle.Oracle(m).chem_step(pr.state.T, pr.state.p, pr.state.Y, hh, 1e-6)
    assert np.all(r.iters == 0) and np.all((r.flags & 1) == 1)
    assert np.array_equal(r.T_new, pr.state.T.astype(np.float64))


def test_newton_first_iterate_is_evaluated_at_the_clamped_start():
    """R10: T_0 = clamp(T_start, T_min, T_max).  One update from T_start = 100 K / 5000 K must equal one update
    written out by hand from 200 K / 3500 K on a QUADRATIC h(T) (a linear one lands on the root from anywhere).
    Catches: the start clamp removed."""
    th = _thermo(5, 17)
    lo = th.nasa_lo.copy()
    lo[:, 2:5] = 0.0
    Y = np.array([0.1, 0.3, 0.2, 0.15, 0.25])
    s = RU / th.W
    A, Bq, Cc = float(np.sum(Y * s * lo[:, 0])), float(np.sum(Y * s * lo[:, 1])), float(np.sum(Y * s * lo[:, 5]))
    hq = lambda T: A * T + Bq * T * T / 2 + Cc
    cq = lambda T: A + Bq * T
    h = hq(1500.0)
    for T_start, T0 in ((100.0, 200.0), (5000.0, 3500.0)):
        want = T0 - (hq(T0) - h) / cq(T0)
        T, it, conv = oracle.newton_T(Y, h, T_start, lo, None, None, th.W, max_iter=1)
        assert it == 1 and not conv and abs(T - want) < 1e-9
        unclamped = T_start - (hq(T_start) - h) / cq(T_start)
        assert abs(unclamped - want) > 1.0               # so a missing clamp cannot pass


# ------------------------------------------------------------------ O8 / O9: reaction rates, HRR, thermal properties (round 2)
def _step_with_derived(n=96, **over):
    pr, h, m = _small_problem(n=n, **over)
    st = pr.state
    orc = oracle.Oracle(m)
    r = orc.chem_step(st.T, st.p, st.Y, h, 1e-6)
    return pr, h, m, r, orc.derived(st.T, st.p, st.Y, 1e-6, r)


def test_density_of_pure_nitrogen_textbook_and_molar_ideal_gas_law():
    """rho of the INPUT state behind RR (R19): a pure-N2 cell at 300 K, 1 atm is 1.138 kg/m3 in any textbook; in molar
    units rho = p M / (R T) with R = 8.314462618 J/(mol K), M in kg/mol.  Catches Y*W for Y/W, T_new for T, a missing p."""
    pr, h, m = _small_problem(n=4)
    th = pr.thermo
    Ns = len(th.W)
    W = th.W.copy()
    W[0] = 28.0134
    T = np.full(4, 300.0, dtype=np.float32)
    p = np.full(4, 101325.0, dtype=np.float32)
    Y = np.zeros((Ns, 4), dtype=np.float32)
    Y[0] = 1.0
    m.W = W
    m.weights = [w.copy() for w in m.weights]
    m.biases = [b.copy() for b in m.biases]
    m.weights[-1][:] = 0.0
    m.biases[-1][:] = 3.0        # species 0 grows in Box-Cox space, the others stay at exactly 0 -> Y_new = Y, T moves with h
    hh = oracle.enthalpy_field(np.full(4, 350.0, np.float32), Y, th.nasa_lo, None, None, W).astype(np.float32)
    orc = oracle.Oracle(m)
    r = orc.chem_step(T, p, Y, hh, 1e-6)
    assert np.all(np.abs(r.T_new - 350.0) < 1e-2)          # the step heats the cell by 50 K
    d = orc.derived(T, p, Y, 1e-6, r)
    rho_new_molar = 101325.0 * 0.0280134 / (8.314462618 * r.T_new)
    assert np.allclose(d.rho_new, rho_new_molar, rtol=1e-9)
    assert abs(101325.0 * 0.0280134 / (8.314462618 * 300.0) - 1.138) < 1e-3      # the textbook figure itself
    assert np.allclose(d.rmix, 8314.46261815324 / 28.0134, rtol=1e-12)            # R_mix = Ru / W for a pure species
    assert np.allclose(d.psi * 101325.0, d.rho_new, rtol=1e-12)


def test_reaction_rates_use_input_density_and_sum_to_the_mass_defect():
    """RR_k dt / (Y_new,k - Y_k) is ONE number per cell, the ideal-gas density of the INPUT state (molar-unit formula below,
    clamped Y); sum_k RR_k = rho (1 - sum_k Y_k) / dt.  Catches rho at T_new, a missing 1/dt, RR from clamped Y."""
    pr, h, m, r, d = _step_with_derived()
    st, th = pr.state, pr.thermo
    Y64, T64, p64 = st.Y.astype(np.float64), st.T.astype(np.float64), st.p.astype(np.float64)
    M_kg_per_mol = 1e-3 / (np.maximum(Y64, 0.0) / th.W[:, None]).sum(axis=0)    # W in g/mol
    rho_in = p64 * M_kg_per_mol / (8.314462618 * T64)
    dY = r.Y_new - Y64
    big = np.abs(dY) > 1e-9
    ratio = d.rr * 1e-6 / np.where(big, dY, 1.0)
    assert np.allclose(ratio[big], np.broadcast_to(rho_in, dY.shape)[big], rtol=1e-9)
    assert np.allclose(d.rr.sum(axis=0) * 1e-6 / rho_in + Y64.sum(axis=0), 1.0, rtol=0, atol=1e-13)
    assert np.abs(r.T_new - T64).max() > 1.0     # T does move, so rho(T_new) would have failed the first assert


def test_hrr_is_the_sensible_heating_of_the_old_mixture():
    """With h conserved, -sum_k h_k(T_new) RR_k = (rho / dt) * integral_{T_old}^{T_new} cp(T; Y_old) dT.  The integral is done by
    scipy.integrate.quad on oracle.mixture_cp (pinned as dh/dT above).  Catches the sign, h_k at T_old (that is the heating
    of the NEW mixture, a few per cent off), a dropped 1/dt or rho."""
    from scipy import integrate
    pr, h, m, r, d = _step_with_derived(n=24)
    st, th = pr.state, pr.thermo
    Y64 = st.Y.astype(np.float64)
    Y64 = Y64 / Y64.sum(axis=0)                      # quad below uses the normalised old composition (1e-7 effect)
    for i in range(24):
        rho_in = float(st.p[i]) / (8314.46261815324 * float(st.T[i]) * (np.maximum(st.Y[:, i].astype(np.float64), 0) / th.W).sum())
        # h handed to the step is the FP32 rounding of h(T_old, Y_old): use the exact old enthalpy on both sides
        h_old = oracle.mixture_h(st.Y[:, i].astype(np.float64), float(st.T[i]), th.nasa_lo, None, None, th.W)
        q, _ = integrate.quad(lambda T: oracle.mixture_cp(st.Y[:, i].astype(np.float64), T, th.nasa_lo, None, None, th.W),
                              float(st.T[i]), r.T_new[i], epsabs=1e-9, epsrel=1e-13)
        # Newton solved sum Y_new h_k(T_new) = h_fp32; the defect h_fp32 - h_old enters once
        want = rho_in / 1e-6 * (q + (h_old - float(h[i])))
        assert abs(d.hrr[i] - want) <= 1e-8 * abs(want) + 1e-3 * rho_in / 1e-6, (i, d.hrr[i], want)
    assert np.abs(d.hrr).max() > 1e6               # it is not trivially zero: MW/m3 scale


def test_hrr_and_rr_vanish_for_the_zero_net_and_for_skipped_cells():
    pr, h, m = _small_problem(n=64)
    m.weights = [w.copy() for w in m.weights]
    m.biases = [b.copy() for b in m.biases]
    m.weights[-1][:] = 0.0
    m.biases[-1][:] = 0.0
    st = pr.state
    orc = oracle.Oracle(m)
    r = orc.chem_step(st.T, st.p, st.Y, h, 1e-6)
    d = orc.derived(st.T, st.p, st.Y, 1e-6, r)
    # Y_new = Y / sum Y: |RR| <= rho |1/sum Y - 1| Y / dt ~ 1e-7 * rho / dt
    assert np.abs(d.rr).max() < 1.0 and np.abs(d.hrr).max() < 5e7 * 1e-1
    pr2, h2, m2 = _small_problem(n=64, T_active=1e4)     # every cell skipped
    orc2 = oracle.Oracle(m2)
    r2 = orc2.chem_step(pr2.state.T, pr2.state.p, pr2.state.Y, h2, 1e-6)
    d2 = orc2.derived(pr2.state.T, pr2.state.p, pr2.state.Y, 1e-6, r2)
    assert np.all(r2.flags == 4) and np.all(d2.rr == 0.0) and np.all(d2.hrr == 0.0)


def test_cp_of_the_new_state_is_dh_dT_and_the_state_equation_closes():
    """cp (O9) against central differences of oracle.mixture_h at (T_new, Y_new); rho_new R_mix T_new = p; R_mix against the
    molar-unit mean molar mass.  Catches cp at T_old or with Y_old, W in place of 1/W."""
    pr, h, m, r, d = _step_with_derived(n=32)
    st, th = pr.state, pr.thermo
    for i in range(32):
        y = r.Y_new[:, i]
        dT = 1e-2
        fd = (oracle.mixture_h(y, r.T_new[i] + dT, th.nasa_lo, None, None, th.W)
              - oracle.mixture_h(y, r.T_new[i] - dT, th.nasa_lo, None, None, th.W)) / (2 * dT)
        assert abs(d.cp[i] - fd) < 1e-6 * abs(fd)
        fd_old = (oracle.mixture_h(y, float(st.T[i]) + dT, th.nasa_lo, None, None, th.W)
                  - oracle.mixture_h(y, float(st.T[i]) - dT, th.nasa_lo, None, None, th.W)) / (2 * dT)
        if abs(r.T_new[i] - float(st.T[i])) > 5.0:
            assert abs(d.cp[i] - fd_old) > 1e-5 * abs(fd)      # the pin can tell T_new from T_old
    assert np.allclose(d.rho_new * d.rmix * r.T_new, st.p.astype(np.float64), rtol=1e-13)
    M_new = 1.0 / (r.Y_new / th.W[:, None]).sum(axis=0)       # g/mol
    assert np.allclose(d.rmix, 8.314462618 / (M_new * 1e-3), rtol=1e-9)
    assert np.allclose(d.psi, d.rho_new / st.p.astype(np.float64), rtol=1e-13)


# ------------------------------------------------------------------ O3': per-species ensemble (R24)
def _ensemble_from_single(m, Ns):
    """Ns one-output nets that all carry the single net's hidden layers and row k of its last layer."""
    import dataclasses
    ws = [[w.copy() for w in m.weights[:-1]] + [m.weights[-1][k:k + 1].copy()] for k in range(Ns)]
    bs = [[b.copy() for b in m.biases[:-1]] + [m.biases[-1][k:k + 1].copy()] for k in range(Ns)]
    return dataclasses.replace(m, sizes=tuple(m.sizes[:-1]) + (1,), weights=ws, biases=bs, ensemble=True)


def test_ensemble_with_shared_hidden_layers_equals_the_single_net():
    pr, h, m = _small_problem(n=96)
    st = pr.state
    Ns = pr.cfg.n_species
    r1 = oracle.Oracle(m).chem_step(st.T, st.p, st.Y, h, 1e-6)
    r2 = oracle.Oracle(_ensemble_from_single(m, Ns)).chem_step(st.T, st.p, st.Y, h, 1e-6)
    assert np.array_equal(r1.o_raw, r2.o_raw) and np.array_equal(r1.Y_new, r2.Y_new) and np.array_equal(r1.T_new, r2.T_new)


def test_ensemble_output_k_is_net_k_alone_and_matches_numpy():
    """Net j != k does not enter o_k (bit-identical after perturbing net j), net k does; and o_k equals the numpy / scipy
    forward pass of net k on the independently built z.  Catches nets indexed by the wrong stride or all outputs from net 0."""
    pr, h, m = _small_problem(n=16)
    st, cfg = pr.state, pr.cfg
    Ns = cfg.n_species
    rng = np.random.default_rng(11)
    sizes = tuple(m.sizes[:-1]) + (1,)
    ws = [[rng.uniform(-0.4, 0.4, (sizes[l + 1], sizes[l])).astype(np.float32) for l in range(len(sizes) - 1)] for _ in range(Ns)]
    bs = [[rng.uniform(-0.3, 0.3, sizes[l + 1]).astype(np.float32) for l in range(len(sizes) - 1)] for _ in range(Ns)]
    import dataclasses
    me = dataclasses.replace(m, sizes=sizes, weights=ws, biases=bs, ensemble=True)
    r = oracle.Oracle(me).chem_step(st.T, st.p, st.Y, h, 1e-6)
    x = np.vstack([st.T.astype(np.float64), st.p.astype(np.float64),
                   special.boxcox(np.maximum(st.Y.astype(np.float64), 0.0), cfg.lam)])
    z = (x - m.in_mean.astype(np.float64)[:, None]) / m.in_std.astype(np.float64)[:, None]
    for k in range(Ns):
        a = z
        for l in range(len(sizes) - 1):
            a = ws[k][l].astype(np.float64) @ a + bs[k][l].astype(np.float64)[:, None]
            if l < len(sizes) - 2:
                a = a * special.ndtr(a)
        assert np.allclose(r.o_raw[k], a[0], rtol=1e-12, atol=1e-13)
    ws2 = [[w.copy() for w in net] for net in ws]
    ws2[3][0][:] += 0.25                                        # perturb net 3 only
    r2 = oracle.Oracle(dataclasses.replace(me, weights=ws2)).chem_step(st.T, st.p, st.Y, h, 1e-6)
    others = [k for k in range(Ns) if k != 3]
    assert np.array_equal(r2.o_raw[others], r.o_raw[others]) and not np.array_equal(r2.o_raw[3], r.o_raw[3])


def test_newton_stops_when_cp_is_exactly_zero_and_empty_batches_are_fine():
    """Two boundaries a systematic mutation run of oracle.c found unpinned: c == 0 exactly must stop the iteration (R10:
    "c <= 0", not "c < 0" -- a division by zero otherwise), and n = 0 is a valid, empty step."""
    th = _thermo(Ns=3)
    lo = np.zeros_like(th.nasa_lo)
    lo[:, 5] = 1.0e3                      # h_k = const, cp_k = 0 for every species
    Y = np.array([0.2, 0.3, 0.5])
    T, it, conv = oracle.newton_T(Y, 123.0, 900.0, lo, None, None, th.W)
    assert T == 900.0 and it == 0 and not conv and np.isfinite(T)
    pr, h, m = _small_problem(n=8)
    st = pr.state
    orc = oracle.Oracle(m)
    r = orc.chem_step(st.T[:0], st.p[:0], st.Y[:, :0], h[:0], 1e-6)
    assert r.T_new.shape == (0,) and r.Y_new.shape == (st.Y.shape[0], 0)
    d = orc.derived(st.T[:0], st.p[:0], st.Y[:, :0], 1e-6, r)
    assert d.hrr.shape == (0,) and d.rr.shape == (st.Y.shape[0], 0)


def test_paper_speedup_arithmetic():
    """context numbers in BASELINE.md are self-consistent (ratio = 32/(1 - reduction))."""
    for red, ratio in read_golden("speedup_arithmetic.txt"):
        assert abs(32.0 / (1.0 - float(red) / 100.0) - float(ratio)) < 1.0
