"""`-m gpu`: the CUDA path (through the C ABI) against the FP64 oracle, element by element, on the seeded inputs of
BASELINE.json configs[0..4] at sizes the oracle finishes in seconds (several tiles + a ragged tail)."""
import numpy as np
import pytest

from paper_2402_18858_b200 import binding as B
from paper_2402_18858_b200 import inputs as I

import gpu_common as G
import oracle

pytestmark = pytest.mark.gpu


def test_c0_fp32_full():
    """configs[0]: 4,096 cells, Ns = 9, 11-64-64-9, FP32 path, the whole config."""
    pr = G.prepare(I.get_config("c0"))
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        worst, dT = G.check_fp32(g, ref)
        dev = G.check_sumY(g.Y_new)
        # the raw FP32 network output is far inside the BF16 criterion as well
        G.check_raw_bf16(g.o_raw, ref.o_raw)
        assert g.stats == (4096, int((ref.flags & 1).sum()), int(((ref.flags & 2) != 0).sum()))
        print(f"c0: Y err/tol {worst:.3f}, dT {dT:.2e} K, sumY dev {dev:.2e}")
    finally:
        B.gpuann_destroy(ctx)


@pytest.mark.parametrize("n", [1, 31, 33, 4096 + 77])
def test_c0_fp32_ragged(n):
    pr = G.prepare(I.get_config("c0"), n=n, seed=100 + n)
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        G.check_fp32(g, ref)
        G.check_sumY(g.Y_new)
    finally:
        B.gpuann_destroy(ctx)


def test_c1_bf16_full():
    """configs[1]: 65,536 cells, Ns = 21, 23-400-200-100-21, BF16 tensor path, the whole config."""
    pr = G.prepare(I.get_config("c1"))
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        w = G.check_all_bf16(g, ref)
        assert g.stats == (65536, int((ref.flags & 1).sum()), 0)
        print(f"c1: {w}")
    finally:
        B.gpuann_destroy(ctx)


@pytest.mark.parametrize("name,n", [("c2", 3 * 128 * 7 + 53), ("c3", 128 * 9 + 1)])
def test_big_nets_reduced_n(name, n):
    """configs[2], [3] nets (23-1600-800-400-21, 38-1600-800-400-36) on a reduced, ragged cell count."""
    pr = G.prepare(I.get_config(name), n=n)
    ctx = G.make_ctx(pr, chunk_cells=1024)  # several chunks + a ragged last chunk
    try:
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        w = G.check_all_bf16(g, ref)
        print(f"{name} n={n}: {w}")
    finally:
        B.gpuann_destroy(ctx)


def test_c4_compaction_reduced_n():
    """configs[4] mixed field: cells with T < 600 K are skipped (bit-identical), the rest match the oracle."""
    n = 128 * 40 + 19
    pr = G.prepare(I.get_config("c4"), n=n)
    ctx = G.make_ctx(pr, chunk_cells=1024)
    try:
        st = pr.prob.state
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        skipped = st.T < np.float32(600.0)
        active = ~skipped
        assert skipped.any() and active.any()
        assert g.stats[0] == int(active.sum())
        assert np.array_equal(g.T_new[skipped].view(np.uint32), st.T[skipped].view(np.uint32))
        assert np.array_equal(g.Y_new[:, skipped].view(np.uint32), st.Y[:, skipped].view(np.uint32))
        assert (ref.flags[skipped] == 4).all()
        w = G.check_all_bf16(g, ref, mask=active, raw_ref=G.run_oracle_all_active(pr))
        print(f"c4 n={n}: active {int(active.sum())}, {w}")
    finally:
        B.gpuann_destroy(ctx)


def _full_field_invariants(cfg, g, active=None):
    """Cheap checks on EVERY cell of a full-size field."""
    sel = slice(None) if active is None else active
    assert np.isfinite(g.T_new).all() and np.isfinite(g.Y_new).all() and np.isfinite(g.o_raw).all()
    assert (g.T_new[sel] >= cfg.T_min).all() and (g.T_new[sel] <= cfg.T_max).all()
    assert (g.Y_new >= 0).all()
    G.check_sumY(g.Y_new, mask=active)


@pytest.mark.parametrize("name", ["c2", "c3"])
def test_full_size_sampled_and_invariants(name):
    """configs[2] (1,048,576 cells, Ns = 21) and configs[3] (4,194,304 cells, Ns = 36, dt = 5e-7, Newton cap 10) at
    their FULL size in the launch configuration bench.py times (default chunk): full-field invariants on every cell,
    oracle parity on the subset S of SURVEY.md 8(d) -- first 4,096 + last 4,096 + 122,880 seed-drawn cells."""
    cfg = I.get_config(name)
    pr = G.prepare(cfg)
    n = cfg.n_cells
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        assert g.stats == (n, 0, 0)
        _full_field_invariants(cfg, g)
        idx = G.sample_indices(n, np.random.default_rng(20260218 + cfg.index), 122880)
        ref, sub = G.subset(pr, g, idx)
        assert int((ref.flags & 3 != 0).sum()) == 0
        w = G.check_all_bf16(sub, ref)
        print(f"{name} full: {idx.size} sampled cells, {w}")
    finally:
        B.gpuann_destroy(ctx)


def test_c4_full_size_compaction_sampled_and_invariants():
    """configs[4] at its FULL size: 8,388,608 cells, device-side compaction (4,096 scan blocks: the carry loop of
    k_compact_scan runs 16 times), several chunks gated by the device-side n_active.  n_active equals the numpy
    count, EVERY skipped cell is bit-identical, oracle parity on S drawn among the active cells."""
    cfg = I.get_config("c4")
    pr = G.prepare(cfg)
    n = cfg.n_cells
    st = pr.prob.state
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        skipped = st.T < np.float32(cfg.T_active)
        active = ~skipped
        n_act = int(active.sum())
        assert 0.45 * n < n_act < 0.50 * n
        assert g.stats == (n_act, 0, 0)
        assert np.array_equal(g.T_new[skipped].view(np.uint32), st.T[skipped].view(np.uint32))
        assert np.array_equal(g.Y_new[:, skipped].view(np.uint32), st.Y[:, skipped].view(np.uint32))
        _full_field_invariants(cfg, g, active)
        assert (g.T_new[active] != st.T[active]).mean() > 0.99          # the active cells were really stepped
        idx = G.sample_indices(n, np.random.default_rng(20260222), 122880, pool=np.flatnonzero(active))
        ref, sub = G.subset(pr, g, idx)
        assert (ref.flags == 0).all()
        w = G.check_all_bf16(sub, ref)
        print(f"c4 full: active {n_act}, {idx.size} sampled active cells, {w}")
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ branches of the BF16 path
def _continuous_two_range(prob, rng):
    """A second NASA-7 range whose cp and h are continuous at a per-species T_mid inside the batch's T range."""
    th = prob.thermo
    Ns = th.W.shape[0]
    T_mid = rng.uniform(900.0, 1600.0, Ns)
    hi = th.nasa_lo.copy()
    d2 = rng.uniform(-4e-4, 4e-4, Ns)
    hi[:, 1] = th.nasa_lo[:, 1] + d2
    hi[:, 0] = th.nasa_lo[:, 0] - d2 * T_mid                 # cp continuous at T_mid
    hi[:, 5] = th.nasa_lo[:, 5] + d2 * T_mid ** 2 / 2.0      # h continuous at T_mid
    th.nasa_hi, th.T_mid = hi, T_mid


def _case(name):
    import dataclasses
    base = I.get_config("c2")
    if name == "lambda0":           # log / exp branch of Eq. 7 (needs Y > 0: log 0 = -inf on both sides)
        def mut(prob):
            prob.state.Y = np.maximum(prob.state.Y, np.float32(1e-30))
        return dataclasses.replace(base, lam=0.0), mut, {}
    if name == "lambda0.3":         # 1/lambda is not an integer: generic pow in the update
        return dataclasses.replace(base, lam=0.3), None, {}
    if name == "two_range":
        return base, (lambda prob: _continuous_two_range(prob, np.random.default_rng(5))), {}
    if name == "negative_Y":        # 5 % of the entries at -1e-9 (LES undershoot), R2
        def mut(prob):
            Y = prob.state.Y
            Y[np.random.default_rng(6).random(Y.shape) < 0.05] = np.float32(-1e-9)
        return base, mut, {}
    if name == "mu_out":
        def mut(prob):
            Ns = prob.out_mean.shape[0]
            prob.out_mean = (np.where(np.arange(Ns) % 2 == 0, 5e3, -5e3) * np.linspace(0.5, 1.5, Ns)).astype(np.float32)
        return base, mut, {}
    if name == "newton_cap2":       # the iteration cap binds: not-converged counts must agree
        return base, None, {"newton_max_iter": 2}
    if name == "degenerate":        # every 1 + lambda (y + dy) <= 0: the vanishing-sum fallback and its counter
        def mut(prob):
            prob.out_mean = np.full_like(prob.out_mean, -1e8)
            prob.state.Y = (prob.state.Y * np.float32(0.8)).astype(np.float32)
        return base, mut, {}
    raise KeyError(name)


@pytest.mark.parametrize("name", ["lambda0", "lambda0.3", "two_range", "negative_Y", "mu_out", "newton_cap2",
                                  "degenerate"])
def test_bf16_branches(name):
    """One small ragged batch (several tiles, two chunks) of the headline net per branch of the GPU path that the
    five configs never take; every BF16 gate plus the statistics counters against the oracle's flags."""
    cfg, mut, over = _case(name)
    n = 128 * 5 + 37
    pr = G.prepare(cfg, n=n, seed=900 + len(name), mutate=mut, **over)
    ctx = G.make_ctx(pr, chunk_cells=512)
    try:
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        w = G.check_all_bf16(g, ref, lam=cfg.lam)
        n_nc, n_deg = int((ref.flags & 1).sum()), int(((ref.flags & 2) != 0).sum())
        if name == "newton_cap2":
            assert n_nc > 0.9 * n
        if name == "degenerate":
            assert n_deg == n
        if name == "two_range":
            tm = pr.prob.thermo.T_mid
            assert ((ref.T_new[:, None] < tm[None, :]).any(axis=1) & (ref.T_new[:, None] >= tm[None, :]).any(axis=1)).any()
        assert g.stats == (n, n_nc, n_deg), (g.stats, n_nc, n_deg)
        print(f"{name}: {w}, not converged {n_nc}, degenerate {n_deg}")
    finally:
        B.gpuann_destroy(ctx)


def test_input_recipe_helpers_match_the_oracle():
    """gpuann_enthalpy / gpuann_input_moments build bench.py's own inputs (G4, G5): compare them with the oracle's
    helpers -- h to 1 FP32 ulp, the moments to 1e-10 relative."""
    import torch
    cfg = I.get_config("c3")
    pr = G.prepare(cfg, n=20000 + 13, mutate=lambda prob: _continuous_two_range(prob, np.random.default_rng(8)))
    st, th = pr.prob.state, pr.prob.thermo
    ctx = G.make_ctx(pr)
    try:
        dev = torch.device("cuda:0")
        dT, dp, dY = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (st.T, st.p, st.Y))
        dh = torch.empty_like(dT)
        n = int(st.T.shape[0])
        B.gpuann_enthalpy(ctx, n, dT.data_ptr(), dY.data_ptr(), dh.data_ptr(), 0)
        torch.cuda.synchronize()
        h64 = oracle.enthalpy_field(st.T, st.Y, th.nasa_lo, th.nasa_hi, th.T_mid, th.W)
        h_gpu = dh.cpu().numpy()
        ulp = np.spacing(np.abs(h64.astype(np.float32)))
        assert (np.abs(h_gpu.astype(np.float64) - h64) <= ulp).all()
        assert (h_gpu == h64.astype(np.float32)).mean() > 0.99
        for lam in (0.1, 0.0):
            Y = np.maximum(st.Y, np.float32(1e-30)) if lam == 0.0 else st.Y
            dYl = torch.from_numpy(np.ascontiguousarray(Y)).to(dev)
            mean, std = B.gpuann_input_moments(ctx, n, cfg.n_species, dT.data_ptr(), dp.data_ptr(), dYl.data_ptr(), lam, 0)
            m_ref, s_ref = oracle.input_moments(st.T, st.p, Y, lam)
            assert np.allclose(mean, m_ref, rtol=1e-10, atol=0) and np.allclose(std, s_ref, rtol=1e-10, atol=0)
    finally:
        B.gpuann_destroy(ctx)


def test_bf16_step_is_deterministic_and_cellwise():
    """Two runs are bit-identical, and a cell's result does not depend on the batch it sits in (permutation)."""
    n = 128 * 6 + 11
    pr = G.prepare(I.get_config("c2"), n=n)
    ctx = G.make_ctx(pr, chunk_cells=512)
    try:
        a = G.run_gpu(ctx, pr, want_raw=False)
        b = G.run_gpu(ctx, pr, want_raw=False)
        assert np.array_equal(a.T_new.view(np.uint32), b.T_new.view(np.uint32))
        assert np.array_equal(a.Y_new.view(np.uint32), b.Y_new.view(np.uint32))
        st = pr.prob.state
        perm = np.random.default_rng(7).permutation(n)
        c = G.run_gpu(ctx, pr, T=st.T[perm], p=st.p[perm], Y=np.ascontiguousarray(st.Y[:, perm]), h=pr.h[perm], want_raw=False)
        assert np.array_equal(c.T_new.view(np.uint32), a.T_new[perm].view(np.uint32))
        assert np.array_equal(c.Y_new.view(np.uint32), a.Y_new[:, perm].view(np.uint32))
    finally:
        B.gpuann_destroy(ctx)


def test_abi_behaviour_on_device():
    """n_cells = 0 is a no-op, chem_step before the loads is NOT_READY, bad arguments are INVALID_ARG (no abort)."""
    import torch
    prm = B.gpuann_default_params()
    ctx = B.gpuann_create(prm)
    try:
        t = torch.zeros(8, dtype=torch.float32, device="cuda:0")
        y = torch.zeros(21 * 8, dtype=torch.float32, device="cuda:0")
        with pytest.raises(B.GpuannError) as e:
            B.gpuann_chem_step(ctx, 8, t.data_ptr(), t.data_ptr(), y.data_ptr(), t.data_ptr(), 1e-6, 0)
        assert e.value.status == B.GPUANN_ERR_NOT_READY
    finally:
        B.gpuann_destroy(ctx)
    pr = G.prepare(I.get_config("c0"), n=64)
    ctx = G.make_ctx(pr)
    try:
        t = torch.zeros(64, dtype=torch.float32, device="cuda:0")
        y = torch.zeros(9 * 64, dtype=torch.float32, device="cuda:0")
        B.gpuann_chem_step(ctx, 0, 0, 0, 0, 0, 1e-6, 0)  # n = 0: pointers are not looked at
        for bad in (dict(n=-1), dict(dt=0.0), dict(T=0)):
            with pytest.raises(B.GpuannError) as e:
                B.gpuann_chem_step(ctx, bad.get("n", 64), bad.get("T", t.data_ptr()), t.data_ptr(), y.data_ptr(),
                                   t.data_ptr(), bad.get("dt", 1e-6), 0)
            assert e.value.status == B.GPUANN_ERR_INVALID_ARG
    finally:
        B.gpuann_destroy(ctx)


@pytest.mark.parametrize("n,chunk", [(128 * 9 + 5, 0), (4 * 128 * 148 + 128 * 300 + 77, 0),
                                     (4 * 128 * 148 + 128 * 41 + 3, 1024)])
def test_host_variant_equals_device_variant(n, chunk):
    """gpuann_chem_step_host (H2D + step + D2H inside; pipelined over slices for large n) returns bit for bit what
    gpuann_chem_step returns on device-resident state -- also when the field needs far more slices than the
    16 the first version allowed (chunk_cells = 1024: 80 slices; a slice must never exceed the scratch chunk)."""
    import torch
    pr = G.prepare(I.get_config("c2"), n=n)
    ctx = G.make_ctx(pr, chunk_cells=chunk)
    try:
        dev = G.run_gpu(ctx, pr, want_raw=False)
        st = pr.prob.state
        Th = torch.from_numpy(st.T.copy()).pin_memory()
        ph = torch.from_numpy(st.p.copy()).pin_memory()
        Yh = torch.from_numpy(np.ascontiguousarray(st.Y).copy()).pin_memory()
        hh = torch.from_numpy(pr.h.copy()).pin_memory()
        B.gpuann_chem_step_host(ctx, n, Th.data_ptr(), ph.data_ptr(), Yh.data_ptr(), hh.data_ptr(), pr.prob.cfg.dt)
        assert np.array_equal(Th.numpy().view(np.uint32), dev.T_new.view(np.uint32))
        assert np.array_equal(Yh.numpy().view(np.uint32), dev.Y_new.view(np.uint32))
        assert np.array_equal(ph.numpy(), st.p) and np.array_equal(hh.numpy(), pr.h)  # read-only inputs untouched
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ gpuann_chem_step_ex: RR, HRR, cp, rho, psi
def test_ex_outputs_fp32_c0():
    pr = G.prepare(I.get_config("c0"))
    ctx = G.make_ctx(pr)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        ref = G.run_oracle(pr)
        G.check_fp32(g, ref)                       # the step itself is unchanged by the extra outputs
        w = G.check_ex(pr, ref, ex, bf16=False)
        print(f"c0 ex: {w}")
    finally:
        B.gpuann_destroy(ctx)


@pytest.mark.parametrize("name,n", [("c2", 128 * 11 + 53), ("c3", 128 * 5 + 1), ("c1", 4099)])
def test_ex_outputs_bf16(name, n):
    pr = G.prepare(I.get_config(name), n=n, seed=77)
    ctx = G.make_ctx(pr)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        ref = G.run_oracle(pr)
        G.check_T_bf16(g, ref)
        G.check_Y_bf16(g, ref)
        G.check_Y_update(g, ref)
        w = G.check_ex(pr, ref, ex, bf16=True)
        # asking for the extra outputs must not change the step: bit-identical T, Y with and without them
        g0 = G.run_gpu(ctx, pr, want_raw=False)
        assert np.array_equal(g0.T_new, g.T_new) and np.array_equal(g0.Y_new, g.Y_new)
        print(f"{name} ex: {w}")
    finally:
        B.gpuann_destroy(ctx)


def test_ex_outputs_subset_and_skipped_cells_c4():
    """Only some outputs requested; cells below T_active are not written (NaN pre-fill survives)."""
    pr = G.prepare(I.get_config("c4"), n=128 * 9 + 17, seed=5)
    ctx = G.make_ctx(pr)
    try:
        g, ex = G.run_gpu_ex(ctx, pr, which=("hrr", "rho"))
        ref = G.run_oracle(pr)
        act = ref.flags != 4
        assert 0 < act.sum() < act.size
        G.check_T_bf16(g, ref, act)
        w = G.check_ex(pr, ref, ex, bf16=True)
        print(f"c4 ex: {w}")
    finally:
        B.gpuann_destroy(ctx)


def test_ex_outputs_two_range_thermo():
    """The generic (non-FAST) instance of the tail kernel: two NASA-7 ranges, T_mid inside the batch's T range."""
    pr = G.prepare(I.get_config("c2"), n=128 * 3 + 9, seed=9,
                   mutate=lambda prob: _continuous_two_range(prob, np.random.default_rng(5)))
    ctx = G.make_ctx(pr)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        ref = G.run_oracle(pr)
        G.check_T_bf16(g, ref)
        w = G.check_ex(pr, ref, ex, bf16=True)
        print(f"two-range ex: {w}")
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ GPUANN_PRECISION_FP16
@pytest.mark.parametrize("name,n", [("c2h", 128 * 13 + 37), ("c1h", 128 * 40 + 5)])
def test_fp16_variant(name, n):
    """The same two kernels with FP16 weights and activations: gates are the BF16 ones scaled by 2^-3 (R23); the BF16 run of
    the same cells must be the looser of the two (the variant really computes in FP16)."""
    pr = G.prepare(I.get_config(name), n=n, seed=21)
    ctx = G.make_ctx(pr)
    try:
        _, variant = B.gpuann_describe(ctx)
        assert variant == "fp16-fused+tail"
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        w = G.check_all_fp16(g, ref)
        assert g.stats == (n, int((ref.flags & 1).sum()), 0)
        print(f"{name}: {w}")
    finally:
        B.gpuann_destroy(ctx)
    ctx = G.make_ctx(pr, precision=B.GPUANN_PRECISION_BF16)    # FP16-representable weights, rounded again to BF16 inside
    try:
        gb = G.run_gpu(ctx, pr)
        d16 = np.abs(g.o_raw.astype(np.float64) - ref.o_raw).max()
        db = np.abs(gb.o_raw.astype(np.float64) - ref.o_raw).max()
        assert d16 < 0.5 * db, (d16, db)
    finally:
        B.gpuann_destroy(ctx)


def test_fp16_unsupported_shapes_fail_loudly():
    pr = G.prepare(I.get_config("c0"), n=64)     # 11-64-64-9: the fused kernel does not take H1 < 128
    prm = B.gpuann_default_params()
    prm.precision = B.GPUANN_PRECISION_FP16
    ctx = B.gpuann_create(prm)
    try:
        with pytest.raises(B.GpuannError) as e:
            B.gpuann_load_net(ctx, 9, pr.prob.net.sizes, pr.prob.net.weights, pr.prob.net.biases, pr.in_mean, pr.in_std,
                              pr.prob.out_mean, pr.prob.out_std, 0.1)
        assert e.value.status == 3
    finally:
        B.gpuann_destroy(ctx)


def test_refused_load_keeps_the_previous_net_and_bad_weights_are_refused():
    """include/gpuann.h, gpuann_load_net: a load that fails with UNSUPPORTED or INVALID_ARG leaves the net loaded earlier
    in place (the step afterwards is bit-identical); weights / biases that are not finite or overflow the operand type are
    INVALID_ARG instead of a silently frozen chemistry."""
    pr = G.prepare(I.get_config("c1h"), n=128 * 3 + 5, seed=3)
    net, cfg = pr.prob.net, pr.prob.cfg
    small = G.prepare(I.get_config("c0"), n=64)

    def load(ctx, weights=None, biases=None):
        B.gpuann_load_net(ctx, cfg.n_species, net.sizes, net.weights if weights is None else weights,
                          net.biases if biases is None else biases, pr.in_mean, pr.in_std, pr.prob.out_mean, pr.prob.out_std, cfg.lam)

    def edited(arrs, l, idx, value):
        out = [np.array(a, dtype=np.float32, copy=True) for a in arrs]
        out[l].reshape(-1)[idx] = value
        return out

    ctx = G.make_ctx(pr)                     # FP16 context, 23-400-200-100-21 on the fused + tail kernels
    try:
        g0 = G.run_gpu(ctx, pr, want_raw=False)
        # (1) a shape the FP16 path does not take
        rng = np.random.default_rng(2)
        sz = [23, 64, 64, 64, 21]             # first hidden layer < 128: not a net of the fused kernel
        ws = [rng.standard_normal((sz[l + 1], sz[l])).astype(np.float32) * 0.1 for l in range(4)]
        bs = [np.zeros(sz[l + 1], dtype=np.float32) for l in range(4)]
        with pytest.raises(B.GpuannError) as e:
            B.gpuann_load_net(ctx, 21, sz, ws, bs, pr.in_mean, pr.in_std, pr.prob.out_mean, pr.prob.out_std, cfg.lam)
        assert e.value.status == B.GPUANN_ERR_UNSUPPORTED
        # (2) NaN weight, inf bias, FP16 overflow of w/2 in a hidden layer and of a first-layer bias
        for weights, biases, what in (
                (edited(net.weights, 2, 17, np.nan), None, "not finite"),
                (None, edited(net.biases, 3, 4, np.inf), "not finite"),
                (edited(net.weights, 1, 5, 140000.0), None, "overflows FP16"),
                (None, edited(net.biases, 0, 7, -70000.0), "overflows FP16")):
            with pytest.raises(B.GpuannError) as e:
                load(ctx, weights, biases)
            assert e.value.status == B.GPUANN_ERR_INVALID_ARG and what in e.value.message, e.value.message
        # 65504 = the largest FP16 value is fine as a first-layer weight, and w = 131008 is as a hidden-layer weight (w/2 = 65504)
        _, variant = B.gpuann_describe(ctx)
        assert variant == "fp16-fused+tail"
        g1 = G.run_gpu(ctx, pr, want_raw=False)
        assert np.array_equal(g0.T_new, g1.T_new) and np.array_equal(g0.Y_new, g1.Y_new)
        load(ctx, edited(net.weights, 1, 5, 131008.0))     # accepted: replaces the net
    finally:
        B.gpuann_destroy(ctx)

    # FP32 context: the ensemble is refused, the FP32 net stays
    ctx = G.make_ctx(small)
    try:
        g0 = G.run_gpu(ctx, small, want_raw=False)
        sz = list(small.prob.net.sizes[:-1]) + [1]
        ws = [[w if l < len(sz) - 2 else w[:1] for l, w in enumerate(small.prob.net.weights)] for _ in range(9)]
        bs = [[b if l < len(sz) - 2 else b[:1] for l, b in enumerate(small.prob.net.biases)] for _ in range(9)]
        with pytest.raises(B.GpuannError) as e:
            B.gpuann_load_net_ensemble(ctx, 9, sz, ws, bs, small.in_mean, small.in_std, small.prob.out_mean, small.prob.out_std, 0.1)
        assert e.value.status == B.GPUANN_ERR_UNSUPPORTED
        g1 = G.run_gpu(ctx, small, want_raw=False)
        assert np.array_equal(g0.T_new, g1.T_new) and np.array_equal(g0.Y_new, g1.Y_new)
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ per-species ensemble (R24)
@pytest.mark.parametrize("name,n", [("c2", 128 * 6 + 19), ("c1", 128 * 20 + 3), ("c4", 128 * 8 + 77)])
def test_ensemble_of_one_output_nets(name, n):
    """Ns nets D-H1-H2-H3-1 through gpuann_load_net_ensemble against the oracle's O3' (n_nets = Ns): every BF16-path gate."""
    import dataclasses
    cfg = I.get_config(name)
    pr = G.prepare(cfg, n=n, seed=31)
    sizes, ws, bs = I.gen_ensemble(cfg, seed=99)
    prm = B.gpuann_default_params()
    prm.precision = cfg.precision
    prm.newton_max_iter, prm.newton_tol = pr.model.newton_max_iter, pr.model.newton_tol
    prm.T_min, prm.T_max, prm.T_active = pr.model.T_min, pr.model.T_max, pr.model.T_active
    ctx = B.gpuann_create(prm)
    try:
        B.gpuann_load_net_ensemble(ctx, cfg.n_species, sizes, ws, bs, pr.in_mean, pr.in_std, pr.prob.out_mean,
                                   pr.prob.out_std, cfg.lam)
        th = pr.prob.thermo
        B.gpuann_load_thermo(ctx, cfg.n_species, th.nasa_lo, th.nasa_hi, th.T_mid, th.W)
        _, variant = B.gpuann_describe(ctx)
        assert variant == "bf16-ensemble"
        g = G.run_gpu(ctx, pr)
        me = dataclasses.replace(pr.model, sizes=sizes, weights=ws, biases=bs, ensemble=True)
        st = pr.prob.state
        ref = oracle.Oracle(me).chem_step(st.T, st.p, st.Y, pr.h, cfg.dt)
        ref.Y_in = st.Y
        raw_ref = oracle.Oracle(dataclasses.replace(me, T_active=0.0)).chem_step(st.T, st.p, st.Y, pr.h, cfg.dt)
        act = ref.flags != 4
        w = G.check_all_bf16(g, ref, mask=act, raw_ref=raw_ref)
        assert np.array_equal(g.T_new[~act], st.T[~act]) and np.array_equal(g.Y_new[:, ~act], st.Y[:, ~act])
        assert g.stats[0] == int(act.sum()) and g.stats[1] == int((ref.flags[act] & 1).sum())
        print(f"{name} ensemble: {w}")
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ race detection by repetition (compute-sanitizer is closed on this pool)
@pytest.mark.parametrize("name,reps", [("c2", 8), ("c4", 3)])
def test_full_size_runs_are_bit_identical(name, reps):
    """The bench launch configuration (full field, default chunk, 74 CTA pairs) repeated: every run must reproduce the first
    bit for bit.  A missing barrier or fence between the issuer, worker and TMA warps of the two tensor kernels shows up
    here as a few differing cells (the parity tests at full size compare sampled cells only)."""
    import torch
    cfg = I.get_config(name)
    pr = G.prepare(cfg)
    ctx = G.make_ctx(pr)
    try:
        dev = torch.device("cuda:0")
        st = pr.prob.state
        T0, p0, Y0, h0 = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (st.T, st.p, st.Y, pr.h))
        stream = torch.cuda.current_stream().cuda_stream
        first = None
        for r in range(reps):
            T, Y = T0.clone(), Y0.clone()
            B.gpuann_chem_step(ctx, cfg.n_cells, T.data_ptr(), p0.data_ptr(), Y.data_ptr(), h0.data_ptr(), cfg.dt, stream)
            torch.cuda.synchronize()
            if first is None:
                first = (T, Y)
                assert bool(torch.isfinite(T).all()) and bool(torch.isfinite(Y).all())
            else:
                assert torch.equal(T.view(torch.int32), first[0].view(torch.int32)), f"run {r}: T differs from run 0"
                assert torch.equal(Y.view(torch.int32), first[1].view(torch.int32)), f"run {r}: Y differs from run 0"
    finally:
        B.gpuann_destroy(ctx)


def test_small_chunks_ex_fp16_and_ensemble():
    """Several chunks per step (chunk_cells = 512 on 1,157 cells): the optional outputs, the FP16 variant and the ensemble
    address their per-chunk scratch and their field-sized outputs correctly."""
    import dataclasses
    n = 128 * 9 + 5
    # optional outputs on the FP16 variant, three chunks
    pr = G.prepare(I.get_config("c2h"), n=n, seed=41)
    ctx = G.make_ctx(pr, chunk_cells=512)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        ref = G.run_oracle(pr)
        g_raw = G.run_gpu(ctx, pr)
        G.check_all_fp16(g_raw, ref)
        assert np.array_equal(g_raw.T_new, g.T_new) and np.array_equal(g_raw.Y_new, g.Y_new)
        print(f"c2h ex: {G.check_ex(pr, ref, ex, bf16=True, tensor_scale=2.0 ** -3)}")
    finally:
        B.gpuann_destroy(ctx)
    # ensemble, three chunks, against the one-chunk run of the same context type (bit-identical) and the oracle
    cfg = I.get_config("c2")
    pr = G.prepare(cfg, n=n, seed=43)
    sizes, ws, bs = I.gen_ensemble(cfg, seed=5)
    res = []
    for chunk in (512, 0):
        prm = B.gpuann_default_params()
        prm.precision, prm.chunk_cells = cfg.precision, chunk
        ctx = B.gpuann_create(prm)
        try:
            B.gpuann_load_net_ensemble(ctx, cfg.n_species, sizes, ws, bs, pr.in_mean, pr.in_std, pr.prob.out_mean,
                                       pr.prob.out_std, cfg.lam)
            th = pr.prob.thermo
            B.gpuann_load_thermo(ctx, cfg.n_species, th.nasa_lo, th.nasa_hi, th.T_mid, th.W)
            res.append(G.run_gpu(ctx, pr))
            if chunk:                                    # the optional outputs of an ensemble come from the update kernel
                g_ex, ex = G.run_gpu_ex(ctx, pr)
                assert np.array_equal(g_ex.T_new, res[-1].T_new) and np.array_equal(g_ex.Y_new, res[-1].Y_new)
        finally:
            B.gpuann_destroy(ctx)
    assert np.array_equal(res[0].T_new, res[1].T_new) and np.array_equal(res[0].Y_new, res[1].Y_new)
    assert np.array_equal(res[0].o_raw, res[1].o_raw)
    me = dataclasses.replace(pr.model, sizes=sizes, weights=ws, biases=bs, ensemble=True)
    st = pr.prob.state
    ref = oracle.Oracle(me).chem_step(st.T, st.p, st.Y, pr.h, cfg.dt)
    ref.Y_in = st.Y
    G.check_all_bf16(res[0], ref)
    pe = dataclasses.replace(pr, model=me)
    print(f"ensemble ex: {G.check_ex(pe, ref, ex, bf16=True)}")


@pytest.mark.parametrize("ns,hidden", [(60, (256, 256, 128)), (50, (96, 80))])
def test_ex_outputs_from_the_standalone_update_kernel(ns, hidden):
    """Nets without a tail kernel (Ns > 48): RR, HRR, cp, rho, psi come from k_post_q (FP64, species split over a quad)."""
    cfg = I.Config(f"x{ns}", 9, 4096, ns, tuple(hidden), precision=1)
    pr = G.prepare(cfg, n=128 * 4 + 33, seed=ns + 1)
    ctx = G.make_ctx(pr, chunk_cells=256)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        ref = G.run_oracle(pr)
        G.check_T_bf16(g, ref)
        G.check_Y_bf16(g, ref)
        G.check_Y_update(g, ref)
        print(f"Ns={ns} ex: {G.check_ex(pr, ref, ex, bf16=True)}")
    finally:
        B.gpuann_destroy(ctx)


def test_full_size_fp16_and_ex_outputs_sampled():
    """configs[2] at its full size once more, (a) as the FP16 variant and (b) with every optional output requested: oracle
    parity on first 4,096 + last 4,096 + 16,384 drawn cells, full-field invariants."""
    # (a)
    cfg = I.get_config("c2h")
    pr = G.prepare(cfg)
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        assert g.stats == (cfg.n_cells, 0, 0)
        _full_field_invariants(cfg, g)
        idx = G.sample_indices(cfg.n_cells, np.random.default_rng(77), 16384)
        ref, sub = G.subset(pr, g, idx)
        print(f"c2h full: {idx.size} sampled cells, {G.check_all_fp16(sub, ref)}")
    finally:
        B.gpuann_destroy(ctx)
    # (b)
    cfg = I.get_config("c2")
    pr = G.prepare(cfg)
    ctx = G.make_ctx(pr)
    try:
        g, ex = G.run_gpu_ex(ctx, pr)
        idx = G.sample_indices(cfg.n_cells, np.random.default_rng(78), 16384)
        st = pr.prob.state
        import dataclasses
        sub_prob = I.Problem(pr.prob.cfg, int(idx.size), I.State(st.T[idx], st.p[idx], np.ascontiguousarray(st.Y[:, idx])),
                             pr.prob.thermo, pr.prob.net, pr.prob.out_mean, pr.prob.out_std)
        sub_pr = dataclasses.replace(pr, prob=sub_prob, h=pr.h[idx])
        ref = G.run_oracle(sub_pr)
        sub = G.GpuResult(g.T_new[idx], np.ascontiguousarray(g.Y_new[:, idx]), None, g.stats)
        G.check_T_bf16(sub, ref)
        G.check_Y_bf16(sub, ref)
        G.check_Y_update(sub, ref)
        ex_sub = {k: (np.ascontiguousarray(v[:, idx]) if v.ndim == 2 else v[idx]) for k, v in ex.items()}
        print(f"c2 full ex: {G.check_ex(sub_pr, ref, ex_sub, bf16=True)}")
        for k, v in ex.items():
            assert np.isfinite(v).all(), k
    finally:
        B.gpuann_destroy(ctx)


# ------------------------------------------------------------------ shapes other than the five configs
@pytest.mark.parametrize("ns,hidden", [
    (10, (144, 336, 48)),      # H1 not a multiple of 64 (zero padded), pass of 336 columns split 176 + 160, narrow layer 3
    (32, (128, 1008, 416)),    # three passes of 336, the widest layer 3 the tail kernel takes (416), Ns padded to 32
    (48, (256, 400, 112)),     # the most species the tail kernel takes, D + 2 = 52 features -> four layer-1 K steps
    (5, (640, 208, 16)),       # one pass of 208 columns, a 16-wide last hidden layer, one 8-species chunk
    (21, (192, 800, 400, 64)), # FIVE weight matrices: fused kernel, one GEMM layer, tail kernel (row-major h2 path)
    (60, (256, 256, 128)),     # Ns > 48: no tail kernel -> fused kernel + layer GEMMs + stand-alone update
    (9, (64, 64)),             # H1 < 128: no fused kernel -> z kernel + layer GEMM + tail kernel (configs[0]'s net in BF16)
    (50, (96, 80)),            # neither: z kernel + three layer GEMMs + stand-alone update
])
def test_other_net_shapes(ns, hidden):
    """The ABI takes any net: whatever combination of fused kernel / layer GEMM / tail kernel / stand-alone update the
    shapes select must meet the same BF16-path gates (several tiles + a ragged tail, two chunks)."""
    cfg = I.Config(f"x{ns}", 9, 4096, ns, tuple(hidden), precision=1)
    pr = G.prepare(cfg, n=128 * 5 + 61, seed=ns)
    ctx = G.make_ctx(pr, chunk_cells=512)
    try:
        _, variant = B.gpuann_describe(ctx)
        g = G.run_gpu(ctx, pr)
        ref = G.run_oracle(pr)
        w = G.check_all_bf16(g, ref)
        assert g.stats == (128 * 5 + 61, int((ref.flags & 1).sum()), 0)
        print(f"Ns={ns} {hidden} [{variant}]: {w}")
    finally:
        B.gpuann_destroy(ctx)
