"""`-m gpu`: the CUDA path (through the C ABI) against the FP64 oracle, element by element, on the seeded inputs of
BASELINE.json configs[0..4] at sizes the oracle finishes in seconds (several tiles + a ragged tail)."""
import numpy as np
import pytest

from paper_2402_18858_b200 import binding as B
from paper_2402_18858_b200 import inputs as I

import gpu_common as G

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
        l2, mx = G.check_raw_bf16(g.o_raw, ref.o_raw)
        dT = G.check_T_bf16(g, ref)
        dev = G.check_sumY(g.Y_new)
        assert g.stats[0] == 65536
        print(f"c1: raw rel-L2 {l2:.2e}, max/colmax {mx:.2e}, dT {dT:.3e} K, sumY dev {dev:.2e}")
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
        l2, mx = G.check_raw_bf16(g.o_raw, ref.o_raw)
        dT = G.check_T_bf16(g, ref)
        dev = G.check_sumY(g.Y_new)
        print(f"{name} n={n}: raw rel-L2 {l2:.2e}, max/colmax {mx:.2e}, dT {dT:.3e} K, sumY dev {dev:.2e}")
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
        G.check_raw_bf16(g.o_raw, G.run_oracle_all_active(pr).o_raw)
        dT = G.check_T_bf16(g, ref, mask=active)
        G.check_sumY(g.Y_new, mask=active)
        print(f"c4 n={n}: active {int(active.sum())}, dT {dT:.3e} K")
    finally:
        B.gpuann_destroy(ctx)


def _sample_indices(n, rng, extra):
    """First 4,096, last 4,096 and `extra` seed-drawn cells: tiles at both ends + scattered ones."""
    head = np.arange(0, min(4096, n))
    tail = np.arange(max(0, n - 4096), n)
    mid = rng.choice(n, size=min(extra, n), replace=False)
    return np.unique(np.concatenate([head, tail, mid]))


def test_c2_full_size_sampled_and_invariants():
    """configs[2] at its FULL size (1,048,576 cells) in the launch configuration bench.py times (default chunk):
    full-field invariants on every cell, oracle parity on a sample the oracle computes cell by cell."""
    cfg = I.get_config("c2")
    pr = G.prepare(cfg)
    n = cfg.n_cells
    ctx = G.make_ctx(pr)
    try:
        g = G.run_gpu(ctx, pr)
        assert g.stats[0] == n and g.stats[1] == 0 and g.stats[2] == 0
        assert np.isfinite(g.T_new).all() and np.isfinite(g.Y_new).all() and np.isfinite(g.o_raw).all()
        assert (g.T_new >= cfg.T_min).all() and (g.T_new <= cfg.T_max).all()
        assert (g.Y_new >= 0).all()
        G.check_sumY(g.Y_new)
        idx = _sample_indices(n, np.random.default_rng(20260218), 8192)
        st = pr.prob.state
        ref = G.run_oracle(pr, T=st.T[idx], p=st.p[idx], Y=np.ascontiguousarray(st.Y[:, idx]), h=pr.h[idx])
        sub = G.GpuResult(g.T_new[idx], np.ascontiguousarray(g.Y_new[:, idx]), np.ascontiguousarray(g.o_raw[:, idx]), g.stats)
        l2, mx = G.check_raw_bf16(sub.o_raw, ref.o_raw)
        dT = G.check_T_bf16(sub, ref)
        print(f"c2 full: {idx.size} sampled cells, raw rel-L2 {l2:.2e}, max/colmax {mx:.2e}, dT {dT:.3e} K")
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


@pytest.mark.parametrize("n", [128 * 9 + 5, 4 * 128 * 148 + 128 * 300 + 77])
def test_host_variant_equals_device_variant(n):
    """gpuann_chem_step_host (H2D + step + D2H inside; pipelined over slices for large n) returns bit for bit what
    gpuann_chem_step returns on device-resident state."""
    import torch
    pr = G.prepare(I.get_config("c2"), n=n)
    ctx = G.make_ctx(pr)
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


def test_experimental_split_variant_matches_oracle():
    """GPUANN_FUSED=split (two CTAs per tile, layer-2 columns split over the cluster, h1 exchanged through distributed
    shared memory; slower than the default, kept for round 2) must give the same parity.  The switch is read once per
    process, so the case runs in a child process."""
    import os
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parents[1]
    code = (
        "import sys; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
        "import gpu_common as G\n"
        "from paper_2402_18858_b200 import inputs as I, binding as B\n"
        "pr = G.prepare(I.get_config('c2'), n=128 * 11 + 29)\n"
        "ctx = G.make_ctx(pr, chunk_cells=1024)\n"
        "g = G.run_gpu(ctx, pr); ref = G.run_oracle(pr)\n"
        "G.check_raw_bf16(g.o_raw, ref.o_raw); G.check_T_bf16(g, ref); G.check_sumY(g.Y_new)\n"
        "B.gpuann_destroy(ctx); print('SPLIT-OK')\n" % (str(root), str(root / "tests")))
    env = dict(os.environ, GPUANN_FUSED="split")
    r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "SPLIT-OK" in r.stdout, r.stdout + r.stderr
