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
