"""`-m gpu`: gpuann_input_moments_static, the input statistics for callers that must not allocate device memory.

Who needs it (include/gpuann.h has the long version): a solver that handed the GPU's memory to its own pools at
start-up, so a later cudaMalloc may fail; a time-step loop with halo exchange and linear solves in flight on other
streams, which every cudaMalloc / cudaFree would stall because both wait for the whole device; codes held to "no
allocation after initialisation".  The ordinary gpuann_input_moments allocates and frees its partial-sum scratch on
every call; the static variant keeps that scratch in a `static __device__` array of the library (271,392 bytes per GPU,
at most 64 species) that all calls share and that keeps the previous call's contents.

What is checked: the static variant returns what gpuann_input_moments returns (1e-10 relative, the tolerance
test_input_recipe_helpers_match_the_oracle holds the moments to; on one GPU the two use the same grid and summation
order, so they are expected to agree to the bit) on TWO calls in a row -- the second on a smaller problem with fewer
species and the other Box-Cox branch, so that sums left in the shared array by the first call would show; that the free
device memory does not shrink across the second call; and that a species count beyond the array is refused with a
message that names the limit instead of being served some other way.

The file sorts last on purpose (pytest -x stops at the first failure; nothing is collected after this).  It builds its
own context and inputs, so it passes alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

from paper_2402_18858_b200 import binding as B
from paper_2402_18858_b200 import inputs as I

import oracle

pytestmark = pytest.mark.gpu

RTOL = 1e-10


def _device_state(cfg_name, n, seed, lam):
    import torch
    cfg = I.get_config(cfg_name)
    st = I.make_problem(cfg, n=n, seed=seed).state
    Y = np.maximum(st.Y, np.float32(1e-30)) if lam == 0.0 else st.Y   # log branch: keep ln Y finite
    dev = torch.device("cuda:0")
    d = tuple(torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (st.T, st.p, Y))
    return cfg.n_species, (st.T, st.p, Y), d


def test_static_scratch_moments_match_the_allocating_path_twice_in_a_row():
    import torch
    torch.cuda.set_device(0)
    ctx = B.gpuann_create()   # the statistics need no net and no thermo table
    try:
        # inputs and reference results first, so that nothing but the entry point under test runs between the two calls
        cases = []
        for cfg_name, n, seed, lam in (("c3", 20000 + 13, 11, 0.1), ("c2", 5000 + 7, 12, 0.0)):
            ns, host, dev = _device_state(cfg_name, n, seed, lam)
            args = (ctx, n, ns, dev[0].data_ptr(), dev[1].data_ptr(), dev[2].data_ptr(), lam, 0)
            want = B.gpuann_input_moments(*args)                       # the existing path (cudaMalloc + cudaFree inside)
            cases.append((cfg_name, host, lam, dev, args, want))
        torch.cuda.synchronize()

        got = [B.gpuann_input_moments_static(*cases[0][4])]            # first call on this device: does the set-up
        free_before, _ = torch.cuda.mem_get_info()
        got.append(B.gpuann_input_moments_static(*cases[1][4]))        # second call, straight after, smaller problem
        free_after, _ = torch.cuda.mem_get_info()

        for (cfg_name, host, lam, _, _, want), (mean, std) in zip(cases, got):
            assert mean.shape == want[0].shape and std.shape == want[1].shape
            assert np.all(np.isfinite(mean)) and np.all(np.isfinite(std)) and np.all(std >= 0), cfg_name
            assert np.allclose(mean, want[0], rtol=RTOL, atol=0), (cfg_name, np.max(np.abs(mean / want[0] - 1)))
            assert np.allclose(std, want[1], rtol=RTOL, atol=0), (cfg_name, np.max(np.abs(std / want[1] - 1)))
            m_ref, s_ref = oracle.input_moments(host[0], host[1], host[2], lam)   # and both against the FP64 oracle
            assert np.allclose(mean, m_ref, rtol=RTOL, atol=0) and np.allclose(std, s_ref, rtol=RTOL, atol=0), cfg_name
            print(f"{cfg_name}: static vs allocating path bit-identical = "
                  f"{bool(np.array_equal(mean, want[0]) and np.array_equal(std, want[1]))}")
        assert free_after >= free_before, f"free device memory shrank by {free_before - free_after} bytes across a call"

        # a third call, the first problem again: the shared array now holds the second call's sums
        mean, std = B.gpuann_input_moments_static(*cases[0][4])
        assert np.array_equal(mean, got[0][0]) and np.array_equal(std, got[0][1])
    finally:
        B.gpuann_destroy(ctx)


def test_static_scratch_refuses_what_does_not_fit():
    import torch
    torch.cuda.set_device(0)
    ctx = B.gpuann_create()
    try:
        ns = B.GPUANN_STATIC_MAX_SPECIES + 1
        n = 256
        rng = np.random.default_rng(5)
        Yh = rng.random((ns, n)).astype(np.float32)
        Yh /= Yh.sum(axis=0, keepdims=True)
        T = torch.from_numpy((300.0 + 2000.0 * rng.random(n)).astype(np.float32)).to("cuda:0")
        p = torch.from_numpy((101325.0 * (1.0 + 0.1 * rng.random(n))).astype(np.float32)).to("cuda:0")
        Y = torch.from_numpy(Yh).to("cuda:0")
        with pytest.raises(B.GpuannError) as ei:
            B.gpuann_input_moments_static(ctx, n, ns, T.data_ptr(), p.data_ptr(), Y.data_ptr(), 0.1, 0)
        assert ei.value.status == B.GPUANN_ERR_UNSUPPORTED
        assert "static scratch" in ei.value.message and str(B.GPUANN_STATIC_MAX_SPECIES) in ei.value.message
        # the largest size that does fit goes through
        ns = B.GPUANN_STATIC_MAX_SPECIES   # (the first 64 rows of Y; their sum is no longer 1, which the statistics ignore)
        mean, std = B.gpuann_input_moments_static(ctx, n, ns, T.data_ptr(), p.data_ptr(), Y.data_ptr(), 0.1, 0)
        want = B.gpuann_input_moments(ctx, n, ns, T.data_ptr(), p.data_ptr(), Y.data_ptr(), 0.1, 0)
        assert np.allclose(mean, want[0], rtol=RTOL, atol=0) and np.allclose(std, want[1], rtol=RTOL, atol=0)
    finally:
        B.gpuann_destroy(ctx)
