// k_tail.cu -- tensor path, last kernel: the LAST TWO layers of S3 and the whole update S4-S8 in one persistent kernel
//     h3 = GELU(h2 W3^T + b3)      [128 x H3]   accumulated in TMEM, never leaves the SM
//     o  = h3 W4^T + b4            [128 x Ns]   accumulated in TMEM
//     dy = dt (o sigma_out + mu_out);  Y* = F^-1(F(Y) + dy);  Y_new = Y* / sum Y*;  Newton for T_new; store in place
//                                                                      (PAPER.md:98-103 Eq. 7, :92, :57; R3, R7-R11)
// Why: the separate layer-3, layer-4 and update kernels moved h3 (0.84 GB at configs[2]) and o through HBM and ran the
// N = 32 layer-4 GEMM at 7 % of the tensor pipe behind an 80 %-of-HBM stream; here h3 goes TMEM -> registers -> a
// 16 KB shared-memory chunk -> the layer-4 MMA, and the update runs on four warps in the shadow of the next tile's MMAs.
//
// Roles (512 threads, one CTA per SM; CTA PAIRS: clusters of 2 whose even CTA, the leader, issues every tcgen05.mma with
// cta_group::2 -- M = 256 = the 128-cell tiles of both CTAs, B read half from each CTA's shared memory, so a CTA stages
// and reads only HALF of every W3 / W4 tile: five ring stages instead of two, half the shared-memory operand traffic):
//   warp 0       TMA (both CTAs): A = own h2 tile k-block [128 x 64], B = own half of the W3 rows of the current column
//                half (ring of 5), completion counted on the LEADER's full barrier; own half of W4 once, resident
//   warp 1       (leader) layer-3 issuer + TMEM owner.  The 400 accumulator columns are two HALVES (192 + 208) with
//                their own K loops (h2 is streamed twice, the second time from L2): while half 1 accumulates, half 0 is
//                drained, and the next tile's half 0 starts as soon as this tile's half 1 is issued -- TMEM cannot hold
//                two 400-column accumulators, so this is how the drain gets out of the tensor pipe's way
//   warp 2       (leader) layer-4 issuer: o[ob] += h3 chunk (smem) x W4 chunk (smem), two o accumulators
//   warps 4-11   drain: tcgen05.ld 32 columns of acc -> + b3 -> 2 GELU -> BF16 -> swizzled 64-column h3 chunk (ring of 2)
//   warps 12-15  update, one thread per cell: state loads (gathered through idx under compaction) issued BEFORE waiting
//                for o; species update in FP32 (Y^lambda by lg2/ex2, integer power 1/lambda), sum of Y* and the NASA-7
//                MIXTURE coefficients sum_k Y_k c_kj accumulated while the species stream by (FP32 in the FAST instance,
//                FP64 in the generic one), then Newton on the two mixture polynomials in FP64: 11 FMAs per iteration
//                instead of 11 Ns (one-range tables; a two-range table re-selects per species and iteration).  The same
//                warps write the optional outputs of gpuann_chem_step_ex (RR_k, HRR, cp, rho, psi).
//                "Precision of the scalar math".
// Barriers the leader's issuers wait on live in the leader and collect arrivals (cluster-scope release) or TMA bytes
// from BOTH CTAs; barriers that release something to a CTA's own warps are signalled in both CTAs by one multicast
// tcgen05.commit.
#include "common.cuh"
#include "ptx.cuh"

namespace gpuann {

constexpr int kTM = 128;            // cells per tile
constexpr int kTK = 64;             // K elements per smem row (128 B)
constexpr int kTStages = 5;
constexpr int kTAccMax = 416;       // TMEM columns of the layer-3 accumulator
constexpr int kTOCol = 416;         // two o accumulators of kTOStride columns follow
constexpr int kTOStride = 48;
constexpr int kTMaxChunks = (kTAccMax + 63) / 64;  // 7
constexpr int kTailThreads = 512;
constexpr uint32_t kTABytes = kTM * 128;            // 16,384
constexpr uint32_t kTBBytes = 128 * 128;            // this CTA's half of a column half: <= 128 rows of 128 B
constexpr uint32_t kTStageBytes = kTABytes + kTBBytes;
constexpr uint32_t kTH3Bytes = kTM * 128;
constexpr uint32_t kTW4Bytes = kTMaxChunks * (kTailMaxNs / 2) * 128;  // this CTA's half of the W4 rows: 21,504
constexpr uint32_t kTOffH3 = kTStages * kTStageBytes;
constexpr uint32_t kTOffW4 = kTOffH3 + 2 * kTH3Bytes;
constexpr uint32_t kTOffBias = kTOffW4 + kTW4Bytes;
constexpr uint32_t kTOffBar = kTOffBias + 2048;
constexpr size_t kTailSmem = 1024 + kTOffBar + 256;

enum {
    tFull = 0, tEmpty = tFull + kTStages, tW4Full = tEmpty + kTStages, tAccFull, tAccEmpty = tAccFull + 2,
    tH3Full = tAccEmpty + 2, tH3Empty = tH3Full + 2, tOFull = tH3Empty + 2, tOEmpty = tOFull + 2, tCount = tOEmpty + 2
};

struct TRing {
    uint32_t st = 0, ph = 0;
    __device__ __forceinline__ void next(uint32_t n) {
        if (++st == n) {
            st = 0;
            ph ^= 1u;
        }
    }
};

__device__ __forceinline__ float powi_f(float x, int n) {
    float r = 1.f;
    while (n) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}

__device__ __forceinline__ double horner5(const double *c, double T) {
    return c[0] + T * (c[1] + T * (c[2] + T * (c[3] + T * c[4])));
}
__device__ __forceinline__ double horner6(const double *c, double T) {
    return c[0] + T * (c[1] + T * (c[2] + T * (c[3] + T * (c[4] + T * c[5]))));
}

// S4 + S5 for one species in FP32 (R3, R7): Y* = Yc (max(1 + lambda dy / Yc^lambda, 0))^(1/lambda); Yc = 0 (or so small that
// Yc^lambda flushes to 0): Y* = max(lambda dy, 0)^(1/lambda); lambda = 0: Y* = Yc exp(dy)
__device__ __forceinline__ float update_species_f32(float yc, float dy, const TailArgs &ta) {
    if (ta.lambda_zero) return yc * expf(dy);
    const float u = yc > 0.f ? ptx::ex2_approx(ta.lambda * ptx::lg2_approx(yc)) : 0.f;
    const float ldy = ta.lambda * dy;
    const bool pos = u > 0.f;
    const float base = fmaxf(pos ? 1.f + __fdividef(ldy, u) : ldy, 0.f);
    float pw;
    if (ta.inv_lambda_int == 10) {
        const float b2 = base * base, b4 = b2 * b2;
        pw = b4 * b4 * b2;
    } else if (ta.inv_lambda_int > 0) {
        pw = powi_f(base, ta.inv_lambda_int);
    } else {
        pw = powf(base, ta.inv_lambda);
    }
    return (pos ? yc : 1.f) * pw;
}

// NSP: species padded to 8.  FAST: lambda > 0 with 1/lambda = 10 and a one-range thermo table.
template <int NSP, bool FAST>
__global__ void __launch_bounds__(kTailThreads, 1)
k_tail(const __grid_constant__ CUtensorMap tmapA /* row-major [rows][K3p] or blocked (common.cuh, FusedNet) */,
       const __grid_constant__ CUtensorMap tmapW3a,
       const __grid_constant__ CUtensorMap tmapW3b, const __grid_constant__ CUtensorMap tmapW4,
       const __grid_constant__ TailArgs ta) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kTOffBar);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + tCount);
    float *sBias = reinterpret_cast<float *>(smem + kTOffBias);
    const uint32_t sbase = ptx::smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // *ta.n_active (written by k_compact_scan) and bias3 (written at load time) are read BEFORE griddepcontrol.wait.
    // That is safe only because launch_tail asks for programmatic dependent launch solely behind a kernel that was itself
    // launched with full stream ordering (fused / pre / layer kernel): no tail CTA can start before that kernel has
    // started, i.e. before everything in front of it -- the compaction -- has completed.  launch_tail enforces this.
    int64_t rows = ta.rows;
    if (ta.n_active) {
        int64_t r = (int64_t)*ta.n_active - ta.c0;
        rows = r < 0 ? 0 : (r < rows ? r : rows);
    }
    const int n_tiles = (int)((rows + kTM - 1) / kTM);
    // both CTAs of a pair walk the same number of tiles (they share every W3 stage); the odd one may get an empty tile
    const uint32_t crank = ptx::cluster_ctarank();
    const int pair_first = (int)blockIdx.x & ~1;
    const int my_tiles = n_tiles > pair_first ? (n_tiles - pair_first + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int nkb = (ta.K3p + kTK - 1) / kTK;
    const int nch = (ta.H3p + 63) / 64;

    const int n_half = ta.n1 > 0 ? 2 : 1;
    const int ch0 = ta.n1 > 0 ? ta.n0 / 64 : nch;  // chunks of column half 0 (n0 is a multiple of 64 when there are two)
    if (threadIdx.x == 0) {
        for (int i = 0; i < kTStages; ++i) { ptx::mbar_init(&bars[tFull + i], 1); ptx::mbar_init(&bars[tEmpty + i], 1); }
        ptx::mbar_init(&bars[tW4Full], 1);
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(&bars[tAccFull + i], 1);
            ptx::mbar_init(&bars[tAccEmpty + i], 16);  // the 8 drain warps of BOTH CTAs
            ptx::mbar_init(&bars[tH3Full + i], 16);
            ptx::mbar_init(&bars[tH3Empty + i], 1);
            ptx::mbar_init(&bars[tOFull + i], 1);
            ptx::mbar_init(&bars[tOEmpty + i], 8);     // the 4 update warps of both CTAs
        }
        ptx::fence_mbar_init();
    }
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmapA);
        ptx::prefetch_tensormap(&tmapW3a);
        ptx::prefetch_tensormap(&tmapW3b);
        ptx::prefetch_tensormap(&tmapW4);
    }
    if (warp == 1) {
        ptx::tmem_alloc_cg2(tmem_slot, 512);
        ptx::tmem_relinquish_cg2();
    }
    for (int i = threadIdx.x; i < ta.H3p && i < kTAccMax; i += kTailThreads) sBias[i] = ta.bias3[i];
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync_all();
    ptx::tc_fence_after_sync();
    // everything above (barriers, TMEM, tensor maps, bias) is independent of the kernel in front; h2 and the state are not
    ptx::griddep_wait();
    const uint32_t tmem_base = *tmem_slot;
    const uint64_t desc0 = ptx::umma_desc_sw128_kmajor(sbase);
    const uint64_t descA0 = ptx::umma_desc_nosw_kmajor(sbase, 2048, 128);  // blocked A stage: [8 kp][128 rows][16 B]
    const uint32_t bars_leader = ptx::mapa_u32(ptx::smem_u32(bars), 0);  // the leader's barrier array, cluster address
    const bool leader = crank == 0;

    // register budget per warpgroup (512 threads x 128 at launch): the update warps hold a cell's whole state in registers
    if (warp < 4) ptx::setmaxnreg_dec<104>();
    else if (warp < 12) ptx::setmaxnreg_dec<104>();
    else ptx::setmaxnreg_inc<200>();

    if (warp == 0) {
        // ================================================================ TMA (both CTAs)
        if (lane == 0) {
            const uint32_t sbase_cl = ptx::mapa_u32(sbase, crank);  // own shared memory in the cluster window
            const int hp = ta.Np / 2;
            if (leader) ptx::mbar_arrive_expect_tx(&bars[tW4Full], (uint32_t)(2 * nch * hp * 128));
            for (int c = 0; c < nch; ++c)
                ptx::tma_load_2d_cg2(&tmapW4, bars_leader + 8u * tW4Full, sbase_cl + kTOffW4 + (uint32_t)(c * hp * 128), c * kTK,
                                     (int)crank * hp);
            TRing st;
            for (int it = 0; it < my_tiles; ++it) {
                const int tile = (int)blockIdx.x + it * (int)gridDim.x;
                for (int hf = 0; hf < n_half; ++hf) {
                    const int nh = (hf ? ta.n1 : ta.n0) / 2;  // rows of this CTA's part of the column half
                    const int row0 = (hf ? ta.n0 : 0) + (int)crank * nh;
                    for (int kb = 0; kb < nkb; ++kb) {
                        ptx::mbar_wait(&bars[tEmpty + st.st], st.ph ^ 1u);
                        if (leader) ptx::mbar_arrive_expect_tx(&bars[tFull + st.st], 2u * (kTABytes + (uint32_t)nh * 128u));
                        const uint32_t full = bars_leader + 8u * (tFull + st.st);
                        const uint32_t sA = sbase_cl + st.st * kTStageBytes;
                        if (ta.a_blocked)  // the [128 x 64] stage is 16 KB contiguous: slabs (tile, 8 kb .. 8 kb + 7), rows of 256 elements
                            ptx::tma_load_2d_cg2(&tmapA, full, sA, 0, (tile * (ta.K3p >> 3) + 8 * kb) * 4);
                        else
                            ptx::tma_load_2d_cg2(&tmapA, full, sA, kb * kTK, tile * kTM);
                        ptx::tma_load_2d_cg2(hf ? &tmapW3b : &tmapW3a, full, sA + kTABytes, kb * kTK, row0);
                        st.next(kTStages);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================================================================ layer-3 MMA issuer (leader; whole warp, uniform)
        if (leader) {
            const uint32_t idesc_h[2] = {ptx::umma_idesc_bf16_f32(2 * kTM, (uint32_t)ta.n0, ta.f16 != 0),
                                         ptx::umma_idesc_bf16_f32(2 * kTM, (uint32_t)(ta.n1 > 0 ? ta.n1 : 16), ta.f16 != 0)};
            TRing st;
            uint32_t acc_ph = 0;
            for (int it = 0; it < my_tiles; ++it) {
                for (int hf = 0; hf < n_half; ++hf) {
                    ptx::mbar_wait_cluster(&bars[tAccEmpty + hf], acc_ph ^ 1u);
                    ptx::tc_fence_after_sync();
                    const uint32_t d_tmem = tmem_base + (uint32_t)(hf ? ta.n0 : 0);
                    const uint32_t idesc = idesc_h[hf];
                    for (int kb = 0; kb < nkb; ++kb) {
                        ptx::mbar_wait_cluster(&bars[tFull + st.st], st.ph);
                        ptx::tc_fence_after_sync();
                        const uint64_t db = desc0 + (uint64_t)((st.st * kTStageBytes + kTABytes) >> 4);
                        // A: 128-byte-swizzled rows (k-step = 32 B) or the blocked core-matrix order (k-step = 2 x 2 KB slabs)
                        const uint64_t da = (ta.a_blocked ? descA0 : desc0) + (uint64_t)((st.st * kTStageBytes) >> 4);
                        const uint64_t ka = ta.a_blocked ? (uint64_t)(4096 >> 4) : 2u;
                        const int ksteps = min(kTK / 16, (ta.K3p - kb * kTK) / 16);
                        if (ptx::elect_one()) {
                            if (ksteps == kTK / 16) {
#pragma unroll
                                for (int k = 0; k < kTK / 16; ++k)
                                    ptx::umma_bf16_ss_cg2(d_tmem, da + ka * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
                            } else {
                                for (int k = 0; k < ksteps; ++k)
                                    ptx::umma_bf16_ss_cg2(d_tmem, da + ka * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
                            }
                            ptx::umma_commit_cg2(&bars[tEmpty + st.st], 3);
                            if (kb == nkb - 1) ptx::umma_commit_cg2(&bars[tAccFull + hf], 3);
                        }
                        __syncwarp();
                        st.next(kTStages);
                    }
                }
                acc_ph ^= 1u;
            }
        }
    } else if (warp == 2) {
        // ================================================================ layer-4 MMA issuer (leader; whole warp, uniform)
        if (leader) {
            const uint32_t idesc4 = ptx::umma_idesc_bf16_f32(2 * kTM, (uint32_t)ta.Np, ta.f16 != 0);
            ptx::mbar_wait_cluster(&bars[tW4Full], 0);
            const uint32_t w4_chunk = (uint32_t)(ta.Np / 2) * 128u;
            uint32_t seq = 0;
            for (int it = 0; it < my_tiles; ++it) {
                const uint32_t ob = (uint32_t)it & 1u, oph = ((uint32_t)it >> 1) & 1u;
                ptx::mbar_wait_cluster(&bars[tOEmpty + ob], oph ^ 1u);
                ptx::tc_fence_after_sync();
                const uint32_t d_tmem = tmem_base + kTOCol + ob * kTOStride;
                for (int c = 0; c < nch; ++c, ++seq) {
                    const uint32_t buf = seq & 1u, ph = (seq >> 1) & 1u;
                    ptx::mbar_wait_cluster(&bars[tH3Full + buf], ph);
                    ptx::tc_fence_after_sync();
                    const uint64_t da = desc0 + (uint64_t)((kTOffH3 + buf * kTH3Bytes) >> 4);
                    const uint64_t db = desc0 + (uint64_t)((kTOffW4 + (uint32_t)c * w4_chunk) >> 4);
                    const int ksteps = min(4, (ta.H3p - c * 64) / 16);
                    if (ptx::elect_one()) {
                        for (int k = 0; k < ksteps; ++k)
                            ptx::umma_bf16_ss_cg2(d_tmem, da + 2 * k, db + 2 * k, idesc4, (c | k) ? 1u : 0u);
                        ptx::umma_commit_cg2(&bars[tH3Empty + buf], 3);
                        if (c == nch - 1) ptx::umma_commit_cg2(&bars[tOFull + ob], 3);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp >= 4 && warp < 12) {
        // ================================================================ drain: acc -> h3 chunks (warps 4..11, both CTAs)
        const int q = warp & 3;           // TMEM lane quarter
        const int hsel = (warp - 4) >> 2; // which 32-column half of every 64-column chunk
        const int r = q * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        const uint32_t swz = (uint32_t)(r & 7);
        const uint32_t row_off = (uint32_t)r * 128u;
        uint32_t acc_ph = 0, seq = 0;
        for (int it = 0; it < my_tiles; ++it) {
#pragma unroll 1
            for (int c = 0; c < nch; ++c, ++seq) {
                if (c == 0 || c == ch0) {  // first chunk of a column half: wait for its accumulator
                    ptx::mbar_wait(&bars[tAccFull + (c == 0 ? 0 : 1)], acc_ph);
                    ptx::tc_fence_after_sync();
                }
                const int cc = c * 64 + hsel * 32;
                const int w = ta.H3p - cc;  // >= 32: full piece; 16: half piece; <= 0: none (widths are multiples of 16)
                uint32_t v[32];
                if (w >= 32) ptx::tmem_ld32(lane_addr + (uint32_t)cc, v);
                else if (w > 0) {
                    uint32_t t[16];
                    ptx::tmem_ld16(lane_addr + (uint32_t)cc, t);
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[j] = t[j];
#pragma unroll
                    for (int j = 16; j < 32; ++j) v[j] = 0u;
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j) v[j] = 0u;
                }
                ptx::tmem_ld_wait();
                if (c == ch0 - 1 || c == nch - 1) {  // last read of a column half by this warp: hand it back to the issuer
                    ptx::tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * (tAccEmpty + ((c == nch - 1 && n_half == 2) ? 1 : 0)));
                }
                uint32_t o[16];
                if (w > 0) {
                    const float4 *b4 = reinterpret_cast<const float4 *>(sBias + cc);
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const float4 b = (w >= 32 || j < 4) ? b4[j] : make_float4(0.f, 0.f, 0.f, 0.f);
                        o[2 * j] = ptx::gelu2_pack(__uint_as_float(v[4 * j]) + b.x, __uint_as_float(v[4 * j + 1]) + b.y, ta.f16 != 0);
                        o[2 * j + 1] = ptx::gelu2_pack(__uint_as_float(v[4 * j + 2]) + b.z, __uint_as_float(v[4 * j + 3]) + b.w, ta.f16 != 0);
                    }
                }
                const uint32_t buf = seq & 1u, ph = (seq >> 1) & 1u;
                ptx::mbar_wait(&bars[tH3Empty + buf], ph ^ 1u);
                if (w > 0) {
                    const uint32_t row_addr = sbase + kTOffH3 + buf * kTH3Bytes + row_off;
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        if (w >= 32 || i < 2)
                            ptx::st_shared_v4(row_addr + ((((uint32_t)(4 * hsel + i)) ^ swz) << 4), o[4 * i], o[4 * i + 1],
                                              o[4 * i + 2], o[4 * i + 3]);
                    ptx::fence_proxy_async_smem();
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * (tH3Full + buf));
            }
            acc_ph ^= 1u;
        }
    } else if (warp >= 12) {
        // ================================================================ update S4-S8 (warps 12..15), one thread per cell
        // Species k >= Ns of the padded range carry Y = 0, o = 0 and all-zero constants: they produce Y* = 0 and drop out
        // of every sum, so the arithmetic below has no per-species guards (only the loads and stores are predicated).
        const int q = warp & 3;
        const int r = q * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16) + kTOCol;
        const int Ns = ta.Ns;
        const bool fwd_only = ta.o_raw != nullptr;
        unsigned nconv_total = 0, ndeg_total = 0;
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int64_t i = (int64_t)tile * kTM + r;
            const bool valid = i < rows;
            int64_t g = ta.c0 + i;
            if (ta.idx) g = valid ? (int64_t)ta.idx[g] : 0;
            if (!valid) g = 0;
            const uint32_t ob = (uint32_t)it & 1u, oph = ((uint32_t)it >> 1) & 1u;
            // state loads first: their latency hides behind the wait for o
            float Yv[NSP];
            float Tin = 300.f, hin = 0.f, pin = 101325.f;
            const bool ex_any = ta.ex.any();  // gpuann_chem_step_ex (include/gpuann.h; R19-R21)
            float inv_w_in = 0.f, inv_w_new = 0.f;
            if (!fwd_only) {
#pragma unroll
                for (int k = 0; k < NSP; ++k) Yv[k] = (valid && k < Ns) ? ta.Y[(int64_t)k * ta.n + g] : 0.f;
                if (valid) {
                    Tin = ta.T[g];
                    hin = ta.h[g];
                    if (ex_any) pin = ta.p[g];
                }
            }
            ptx::mbar_wait(&bars[tOFull + ob], oph);
            ptx::tc_fence_after_sync();
            // S4 + S5 (R3, R7) in FP32; sum of Y* and the mixture coefficients sum_k Y*_k c_kj in FP64; o is read from TMEM
            // eight species at a time
            double S = 0.0;
            double Ch[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, Cc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
            // FAST: the sum and the mixture coefficients are accumulated in FP32 (DESIGN.md "Precision of the scalar math":
            // the FP64 pipe of this part runs ~1 warp instruction per 40 clk, and 11 DFMAs per species made the update the
            // slowest stage of the kernel; the rounding adds ~4e-3 K to T against the 0.5 K budget of the tensor path)
            float Sf = 0.f;
            float Chf[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, Ccf[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int pc = 0; pc < NSP / 8; ++pc) {
                uint32_t t8[8];
                ptx::tmem_ld8(lane_addr + ob * kTOStride + (uint32_t)(8 * pc), t8);
                ptx::tmem_ld_wait();
                if (pc == NSP / 8 - 1) {  // o is in registers: hand the accumulator back to the layer-4 issuer
                    ptx::tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * (tOEmpty + ob));
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k = 8 * pc + j;
                    const float o = __uint_as_float(t8[j]);
                    if (fwd_only) {
                        if (valid && k < Ns) ta.o_raw[(int64_t)k * ta.o_stride + i] = o + ta.b4[k];
                        continue;
                    }
                    const float yc = fmaxf(Yv[k], 0.f);
                    const float dy = fmaf(o, ta.sA[k], ta.sC[k]);
                    float ys;
                    if (FAST) {
                        // lambda = 1/10: Y* = Yc (max(1 + lambda dy / u, 0))^10, u = Yc^lambda = ex2(lambda lg2 Yc); Yc = 0 (or
                        // so small that u flushes to 0): Y* = max(lambda dy, 0)^10.  lg2(0) = -inf, ex2(-inf) = 0: no guard
                        const float u = ptx::ex2_approx(ta.lambda * ptx::lg2_approx(yc));
                        const float ldy = ta.lambda * dy;
                        const bool pos = u > 0.f;
                        const float base = fmaxf(pos ? fmaf(ldy, ptx::rcp_approx(u), 1.f) : ldy, 0.f);
                        const float b2 = base * base, b4 = b2 * b2;
                        ys = (pos ? yc : 1.f) * (b4 * b4 * b2);
                    } else {
                        ys = update_species_f32(yc, dy, ta);
                    }
                    Yv[k] = ys;
                    if (ex_any) {
                        inv_w_in = fmaf(yc, ta.invW[k], inv_w_in);
                        inv_w_new = fmaf(ys, ta.invW[k], inv_w_new);
                    }
                    if (FAST) {
                        Sf += ys;
#pragma unroll
                        for (int m = 0; m < 6; ++m) Chf[m] = fmaf(ys, ta.hhf[k][m], Chf[m]);
#pragma unroll
                        for (int m = 0; m < 5; ++m) Ccf[m] = fmaf(ys, ta.cpf[k][m], Ccf[m]);
                        continue;
                    }
                    const double yd = (double)ys;
                    S += yd;
                    if (!ta.two_ranges) {
#pragma unroll
                        for (int m = 0; m < 6; ++m) Ch[m] = fma(yd, ta.th.hh[k][0][m], Ch[m]);
#pragma unroll
                        for (int m = 0; m < 5; ++m) Cc[m] = fma(yd, ta.th.cp[k][0][m], Cc[m]);
                    }
                }
            }
            if (fwd_only) continue;
            // S6 (R8): divide by the sum; a vanishing sum falls back to max(Y,0)/sum (rare: the inputs are re-read)
            const bool degenerate = FAST ? !(Sf > 0.f) : !(S > 0.0);
            if (degenerate) {
                S = 0.0;
#pragma unroll
                for (int m = 0; m < 6; ++m) Ch[m] = 0.0;
#pragma unroll
                for (int m = 0; m < 5; ++m) Cc[m] = 0.0;
#pragma unroll 1
                for (int k = 0; k < Ns; ++k) S += (double)fmaxf(valid ? ta.Y[(int64_t)k * ta.n + g] : 0.f, 0.f);
                inv_w_new = 0.f;
#pragma unroll
                for (int k = 0; k < NSP; ++k) {
                    Yv[k] = (valid && k < Ns) ? fmaxf(ta.Y[(int64_t)k * ta.n + g], 0.f) : 0.f;
                    inv_w_new = fmaf(Yv[k], ta.invW[k], inv_w_new);
                    const double yd = (double)Yv[k];
#pragma unroll
                    for (int m = 0; m < 6; ++m) Ch[m] = fma(yd, ta.th.hh[k][0][m], Ch[m]);
#pragma unroll
                    for (int m = 0; m < 5; ++m) Cc[m] = fma(yd, ta.th.cp[k][0][m], Cc[m]);
                }
            }
            double rS;
            float rSf;
            if (FAST && !degenerate) {
                rSf = 1.f / Sf;
                rS = (double)rSf;
#pragma unroll
                for (int m = 0; m < 6; ++m) Ch[m] = (double)(Chf[m] * rSf);
#pragma unroll
                for (int m = 0; m < 5; ++m) Cc[m] = (double)(Ccf[m] * rSf);
            } else {
                rS = 1.0 / S;
                rSf = (float)rS;
#pragma unroll
                for (int m = 0; m < 6; ++m) Ch[m] *= rS;
#pragma unroll
                for (int m = 0; m < 5; ++m) Cc[m] *= rS;
            }
            // S7 (R9-R11): Newton on h(T) = sum_k Y_k h_k(T), FP64
            double Tn = fmin(fmax((double)Tin, ta.T_min), ta.T_max);
            bool conv = false;
            const double hc = (double)hin;
            for (int itn = 0; itn < ta.newton_max_iter; ++itn) {
                double f, c;
                if (FAST || !ta.two_ranges) {
                    f = horner6(Ch, Tn) - hc;
                    c = horner5(Cc, Tn);
                } else {
                    f = 0.0;
                    c = 0.0;
#pragma unroll
                    for (int k = 0; k < NSP; ++k) {
                        const int rg = (k < Ns && !(Tn < ta.th.T_mid[k])) ? 1 : 0;
                        const double yd = (double)Yv[k] * rS;
                        f = fma(yd, horner6(ta.th.hh[k][rg], Tn), f);
                        c = fma(yd, horner5(ta.th.cp[k][rg], Tn), c);
                    }
                    f -= hc;
                }
                if (!(c > 0.0)) break;  // R10: stop, not converged
                double dT;
                if (FAST) {
                    // -f / c through an FP32 reciprocal refined twice in FP64 (relative error ~1e-16): 5 FP64 instructions
                    // instead of the ~12 of the division sequence
                    double rc = (double)ptx::rcp_approx((float)c);
                    rc = fma(rc, fma(-c, rc, 1.0), rc);
                    rc = fma(rc, fma(-c, rc, 1.0), rc);
                    dT = -f * rc;
                } else {
                    dT = -f / c;
                }
                Tn = fmin(fmax(Tn + dT, ta.T_min), ta.T_max);
                if (fabs(dT) < ta.newton_tol) {
                    conv = true;
                    break;
                }
            }
            // gpuann_chem_step_ex: the inputs are read once more (cache hits) before they are overwritten
            if (ex_any && valid) {
                const float Tnf = (float)Tn;
                const float rate = pin / (8314.46261815324f * Tin * inv_w_in) * ta.inv_dt;  // rho of the input state / dt
                float q = 0.f, cpm = 0.f;
#pragma unroll
                for (int k = 0; k < NSP; ++k) {
                    if (k < Ns) {
                        const float ynew = FAST ? Yv[k] * rSf : (float)((double)Yv[k] * rS);
                        const float rr = rate * (ynew - ta.Y[(int64_t)k * ta.n + g]);
                        float hk;
                        if (FAST || !ta.two_ranges) {
                            const float *hh = ta.hhf[k];
                            hk = hh[0] + Tnf * (hh[1] + Tnf * (hh[2] + Tnf * (hh[3] + Tnf * (hh[4] + Tnf * hh[5]))));
                        } else {
                            const int rg = !(Tn < ta.th.T_mid[k]) ? 1 : 0;
                            hk = (float)horner6(ta.th.hh[k][rg], Tn);
                            cpm = fmaf(ynew, (float)horner5(ta.th.cp[k][rg], Tn), cpm);
                        }
                        q = fmaf(-hk, rr, q);
                        if (ta.ex.rr) ta.ex.rr[(int64_t)k * ta.n + g] = rr;
                    }
                }
                if (FAST || !ta.two_ranges) cpm = (float)horner5(Cc, Tn);  // the mixture coefficients are already those of Y_new
                const float psi = 1.f / (8314.46261815324f * (inv_w_new * rSf) * Tnf);
                if (ta.ex.hrr) ta.ex.hrr[g] = q;
                if (ta.ex.cp) ta.ex.cp[g] = cpm;
                if (ta.ex.rho) ta.ex.rho[g] = pin * psi;
                if (ta.ex.psi) ta.ex.psi[g] = psi;
            }
            // S8: store in place (skipped / out-of-range cells are never touched)
            if (valid) {
#pragma unroll
                for (int k = 0; k < NSP; ++k)
                    if (k < Ns) ta.Y[(int64_t)k * ta.n + g] = FAST ? Yv[k] * rSf : (float)((double)Yv[k] * rS);
                ta.T[g] = (float)Tn;
                if (!conv) ++nconv_total;
                if (degenerate) ++ndeg_total;
            }
        }
        // statistics: one atomic per warp and counter, only when something happened
        nconv_total = __reduce_add_sync(0xffffffffu, nconv_total);
        ndeg_total = __reduce_add_sync(0xffffffffu, ndeg_total);
        if (lane == 0) {
            if (nconv_total) atomicAdd(&ta.counters->n_not_converged, (unsigned long long)nconv_total);
            if (ndeg_total) atomicAdd(&ta.counters->n_degenerate, (unsigned long long)ndeg_total);
        }
    }

    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync_all();  // no CTA leaves while its peer may still signal its barriers or the pair's MMAs run
    if (warp == 1) {
        ptx::tc_fence_after_sync();
        ptx::tmem_dealloc_cg2(tmem_base, 512);
    }
}

// ---------------------------------------------------------------- host side
typedef void (*TailKernel)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const CUtensorMap, const TailArgs);

static TailKernel tail_kernel(int Ns, bool fast) {
    switch ((Ns + 7) / 8) {
        case 1: return fast ? k_tail<8, true> : k_tail<8, false>;
        case 2: return fast ? k_tail<16, true> : k_tail<16, false>;
        case 3: return fast ? k_tail<24, true> : k_tail<24, false>;
        case 4: return fast ? k_tail<32, true> : k_tail<32, false>;
        case 5: return fast ? k_tail<40, true> : k_tail<40, false>;
        default: return fast ? k_tail<48, true> : k_tail<48, false>;
    }
}

cudaError_t tail_setup(Ctx *c) {
    (void)c;
    for (int ns = 8; ns <= kTailMaxNs; ns += 8)
        for (int fast = 0; fast < 2; ++fast) {
            cudaError_t e = cudaFuncSetAttribute(tail_kernel(ns, fast != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmem);
            if (e != cudaSuccess) return e;
        }
    return cudaSuccess;
}

bool tail_supported(int K3p, int H3p, int Ns) {
    return K3p >= 16 && K3p % 16 == 0 && H3p >= 16 && H3p % 16 == 0 && H3p <= kTAccMax && Ns >= 1 && Ns <= kTailMaxNs;
}

// column halves of the layer-3 accumulator: one (<= 256 columns), or two with the first on a 64-column chunk boundary
void tail_plan(int H3p, int *n0, int *n1) {
    int a = H3p, b = 0;
    if (H3p > 256) {
        a = ((H3p + 63) / 64 / 2) * 64;
        b = H3p - a;
    }
    *n0 = a;
    *n1 = b;
}

cudaError_t launch_tail(Ctx *c, int64_t n, int64_t c0, int64_t cn, float *T, const float *p, float *Y, const float *h,
                        double dt, float *o_raw, int64_t o_stride, bool use_idx, const ExtraOut &ex, cudaStream_t s) {
    if (cn <= 0) return cudaSuccess;
    TailNet &tn = c->cur->tail;
    TailArgs &ta = tn.args;  // the constant part (thermo, net parameters) was filled at load time
    const LayerBf16 &l3 = c->cur->lay[c->L - 2], &l4 = c->cur->lay[c->L - 1];
    ta.n = n;
    ta.c0 = c0;
    ta.rows = cn;
    ta.n_active = use_idx ? c->n_active_dev : nullptr;
    ta.idx = use_idx ? c->idx : nullptr;
    ta.T = T;
    ta.Y = Y;
    ta.h = h;
    ta.p = p;
    ta.ex = ex;
    ta.inv_dt = (float)(1.0 / dt);
    ta.f16 = c->prm.precision == GPUANN_PRECISION_FP16 ? 1 : 0;
    ta.o_raw = o_raw;
    ta.o_stride = o_stride;
    ta.counters = c->counters;
    for (int k = 0; k < ta.Ns; ++k) {
        ta.sA[k] = (float)(dt * (double)c->post.out_std[k]);
        ta.sC[k] = (float)(dt * ((double)c->post.out_std[k] * (double)ta.b4[k] + (double)c->post.out_mean[k]));
    }
    const int64_t tiles = (cn + kTM - 1) / kTM;
    int grid = (int)(tiles < c->sm_count ? tiles : c->sm_count);
    grid = (grid + 1) & ~1;
    // INVARIANT of the kernel's prologue (it reads *n_active before griddepcontrol.wait): PDL only directly behind a kernel
    // of this context that was launched with full stream ordering and writes neither n_active nor the thermo / bias
    // tables.  Behind anything else (the compaction kernels, another tail kernel, nothing) the launch is an ordinary one.
    const bool pdl = c->last_cls == kClsFused || c->last_cls == kClsPre || (c->last_cls >= kClsLayer0 && c->last_cls < kClsLayer0 + kMaxLayers);
    LaunchScope ls(c, kClsTail, s);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kTailThreads);
    cfg.dynamicSmemBytes = kTailSmem;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // programmatic dependent launch: a tail CTA may start its prologue on an SM as soon as that SM's CTA of the kernel in
    // front has exited; the kernel itself waits (griddepcontrol.wait) before it touches h2 or the state
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 2 : 1;
    (void)l4;
    // species beyond Ns of the padded range must carry all-zero constants (the kernel's arithmetic is unguarded)
    for (int k = ta.Ns; k < kTailMaxNs; ++k) ta.sA[k] = ta.sC[k] = 0.f;
    const bool fast = !ta.lambda_zero && ta.inv_lambda_int == 10 && !ta.two_ranges;
    return cudaLaunchKernelEx(&cfg, tail_kernel(ta.Ns, fast), ta.a_blocked ? tn.tmapAb : l3.tmapA, tn.tmapW3a, tn.tmapW3b, tn.tmapW4, ta);
}

}  // namespace gpuann
