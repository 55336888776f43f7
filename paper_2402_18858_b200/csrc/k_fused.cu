// k_fused.cu -- "bf16-fused" variant, first kernel: S1 + S2 + the first TWO layers of S3 in one persistent kernel
//     z  = normalise(Box-Cox(state))                      (Eq. 7; R1, R2, R4)
//     h1 = GELU(z W1^T + b1)     [128 x H1]   never leaves the SM
//     h2 = GELU(h1 W2^T + b2)    [128 x H2]   -> global scratch, BF16 (input of the next layer kernel)
// Why: layer 2 holds 78 % of the FLOPs and its A operand h1 (3.2 KB/cell) is the largest
// activation; producing it on the fly from the 64-byte z row removes the h1 round trip and leaves the weights
// as the only L2 -> SMEM stream.  TMEM (512 columns) cannot hold a 128 x 800 FP32 accumulator, so the H2
// columns are processed in n_pass passes of <= 416 columns and h1 is recomputed per pass (layer 1 is 2 % of
// the FLOPs; its GELU runs on otherwise idle ALUs under the layer-2 MMAs).
//
// Roles (384 threads, one CTA per SM, tiles of 128 cells walked with stride gridDim.x):
//   warp 0      TMA: W2 k-block [pass_w x 64] ring of 2, W1 rows [64 x 64] ring of 4 (runs 2 chunks ahead)
//   warp 1      tcgen05.mma issuer (one lane) + TMEM owner
//                 L1: D = L1acc[slot] (128 x 32 FP32), A = z tile (smem), B = W1 rows; bias b1 rides in two
//                     extra K columns of W1 against two constant-1 columns of z (hi + lo BF16 split)
//                 L2: D = acc[0..pass_w), A = h1 chunk (smem, written by the producers), B = W2 k-block
//   warps 2-3   z builder: state (SoA, gathered through idx when compaction is on) -> Box-Cox -> z-score ->
//               BF16 -> 128-byte-swizzled smem tile, double buffered across tiles
//   warps 4-11  producers / epilogue: tcgen05.ld of an L1 sub-chunk -> GELU -> BF16 -> swizzled A chunk;
//               after a pass: tcgen05.ld of acc -> + b2 -> GELU -> BF16 -> smem staging -> coalesced 16-byte
//               global stores of h2.
#include "common.cuh"
#include "post.cuh"
#include "ptx.cuh"

namespace gpuann {

constexpr int kFM = 128;         // cells per tile
constexpr int kFK = 64;          // K elements per smem row (128 B) = h1 columns per chunk
constexpr int kSub = 32;         // h1 columns per L1 sub-chunk (one TMEM slot)
constexpr int kW2Stages = 2;
constexpr int kW1Stages = 4;
constexpr int kAStages = 3;
constexpr int kL1Slots = 3;
constexpr int kAccCols = 416;    // TMEM columns of the layer-2 accumulator (max pass width)
constexpr int kL1Col = kAccCols; // L1 slots live in columns 416..511
constexpr int kFusedThreads = 384;
constexpr int kProdThreads = 256;

constexpr uint32_t kW2StageBytes = kAccCols * 128;  // 53,248
constexpr uint32_t kW1StageBytes = kFK * 128;       // 8,192
constexpr uint32_t kAStageBytes = kFM * 128;        // 16,384
constexpr uint32_t kZBytes = kFM * 128;             // 16,384
constexpr uint32_t kBias2Bytes = 4096;
constexpr uint32_t kOffW2 = 0;
constexpr uint32_t kOffW1 = kOffW2 + kW2Stages * kW2StageBytes;
constexpr uint32_t kOffA = kOffW1 + kW1Stages * kW1StageBytes;
constexpr uint32_t kOffZ = kOffA + kAStages * kAStageBytes;
constexpr uint32_t kOffBias = kOffZ + 2 * kZBytes;
constexpr uint32_t kOffBar = kOffBias + kBias2Bytes;
constexpr size_t kFusedSmem = 1024 + kOffBar + 512;

// barrier indices
enum {
    bW2Full = 0, bW2Empty = bW2Full + kW2Stages, bW1Full = bW2Empty + kW2Stages, bW1Empty = bW1Full + kW1Stages,
    bAFull = bW1Empty + kW1Stages, bAEmpty = bAFull + kAStages, bL1Full = bAEmpty + kAStages,
    bL1Empty = bL1Full + kL1Slots, bZFull = bL1Empty + kL1Slots, bZEmpty = bZFull + 2, bAccFull = bZEmpty + 2,
    bAccEmpty = bAccFull + 1, bCount = bAccEmpty + 1
};

struct FusedArgs {
    int64_t n;               // cells of the whole field (row stride of Y)
    int64_t c0;              // first (compacted) cell of this chunk
    int64_t rows;            // cells of this chunk (upper bound when n_active is given)
    const int32_t *n_active; // DEVICE or nullptr
    const int32_t *idx;      // DEVICE or nullptr: compacted -> field cell index
    const float *T, *p, *Y;
    int D, Kz;               // 2 + Ns; K-steps of layer 1 = ceil((D + 2) / 16)
    int H1, H2p;             // H1 % 64 == 0; padded H2
    int n_pass, pass_w, n0, n1;
    const float *bias2;      // [H2p]
    __nv_bfloat16 *h2;       // [rows][H2p]
    PreParams pre;
};

__device__ __forceinline__ float gelu_tanh_f(float v) {
    const float u = v * (0.7978845608028654f + 0.0356774081363001f * v * v);
    const float hv = 0.5f * v;
    return fmaf(hv, ptx::tanh_approx(u), hv);
}

__global__ void __launch_bounds__(kFusedThreads, 1)
k_fused_l1l2(const __grid_constant__ CUtensorMap tmapW1, const __grid_constant__ CUtensorMap tmapW2a,
             const __grid_constant__ CUtensorMap tmapW2b, const FusedArgs fa) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kOffBar);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + bCount);
    float *sBias = reinterpret_cast<float *>(smem + kOffBias);
    const uint32_t sbase = ptx::smem_u32(smem);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    int64_t rows = fa.rows;
    if (fa.n_active) {
        int64_t r = (int64_t)*fa.n_active - fa.c0;
        rows = r < 0 ? 0 : (r < rows ? r : rows);
    }
    const int n_tiles = (int)((rows + kFM - 1) / kFM);
    const int my_tiles = n_tiles > (int)blockIdx.x ? (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int n_chunks = fa.H1 / kFK;
    const int n_sub = 2 * n_chunks;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kW2Stages; ++i) { ptx::mbar_init(&bars[bW2Full + i], 1); ptx::mbar_init(&bars[bW2Empty + i], 1); }
        for (int i = 0; i < kW1Stages; ++i) { ptx::mbar_init(&bars[bW1Full + i], 1); ptx::mbar_init(&bars[bW1Empty + i], 1); }
        for (int i = 0; i < kAStages; ++i) { ptx::mbar_init(&bars[bAFull + i], 8); ptx::mbar_init(&bars[bAEmpty + i], 1); }
        for (int i = 0; i < kL1Slots; ++i) { ptx::mbar_init(&bars[bL1Full + i], 1); ptx::mbar_init(&bars[bL1Empty + i], 4); }
        for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars[bZFull + i], 2); ptx::mbar_init(&bars[bZEmpty + i], 1); }
        ptx::mbar_init(&bars[bAccFull], 1);
        ptx::mbar_init(&bars[bAccEmpty], 8);
        ptx::fence_mbar_init();
    }
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmapW1);
        ptx::prefetch_tensormap(&tmapW2a);
        ptx::prefetch_tensormap(&tmapW2b);
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, 512);
        ptx::tmem_relinquish();
    }
    for (int i = threadIdx.x; i < fa.H2p && i < (int)(kBias2Bytes / 4); i += kFusedThreads) sBias[i] = fa.bias2[i];
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ================================================================ TMA: weights only (tile independent)
        if (lane == 0) {
            const int per_tile = fa.n_pass * n_chunks;
            const int64_t total = (int64_t)my_tiles * per_tile;
            const uint32_t w2_bytes = (uint32_t)(fa.n0 + fa.n1) * 128u;
            for (int64_t i = 0; i < total + 2; ++i) {
                if (i < total) {
                    const int st = (int)(i & (kW1Stages - 1));
                    ptx::mbar_wait(&bars[bW1Empty + st], (uint32_t)((i / kW1Stages) & 1) ^ 1u);
                    ptx::mbar_arrive_expect_tx(&bars[bW1Full + st], kW1StageBytes);
                    ptx::tma_load_2d(&tmapW1, &bars[bW1Full + st], smem + kOffW1 + st * kW1StageBytes, 0,
                                     (int)(i % n_chunks) * kFK);
                }
                if (i >= 2) {
                    const int64_t j = i - 2;
                    const int st = (int)(j % kW2Stages);
                    const int chunk = (int)(j % n_chunks);
                    const int pass = (int)((j / n_chunks) % fa.n_pass);
                    ptx::mbar_wait(&bars[bW2Empty + st], (uint32_t)((j / kW2Stages) & 1) ^ 1u);
                    ptx::mbar_arrive_expect_tx(&bars[bW2Full + st], w2_bytes);
                    unsigned char *dst = smem + kOffW2 + st * kW2StageBytes;
                    ptx::tma_load_2d(&tmapW2a, &bars[bW2Full + st], dst, chunk * kFK, pass * fa.pass_w);
                    if (fa.n1 > 0)
                        ptx::tma_load_2d(&tmapW2b, &bars[bW2Full + st], dst + (size_t)fa.n0 * 128, chunk * kFK,
                                         pass * fa.pass_w + fa.n0);
                }
            }
        }
    } else if (warp == 1) {
        // ================================================================ MMA issuer
        if (lane == 0) {
            const uint32_t idesc_l1 = ptx::umma_idesc_bf16_f32(kFM, kSub);
            const uint32_t idesc_n0 = ptx::umma_idesc_bf16_f32(kFM, (uint32_t)fa.n0);
            const uint32_t idesc_n1 = ptx::umma_idesc_bf16_f32(kFM, (uint32_t)(fa.n1 > 0 ? fa.n1 : 16));
            uint32_t g1 = 0;   // L1 sub-chunks issued so far (ring of kL1Slots)
            uint32_t gw = 0;   // chunk sequence number at the start of the current pass
            uint32_t gc = 0;   // L2 chunks issued so far
            uint32_t acc_use = 0;
            for (int it = 0; it < my_tiles; ++it) {
                const int zb = it & 1;
                ptx::mbar_wait(&bars[bZFull + zb], (uint32_t)(it >> 1) & 1u);
                ptx::tc_fence_after_sync();
                const uint32_t z_addr = sbase + kOffZ + zb * kZBytes;
                for (int pass = 0; pass < fa.n_pass; ++pass) {
                    ptx::mbar_wait(&bars[bAccEmpty], (acc_use & 1u) ^ 1u);
                    ptx::tc_fence_after_sync();
                    auto issue_l1 = [&](int s) {
                        const uint32_t cw = gw + (uint32_t)(s >> 1);
                        const int wst = (int)(cw % kW1Stages);
                        if ((s & 1) == 0) {
                            ptx::mbar_wait(&bars[bW1Full + wst], (cw / kW1Stages) & 1u);
                            ptx::tc_fence_after_sync();
                        }
                        const int slot = (int)(g1 % kL1Slots);
                        ptx::mbar_wait(&bars[bL1Empty + slot], ((g1 / kL1Slots) & 1u) ^ 1u);
                        ptx::tc_fence_after_sync();
                        const uint32_t b_addr = sbase + kOffW1 + wst * kW1StageBytes + (uint32_t)(s & 1) * (kSub * 128);
                        const uint32_t d_tmem = tmem_base + kL1Col + (uint32_t)slot * kSub;
                        for (int k = 0; k < fa.Kz; ++k)
                            ptx::umma_bf16_ss(d_tmem, ptx::umma_desc_sw128_kmajor(z_addr + k * 32),
                                              ptx::umma_desc_sw128_kmajor(b_addr + k * 32), idesc_l1, k ? 1u : 0u);
                        ptx::umma_commit(&bars[bL1Full + slot]);
                        ++g1;
                    };
                    issue_l1(0);
                    issue_l1(1);
                    for (int c = 0; c < n_chunks; ++c) {
                        if (c + 1 < n_chunks) {
                            issue_l1(2 * c + 2);
                            issue_l1(2 * c + 3);
                        }
                        const int ast = (int)(gc % kAStages), wst2 = (int)(gc % kW2Stages);
                        ptx::mbar_wait(&bars[bW2Full + wst2], (gc / kW2Stages) & 1u);
                        ptx::mbar_wait(&bars[bAFull + ast], (gc / kAStages) & 1u);
                        ptx::tc_fence_after_sync();
                        const uint32_t a_addr = sbase + kOffA + ast * kAStageBytes;
                        const uint32_t b_addr = sbase + kOffW2 + wst2 * kW2StageBytes;
#pragma unroll
                        for (int k = 0; k < kFK / 16; ++k) {
                            const uint64_t da = ptx::umma_desc_sw128_kmajor(a_addr + k * 32);
                            ptx::umma_bf16_ss(tmem_base, da, ptx::umma_desc_sw128_kmajor(b_addr + k * 32), idesc_n0,
                                              (c | k) ? 1u : 0u);
                            if (fa.n1 > 0)
                                ptx::umma_bf16_ss(tmem_base + (uint32_t)fa.n0, da,
                                                  ptx::umma_desc_sw128_kmajor(b_addr + (uint32_t)fa.n0 * 128 + k * 32),
                                                  idesc_n1, (c | k) ? 1u : 0u);
                        }
                        ptx::umma_commit(&bars[bAEmpty + ast]);
                        ptx::umma_commit(&bars[bW2Empty + wst2]);
                        ptx::umma_commit(&bars[bW1Empty + (int)((gw + (uint32_t)c) % kW1Stages)]);
                        ++gc;
                    }
                    if (pass == fa.n_pass - 1) ptx::umma_commit(&bars[bZEmpty + zb]);
                    ptx::umma_commit(&bars[bAccFull]);
                    gw += (uint32_t)n_chunks;
                    ++acc_use;
                }
            }
        }
    } else if (warp < 4) {
        // ================================================================ z builder (64 threads, 2 cells each)
        const int zt = (int)threadIdx.x - 64;
        const int D = fa.D;
        const int n_units = 2 * fa.Kz;  // 16-byte units (8 features) that carry data
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int zb = it & 1;
            ptx::mbar_wait(&bars[bZEmpty + zb], ((uint32_t)(it >> 1) & 1u) ^ 1u);
            const uint32_t z_addr = sbase + kOffZ + zb * kZBytes;
#pragma unroll 1
            for (int rr = zt; rr < kFM; rr += 64) {
                const int64_t i = (int64_t)tile * kFM + rr;
                const bool valid = i < rows;
                int64_t g = fa.c0 + i;
                if (fa.idx) g = valid ? (int64_t)fa.idx[g] : 0;
                const uint32_t row_addr = z_addr + (uint32_t)rr * 128u;
                for (int u = 0; u < 8; ++u) {
                    float v[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const int j = u * 8 + q;
                        float x = 0.f;
                        if (valid && u < n_units) {
                            if (j < D) {
                                if (j == 0) x = fa.T[g];
                                else if (j == 1) x = fa.p[g];
                                else {
                                    const float Yc = fmaxf(fa.Y[(int64_t)(j - 2) * fa.n + g], 0.f);
                                    x = boxcox_y(Yc, boxcox_u(Yc, fa.pre.lambda), fa.pre);
                                }
                                x = (x - fa.pre.mean[j]) * fa.pre.inv_std[j];
                            } else if (j < D + 2) {
                                x = 1.f;  // multiplies the hi / lo halves of b1 stored in W1 columns D, D+1
                            }
                        }
                        v[q] = x;
                    }
                    ptx::st_shared_v4(row_addr + (uint32_t)((u ^ (rr & 7)) << 4), ptx::pack_bf16x2(v[0], v[1]),
                                      ptx::pack_bf16x2(v[2], v[3]), ptx::pack_bf16x2(v[4], v[5]),
                                      ptx::pack_bf16x2(v[6], v[7]));
                }
            }
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&bars[bZFull + zb]);
        }
    } else {
        // ================================================================ producers / epilogue (warps 4..11)
        const int q = warp & 3;             // TMEM lane quarter
        const int set = (warp - 4) >> 2;    // which 32-column half of a 64-column chunk / piece
        const int r = q * 32 + lane;        // row of the tile
        const int pt = (int)threadIdx.x - 128;  // 0..255
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        const uint32_t swz = (uint32_t)(r & 7);
        uint32_t gsub = 0, gch = 0, acc_use = 0;
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            for (int pass = 0; pass < fa.n_pass; ++pass) {
                // ---------------- h1 sub-chunks of this warp set
                for (int s = set; s < n_sub; s += 2) {
                    const uint32_t g = gsub + (uint32_t)s;
                    const int slot = (int)(g % kL1Slots);
                    ptx::mbar_wait(&bars[bL1Full + slot], (g / kL1Slots) & 1u);
                    ptx::tc_fence_after_sync();
                    uint32_t v[32];
                    ptx::tmem_ld32(lane_addr + kL1Col + (uint32_t)slot * kSub, v);
                    ptx::tmem_ld_wait();
                    ptx::tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(&bars[bL1Empty + slot]);
                    uint32_t o[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        o[j] = ptx::pack_bf16x2(gelu_tanh_f(__uint_as_float(v[2 * j])),
                                                gelu_tanh_f(__uint_as_float(v[2 * j + 1])));
                    const uint32_t gc = gch + (uint32_t)(s >> 1);
                    const int ast = (int)(gc % kAStages);
                    ptx::mbar_wait(&bars[bAEmpty + ast], ((gc / kAStages) & 1u) ^ 1u);
                    const uint32_t row_addr = sbase + kOffA + ast * kAStageBytes + (uint32_t)r * 128u;
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        ptx::st_shared_v4(row_addr + ((((uint32_t)(4 * set + i)) ^ swz) << 4), o[4 * i], o[4 * i + 1],
                                          o[4 * i + 2], o[4 * i + 3]);
                    ptx::fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(&bars[bAFull + ast]);
                }
                gsub += (uint32_t)n_sub;
                gch += (uint32_t)n_chunks;

                // ---------------- epilogue of the pass: acc -> + b2 -> GELU -> BF16 -> staging -> global
                ptx::mbar_wait(&bars[bAccFull], acc_use & 1u);
                ptx::tc_fence_after_sync();
                ++acc_use;
                const int col_base = pass * fa.pass_w;
                int cur_w = fa.H2p - col_base;
                cur_w = cur_w < fa.pass_w ? cur_w : fa.pass_w;
                const int n_pieces = (cur_w + kFK - 1) / kFK;
                // last piece in which this warp set still reads the accumulator (-1: it reads nothing)
                const int last_pc = cur_w > set * kSub ? (cur_w - set * kSub - 1) / kFK : -1;
                if (last_pc < 0) {
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(&bars[bAccEmpty]);
                }
                for (int pc = 0; pc < n_pieces; ++pc) {
                    const int col_lo = pc * kFK + set * kSub;  // within the pass
                    const uint32_t stage_addr = sbase + kOffA + (uint32_t)(pc % kAStages) * kAStageBytes;
                    if (col_lo < cur_w) {
                        uint32_t v[32];
                        ptx::tmem_ld32(lane_addr + (uint32_t)col_lo, v);
                        ptx::tmem_ld_wait();
                        if (pc == last_pc) {
                            // last accumulator read of this warp: hand the accumulator back to the MMA warp
                            ptx::tc_fence_before_sync();
                            __syncwarp();
                            if (lane == 0) ptx::mbar_arrive(&bars[bAccEmpty]);
                        }
                        const float4 *b4 = reinterpret_cast<const float4 *>(sBias + col_base + col_lo);
                        uint32_t o[16];
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const float4 b = b4[j];
                            o[2 * j] = ptx::pack_bf16x2(gelu_tanh_f(__uint_as_float(v[4 * j]) + b.x),
                                                        gelu_tanh_f(__uint_as_float(v[4 * j + 1]) + b.y));
                            o[2 * j + 1] = ptx::pack_bf16x2(gelu_tanh_f(__uint_as_float(v[4 * j + 2]) + b.z),
                                                            gelu_tanh_f(__uint_as_float(v[4 * j + 3]) + b.w));
                        }
                        const uint32_t row_addr = stage_addr + (uint32_t)r * 128u;
#pragma unroll
                        for (int i = 0; i < 4; ++i)
                            ptx::st_shared_v4(row_addr + ((((uint32_t)(4 * set + i)) ^ swz) << 4), o[4 * i],
                                              o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
                    }
                    ptx::named_bar_sync(1, kProdThreads);
                    // copy the 128 x 64 piece out: unit = 16 bytes = 8 columns; a warp covers 4 rows x 128 bytes
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int unit = pt + i * kProdThreads;
                        const int row = unit >> 3, u = unit & 7;
                        const int col = pc * kFK + u * 8;
                        const int64_t grow = (int64_t)tile * kFM + row;
                        if (col < cur_w && grow < rows) {
                            const uint4 val = ptx::ld_shared_v4(stage_addr + (uint32_t)row * 128u + (uint32_t)((u ^ (row & 7)) << 4));
                            *reinterpret_cast<uint4 *>(fa.h2 + grow * fa.H2p + col_base + col) = val;
                        }
                    }
                }
                // staging aliases the A stages: nobody may start the next pass's producer stores before every
                // thread has finished reading the last piece
                ptx::named_bar_sync(1, kProdThreads);
            }
        }
    }

    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after_sync();
        ptx::tmem_dealloc(tmem_base, 512);
    }
}

// ---------------------------------------------------------------- host side
cudaError_t fused_setup(Ctx *c) {
    (void)c;
    return cudaFuncSetAttribute(k_fused_l1l2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
}

bool fused_supported(int D, int H1, int H2p) {
    return D + 2 <= kFK && H1 >= 2 * kFK && H1 % kFK == 0 && H2p >= 16 && H2p <= (int)(kBias2Bytes / 4) && H2p % 16 == 0;
}

void fused_plan(int H2p, int *n_pass, int *pass_w, int *n0, int *n1) {
    const int np = (H2p + kAccCols - 1) / kAccCols;
    int pw = ((H2p + np - 1) / np + 15) / 16 * 16;
    int a = pw, b = 0;
    if (pw > 256) {
        a = ((pw / 2) + 15) / 16 * 16;
        b = pw - a;
    }
    *n_pass = np;
    *pass_w = pw;
    *n0 = a;
    *n1 = b;
}

cudaError_t launch_fused_l1l2(Ctx *c, int64_t n, int64_t c0, int64_t cn, const float *T, const float *p, const float *Y,
                              bool use_idx, cudaStream_t s) {
    if (cn <= 0) return cudaSuccess;
    const FusedNet &fn = c->fused;
    FusedArgs fa{};
    fa.n = n;
    fa.c0 = c0;
    fa.rows = cn;
    fa.n_active = use_idx ? c->n_active_dev : nullptr;
    fa.idx = use_idx ? c->idx : nullptr;
    fa.T = T;
    fa.p = p;
    fa.Y = Y;
    fa.D = c->sizes[0];
    fa.Kz = (c->sizes[0] + 2 + 15) / 16;
    fa.H1 = c->sizes[1];
    fa.H2p = c->lay[1].Np;
    fa.n_pass = fn.n_pass;
    fa.pass_w = fn.pass_w;
    fa.n0 = fn.n0;
    fa.n1 = fn.n1;
    fa.bias2 = c->lay[1].bias;
    fa.h2 = c->act[0];
    fa.pre = c->pre;
    const int64_t tiles = (cn + kFM - 1) / kFM;
    const int grid = (int)(tiles < c->sm_count ? tiles : c->sm_count);
    LaunchScope ls(c, kClsFused, s);
    k_fused_l1l2<<<grid, kFusedThreads, kFusedSmem, s>>>(fn.tmapW1, fn.tmapW2a, fn.tmapW2b, fa);
    return cudaGetLastError();
}

}  // namespace gpuann
