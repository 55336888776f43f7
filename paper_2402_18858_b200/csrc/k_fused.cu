// k_fused.cu -- "bf16-fused" variant, first kernel: S1 + S2 + the first TWO layers of S3 in one persistent kernel
//     z  = normalise(Box-Cox(state))                      (Eq. 7; R1, R2, R4)
//     h1 = GELU(z W1^T + b1)     [128 x H1]   never leaves the SM
//     h2 = GELU(h1 W2^T + b2)    [128 x H2]   -> global scratch, BF16 (input of the next layer kernel)
// Why: layer 2 holds 78 % of the FLOPs and its A operand h1 (3.2 KB/cell) is the largest
// activation; producing it on the fly from the 64-byte z row removes the h1 round trip and leaves the weights
// as the only L2 -> SMEM stream.  TMEM (512 columns) cannot hold a 128 x 800 FP32 accumulator, so the H2
// columns are processed in n_pass passes of <= 416 columns and h1 is recomputed per pass.
//
// Roles (512 threads, one CTA per SM, tiles of 128 cells walked with stride gridDim.x):
//   warp 0      TMA: W2 k-block [pass_w x 64] ring of 2, W1 rows [64 x 64] ring of 4 (runs 2 chunks ahead)
//   warp 1      layer-2 tcgen05.mma issuer + TMEM owner:  acc[0..pass_w) += h1 chunk (smem) x W2 k-block
//   warp 2      layer-1 tcgen05.mma issuer:  L1acc[slot] (128 x 32 FP32) = z tile (smem) x W1 rows; bias b1
//               rides in two extra K columns of W1 against two constant-1 columns of z (hi + lo BF16 split)
//   warp 3      z builder: state (SoA, gathered through idx when compaction is on) -> Box-Cox -> z-score ->
//               BF16 -> 128-byte-swizzled smem tile, double buffered across tiles
//   warps 4-11  h1 producers: tcgen05.ld of an L1 sub-chunk -> GELU -> BF16 -> swizzled A chunk
//   warps 12-15 pass epilogue: tcgen05.ld of acc -> + b2 -> GELU -> BF16 -> 64-byte row segments of h2 (global)
// The two MMA warps run warp-uniform loops and predicate only the tcgen05 instructions on one lane: inside an
// `if (lane == 0)` branch ptxas cannot use the uniform datapath and spends ~20 vector instructions + R2UR
// per MMA, which made ONE thread the bottleneck of the first version of this kernel (465 SASS instructions
// per 64-column chunk, ~3000 clk against 800 clk of MMA work; profiles/r01_fused_l1l2_v1.md).
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
constexpr int kFusedThreads = 512;

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


// ring position: stage index + phase bit, advanced without integer division
struct Ring {
    uint32_t st = 0, ph = 0;
    __device__ __forceinline__ void next(uint32_t n) {
        if (++st == n) {
            st = 0;
            ph ^= 1u;
        }
    }
};

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
    // CTAs run in clusters of two that share every weight tile: each CTA loads HALF of a W1 / W2 stage and multicasts
    // it to both (the kernel is bound by the L2 -> SM weight stream: 2.97 MB per 128-cell tile, 8.9 TB/s measured
    // against an L2 slice throughput cap of ~10-12 TB/s; profiles/r01_fused_l1l2.md).  Both CTAs of a pair must walk
    // the same number of tiles; the odd one may get a tile index past the end, which it processes as an empty tile.
    const uint32_t crank = ptx::cluster_ctarank();
    const int pair_first = (int)blockIdx.x & ~1;
    const int my_tiles = n_tiles > pair_first ? (n_tiles - pair_first + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int n_chunks = fa.H1 / kFK;

    if (threadIdx.x == 0) {
        // "empty" barriers of the weight rings collect one tcgen05.commit from EACH CTA of the pair
        for (int i = 0; i < kW2Stages; ++i) { ptx::mbar_init(&bars[bW2Full + i], 1); ptx::mbar_init(&bars[bW2Empty + i], 2); }
        for (int i = 0; i < kW1Stages; ++i) { ptx::mbar_init(&bars[bW1Full + i], 1); ptx::mbar_init(&bars[bW1Empty + i], 2); }
        for (int i = 0; i < kAStages; ++i) { ptx::mbar_init(&bars[bAFull + i], 8); ptx::mbar_init(&bars[bAEmpty + i], 1); }
        for (int i = 0; i < kL1Slots; ++i) { ptx::mbar_init(&bars[bL1Full + i], 1); ptx::mbar_init(&bars[bL1Empty + i], 4); }
        for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars[bZFull + i], 1); ptx::mbar_init(&bars[bZEmpty + i], 1); }
        ptx::mbar_init(&bars[bAccFull], 1);
        ptx::mbar_init(&bars[bAccEmpty], 4);
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
    ptx::cluster_sync_all();  // the peer's barriers are initialised before anything of ours can reach them
    ptx::tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    const uint64_t desc0 = ptx::umma_desc_sw128_kmajor(sbase);  // + (byte offset >> 4) addresses any tile below

    if (warp == 0) {
        // ================================================================ TMA: weights only (tile independent)
        if (lane == 0) {
            const int64_t total = (int64_t)my_tiles * fa.n_pass * n_chunks;
            const uint32_t w2_bytes = (uint32_t)(fa.n0 + fa.n1) * 128u;
            Ring w1, w2;
            int c1 = 0;           // chunk of the W1 sequence
            int c2 = 0, p2 = 0;   // chunk / pass of the W2 sequence
            for (int64_t i = 0; i < total + 2; ++i) {
                if (i < total) {
                    ptx::mbar_wait(&bars[bW1Empty + w1.st], w1.ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(&bars[bW1Full + w1.st], kW1StageBytes);
                    ptx::tma_load_2d_multicast(&tmapW1, &bars[bW1Full + w1.st],
                                               smem + kOffW1 + w1.st * kW1StageBytes + crank * (kW1StageBytes / 2), 0,
                                               c1 * kFK + (int)crank * (kFK / 2), 3);
                    w1.next(kW1Stages);
                    if (++c1 == n_chunks) c1 = 0;
                }
                if (i >= 2) {
                    ptx::mbar_wait(&bars[bW2Empty + w2.st], w2.ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(&bars[bW2Full + w2.st], w2_bytes);
                    unsigned char *dst = smem + kOffW2 + w2.st * kW2StageBytes;
                    const int h0 = fa.n0 / 2, h1 = fa.n1 / 2;  // rows of this CTA's halves of the two boxes
                    ptx::tma_load_2d_multicast(&tmapW2a, &bars[bW2Full + w2.st], dst + (size_t)crank * h0 * 128, c2 * kFK,
                                               p2 * fa.pass_w + (int)crank * h0, 3);
                    if (fa.n1 > 0)
                        ptx::tma_load_2d_multicast(&tmapW2b, &bars[bW2Full + w2.st],
                                                   dst + (size_t)fa.n0 * 128 + (size_t)crank * h1 * 128, c2 * kFK,
                                                   p2 * fa.pass_w + fa.n0 + (int)crank * h1, 3);
                    w2.next(kW2Stages);
                    if (++c2 == n_chunks) {
                        c2 = 0;
                        if (++p2 == fa.n_pass) p2 = 0;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================================================================ layer-2 MMA issuer (whole warp, uniform)
        const uint32_t idesc_n0 = ptx::umma_idesc_bf16_f32(kFM, (uint32_t)fa.n0);
        const uint32_t idesc_n1 = ptx::umma_idesc_bf16_f32(kFM, (uint32_t)(fa.n1 > 0 ? fa.n1 : 16));

        const uint64_t b1_off = (uint64_t)((uint32_t)fa.n0 * 128u >> 4);
        Ring a, w2;
        uint32_t acc_ph = 0;
        for (int it = 0; it < my_tiles; ++it) {
            for (int pass = 0; pass < fa.n_pass; ++pass) {
                ptx::mbar_wait(&bars[bAccEmpty], acc_ph ^ 1u);
                ptx::tc_fence_after_sync();
                for (int c = 0; c < n_chunks; ++c) {
                    ptx::mbar_wait(&bars[bW2Full + w2.st], w2.ph);
                    ptx::mbar_wait(&bars[bAFull + a.st], a.ph);
                    ptx::tc_fence_after_sync();
                    const uint64_t da = desc0 + (uint64_t)((kOffA + a.st * kAStageBytes) >> 4);
                    const uint64_t db = desc0 + (uint64_t)((kOffW2 + w2.st * kW2StageBytes) >> 4);
                    if (ptx::elect_one()) {
#pragma unroll
                        for (int k = 0; k < kFK / 16; ++k) {
                            const uint32_t accum = (c | k) ? 1u : 0u;
                            ptx::umma_bf16_ss(tmem_base, da + 2 * k, db + 2 * k, idesc_n0, accum);
                            if (fa.n1 > 0)
                                ptx::umma_bf16_ss(tmem_base + (uint32_t)fa.n0, da + 2 * k, db + b1_off + 2 * k, idesc_n1, accum);
                        }
                        ptx::umma_commit(&bars[bAEmpty + a.st]);
                        ptx::umma_commit_multicast(&bars[bW2Empty + w2.st], 3);
                    }
                    __syncwarp();
                    a.next(kAStages);
                    w2.next(kW2Stages);
                }
                if (ptx::elect_one()) ptx::umma_commit(&bars[bAccFull]);
                __syncwarp();
                acc_ph ^= 1u;
            }
        }
    } else if (warp == 2) {
        // ================================================================ layer-1 MMA issuer (whole warp, uniform)
        const uint32_t idesc_l1 = ptx::umma_idesc_bf16_f32(kFM, kSub);
        Ring w1, slot;
        for (int it = 0; it < my_tiles; ++it) {
            const uint32_t zb = (uint32_t)it & 1u;
            ptx::mbar_wait(&bars[bZFull + zb], ((uint32_t)it >> 1) & 1u);
            ptx::tc_fence_after_sync();
            const uint64_t dz = desc0 + (uint64_t)((kOffZ + zb * kZBytes) >> 4);
            for (int pass = 0; pass < fa.n_pass; ++pass) {
                for (int c = 0; c < n_chunks; ++c) {
                    ptx::mbar_wait(&bars[bW1Full + w1.st], w1.ph);
                    const uint64_t dw = desc0 + (uint64_t)((kOffW1 + w1.st * kW1StageBytes) >> 4);
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        ptx::mbar_wait(&bars[bL1Empty + slot.st], slot.ph ^ 1u);
                        ptx::tc_fence_after_sync();
                        const uint32_t d_tmem = tmem_base + kL1Col + slot.st * kSub;
                        const uint64_t dws = dw + (uint64_t)(s * ((kSub * 128) >> 4));
                        if (ptx::elect_one()) {
                            for (int k = 0; k < fa.Kz; ++k)
                                ptx::umma_bf16_ss(d_tmem, dz + 2 * k, dws + 2 * k, idesc_l1, k ? 1u : 0u);
                            ptx::umma_commit(&bars[bL1Full + slot.st]);
                        }
                        __syncwarp();
                        slot.next(kL1Slots);
                    }
                    if (ptx::elect_one()) ptx::umma_commit_multicast(&bars[bW1Empty + w1.st], 3);
                    __syncwarp();
                    w1.next(kW1Stages);
                }
            }
            if (ptx::elect_one()) ptx::umma_commit(&bars[bZEmpty + zb]);
            __syncwarp();
        }
    } else if (warp == 3) {
        // ================================================================ z builder (32 threads, 4 cells each)
        const int D = fa.D;
        const int n_units = 2 * fa.Kz;  // 16-byte units (8 features) that carry data
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int zb = it & 1;
            ptx::mbar_wait(&bars[bZEmpty + zb], ((uint32_t)(it >> 1) & 1u) ^ 1u);
            const uint32_t z_addr = sbase + kOffZ + zb * kZBytes;
            // 4 rows per lane (rr = lane + 32 q).  Loads first, arithmetic after: the 32 independent loads of a
            // unit (8 features x 4 rows) are in flight together -- one memory latency per unit instead of one per
            // load (the first version waited for every load in turn and needed ~100k clk per tile)
            int64_t g4[4];
            bool ok4[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int64_t i = (int64_t)tile * kFM + lane + 32 * q;
                ok4[q] = i < rows;
                int64_t g = fa.c0 + i;
                if (fa.idx) g = ok4[q] ? (int64_t)fa.idx[g] : 0;
                g4[q] = ok4[q] ? g : 0;
            }
#pragma unroll 1
            for (int u = 0; u < 8; ++u) {
                float x[4][8];
                if (u < n_units) {
#pragma unroll
                    for (int f = 0; f < 8; ++f) {
                        const int j = u * 8 + f;
                        const float *src = j == 0 ? fa.T : (j == 1 ? fa.p : fa.Y + (int64_t)(j - 2) * fa.n);
#pragma unroll
                        for (int q = 0; q < 4; ++q) x[q][f] = (j < D && ok4[q]) ? src[g4[q]] : 0.f;
                    }
#pragma unroll
                    for (int f = 0; f < 8; ++f) {
                        const int j = u * 8 + f;
                        const float mu = j < D ? fa.pre.mean[j] : 0.f, is = j < D ? fa.pre.inv_std[j] : 0.f;
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            float t = x[q][f];
                            if (j >= 2 && j < D) {
                                // z is rounded to BF16 (2^-9): the approximate lg2 / ex2 pair (2^-22) is ample here;
                                // Y = 0 still maps to exactly -1/lambda (R1, R2)
                                const float Yc = fmaxf(t, 0.f);
                                if (fa.pre.lambda_zero) t = logf(Yc);
                                else {
                                    const float uu = Yc > 0.f ? ptx::ex2_approx(fa.pre.lambda * ptx::lg2_approx(Yc)) : 0.f;
                                    t = (uu - 1.f) * fa.pre.inv_lambda;
                                }
                            }
                            t = (t - mu) * is;
                            if (j >= D && j < D + 2) t = 1.f;  // multiplies the hi / lo halves of b1 in W1 columns D, D+1
                            x[q][f] = ok4[q] ? t : 0.f;
                        }
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
#pragma unroll
                        for (int f = 0; f < 8; ++f) x[q][f] = 0.f;
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int rr = lane + 32 * q;
                    ptx::st_shared_v4(z_addr + (uint32_t)rr * 128u + (uint32_t)((u ^ (rr & 7)) << 4),
                                      ptx::pack_bf16x2(x[q][0], x[q][1]), ptx::pack_bf16x2(x[q][2], x[q][3]),
                                      ptx::pack_bf16x2(x[q][4], x[q][5]), ptx::pack_bf16x2(x[q][6], x[q][7]));
                }
            }
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&bars[bZFull + zb]);
        }
    } else if (warp < 12) {
        // ================================================================ h1 producers (warps 4..11)
        const int q = warp & 3;             // TMEM lane quarter
        const int set = (warp - 4) >> 2;    // which 32-column half of a 64-column chunk
        const int r = q * 32 + lane;        // row of the tile
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16) + kL1Col;
        const uint32_t swz = (uint32_t)(r & 7);
        const uint32_t row_off = (uint32_t)r * 128u;
        uint32_t slot = (uint32_t)set, slot_ph = 0;  // sub-chunk g = 2 c + set lives in slot g % 3, phase (g / 3) & 1
        Ring a;
        const int total_chunks = my_tiles * fa.n_pass * n_chunks;
#pragma unroll 1
        for (int c = 0; c < total_chunks; ++c) {
            ptx::mbar_wait(&bars[bL1Full + slot], slot_ph);
            ptx::tc_fence_after_sync();
            uint32_t v[32];
            ptx::tmem_ld32(lane_addr + slot * kSub, v);
            ptx::tmem_ld_wait();
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&bars[bL1Empty + slot]);
            uint32_t o[16];
#pragma unroll
            for (int j = 0; j < 16; ++j)
                o[j] = ptx::gelu2_pack(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
            ptx::mbar_wait(&bars[bAEmpty + a.st], a.ph ^ 1u);
            const uint32_t row_addr = sbase + kOffA + a.st * kAStageBytes + row_off;
#pragma unroll
            for (int i = 0; i < 4; ++i)
                ptx::st_shared_v4(row_addr + ((((uint32_t)(4 * set + i)) ^ swz) << 4), o[4 * i], o[4 * i + 1],
                                  o[4 * i + 2], o[4 * i + 3]);
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&bars[bAFull + a.st]);
            a.next(kAStages);
            slot += 2;
            if (slot >= kL1Slots) {
                slot -= kL1Slots;
                slot_ph ^= 1u;
            }
        }
    } else {
        // ================================================================ pass epilogue (warps 12..15)
        const int q = warp & 3;
        const int r = q * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        uint32_t acc_ph = 0;
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int64_t grow = (int64_t)tile * kFM + r;
            const bool row_ok = grow < rows;
            for (int pass = 0; pass < fa.n_pass; ++pass) {
                ptx::mbar_wait(&bars[bAccFull], acc_ph);
                ptx::tc_fence_after_sync();
                acc_ph ^= 1u;
                const int col_base = pass * fa.pass_w;
                int cur_w = fa.H2p - col_base;
                cur_w = cur_w < fa.pass_w ? cur_w : fa.pass_w;
                __nv_bfloat16 *dst_row = fa.h2 + grow * fa.H2p + col_base;
#pragma unroll 1
                for (int cc = 0; cc < cur_w; cc += 32) {
                    const bool full = cc + 32 <= cur_w;  // widths are multiples of 16: the tail piece has 16 columns
                    uint32_t v[32];
                    if (full) ptx::tmem_ld32(lane_addr + (uint32_t)cc, v);
                    else {
                        uint32_t w[16];
                        ptx::tmem_ld16(lane_addr + (uint32_t)cc, w);
#pragma unroll
                        for (int j = 0; j < 16; ++j) v[j] = w[j];
#pragma unroll
                        for (int j = 16; j < 32; ++j) v[j] = 0u;
                    }
                    ptx::tmem_ld_wait();
                    if (cc + 32 >= cur_w) {
                        // last accumulator read of this warp: hand the accumulator back to the MMA warp
                        ptx::tc_fence_before_sync();
                        __syncwarp();
                        if (lane == 0) ptx::mbar_arrive(&bars[bAccEmpty]);
                    }
                    const float4 *b4 = reinterpret_cast<const float4 *>(sBias + col_base + cc);
                    uint32_t o[16];
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const float4 b = (full || j < 4) ? b4[j] : make_float4(0.f, 0.f, 0.f, 0.f);
                        o[2 * j] = ptx::gelu2_pack(__uint_as_float(v[4 * j]) + b.x, __uint_as_float(v[4 * j + 1]) + b.y);
                        o[2 * j + 1] = ptx::gelu2_pack(__uint_as_float(v[4 * j + 2]) + b.z, __uint_as_float(v[4 * j + 3]) + b.w);
                    }
                    if (row_ok) {
                        uint4 *dst = reinterpret_cast<uint4 *>(dst_row + cc);
                        dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
                        dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
                        if (full) {
                            dst[2] = make_uint4(o[8], o[9], o[10], o[11]);
                            dst[3] = make_uint4(o[12], o[13], o[14], o[15]);
                        }
                    }
                }
            }
        }
    }

    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync_all();  // no CTA leaves while its peer may still multicast into it or signal its barriers
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
    int grid = (int)(tiles < c->sm_count ? tiles : c->sm_count);
    grid = (grid + 1) & ~1;  // clusters of two CTAs
    LaunchScope ls(c, kClsFused, s);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kFusedThreads);
    cfg.dynamicSmemBytes = kFusedSmem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_fused_l1l2, fn.tmapW1, fn.tmapW2a, fn.tmapW2b, fa);
}

}  // namespace gpuann
