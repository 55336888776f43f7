// k_fused.cu -- tensor path, first kernel: S1 + S2 + the first TWO layers of S3 in one persistent kernel
//     z  = normalise(Box-Cox(state))                      (Eq. 7; R1, R2, R4)
//     h1 = GELU(z W1^T + b1)     [128 x H1]   never leaves the SM -- not even into shared memory
//     h2 = GELU(h1 W2^T + b2)    [128 x H2]   -> global scratch, BF16 (input of the tail kernel)
// Why: layer 2 holds 78 % of the FLOPs and its A operand h1 (3.2 KB/cell) is the largest activation.
// TMEM (512 columns) cannot hold a 128 x 800 FP32 accumulator, so the H2 columns are processed in n_pass passes of
// <= 400 columns and h1 is recomputed per pass (4 % more MMA work; the alternatives -- h1 through L2 or through
// distributed shared memory -- cost more bandwidth than either has).
//
// Data path of one 32-column piece of h1 ("slot step"; TMEM columns 400..511: two layer-1 accumulators of 32 FP32 columns
// and three A slots of 16 columns):
//     tcgen05.mma  L1acc[g & 1] (128 x 32 FP32, TMEM) = z tile (smem) x W1 rows (smem); b1 rides in two extra K columns
//     workers      tcgen05.ld (accumulator free again) -> 2 GELU -> BF16 pairs -> tcgen05.st into A slot g % 3
//     tcgen05.mma  acc[0..pass_w) += A slot (A operand read from TENSOR MEMORY) x W2 k-slab (smem)
// so h1 costs no shared-memory bandwidth at all: the only shared-memory streams left are the W2 / W1 slabs written by
// TMA and read by the MMAs (the first version of this kernel kept h1 in a shared-memory ring and ran the MMAs' operand
// reads + TMA writes + the producers' stores at ~120 % of the 128 B/clk the shared memory delivers at full tensor rate).
// Five pieces are in flight (two accumulators + three slots), so neither issuer waits for a conversion in steady state.
//
// CTA PAIRS: clusters of 2 whose even CTA (the leader) issues every tcgen05.mma with cta_group::2 -- M = 256 = the
// 128-cell tiles of both CTAs, B read half from each CTA's shared memory: a CTA stages and reads HALF of every W1 / W2
// slab (six W2 stages instead of two).
//
// Roles (512 threads, one CTA per SM, tiles of 128 cells walked with stride gridDim.x):
//   warp 14     TMA (both CTAs): own half of each W2 k-slab [pass_w/2 x 64] (ring of 6) and of each W1 row block (ring
//               of 4); completion is counted on the LEADER's full barriers
//   warp 15     (leader) layer-2 issuer: acc += A slot (TMEM) x W2 slab; its commit hands the slot back to the workers
//   warp 13     (leader) layer-1 issuer: runs up to two accumulators ahead of the workers.  Two issuer warps because ONE
//               warp's instruction stream (waits ~90 clk each, descriptor set-up, 6 MMAs, 2-3 commits) took ~1000 clk
//               per step against the 480 clk the tensor pipe needs (profiles/r02_ncu_full_c2.md)
//   warp 12     z builder: state (SoA, 128-bit loads; gathered through idx under compaction) -> Box-Cox -> z-score ->
//               BF16 -> 128-byte-swizzled smem tile, double buffered across tiles
//   warps 0-11  workers, three groups of four warps (one per TMEM lane quarter); group s converts steps g = s mod 3 into A
//               slot s.  At the end of
//               a pass ALL twelve drain the accumulator (tcgen05.ld -> + b2 -> 2 GELU -> BF16 -> h2), every third
//               32-column block each: the drain is bound by the SFU (one tanh per element), so it takes all four SM
//               sub-partitions to keep the tensor pipe's idle time per pass near 51,200 / 14 per clk = 3.7 k clk
// Barriers the leader's issuer waits on live in the leader and collect arrivals (cluster-scope release) or TMA bytes
// from BOTH CTAs; barriers that release something to a CTA's own warps are signalled in both CTAs by one multicast
// tcgen05.commit.
#include <type_traits>
#include "common.cuh"
#include "ptx.cuh"

namespace gpuann {

constexpr int kFM = 128;         // cells per tile
constexpr int kFK = 64;          // K elements per shared-memory row (128 B) = h1 columns per weight stage
constexpr int kSub = 32;         // h1 columns per slot step
constexpr int kW2Stages = 6;
constexpr int kW1Stages = 4;
constexpr int kL1Accs = 2;       // layer-1 accumulators (32 FP32 columns each)
constexpr int kASlots = 3;       // converted h1 pieces = A operands of layer 2 (16 columns of BF16 pairs each)
constexpr int kAccCols = 400;    // TMEM columns of the layer-2 accumulator (max pass width)
constexpr int kL1Col = kAccCols;                   // 400..463: the two layer-1 accumulators
constexpr int kACol = kL1Col + kL1Accs * kSub;     // 464..511: the three A slots
constexpr int kFusedThreads = 512;
constexpr int kWorkerGroups = 3;
// Warp numbering follows the issue arbiter, which serves the HIGHEST warp id of a sub-partition first (measured: as warp 1,
// behind three GELU-dense worker warps on its sub-partition, the MMA issuer got an issue slot every ~10 clk and needed
// 1000 clk per slot step): workers are warps 0..11, the latency-critical single-thread roles sit on
// top, one per sub-partition.
constexpr int kWarpZ = 12;
constexpr int kWarpMma1 = 13;  // layer-1 issuer
constexpr int kWarpTma = 14;
constexpr int kWarpMma2 = 15;  // layer-2 issuer, TMEM owner

constexpr uint32_t kW2StageBytes = (kAccCols / 2) * 128;   // this CTA's half of the rows of a pass: 26,624
constexpr uint32_t kW1SubBytes = (kSub / 2) * 128;         // this CTA's 16 of the 32 W1 rows of a slot step: 2,048
constexpr uint32_t kW1StageBytes = 2 * kW1SubBytes;        // two slot steps
constexpr uint32_t kZBytes = kFM * 128;                    // 16,384
constexpr uint32_t kBias2Bytes = 4096;
constexpr uint32_t kOffW2 = 0;
constexpr uint32_t kOffW1 = kOffW2 + kW2Stages * kW2StageBytes;
constexpr uint32_t kOffZ = kOffW1 + kW1Stages * kW1StageBytes;
constexpr uint32_t kOffBias = kOffZ + 2 * kZBytes;
constexpr uint32_t kOffBar = kOffBias + kBias2Bytes;
constexpr size_t kFusedSmem = 1024 + kOffBar + 512;

// barrier indices
enum {
    bW2Full = 0, bW2Empty = bW2Full + kW2Stages, bW1Full = bW2Empty + kW2Stages, bW1Empty = bW1Full + kW1Stages,
    bL1Full = bW1Empty + kW1Stages, bL1Free = bL1Full + kASlots, bAFull = bL1Free + kL1Accs, bAFree = bAFull + kASlots,
    bZFull = bAFree + kASlots, bZEmpty = bZFull + 2,
    bAccFull = bZEmpty + 2, bAccEmpty = bAccFull + 1, bCount = bAccEmpty + 1
};

struct FusedArgs {
    int64_t n;               // cells of the whole field (row stride of Y)
    int64_t c0;              // first (compacted) cell of this chunk
    int64_t rows;            // cells of this chunk (upper bound when n_active is given)
    const int32_t *n_active; // DEVICE or nullptr
    const int32_t *idx;      // DEVICE or nullptr: compacted -> field cell index
    const float *T, *p, *Y;
    int D, Kz;               // 2 + Ns; K-steps of layer 1 = ceil((D + 2) / 16)
    int H1p, H2p;            // H1 padded to a multiple of 64 (zero rows of W1, zero-filled K columns of W2); padded H2
    int n_pass, pass_w, n0, n1;
    const float *bias2;      // [H2p]
    __nv_bfloat16 *h2;       // [rows][H2p] row-major, or blocked [tile][H2p / 8][128][8] (common.cuh, FusedNet)
    int h2_blocked;
    int f16;                 // 1: FP16 operands (GPUANN_PRECISION_FP16), 0: BF16
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

// F16: FP16 operands (GPUANN_PRECISION_FP16) instead of BF16 -- a template parameter so that the BF16 instance pays nothing
template <bool F16>
__global__ void __launch_bounds__(kFusedThreads, 1)
k_fused_l1l2(const __grid_constant__ CUtensorMap tmapW1, const __grid_constant__ CUtensorMap tmapW2a,
             const __grid_constant__ CUtensorMap tmapW2b, const __grid_constant__ FusedArgs fa) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kOffBar);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + bCount);
    float *sBias = reinterpret_cast<float *>(smem + kOffBias);
    const uint32_t sbase = ptx::smem_u32(smem);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr bool f16 = F16;

    int64_t rows = fa.rows;
    if (fa.n_active) {
        int64_t r = (int64_t)*fa.n_active - fa.c0;
        rows = r < 0 ? 0 : (r < rows ? r : rows);
    }
    const int n_tiles = (int)((rows + kFM - 1) / kFM);
    // both CTAs of a pair walk the same number of tiles (every MMA covers both); the odd one may get a tile index past
    // the end, which it processes as an empty tile
    const uint32_t crank = ptx::cluster_ctarank();
    const bool leader = crank == 0;
    const int pair_first = (int)blockIdx.x & ~1;
    const int my_tiles = n_tiles > pair_first ? (n_tiles - pair_first + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int n_chunks = fa.H1p / kFK;
    const int nsteps = fa.H1p / kSub;                      // slot steps per pass (even, >= 4)
    const int total_steps = my_tiles * fa.n_pass * nsteps;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kW2Stages; ++i) { ptx::mbar_init(&bars[bW2Full + i], 1); ptx::mbar_init(&bars[bW2Empty + i], 1); }
        for (int i = 0; i < kW1Stages; ++i) { ptx::mbar_init(&bars[bW1Full + i], 1); ptx::mbar_init(&bars[bW1Empty + i], 1); }
        for (int i = 0; i < kASlots; ++i) {
            ptx::mbar_init(&bars[bL1Full + i], 1);  // one per worker group: "your step's layer-1 accumulator is complete"
            ptx::mbar_init(&bars[bAFull + i], 8);   // the four warps of the slot's group in BOTH CTAs
            ptx::mbar_init(&bars[bAFree + i], 1);
        }
        for (int i = 0; i < kL1Accs; ++i) ptx::mbar_init(&bars[bL1Free + i], 8);
        for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars[bZFull + i], 2); ptx::mbar_init(&bars[bZEmpty + i], 1); }
        ptx::mbar_init(&bars[bAccFull], 1);
        ptx::mbar_init(&bars[bAccEmpty], 2 * 4 * kWorkerGroups);
        ptx::fence_mbar_init();
    }
    if (warp == kWarpTma && lane == 0) {
        ptx::prefetch_tensormap(&tmapW1);
        ptx::prefetch_tensormap(&tmapW2a);
        ptx::prefetch_tensormap(&tmapW2b);
    }
    if (warp == kWarpMma2) {
        ptx::tmem_alloc_cg2(tmem_slot, 512);
        ptx::tmem_relinquish_cg2();
    }
    for (int i = threadIdx.x; i < fa.H2p && i < (int)(kBias2Bytes / 4); i += kFusedThreads) sBias[i] = fa.bias2[i];
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync_all();  // the peer's barriers are initialised before anything of ours can reach them
    ptx::tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;
    const uint64_t desc0 = ptx::umma_desc_sw128_kmajor(sbase);  // + (byte offset >> 4) addresses any tile below
    const uint32_t bars_leader = ptx::mapa_u32(ptx::smem_u32(bars), 0);  // the leader's barrier array, cluster address

    if (warp == kWarpTma) {
        // ================================================================ TMA: weights only (tile independent), both CTAs
        if (lane == 0) {
            const uint32_t sbase_cl = ptx::mapa_u32(sbase, crank);  // own shared memory in the cluster window
            const int64_t total = (int64_t)my_tiles * fa.n_pass * n_chunks;
            const int h0 = fa.n0 / 2, h1 = fa.n1 / 2;  // rows of this CTA's halves of the two column blocks
            const uint32_t w2_bytes = (uint32_t)(fa.n0 + fa.n1) * 128u;  // both CTAs' halves together
            Ring w1, w2;
            int c1 = 0;           // chunk of the W1 sequence
            int c2 = 0, p2 = 0;   // chunk / pass of the W2 sequence
            for (int64_t i = 0; i < total + 2; ++i) {
                if (i < total) {  // W1 runs two chunks ahead of W2: layer 1 is issued three slot steps ahead of layer 2
                    ptx::mbar_wait(&bars[bW1Empty + w1.st], w1.ph ^ 1u);
                    if (leader) ptx::mbar_arrive_expect_tx(&bars[bW1Full + w1.st], 2u * kW1StageBytes);
                    const uint32_t full = bars_leader + 8u * (bW1Full + w1.st);
                    const uint32_t dst = sbase_cl + kOffW1 + w1.st * kW1StageBytes;
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        ptx::tma_load_2d_cg2(&tmapW1, full, dst + s * kW1SubBytes, 0, c1 * kFK + s * kSub + (int)crank * (kSub / 2));
                    w1.next(kW1Stages);
                    if (++c1 == n_chunks) c1 = 0;
                }
                if (i >= 2) {
                    ptx::mbar_wait(&bars[bW2Empty + w2.st], w2.ph ^ 1u);
                    if (leader) ptx::mbar_arrive_expect_tx(&bars[bW2Full + w2.st], w2_bytes);
                    const uint32_t full = bars_leader + 8u * (bW2Full + w2.st);
                    const uint32_t dst = sbase_cl + kOffW2 + w2.st * kW2StageBytes;
                    ptx::tma_load_2d_cg2(&tmapW2a, full, dst, c2 * kFK, p2 * fa.pass_w + (int)crank * h0);
                    if (fa.n1 > 0)
                        ptx::tma_load_2d_cg2(&tmapW2b, full, dst + (uint32_t)h0 * 128u, c2 * kFK, p2 * fa.pass_w + fa.n0 + (int)crank * h1);
                    w2.next(kW2Stages);
                    if (++c2 == n_chunks) {
                        c2 = 0;
                        if (++p2 == fa.n_pass) p2 = 0;
                    }
                }
            }
        }
    } else if (warp == kWarpMma2) {
        // ================================================================ layer-2 MMA issuer (leader; whole warp, uniform)
        if (leader && total_steps > 0) {
            const uint32_t idesc_n0 = ptx::umma_idesc_bf16_f32(2 * kFM, (uint32_t)fa.n0, F16);
            const uint32_t idesc_n1 = ptx::umma_idesc_bf16_f32(2 * kFM, (uint32_t)(fa.n1 > 0 ? fa.n1 : 16), F16);
            const uint64_t b1_off = (uint64_t)((uint32_t)(fa.n0 / 2) * 128u >> 4);
            Ring w2;
            uint32_t slot = 0, a_ph = 0 /* bit s: parity of slot s's next "converted" phase */, acc_ph = 0;
            int j = 0;
            for (int g = 0; g < total_steps; ++g) {
                if (j == 0) ptx::mbar_wait(&bars[bAccEmpty], acc_ph ^ 1u);
                // both barriers of the step are polled together: a successful try_wait alone costs ~90 clk of this warp
                ptx::mbar_wait2(&bars[bAFull + slot], (a_ph >> slot) & 1u, &bars[bW2Full + w2.st], w2.ph);
                ptx::tc_fence_after_sync();
                a_ph ^= 1u << slot;
                const uint32_t a_tmem = tmem_base + kACol + slot * (kSub / 2);
                const uint64_t db = desc0 + (uint64_t)((kOffW2 + w2.st * kW2StageBytes) >> 4) + (uint64_t)((j & 1) * (kSub * 2 / 16));
                const bool last_of_pass = j == nsteps - 1;
                if (ptx::elect_one()) {
#pragma unroll
                    for (int k = 0; k < kSub / 16; ++k) {
                        const uint32_t accum = (j | k) ? 1u : 0u;
                        ptx::umma_bf16_ts_cg2(tmem_base, a_tmem + 8u * k, db + 2 * k, idesc_n0, accum);
                        if (fa.n1 > 0)
                            ptx::umma_bf16_ts_cg2(tmem_base + (uint32_t)fa.n0, a_tmem + 8u * k, db + b1_off + 2 * k, idesc_n1, accum);
                    }
                    ptx::umma_commit_cg2(&bars[bAFree + slot], 3);  // the slot may be rewritten once these MMAs have read it
                    if (j & 1) ptx::umma_commit_cg2(&bars[bW2Empty + w2.st], 3);
                    if (last_of_pass) ptx::umma_commit_cg2(&bars[bAccFull], 3);
                }
                __syncwarp();
                if (j & 1) w2.next(kW2Stages);
                if (++slot == kASlots) slot = 0;
                if (++j == nsteps) {
                    j = 0;
                    acc_ph ^= 1u;
                }
            }
        }
    } else if (warp == kWarpMma1) {
        // ================================================================ layer-1 MMA issuer (leader; whole warp, uniform)
        if (leader && total_steps > 0) {
            const uint32_t idesc_l1 = ptx::umma_idesc_bf16_f32(2 * kFM, kSub, F16);
            Ring w1;
            int j1 = 0, pass1 = 0, it1 = 0;
            uint32_t grp1 = 0, acc1 = 0, f_ph = 0x3u;  // first use of either accumulator: nothing to wait for
            for (int g = 0; g < total_steps; ++g) {
                const uint32_t zb = (uint32_t)it1 & 1u;
                if (j1 == 0 && pass1 == 0) ptx::mbar_wait(&bars[bZFull + zb], ((uint32_t)it1 >> 1) & 1u);
                ptx::mbar_wait2(&bars[bL1Free + acc1], (f_ph >> acc1) & 1u, &bars[bW1Full + w1.st], w1.ph);
                ptx::tc_fence_after_sync();
                f_ph ^= 1u << acc1;
                const uint64_t dz = desc0 + (uint64_t)((kOffZ + zb * kZBytes) >> 4);
                const uint64_t dw = desc0 + (uint64_t)((kOffW1 + w1.st * kW1StageBytes + (uint32_t)(j1 & 1) * kW1SubBytes) >> 4);
                const uint32_t d_tmem = tmem_base + kL1Col + acc1 * kSub;
                const bool last_of_tile = pass1 == fa.n_pass - 1 && j1 == nsteps - 1;
                if (ptx::elect_one()) {
                    if (fa.Kz == 2) {
                        ptx::umma_bf16_ss_cg2(d_tmem, dz, dw, idesc_l1, 0u);
                        ptx::umma_bf16_ss_cg2(d_tmem, dz + 2, dw + 2, idesc_l1, 1u);
                    } else {
                        for (int k = 0; k < fa.Kz; ++k) ptx::umma_bf16_ss_cg2(d_tmem, dz + 2 * k, dw + 2 * k, idesc_l1, k ? 1u : 0u);
                    }
                    ptx::umma_commit_cg2(&bars[bL1Full + grp1], 3);
                    if (j1 & 1) ptx::umma_commit_cg2(&bars[bW1Empty + w1.st], 3);
                    if (last_of_tile) ptx::umma_commit_cg2(&bars[bZEmpty + zb], 3);
                }
                __syncwarp();
                if (j1 & 1) w1.next(kW1Stages);
                if (++grp1 == kASlots) grp1 = 0;
                acc1 ^= 1u;
                if (++j1 == nsteps) {
                    j1 = 0;
                    if (++pass1 == fa.n_pass) {
                        pass1 = 0;
                        ++it1;
                    }
                }
            }
        }
    } else if (warp == kWarpZ) {
        // ================================================================ z builder (one warp): 4 consecutive cells per lane
        const int D = fa.D;
        const int n_units = 2 * fa.Kz;  // 16-byte units (8 features) that carry data
        const bool vec_ok = fa.idx == nullptr && (fa.n & 3) == 0 && (fa.c0 & 3) == 0 &&
                            ((reinterpret_cast<uintptr_t>(fa.T) | reinterpret_cast<uintptr_t>(fa.p) | reinterpret_cast<uintptr_t>(fa.Y)) & 15) == 0;
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int zb = it & 1;
            ptx::mbar_wait(&bars[bZEmpty + zb], ((uint32_t)(it >> 1) & 1u) ^ 1u);
            const uint32_t z_addr = sbase + kOffZ + zb * kZBytes;
            const int64_t i0 = (int64_t)tile * kFM + 4 * lane;  // this lane's rows: i0 .. i0 + 3
            const bool all4 = i0 + 3 < rows;
            int64_t g4[4];
            bool ok4[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                ok4[q] = i0 + q < rows;
                int64_t g = fa.c0 + i0 + q;
                if (fa.idx) g = ok4[q] ? (int64_t)fa.idx[g] : 0;
                g4[q] = ok4[q] ? g : 0;
            }
            // raw loads of one unit (8 features x 4 rows; one LDG.128 per feature on the aligned path).  The path is chosen
            // ONCE per unit, not per feature: per-feature branches keep the compiler from overlapping the eight loads
            auto load_unit = [&](int u, float (&x)[4][8]) {
                if (vec_ok && all4) {
#pragma unroll
                    for (int f = 0; f < 8; ++f) {
                        const int j = u * 8 + f;
                        const float *src = j == 0 ? fa.T : (j == 1 ? fa.p : fa.Y + (int64_t)(j - 2) * fa.n);
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (j < D) v = *reinterpret_cast<const float4 *>(src + fa.c0 + i0);
                        x[0][f] = v.x;
                        x[1][f] = v.y;
                        x[2][f] = v.z;
                        x[3][f] = v.w;
                    }
                } else {
#pragma unroll
                    for (int f = 0; f < 8; ++f) {
                        const int j = u * 8 + f;
                        const float *src = j == 0 ? fa.T : (j == 1 ? fa.p : fa.Y + (int64_t)(j - 2) * fa.n);
#pragma unroll
                        for (int q = 0; q < 4; ++q) x[q][f] = (j < D && ok4[q]) ? src[g4[q]] : 0.f;
                    }
                }
            };
            // software pipeline over the units: the loads of unit u + 1 are in flight while unit u is transformed (with one
            // unit at a time the builder needed ~14 k clk per tile -- four exposed memory latencies -- which is longer than
            // a whole tile of a small net like configs[1])
            float xa[4][8];
            load_unit(0, xa);
#pragma unroll 1
            for (int u = 0; u < n_units; ++u) {
                float x[4][8];
#pragma unroll
                for (int q = 0; q < 4; ++q)
#pragma unroll
                    for (int f = 0; f < 8; ++f) x[q][f] = xa[q][f];
                if (u + 1 < n_units) load_unit(u + 1, xa);
                // Box-Cox + z-score of the 32 values of the unit.  The lambda = 0 (log) variant is a separate copy of the loop:
                // a branch per element serialised the eight features (ILP 4 instead of 32: ~3 k clk per unit)
                auto transform = [&](auto lz) {
                    constexpr bool kLambdaZero = decltype(lz)::value;
#pragma unroll
                    for (int f = 0; f < 8; ++f) {
                        const int j = u * 8 + f;
                        const float mu = j < D ? fa.pre.mean[j] : 0.f, is = j < D ? fa.pre.inv_std[j] : 0.f;
                        const bool species = j >= 2 && j < D, one = j >= D && j < D + 2;
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            float t = x[q][f];
                            // z is rounded to BF16 (2^-9): the approximate lg2 / ex2 pair (2^-22) is ample here;
                            // Y = 0 still maps to exactly -1/lambda (R1, R2): lg2(0) = -inf, ex2(-inf) = 0
                            const float Yc = fmaxf(t, 0.f);
                            float y;
                            if (kLambdaZero) y = logf(Yc);
                            else y = (ptx::ex2_approx(fa.pre.lambda * ptx::lg2_approx(Yc)) - 1.f) * fa.pre.inv_lambda;
                            t = species ? y : t;
                            t = (t - mu) * is;
                            t = one ? 1.f : t;  // multiplies the hi / lo halves of b1 in W1 columns D, D+1
                            x[q][f] = ok4[q] ? t : 0.f;
                        }
                    }
                };
                if (fa.pre.lambda_zero) transform(std::true_type{});
                else transform(std::false_type{});
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int rr = 4 * lane + q;
                    ptx::st_shared_v4(z_addr + (uint32_t)rr * 128u + (uint32_t)((u ^ (rr & 7)) << 4),
                                      ptx::pack_half2(x[q][0], x[q][1], f16), ptx::pack_half2(x[q][2], x[q][3], f16),
                                      ptx::pack_half2(x[q][4], x[q][5], f16), ptx::pack_half2(x[q][6], x[q][7], f16));
                }
            }
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * (bZFull + zb));
        }
    } else {
        // ================================================================ workers (warps 0..11): three groups of four
        const int q = warp & 3;                  // TMEM lane quarter
        const int grp = warp >> 2;         // slot this group owns; every third 32-column block of the drain
        const int r = q * 32 + lane;             // row of the tile
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        const uint32_t a_addr = lane_addr + kACol + (uint32_t)grp * (kSub / 2);
        const uint32_t afull = bars_leader + 8u * (bAFull + grp);
        uint32_t afree_ph = 1u;  // first use of the slot: nothing to wait for
        const int total_passes = my_tiles * fa.n_pass;
        int pass_idx = 0;       // passes drained so far (over all tiles)
        uint32_t l1_ph = 0;

        // the drain of one pass: acc -> + b2 -> 2 GELU -> BF16 -> 64-byte row segments of h2 (global)
        auto drain = [&]() {
            const int it = pass_idx / fa.n_pass, pass = pass_idx - it * fa.n_pass;
            const int tile = (int)blockIdx.x + it * (int)gridDim.x;
            const int64_t grow = (int64_t)tile * kFM + r;
            const bool row_ok = grow < rows;
            ptx::mbar_wait(&bars[bAccFull], (uint32_t)pass_idx & 1u);
            ptx::tc_fence_after_sync();
            const int col_base = pass * fa.pass_w;
            int cur_w = fa.H2p - col_base;
            cur_w = cur_w < fa.pass_w ? cur_w : fa.pass_w;
            __nv_bfloat16 *dst_row = fa.h2 + grow * fa.H2p + col_base;
            // work split over the three groups: every third full 32-column block, and the 16-column remainder of a pass
            // (widths are multiples of 16) as two 8-column units for groups 0 and 1 -- 4.25 / 4.25 / 4 blocks at 400 columns
            const int n_full = cur_w >> 5, rem = cur_w & 31;
            const bool has_tail = rem > 0 && grp < (rem >> 3);
            const int my_last = n_full > grp ? ((n_full - 1 - grp) / kWorkerGroups) * kWorkerGroups + grp : -1;
            if (my_last < 0 && !has_tail) {
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * bAccEmpty);
            }
#pragma unroll 1
            for (int b = grp; b < n_full; b += kWorkerGroups) {
                const int cc = b * 32;
                uint32_t v[32];
                ptx::tmem_ld32(lane_addr + (uint32_t)cc, v);
                ptx::tmem_ld_wait();
                if (b == my_last && !has_tail) {
                    // last accumulator read of this warp: hand the accumulator back to the issuer
                    ptx::tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * bAccEmpty);
                }
                const float4 *b4 = reinterpret_cast<const float4 *>(sBias + col_base + cc);
                uint32_t o[16];
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) {
                    const float4 bb = b4[jj];
                    o[2 * jj] = ptx::gelu2_pack(__uint_as_float(v[4 * jj]) + bb.x, __uint_as_float(v[4 * jj + 1]) + bb.y, f16);
                    o[2 * jj + 1] = ptx::gelu2_pack(__uint_as_float(v[4 * jj + 2]) + bb.z, __uint_as_float(v[4 * jj + 3]) + bb.w, f16);
                }
                if (fa.h2_blocked) {
                    // lane = row, one 16-byte piece per instruction: 512 contiguous bytes per warp instruction.  Rows past
                    // the end of a real tile are stored too (the buffer holds whole tiles; they are zeros)
                    if (tile < n_tiles) {
                        uint4 *dst = reinterpret_cast<uint4 *>(fa.h2) + ((int64_t)tile * (fa.H2p >> 3) + ((col_base + cc) >> 3)) * kFM + r;
                        dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
                        dst[kFM] = make_uint4(o[4], o[5], o[6], o[7]);
                        dst[2 * kFM] = make_uint4(o[8], o[9], o[10], o[11]);
                        dst[3 * kFM] = make_uint4(o[12], o[13], o[14], o[15]);
                    }
                } else if (row_ok) {
                    uint4 *dst = reinterpret_cast<uint4 *>(dst_row + cc);
                    dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
                    dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
                    dst[2] = make_uint4(o[8], o[9], o[10], o[11]);
                    dst[3] = make_uint4(o[12], o[13], o[14], o[15]);
                }
            }
            if (has_tail) {
                const int cc = n_full * 32 + grp * 8;
                uint32_t v[8];
                ptx::tmem_ld8(lane_addr + (uint32_t)cc, v);
                ptx::tmem_ld_wait();
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * bAccEmpty);
                const float4 *b4 = reinterpret_cast<const float4 *>(sBias + col_base + cc);
                const float4 b0 = b4[0], b1 = b4[1];
                const uint4 o = make_uint4(ptx::gelu2_pack(__uint_as_float(v[0]) + b0.x, __uint_as_float(v[1]) + b0.y, f16),
                                           ptx::gelu2_pack(__uint_as_float(v[2]) + b0.z, __uint_as_float(v[3]) + b0.w, f16),
                                           ptx::gelu2_pack(__uint_as_float(v[4]) + b1.x, __uint_as_float(v[5]) + b1.y, f16),
                                           ptx::gelu2_pack(__uint_as_float(v[6]) + b1.z, __uint_as_float(v[7]) + b1.w, f16));
                if (fa.h2_blocked) {
                    if (tile < n_tiles)
                        *(reinterpret_cast<uint4 *>(fa.h2) + ((int64_t)tile * (fa.H2p >> 3) + ((col_base + cc) >> 3)) * kFM + r) = o;
                } else if (row_ok) {
                    *reinterpret_cast<uint4 *>(dst_row + cc) = o;
                }
            }
            ++pass_idx;
        };

        int boundary = nsteps;  // first global step of the next pass
#pragma unroll 1
        for (int g = grp; g < total_steps; g += kASlots) {
            // ---- convert this group's step: layer-1 accumulator (g & 1) -> 2 GELU -> BF16 pairs -> A slot `grp`
            const uint32_t acc = (uint32_t)g & 1u;
            ptx::mbar_wait(&bars[bL1Full + grp], l1_ph);
            l1_ph ^= 1u;
            ptx::tc_fence_after_sync();
            uint32_t v[32];
            ptx::tmem_ld32(lane_addr + kL1Col + acc * kSub, v);
            ptx::tmem_ld_wait();
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster(bars_leader + 8u * (bL1Free + acc));  // the accumulator is in registers
            uint32_t o[16];
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) o[jj] = ptx::gelu2_pack(__uint_as_float(v[2 * jj]), __uint_as_float(v[2 * jj + 1]), f16);
            ptx::mbar_wait(&bars[bAFree + grp], afree_ph);  // the layer-2 MMAs of this slot's previous piece have completed
            afree_ph ^= 1u;
            ptx::tc_fence_after_sync();
            ptx::tmem_st16(a_addr, o);
            ptx::tmem_st_wait();
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster(afull);
            // ---- the first step of a new pass is converted BEFORE the old pass is drained (its layer-1 MMAs were issued
            // under the old pass's last layer-2 MMAs), so layer 2 restarts the moment the accumulator is free
            if (g >= boundary) {
                drain();
                boundary += nsteps;
            }
        }
        while (pass_idx < total_passes) drain();
    }

    ptx::griddep_launch_dependents();  // the tail kernel's CTAs may be scheduled as SMs free up (it waits for this grid's end)
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync_all();  // no CTA leaves while its peer may still signal its barriers or the pair's MMAs run
    if (warp == kWarpMma2) {
        ptx::tc_fence_after_sync();
        ptx::tmem_dealloc_cg2(tmem_base, 512);
    }
}
// ---------------------------------------------------------------- host side
cudaError_t fused_setup(Ctx *c) {
    (void)c;
    cudaError_t e = cudaFuncSetAttribute(k_fused_l1l2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_fused_l1l2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
}

// H1 need not be a multiple of 64: W1 gets zero rows up to the next multiple (h1 = 2 GELU(0) = 0 there) and TMA zero-fills
// the K columns of W2 past the tensor's edge
bool fused_supported(int D, int H1, int H2p) {
    return D + 2 <= kFK && H1 >= 2 * kFK && H1 % 16 == 0 && H2p >= 16 && H2p <= (int)(kBias2Bytes / 4) && H2p % 16 == 0;
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
    const FusedNet &fn = c->cur->fused;
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
    fa.H1p = (c->sizes[1] + kFK - 1) / kFK * kFK;
    fa.H2p = c->cur->lay[1].Np;
    fa.n_pass = fn.n_pass;
    fa.pass_w = fn.pass_w;
    fa.n0 = fn.n0;
    fa.n1 = fn.n1;
    fa.bias2 = c->cur->lay[1].bias;
    fa.h2 = c->act[0];
    fa.h2_blocked = fn.h2_blocked ? 1 : 0;
    fa.f16 = c->prm.precision == GPUANN_PRECISION_FP16 ? 1 : 0;
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
    if (fa.f16) return cudaLaunchKernelEx(&cfg, k_fused_l1l2<true>, fn.tmapW1, fn.tmapW2a, fn.tmapW2b, fa);
    return cudaLaunchKernelEx(&cfg, k_fused_l1l2<false>, fn.tmapW1, fn.tmapW2a, fn.tmapW2b, fa);
}

}  // namespace gpuann
