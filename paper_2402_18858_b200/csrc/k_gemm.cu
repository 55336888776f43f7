// k_gemm.cu -- one fully connected layer of S3 on the 5th-generation tensor cores ("bf16-layerwise" variant):
//     out[r][j] = act( sum_i A[r][i] W[j][i] + b[j] ),   A: [rows][Kp] BF16, W: [Np][Kp] BF16, FP32 accumulate
// (PAPER.md:103 hidden sizes / GELU; PAPER.md:56 half-precision inference).  Persistent, warp-specialised:
//   warp 0    TMA producer: A tile 128 x 64 and W tile n_tile x 64 (128-byte swizzle) into a 4-stage ring
//   warp 1    allocates TMEM (512 columns = 2 accumulators of <= 256 columns) and issues tcgen05.mma
//             (M = 128, N = n_tile, K = 16), committing each stage back to the producer and each finished
//             accumulator to the epilogue
//   warps 2-9 epilogue (two per TMEM lane quarter): tcgen05.ld 32 lanes x 32 columns, + bias (smem), GELU, BF16 pack, 64-byte row segments
//             (hidden layers) or FP32 species-major stores (last layer); overlaps the next tile's MMAs.
// Tiles are walked n-fastest so that CTAs running together share the A rows and the whole W in L2.
#include "common.cuh"
#include "ptx.cuh"

namespace gpuann {

constexpr int kBM = 128;
constexpr int kBK = 64;
constexpr int kStages = 4;
constexpr int kMaxNT = 256;
constexpr int kGemmThreads = 320;   // TMA, MMA, 8 epilogue warps
constexpr uint32_t kABytes = kBM * kBK * 2;        // 16 KB
constexpr uint32_t kBBytesMax = kMaxNT * kBK * 2;  // 32 KB
constexpr int kBiasMax = 4096;  // = GPUANN_MAX_WIDTH floats staged in shared memory
// "wide" tiles (n_tile > 256: two MMAs per k-step into ONE accumulator of up to 416 columns, A read once for the
// whole row of W): 3 stages of A 16 KB + B 52 KB; narrow tiles: 4 stages of 16 + 32 KB and two accumulators
constexpr int kWideStages = 3;
constexpr uint32_t kBBytesWide = 416 * kBK * 2;  // 53,248
constexpr size_t kRegion = (size_t)kWideStages * (kABytes + kBBytesWide) > (size_t)kStages * (kABytes + kBBytesMax)
                               ? (size_t)kWideStages * (kABytes + kBBytesWide)
                               : (size_t)kStages * (kABytes + kBBytesMax);
constexpr size_t kGemmSmem = 1024 /*align slack*/ + kRegion + 256 + kBiasMax * 4;

struct GemmArgs {
    int Kp, Np, N;          // padded K, padded N, true N
    int n_tile, tiles_n;
    int n0;                 // wide tiles (n_tile > 256): columns of the first MMA (= TMA box rows); 0 = narrow
    int64_t rows;           // valid rows when n_active == nullptr
    int64_t c0;             // first (compacted) cell of this chunk, for the n_active test
    const int32_t *n_active;  // DEVICE or nullptr: rows = clamp(*n_active - c0, 0, rows)
    const float *bias;      // [Np]
    __nv_bfloat16 *out_bf16;  // [rows][out_ld] or nullptr
    int out_ld;
    float *out_f32;         // [N][out_f32_stride] (species-major) or nullptr
    int64_t out_f32_stride;
    int apply_gelu;
};

__global__ void __launch_bounds__(kGemmThreads, 1)
k_layer_bf16(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapW, const GemmArgs ga) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    unsigned char *sA = smem;
    const bool wide = ga.n0 > 0;
    const int nst = wide ? kWideStages : kStages;
    const uint32_t bsz = wide ? kBBytesWide : kBBytesMax;
    unsigned char *sB = smem + (size_t)nst * kABytes;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kRegion);
    uint64_t *full = bars, *empty = bars + kStages, *tfull = bars + 2 * kStages, *tempty = bars + 2 * kStages + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 2 * kStages + 4);
    float *sBias = reinterpret_cast<float *>(smem + kRegion + 256);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    int64_t rows = ga.rows;
    if (ga.n_active) {
        int64_t r = (int64_t)*ga.n_active - ga.c0;
        rows = r < 0 ? 0 : (r < rows ? r : rows);
    }
    const int tiles_m = (int)((rows + kBM - 1) / kBM);
    const int n_tiles = tiles_m * ga.tiles_n;
    const int num_kb = (ga.Kp + kBK - 1) / kBK;
    const uint32_t b_bytes = (wide ? 2u * (uint32_t)ga.n0 : (uint32_t)ga.n_tile) * kBK * 2;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], 1);
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(&tfull[a], 1);
            ptx::mbar_init(&tempty[a], 8);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmapA);
        ptx::prefetch_tensormap(&tmapW);
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, 512);
        ptx::tmem_relinquish();
    }
    for (int i = threadIdx.x; i < ga.Np && i < kBiasMax; i += kGemmThreads) sBias[i] = ga.bias[i];
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================================================== TMA producer
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                const int mt = tile / ga.tiles_n, nt = tile % ga.tiles_n;
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait(&empty[stage], phase ^ 1);
                    ptx::mbar_arrive_expect_tx(&full[stage], kABytes + b_bytes);
                    ptx::tma_load_2d(&tmapA, &full[stage], sA + (size_t)stage * kABytes, kb * kBK, mt * kBM);
                    ptx::tma_load_2d(&tmapW, &full[stage], sB + (size_t)stage * bsz, kb * kBK, nt * ga.n_tile);
                    if (wide)  // second box: rows n0.. (rows beyond Np are zero filled)
                        ptx::tma_load_2d(&tmapW, &full[stage], sB + (size_t)stage * bsz + (size_t)ga.n0 * 128, kb * kBK,
                                         nt * ga.n_tile + ga.n0);
                    if (++stage == nst) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===================================================== MMA issuer (whole warp; one elected lane issues)
        // warp-uniform control flow + one elect.sync branch per k-block lets ptxas keep the descriptors in uniform
        // registers and emit the UTCHMMAs back to back (profiles/r01_fused_l1l2.md)
        {
            int stage = 0;
            uint32_t phase = 0;
            int it = 0;
            const uint64_t desc0 = ptx::umma_desc_sw128_kmajor(ptx::smem_u32(smem));
            for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
                const int nt = tile % ga.tiles_n;
                const int n_cur = min(ga.n_tile, ga.Np - nt * ga.n_tile);
                const int n0_cur = wide ? min(ga.n0, n_cur) : n_cur, n1_cur = n_cur - n0_cur;
                const uint32_t idesc = ptx::umma_idesc_bf16_f32(kBM, (uint32_t)n0_cur);
                const uint32_t idesc1 = ptx::umma_idesc_bf16_f32(kBM, (uint32_t)(n1_cur > 0 ? n1_cur : 16));
                const uint64_t b1_off = (uint64_t)(((uint32_t)ga.n0 * 128u) >> 4);
                const int acc = wide ? 0 : (it & 1);
                const uint32_t acc_phase = wide ? ((uint32_t)it & 1) : ((uint32_t)(it >> 1) & 1);
                ptx::mbar_wait(&tempty[acc], acc_phase ^ 1);
                ptx::tc_fence_after_sync();
                const uint32_t d_tmem = tmem_base + (uint32_t)acc * kMaxNT;
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait(&full[stage], phase);
                    ptx::tc_fence_after_sync();
                    const uint64_t da = desc0 + (uint64_t)(((uint32_t)stage * kABytes) >> 4);
                    const uint64_t db = desc0 + (uint64_t)(((uint32_t)nst * kABytes + (uint32_t)stage * bsz) >> 4);
                    const int ksteps = min(kBK / 16, (ga.Kp - kb * kBK) / 16);
                    if (ptx::elect_one()) {
                        if (ksteps == kBK / 16) {
#pragma unroll
                            for (int k = 0; k < kBK / 16; ++k) {
                                ptx::umma_bf16_ss(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
                                if (n1_cur > 0)
                                    ptx::umma_bf16_ss(d_tmem + (uint32_t)ga.n0, da + 2 * k, db + b1_off + 2 * k, idesc1, (kb | k) ? 1u : 0u);
                            }
                        } else {
                            for (int k = 0; k < ksteps; ++k) {
                                ptx::umma_bf16_ss(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
                                if (n1_cur > 0)
                                    ptx::umma_bf16_ss(d_tmem + (uint32_t)ga.n0, da + 2 * k, db + b1_off + 2 * k, idesc1, (kb | k) ? 1u : 0u);
                            }
                        }
                        ptx::umma_commit(&empty[stage]);  // frees the smem slot when these MMAs have read it
                        if (kb == num_kb - 1) ptx::umma_commit(&tfull[acc]);  // accumulator complete -> epilogue
                    }
                    __syncwarp();
                    if (++stage == nst) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
    } else {
        // ===================================================== epilogue (warps 2..9)
        // two warps per TMEM lane quarter: 32-column pieces of the accumulator alternate between them
        const int q = warp & 3;          // TMEM lane quarter this warp may access
        const int hsel = (warp - 2) >> 2;  // 0 / 1: which pieces
        int it = 0;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
            const int mt = tile / ga.tiles_n, nt = tile % ga.tiles_n;
            const int n_cur = min(ga.n_tile, ga.Np - nt * ga.n_tile);
            const int acc = wide ? 0 : (it & 1);
            const uint32_t acc_phase = wide ? ((uint32_t)it & 1) : ((uint32_t)(it >> 1) & 1);
            ptx::mbar_wait(&tfull[acc], acc_phase);
            ptx::tc_fence_after_sync();
            const int64_t r = (int64_t)mt * kBM + q * 32 + lane;
            const bool row_ok = r < rows;
            const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)acc * kMaxNT;
            const int col0 = nt * ga.n_tile;
            const int n_pieces = (n_cur + 31) >> 5;
            for (int pc = hsel; pc < n_pieces; pc += 2) {
                const int cc = pc << 5;
                const bool full = cc + 32 <= n_cur;  // widths are multiples of 16: a tail piece has 16 columns
                uint32_t v[32];
                if (full) ptx::tmem_ld32(t_addr + cc, v);
                else {
                    uint32_t w[16];
                    ptx::tmem_ld16(t_addr + cc, w);
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[j] = w[j];
#pragma unroll
                    for (int j = 16; j < 32; ++j) v[j] = 0u;
                }
                ptx::tmem_ld_wait();
                if (pc + 2 >= n_pieces) {  // last accumulator read of this warp
                    ptx::tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(&tempty[acc]);
                }
                float f[32];
                const float4 *b4 = reinterpret_cast<const float4 *>(sBias + col0 + cc);
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float4 b = (full || j < 4) ? b4[j] : make_float4(0.f, 0.f, 0.f, 0.f);
                    f[4 * j + 0] = __uint_as_float(v[4 * j + 0]) + b.x;
                    f[4 * j + 1] = __uint_as_float(v[4 * j + 1]) + b.y;
                    f[4 * j + 2] = __uint_as_float(v[4 * j + 2]) + b.z;
                    f[4 * j + 3] = __uint_as_float(v[4 * j + 3]) + b.w;
                }
                if (ga.out_bf16) {
                    // hidden layer: 2 GELU(.) packed to BF16 (the 1/2 is in the next layer's weights, api.cu)
                    if (row_ok) {
                        uint4 *dst = reinterpret_cast<uint4 *>(ga.out_bf16 + r * ga.out_ld + col0 + cc);
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            if (full || j < 2) {
                                uint4 o;
                                if (ga.apply_gelu) {
                                    o = make_uint4(ptx::gelu2_pack(f[8 * j], f[8 * j + 1]), ptx::gelu2_pack(f[8 * j + 2], f[8 * j + 3]),
                                                   ptx::gelu2_pack(f[8 * j + 4], f[8 * j + 5]), ptx::gelu2_pack(f[8 * j + 6], f[8 * j + 7]));
                                } else {
                                    o = make_uint4(ptx::pack_bf16x2(f[8 * j], f[8 * j + 1]), ptx::pack_bf16x2(f[8 * j + 2], f[8 * j + 3]),
                                                   ptx::pack_bf16x2(f[8 * j + 4], f[8 * j + 5]), ptx::pack_bf16x2(f[8 * j + 6], f[8 * j + 7]));
                                }
                                dst[j] = o;
                            }
                        }
                    }
                } else if (row_ok) {
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int col = col0 + cc + j;
                        if (col < ga.N) ga.out_f32[(int64_t)col * ga.out_f32_stride + r] = f[j];
                    }
                }
            }
            if (hsel >= n_pieces) {  // this warp had no piece in this tile: still release the accumulator
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(&tempty[acc]);
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
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode_fn(std::string *err) {
    static PFN_encodeTiled fn = nullptr;
    if (fn) return fn;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !p) {
        if (err) *err = std::string("cuTensorMapEncodeTiled is not available: ") + cudaGetErrorString(e);
        return nullptr;
    }
    fn = reinterpret_cast<PFN_encodeTiled>(p);
    return fn;
}

bool encode_tmap_bf16(CUtensorMap *out, const void *base, uint64_t cols, uint64_t rows, uint64_t row_pitch_bytes,
                      uint32_t box_rows, std::string *err) {
    PFN_encodeTiled fn = get_encode_fn(err);
    if (!fn) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {row_pitch_bytes};
    cuuint32_t box[2] = {(cuuint32_t)kBK, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        if (err) *err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
        return false;
    }
    return true;
}

bool encode_tmap_bf16_linear(CUtensorMap *out, const void *base, uint64_t total_elems, std::string *err) {
    PFN_encodeTiled fn = get_encode_fn(err);
    if (!fn) return false;
    cuuint64_t dims[2] = {256, total_elems / 256};
    cuuint64_t strides[1] = {512};
    cuuint32_t box[2] = {256, 32};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        if (err) *err = "cuTensorMapEncodeTiled (linear) failed with CUresult " + std::to_string((int)r);
        return false;
    }
    return true;
}

cudaError_t gemm_setup(Ctx *c) {
    (void)c;
    return cudaFuncSetAttribute(k_layer_bf16, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGemmSmem);
}

cudaError_t launch_layer_bf16(Ctx *c, int layer, int64_t rows, const CUtensorMap *tmapA, __nv_bfloat16 *out_bf16,
                              int out_ld, float *out_f32, int64_t out_f32_stride, int64_t c0, bool use_count,
                              cudaStream_t s) {
    if (rows <= 0) return cudaSuccess;
    const LayerBf16 &ly = c->cur->lay[layer];
    GemmArgs ga{};
    ga.Kp = ly.Kp;
    ga.Np = ly.Np;
    ga.N = ly.N;
    ga.n_tile = ly.n_tile;
    ga.tiles_n = ly.tiles_n;
    ga.n0 = ly.n0;
    ga.rows = rows;
    ga.c0 = c0;
    ga.n_active = use_count ? c->n_active_dev : nullptr;
    ga.bias = ly.bias;
    ga.out_bf16 = out_bf16;
    ga.out_ld = out_ld;
    ga.out_f32 = out_f32;
    ga.out_f32_stride = out_f32_stride;
    ga.apply_gelu = (layer < c->L - 1) ? 1 : 0;
    const int64_t tiles = ((rows + kBM - 1) / kBM) * ly.tiles_n;
    const int grid = (int)(tiles < c->sm_count ? tiles : c->sm_count);
    LaunchScope ls(c, kClsLayer0 + layer, s);
    k_layer_bf16<<<grid, kGemmThreads, kGemmSmem, s>>>(*tmapA, ly.tmapW, ga);
    return cudaGetLastError();
}

}  // namespace gpuann
