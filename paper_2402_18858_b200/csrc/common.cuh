// common.cuh -- internal declarations shared by the translation units of libgpuann.so
// (context, device-side parameter blocks, launch prototypes).  Not part of the public ABI.
#pragma once
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>

#include "../../include/gpuann.h"

namespace gpuann {

constexpr int kMaxSpecies = GPUANN_MAX_SPECIES;
constexpr int kMaxLayers = GPUANN_MAX_LAYERS;
constexpr double kRu = 8314.46261815324;  // J/(kmol K)

// ---------------------------------------------------------------- device-side parameter blocks
// Thermo table in the form the T-solve evaluates: per species and range, pre-scaled by Ru/W_k:
//   cp_k(T) = c[0] + T (c[1] + T (c[2] + T (c[3] + T c[4])))
//   h_k(T)  = c[5] + T (c[0] + T (c[1]/2 + T (c[2]/3 + T (c[3]/4 + T c[4]/5))))  -- the /j factors are stored in d[]
struct ThermoDev {
    double cp[kMaxSpecies][2][5];  // (Ru/W) a1..a5
    double hh[kMaxSpecies][2][6];  // (Ru/W) {a6, a1, a2/2, a3/3, a4/4, a5/5}
    double T_mid[kMaxSpecies];
    double inv_W[kMaxSpecies];     // 1 / W_k [kmol/kg] (density, R_mix)
    int n_species;
    int two_ranges;
};

// optional outputs of gpuann_chem_step_ex (device pointers or nullptr)
struct ExtraOut {
    float *rr = nullptr, *hrr = nullptr, *cp = nullptr, *rho = nullptr, *psi = nullptr;
    __host__ __device__ bool any() const { return rr || hrr || cp || rho || psi; }
};

// Everything the update S4-S7 needs besides the thermo table.
struct PostParams {
    int n_species;
    int newton_max_iter;
    int inv_lambda_int;  // > 0: 1/lambda is this integer (power by repeated squaring); 0: generic pow
    int lambda_zero;     // 1: log/exp branch of Eq. 7
    double lambda;
    double inv_lambda;
    double newton_tol;
    double T_min, T_max;
    float out_mean[kMaxSpecies];
    float out_std[kMaxSpecies];
};

// Input side S1-S2: z_j = (x_j - mean_j) * inv_std_j
struct PreParams {
    int n_species;
    int lambda_zero;
    float lambda;
    float inv_lambda;
    float mean[kMaxSpecies + 2];
    float inv_std[kMaxSpecies + 2];
};

struct Counters {
    unsigned long long n_active;
    unsigned long long n_not_converged;
    unsigned long long n_degenerate;
    unsigned long long pad;
};

// One layer of the BF16 tensor path.
struct LayerBf16 {
    int K, N;            // true fan-in / fan-out
    int Kp, Np;          // padded to multiples of 16
    int n_tile;          // columns of a full tile (multiple of 16, <= 416)
    int n0;              // n_tile > 256: columns of the first of the two MMAs per k-step (= TMA box rows); else 0
    int tiles_n;         // ceil(Np / n_tile)
    __nv_bfloat16 *W;    // DEVICE [Np][Kp] row-major, zero padded
    float *bias;         // DEVICE [Np], zero padded
    CUtensorMap tmapW;   // box {64, n_tile}, SWIZZLE_128B
    CUtensorMap tmapA;   // this layer's input: activation buffer [chunk][Kp], box {64, 128}
};

// "bf16-fused" variant: S1 + S2 + layers 1-2 in one kernel (k_fused.cu)
struct FusedNet {
    bool on = false;
    __nv_bfloat16 *W1p = nullptr;  // DEVICE [H1][64]: W1 zero padded to K = 64, b1 (hi, lo) in columns D, D+1
    CUtensorMap tmapW1{};          // box {64, 64}
    CUtensorMap tmapW2a{}, tmapW2b{};  // W2 [H2p][H1]: box {64, n0}, box {64, n1}
    int n_pass = 0, pass_w = 0, n0 = 0, n1 = 0;
    // h2 layout in HBM when the tail kernel consumes it directly: BLOCKED in the MMA's canonical core-matrix order,
    //     h2b[tile][kp = column / 8][row 0..127][8 columns]   (16-byte pieces; a (tile, kp) slab is 2 KB)
    // so that (a) a drain warp's store instruction -- lane = row, one 16-byte piece -- writes 512 contiguous bytes instead
    // of 32 pieces 1600 bytes apart (the row-major stores cost 6,400 LSU line transactions per pass and made the drain
    // 10 k clk long), and (b) a [128 x 64] A stage of the tail kernel is ONE contiguous 16 KB
    // piece of global memory, read by the MMA through a no-swizzle descriptor (LBO 2048, SBO 128).
    bool h2_blocked = false;
};

// tail kernel (k_tail.cu): the last two layers + S4-S8.  TailArgs is the kernel's by-value parameter block: the
// thermo table and the per-species constants sit in the constant bank, where warp-uniform reads cost nothing.
constexpr int kTailMaxNs = 48;
struct TailThermo {
    double cp[kTailMaxNs][2][5];  // as ThermoDev
    double hh[kTailMaxNs][2][6];
    double T_mid[kTailMaxNs];
};
struct TailArgs {
    int64_t n, c0, rows;
    const int32_t *n_active, *idx;
    float *T, *Y;
    const float *h;
    float *o_raw;  // != nullptr: forward only, o + b4 -> o_raw[k * o_stride + local cell]
    int64_t o_stride;
    int Ns, Np;    // species, padded to 16
    int K3p, H3p, n0, n1;
    int f16;        // 1: FP16 operands (GPUANN_PRECISION_FP16), 0: BF16
    int a_blocked;  // 1: the input activation is in the blocked layout the fused kernel writes (see FusedNet)
    const float *bias3;
    int newton_max_iter, inv_lambda_int, lambda_zero, two_ranges;
    float lambda, inv_lambda;
    double newton_tol, T_min, T_max;
    float sA[kTailMaxNs];  // dt sigma_out,k
    float sC[kTailMaxNs];  // dt (sigma_out,k b4,k + mu_out,k)
    float b4[kTailMaxNs];
    Counters *counters;
    TailThermo th;
    // FP32 copies of the one-range table for the FAST instance of the kernel (mixture coefficients accumulated in FP32)
    float hhf[kTailMaxNs][6];
    float cpf[kTailMaxNs][5];
    // gpuann_chem_step_ex
    const float *p;
    ExtraOut ex;
    float invW[kTailMaxNs];
    float inv_dt;
};
struct TailNet {
    bool on = false;
    CUtensorMap tmapW3a{}, tmapW3b{}, tmapW4{};  // per-CTA boxes: W3 {64, n0/2}, {64, n1/2}; W4 {64, Np/2}
    CUtensorMap tmapAb{};                        // the kernel's input in the BLOCKED layout (see h2 layout below)
    TailArgs args{};
};

// One network of the tensor path: its layers, the fused-kernel and tail-kernel set-up.  A context holds ONE (the net of
// gpuann_load_net) or Ns (the per-species ensemble of gpuann_load_net_ensemble, each with a single output).
struct SubNet {
    int n_out = 0;                 // outputs of this net: Ns, or 1 in an ensemble
    LayerBf16 lay[kMaxLayers]{};
    FusedNet fused;
    TailNet tail;
};

struct Ctx {
    gpuann_params prm{};
    int device = 0;
    int sm_count = 0;
    std::string err;

    // net
    bool net_loaded = false;
    int Ns = 0, L = 0;
    int sizes[kMaxLayers + 1]{};
    double lambda = 0.1;
    PreParams pre{};
    PostParams post{};
    // FP32 path
    float *w32 = nullptr;        // DEVICE concatenated [out][in] per layer
    float *b32 = nullptr;        // DEVICE concatenated
    size_t w32_count = 0, b32_count = 0;
    int max_width = 0;
    // BF16 path
    SubNet net0;                              // gpuann_load_net
    std::vector<SubNet> ens;                  // gpuann_load_net_ensemble: net k yields o_k (R24)
    SubNet *cur = &net0;                      // the net the launchers below read (set before every launch)
    int64_t chunk = 0;                        // cells per pass
    __nv_bfloat16 *act[2] = {nullptr, nullptr};  // ping-pong activation buffers [chunk][maxKp]
    size_t act_elems = 0;
    float *o_buf = nullptr;                   // [Ns][chunk] raw output of the chunk
    int64_t issued_mac_per_cell = 0;
    const char *variant = "none";

    // thermo
    bool thermo_loaded = false;
    int thermo_Ns = 0;
    ThermoDev *thermo_dev = nullptr;  // DEVICE

    // compaction scratch (S0)
    int32_t *idx = nullptr;       // DEVICE [idx_cap] active cell indices
    int64_t idx_cap = 0;
    int32_t *blk_counts = nullptr;  // DEVICE per-block counts / offsets
    int64_t blk_cap = 0;
    int32_t *n_active_dev = nullptr;  // DEVICE int32: number of active cells of the current step

    // host-variant staging
    float *stage = nullptr;
    size_t stage_floats = 0;

    Counters *counters = nullptr;  // DEVICE
    int64_t host_active = 0;       // cells counted as active without a device-side compaction
    cudaStream_t own_stream = nullptr;  // used by gpuann_chem_step_host
    cudaStream_t copy_in = nullptr, copy_out = nullptr;  // copy streams of the pipelined host variant
    std::vector<cudaEvent_t> slice_events;
    cudaStream_t last_stream = nullptr;
    int64_t launches = 0;
    int last_cls = -1;  // KernelClass of the launch enqueued last (LaunchScope); launch_tail decides on it whether PDL is safe

    // per-kernel-class device timing (gpuann_timing_enable / gpuann_timing_read): CUDA events around every launch
    bool timing = false;
    struct TimedLaunch {
        int cls;
        cudaEvent_t e0, e1;
    };
    std::vector<TimedLaunch> timed;       // launches recorded since timing was enabled
    std::vector<cudaEvent_t> event_pool;  // recycled events
};

// Kernel classes of the timing hook (index into gpuann_timing_read's arrays)
enum KernelClass {
    kClsCompact = 0,
    kClsPre = 1,
    kClsLayer0 = 2,  // + layer index (0..7)
    kClsPost = 10,
    kClsFp32 = 11,
    kClsFused = 12,
    kClsAux = 13,
    kClsTail = 14,
    kNumKernelClasses = 15
};

// RAII: counts the launch and, when timing is on, brackets it with two events on the launching stream.
struct LaunchScope {
    Ctx *c;
    cudaStream_t s;
    cudaEvent_t e1 = nullptr;
    LaunchScope(Ctx *ctx, int cls, cudaStream_t stream, int n_launches = 1) : c(ctx), s(stream) {
        c->launches += n_launches;
        c->last_cls = cls;
        if (!c->timing) return;
        cudaEvent_t ev[2] = {nullptr, nullptr};
        for (int i = 0; i < 2; ++i) {
            if (!c->event_pool.empty()) {
                ev[i] = c->event_pool.back();
                c->event_pool.pop_back();
            } else if (cudaEventCreate(&ev[i]) != cudaSuccess) {
                ev[i] = nullptr;
            }
        }
        if (!ev[0] || !ev[1]) return;
        cudaEventRecord(ev[0], s);
        e1 = ev[1];
        c->timed.push_back({cls, ev[0], ev[1]});
    }
    ~LaunchScope() {
        if (e1) cudaEventRecord(e1, s);
    }
};

// ---------------------------------------------------------------- kernel launchers (defined in the .cu files)
// k_fp32.cu
cudaError_t launch_chem_fp32(Ctx *c, int64_t n, float *T, const float *p, float *Y, const float *h, double dt,
                             float *o_raw, bool forward_only, const ExtraOut &ex, cudaStream_t s);
size_t fp32_smem_bytes(const Ctx *c, int *cells_per_block);

// k_aux.cu
cudaError_t launch_compact(Ctx *c, int64_t n, const float *T, float T_active, cudaStream_t s);
cudaError_t launch_pre_bf16(Ctx *c, int64_t n, int64_t c0, int64_t cn, const float *T, const float *p, const float *Y,
                            bool use_idx, __nv_bfloat16 *z, int Kp, cudaStream_t s);
cudaError_t launch_post(Ctx *c, int64_t n, int64_t c0, int64_t cn, float *T, float *Y, const float *h, const float *o,
                        int64_t o_stride, double dt, bool use_idx, const float *p, const ExtraOut &ex, cudaStream_t s);
cudaError_t launch_enthalpy(Ctx *c, int64_t n, const float *T, const float *Y, float *h_out, cudaStream_t s);
cudaError_t launch_moments(Ctx *c, int64_t n, int Ns, const float *T, const float *p, const float *Y, double lambda,
                           double *mean_out, double *std_out, cudaStream_t s);
cudaError_t launch_moments_static(Ctx *c, int64_t n, int Ns, const float *T, const float *p, const float *Y, double lambda,
                                  double *mean_out, double *std_out, cudaStream_t s);  // scratch in a static __device__ array

// k_gemm.cu
cudaError_t gemm_setup(Ctx *c);  // opt-in shared memory etc.
cudaError_t launch_layer_bf16(Ctx *c, int layer, int64_t rows_cap, const CUtensorMap *tmapA, __nv_bfloat16 *out_bf16,
                              int out_ld, float *out_f32, int64_t out_f32_stride, int64_t c0, bool use_count,
                              cudaStream_t s);

// k_fused.cu
cudaError_t fused_setup(Ctx *c);
bool fused_supported(int D, int H1, int H2p);
void fused_plan(int H2p, int *n_pass, int *pass_w, int *n0, int *n1);
cudaError_t launch_fused_l1l2(Ctx *c, int64_t n, int64_t c0, int64_t cn, const float *T, const float *p, const float *Y,
                              bool use_idx, cudaStream_t s);

// k_tail.cu
cudaError_t tail_setup(Ctx *c);
bool tail_supported(int K3p, int H3p, int Ns);
void tail_plan(int H3p, int *n0, int *n1);
cudaError_t launch_tail(Ctx *c, int64_t n, int64_t c0, int64_t cn, float *T, const float *p, float *Y, const float *h,
                        double dt, float *o_raw, int64_t o_stride, bool use_idx, const ExtraOut &ex, cudaStream_t s);

// encodes a 2-D BF16 row-major tensor map {inner = cols, outer = rows}, box {64, box_rows}, 128-byte swizzle
bool encode_tmap_bf16(CUtensorMap *out, const void *base, uint64_t cols, uint64_t rows, uint64_t row_pitch_bytes,
                      uint32_t box_rows, std::string *err);

// 2-D map over `total_elems` contiguous BF16 viewed as rows of 256: box {256, 32} = 16 KB contiguous, no swizzle
bool encode_tmap_bf16_linear(CUtensorMap *out, const void *base, uint64_t total_elems, std::string *err);

}  // namespace gpuann
