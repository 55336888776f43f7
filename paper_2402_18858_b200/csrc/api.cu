// api.cu -- the C ABI of libgpuann.so (include/gpuann.h): argument validation, context, weight / thermo
// packing, the chunk loop of the tensor path.  Every step of the hot path runs in the kernels of k_*.cu.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include <cuda_fp16.h>
#include "common.cuh"

using namespace gpuann;

struct gpuann_ctx : public Ctx {};

namespace {

thread_local std::string g_create_err;

int fail(Ctx *c, int status, const std::string &msg) {
    if (c) c->err = msg;
    else g_create_err = msg;
    return status;
}

int fail_cuda(Ctx *c, cudaError_t e, const char *what) {
    cudaGetLastError();  // clear the sticky-less error state
    return fail(c, e == cudaErrorMemoryAllocation ? GPUANN_ERR_ALLOC : GPUANN_ERR_CUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU_TRY(ctx, call, what)                                   \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return fail_cuda(ctx, e__, what); \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};

inline int pad16(int x) { return (x + 15) / 16 * 16; }

// FP32 -> BF16 bits, round to nearest even (NaN stays NaN)
inline uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    std::memcpy(&u, &f, 4);
    if ((u & 0x7F800000u) == 0x7F800000u && (u & 0x007FFFFFu)) return (uint16_t)((u >> 16) | 0x0040u);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

// FP32 -> FP16 bits, round to nearest even (overflow -> inf, subnormals kept)
inline uint16_t f32_to_f16_rne(float f) {
    const __half h = __float2half_rn(f);
    uint16_t u;
    std::memcpy(&u, &h, 2);
    return u;
}
inline float f16_bits_to_f32(uint16_t u) {
    __half h;
    std::memcpy(&h, &u, 2);
    return __half2float(h);
}

void free_net(Ctx *c) {
    cudaFree(c->w32);
    cudaFree(c->b32);
    c->w32 = c->b32 = nullptr;
    c->w32_count = c->b32_count = 0;
    auto free_sub = [](SubNet &sn) {
        for (int l = 0; l < kMaxLayers; ++l) {
            cudaFree(sn.lay[l].W);
            cudaFree(sn.lay[l].bias);
        }
        cudaFree(sn.fused.W1p);
        sn = SubNet{};
    };
    {   // the thermo table of the tail kernel survives a reload of the net (gpuann_load_thermo may have come first)
        const TailThermo th = c->net0.tail.args.th;
        const int two = c->net0.tail.args.two_ranges;
        TailArgs keep = c->net0.tail.args;
        free_sub(c->net0);
        std::memcpy(c->net0.tail.args.hhf, keep.hhf, sizeof(keep.hhf));
        std::memcpy(c->net0.tail.args.cpf, keep.cpf, sizeof(keep.cpf));
        std::memcpy(c->net0.tail.args.invW, keep.invW, sizeof(keep.invW));
        c->net0.tail.args.th = th;
        c->net0.tail.args.two_ranges = two;
    }
    for (SubNet &sn : c->ens) free_sub(sn);
    c->ens.clear();
    c->cur = &c->net0;
    cudaFree(c->act[0]);
    cudaFree(c->act[1]);
    cudaFree(c->o_buf);
    c->act[0] = c->act[1] = nullptr;
    c->o_buf = nullptr;
    c->act_elems = 0;
    c->net_loaded = false;
    c->variant = "none";
    c->issued_mac_per_cell = 0;
}

bool finite_f(float x) { return std::isfinite(x); }


// which kernels a net of these sizes runs, and its scratch: sets c->chunk, allocates the activation buffers (shared by all
// nets of an ensemble) and, when no tail kernel consumes the raw output in place (or `need_obuf`), the o buffer
int plan_and_alloc(Ctx *c, int n_species, int n_layers, const int *sizes, bool need_obuf) {
    const bool f16 = c->prm.precision == GPUANN_PRECISION_FP16;
    const bool fused = n_layers >= 3 && fused_supported(sizes[0], sizes[1], pad16(sizes[2]));
    const bool tail = n_layers >= (fused ? 4 : 2) &&
                      tail_supported(pad16(sizes[n_layers - 2]), pad16(sizes[n_layers - 1]), sizes[n_layers]);
    if (f16 && !(fused && tail && n_layers == 4))
        return fail(c, GPUANN_ERR_UNSUPPORTED, "gpuann_load_net: GPUANN_PRECISION_FP16 needs a net the fused + tail kernels run (4 weight matrices)");
    int64_t chunk = c->prm.chunk_cells > 0 ? c->prm.chunk_cells : (int64_t)c->sm_count * 128 * (fused ? 56 : 1);
    chunk = (chunk + 127) / 128 * 128;
    c->chunk = chunk;
    int maxKp = 0;
    for (int l = 0; l < n_layers; ++l)
        if (!fused || l >= 2) maxKp = pad16(sizes[l]) > maxKp ? pad16(sizes[l]) : maxKp;
    // activation scratch: ping-pong buffers [chunk][maxKp]; with the fused kernel in front and the tail kernel behind
    // only ONE of them is ever used (h2), and the raw output never leaves the SM
    c->act_elems = (size_t)chunk * (size_t)maxKp;
    const bool one_buffer = fused && tail && n_layers == 4;
    for (int b = 0; b < (one_buffer ? 1 : 2); ++b) {
        CU_TRY(c, cudaMalloc(&c->act[b], c->act_elems * sizeof(__nv_bfloat16)), "cudaMalloc(activations)");
        CU_TRY(c, cudaMemset(c->act[b], 0, c->act_elems * sizeof(__nv_bfloat16)), "cudaMemset(activations)");
    }
    if (!tail || need_obuf) {
        CU_TRY(c, cudaMalloc(&c->o_buf, (size_t)n_species * chunk * sizeof(float)), "cudaMalloc(o_buf)");
        CU_TRY(c, cudaMemset(c->o_buf, 0, (size_t)n_species * chunk * sizeof(float)), "cudaMemset(o_buf)");
    }
    return GPUANN_OK;
}

// pads, rounds (RNE) and uploads one net of the tensor path and encodes its tensor maps (against the context's shared
// activation buffers: plan_and_alloc first).  n_out = sizes[n_layers].  *mac_out: MACs issued per cell including padding.
int build_subnet(Ctx *c, SubNet &sn, int n_out, int n_layers, const int *sizes, const float *const *weights,
                 const float *const *biases, int64_t *mac_out) {
    const PreParams &pre = c->pre;
    const PostParams &po = c->post;
    const int64_t chunk = c->chunk;
    sn.n_out = n_out;
    const bool f16 = c->prm.precision == GPUANN_PRECISION_FP16;
    auto to_half = [f16](float v) { return f16 ? f32_to_f16_rne(v) : f32_to_bf16_rne(v); };
    const bool fused = n_layers >= 3 && fused_supported(sizes[0], sizes[1], pad16(sizes[2]));
    const bool tail = n_layers >= (fused ? 4 : 2) &&
                      tail_supported(pad16(sizes[n_layers - 2]), pad16(sizes[n_layers - 1]), n_out);
    int64_t mac = 0;
    for (int l = 0; l < n_layers; ++l) {
        LayerBf16 &ly = sn.lay[l];
        ly.K = sizes[l];
        ly.N = sizes[l + 1];
        ly.Kp = pad16(ly.K);
        ly.Np = pad16(ly.N);
        ly.tiles_n = (ly.Np + 415) / 416;
        ly.n_tile = pad16((ly.Np + ly.tiles_n - 1) / ly.tiles_n);
        ly.tiles_n = (ly.Np + ly.n_tile - 1) / ly.n_tile;
        ly.n0 = ly.n_tile > 256 ? pad16((ly.n_tile + 1) / 2) : 0;
        mac += (int64_t)ly.Kp * ly.Np;
        std::vector<uint16_t> hw((size_t)ly.Np * ly.Kp, 0);
        std::vector<float> hb((size_t)ly.Np, 0.f);
        // every hidden activation is stored as 2 GELU(.) (ptx::gelu2_pack): its consumer W_l, l >= 1, carries the 1/2
        const float wscale = l >= 1 ? 0.5f : 1.f;
        for (int j = 0; j < ly.N; ++j) {
            for (int i = 0; i < ly.K; ++i) hw[(size_t)j * ly.Kp + i] = to_half(wscale * weights[l][(size_t)j * ly.K + i]);
            hb[j] = biases[l][j];
        }
        CU_TRY(c, cudaMalloc(&ly.W, hw.size() * sizeof(uint16_t)), "cudaMalloc(W bf16)");
        CU_TRY(c, cudaMalloc(&ly.bias, hb.size() * sizeof(float)), "cudaMalloc(bias)");
        CU_TRY(c, cudaMemcpy(ly.W, hw.data(), hw.size() * sizeof(uint16_t), cudaMemcpyHostToDevice), "cudaMemcpy(W)");
        CU_TRY(c, cudaMemcpy(ly.bias, hb.data(), hb.size() * sizeof(float), cudaMemcpyHostToDevice), "cudaMemcpy(bias)");
        std::string terr;
        if (!encode_tmap_bf16(&ly.tmapW, ly.W, (uint64_t)ly.Kp, (uint64_t)ly.Np, (uint64_t)ly.Kp * 2, (uint32_t)(ly.n0 > 0 ? ly.n0 : ly.n_tile), &terr))
            return fail(c, GPUANN_ERR_CUDA, "gpuann_load_net: " + terr);
    }
    if (fused) {
        FusedNet &fn = sn.fused;
        const int D = sizes[0], H1 = sizes[1];
        fused_plan(sn.lay[1].Np, &fn.n_pass, &fn.pass_w, &fn.n0, &fn.n1);
        // W1 padded to K = 64 with the bias in two extra columns: b1 = hi + lo, both BF16, multiplied by the
        // constant-1 features z[D], z[D+1] the kernel appends (bias error <= 2^-17 |b1|)
        const int H1p = (H1 + 63) / 64 * 64;  // rows up to the next multiple of 64 stay zero: h1 = 0 there (k_fused.cu)
        std::vector<uint16_t> w1((size_t)H1p * 64, 0);
        for (int j = 0; j < H1; ++j) {
            for (int i = 0; i < D; ++i) w1[(size_t)j * 64 + i] = to_half(weights[0][(size_t)j * D + i]);
            const float b = biases[0][j];
            const uint16_t hi = to_half(b);
            float hf;
            if (f16) {
                hf = f16_bits_to_f32(hi);
            } else {
                uint32_t hbits = (uint32_t)hi << 16;
                std::memcpy(&hf, &hbits, 4);
            }
            w1[(size_t)j * 64 + D] = hi;
            w1[(size_t)j * 64 + D + 1] = to_half(b - hf);
        }
        CU_TRY(c, cudaMalloc(&fn.W1p, w1.size() * sizeof(uint16_t)), "cudaMalloc(W1 padded)");
        CU_TRY(c, cudaMemcpy(fn.W1p, w1.data(), w1.size() * sizeof(uint16_t), cudaMemcpyHostToDevice), "cudaMemcpy(W1 padded)");
        std::string terr;
        const LayerBf16 &l2 = sn.lay[1];
        // boxes are a CTA's HALF of a stage: the pair's MMAs (cta_group::2) read half of B from each CTA (k_fused.cu)
        if (!encode_tmap_bf16(&fn.tmapW1, fn.W1p, 64, (uint64_t)H1p, 128, 16, &terr) ||
            !encode_tmap_bf16(&fn.tmapW2a, l2.W, (uint64_t)l2.Kp, (uint64_t)l2.Np, (uint64_t)l2.Kp * 2, (uint32_t)(fn.n0 / 2), &terr) ||
            !encode_tmap_bf16(&fn.tmapW2b, l2.W, (uint64_t)l2.Kp, (uint64_t)l2.Np, (uint64_t)l2.Kp * 2,
                              (uint32_t)(fn.n1 > 0 ? fn.n1 / 2 : 8), &terr))
            return fail(c, GPUANN_ERR_CUDA, "gpuann_load_net: " + terr);
        fn.on = true;
        // MACs issued: layer 1 once per pass over 16 * Kz columns, layer 2 over n_pass * pass_w columns
        const int Kz16 = ((D + 2 + 15) / 16) * 16;
        mac += (int64_t)fn.n_pass * H1p * Kz16 - (int64_t)sn.lay[0].Kp * sn.lay[0].Np;
        mac += (int64_t)H1p * (int64_t)fn.n_pass * fn.pass_w - (int64_t)l2.Kp * l2.Np;
    }
    const bool one_buffer = fused && tail && n_layers == 4;
    for (int l = fused ? 2 : 0; l < n_layers; ++l) {
        // tmapA is read by the layer kernel and by the tail kernel's row-major input.  Not encoded where nothing reads it:
        // the last layer under a tail kernel (h3 stays in shared memory), and the tail kernel's input when it is the
        // blocked h2 (tmapAb below) -- in that mode act[1] does not even exist.
        if (tail && (l == n_layers - 1 || (l == n_layers - 2 && one_buffer))) continue;
        LayerBf16 &ly = sn.lay[l];
        std::string terr;
        if (!encode_tmap_bf16(&ly.tmapA, c->act[l & 1], (uint64_t)ly.Kp, (uint64_t)chunk, (uint64_t)ly.Kp * 2, 128, &terr))
            return fail(c, GPUANN_ERR_CUDA, "gpuann_load_net: " + terr);
    }
    if (tail) {
        TailNet &tn = sn.tail;
        const LayerBf16 &l3 = sn.lay[n_layers - 2], &l4 = sn.lay[n_layers - 1];
        TailArgs &ta = tn.args;
        ta.Ns = n_out;
        ta.Np = l4.Np;
        ta.K3p = l3.Kp;
        ta.H3p = l3.Np;
        tail_plan(l3.Np, &ta.n0, &ta.n1);
        ta.bias3 = l3.bias;
        ta.newton_max_iter = po.newton_max_iter;
        ta.inv_lambda_int = po.inv_lambda_int;
        ta.lambda_zero = po.lambda_zero;
        ta.lambda = pre.lambda;
        ta.inv_lambda = pre.inv_lambda;
        ta.newton_tol = po.newton_tol;
        ta.T_min = po.T_min;
        ta.T_max = po.T_max;
        for (int k = 0; k < kTailMaxNs; ++k) ta.b4[k] = k < n_out ? biases[n_layers - 1][k] : 0.f;
        std::string terr;
        if (!encode_tmap_bf16(&tn.tmapW3a, l3.W, (uint64_t)l3.Kp, (uint64_t)l3.Np, (uint64_t)l3.Kp * 2, (uint32_t)(ta.n0 / 2), &terr) ||
            !encode_tmap_bf16(&tn.tmapW3b, l3.W, (uint64_t)l3.Kp, (uint64_t)l3.Np, (uint64_t)l3.Kp * 2,
                              (uint32_t)(ta.n1 > 0 ? ta.n1 / 2 : 8), &terr) ||
            !encode_tmap_bf16(&tn.tmapW4, l4.W, (uint64_t)l4.Kp, (uint64_t)l4.Np, (uint64_t)l4.Kp * 2, (uint32_t)(l4.Np / 2), &terr))
            return fail(c, GPUANN_ERR_CUDA, "gpuann_load_net: " + terr);
        // fused kernel directly in front: h2 travels in the blocked layout (common.cuh, FusedNet)
        ta.a_blocked = one_buffer ? 1 : 0;
        sn.fused.h2_blocked = one_buffer;
        if (one_buffer && !encode_tmap_bf16_linear(&tn.tmapAb, c->act[0], (uint64_t)chunk * (uint64_t)l3.Kp, &terr))
            return fail(c, GPUANN_ERR_CUDA, "gpuann_load_net: " + terr);
        tn.on = true;
    }
    if (mac_out) *mac_out = mac;
    return GPUANN_OK;
}

}  // namespace

extern "C" {

void gpuann_default_params(gpuann_params *p) {
    if (!p) return;
    p->precision = GPUANN_PRECISION_BF16;
    p->newton_max_iter = 20;
    p->newton_tol = 1e-6;
    p->T_min = 200.0;
    p->T_max = 3500.0;
    p->T_active = 0.0;
    p->device = -1;
    p->chunk_cells = 0;
}

int gpuann_create(const gpuann_params *params, gpuann_ctx **out) {
    if (!out) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_create: out is NULL");
    *out = nullptr;
    gpuann_params prm;
    gpuann_default_params(&prm);
    if (params) prm = *params;
    if (prm.precision != GPUANN_PRECISION_FP32 && prm.precision != GPUANN_PRECISION_BF16 && prm.precision != GPUANN_PRECISION_FP16)
        return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_create: precision must be 0 (FP32), 1 (BF16) or 2 (FP16)");
    if (prm.newton_max_iter < 0 || !(prm.newton_tol > 0.0) || !(prm.T_min > 0.0) || !(prm.T_max > prm.T_min) ||
        !std::isfinite(prm.T_active))
        return fail(nullptr, GPUANN_ERR_INVALID_ARG,
                    "gpuann_create: need newton_max_iter >= 0, newton_tol > 0, 0 < T_min < T_max, finite T_active");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev <= 0) {
        cudaGetLastError();
        return fail(nullptr, GPUANN_ERR_UNSUPPORTED,
                    std::string("gpuann_create: no CUDA device (there is no CPU fallback): ") + cudaGetErrorString(e));
    }
    int dev = prm.device;
    if (dev < 0) {
        if (cudaGetDevice(&dev) != cudaSuccess) dev = 0;
    }
    if (dev >= ndev) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_create: device ordinal out of range");
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return fail_cuda(nullptr, e, "cudaGetDeviceProperties");
    if (prop.major != 10)
        return fail(nullptr, GPUANN_ERR_UNSUPPORTED,
                    "gpuann_create: device compute capability " + std::to_string(prop.major) + "." +
                        std::to_string(prop.minor) + " is not 10.x (this library is sm_100a only)");
    gpuann_ctx *c = new (std::nothrow) gpuann_ctx();
    if (!c) return fail(nullptr, GPUANN_ERR_ALLOC, "gpuann_create: host allocation failed");
    c->prm = prm;
    c->device = dev;
    c->sm_count = prop.multiProcessorCount;
    DeviceGuard g(dev);
    if (!g.ok) {
        delete c;
        return fail(nullptr, GPUANN_ERR_CUDA, "gpuann_create: cudaSetDevice failed");
    }
    e = cudaMalloc(&c->counters, sizeof(Counters));
    if (e == cudaSuccess) e = cudaMemset(c->counters, 0, sizeof(Counters));
    if (e == cudaSuccess) e = cudaMalloc(&c->n_active_dev, sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(c->n_active_dev, 0, sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&c->thermo_dev, sizeof(ThermoDev));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess && prm.precision != GPUANN_PRECISION_FP32) e = gemm_setup(c);
    if (e == cudaSuccess && prm.precision != GPUANN_PRECISION_FP32) e = fused_setup(c);
    if (e == cudaSuccess && prm.precision != GPUANN_PRECISION_FP32) e = tail_setup(c);
    if (e != cudaSuccess) {
        int rc = fail_cuda(nullptr, e, "gpuann_create");
        gpuann_destroy(c);
        return rc;
    }
    *out = c;
    return GPUANN_OK;
}

// which kernels would run a net of these sizes, and whether this context's precision takes it (the same decisions as
// plan_and_alloc / build_subnet / the FP32 branch of gpuann_load_net, taken here without touching the context)
static int check_net_supported(gpuann_ctx *c, const char *fn, int n_layers, const int *sizes, int n_out, int n_nets, int maxw) {
    const std::string f(fn);
    if (c->prm.precision == GPUANN_PRECISION_FP32) {
        if (n_nets > 1) return fail(c, GPUANN_ERR_UNSUPPORTED, f + ": tensor path only (BF16 or FP16 context)");
        // fp32_smem_bytes: two activation rows of the widest layer for 8 cells must fit 200 KB of shared memory
        if (2ull * (size_t)maxw * 8 * sizeof(float) > 200 * 1024)
            return fail(c, GPUANN_ERR_UNSUPPORTED, f + ": layer too wide for the FP32 path (max width 3200)");
        return GPUANN_OK;
    }
    const bool fused = n_layers >= 3 && fused_supported(sizes[0], sizes[1], pad16(sizes[2]));
    const bool tail = n_layers >= (fused ? 4 : 2) && tail_supported(pad16(sizes[n_layers - 2]), pad16(sizes[n_layers - 1]), n_out);
    const bool two_kernels = fused && tail && n_layers == 4;
    if (c->prm.precision == GPUANN_PRECISION_FP16 && !two_kernels)
        return fail(c, GPUANN_ERR_UNSUPPORTED, f + ": GPUANN_PRECISION_FP16 needs a net the fused + tail kernels run (4 weight matrices)");
    if (n_nets > 1 && !two_kernels)
        return fail(c, GPUANN_ERR_UNSUPPORTED,
                    f + ": every net must run the fused + tail kernels (4 weight matrices, first hidden layer >= 128, last <= 416)");
    return GPUANN_OK;
}

// weights and biases must be finite, and on the tensor path they must stay finite in the operand type: a hidden-layer
// weight is stored as BF16 / FP16 of w/2 (build_subnet), the first-layer bias of the fused kernel as two such values.
// An inf operand would make the raw output NaN, every cell would take the vanishing-sum fallback and the chemistry would
// freeze with nothing but a counter to show for it -- so it is an error here.
static int check_net_values(gpuann_ctx *c, const char *fn, int n_layers, const int *sizes, int n_out, int n_nets,
                            const float *const *weights, const float *const *biases) {
    (void)n_out;
    const std::string f(fn);
    const int prec = c->prm.precision;
    const bool tensor = prec != GPUANN_PRECISION_FP32;
    const bool f16 = prec == GPUANN_PRECISION_FP16;
    const bool fused = tensor && n_layers >= 3 && fused_supported(sizes[0], sizes[1], pad16(sizes[2]));
    auto overflows = [f16](float v) {
        return f16 ? (f32_to_f16_rne(v) & 0x7C00u) == 0x7C00u : (f32_to_bf16_rne(v) & 0x7F80u) == 0x7F80u;
    };
    const char *type = f16 ? "FP16" : "BF16";
    for (int k = 0; k < n_nets; ++k)
        for (int l = 0; l < n_layers; ++l) {
            const float *w = weights[(size_t)k * n_layers + l], *b = biases[(size_t)k * n_layers + l];
            const size_t cnt = (size_t)sizes[l] * sizes[l + 1];
            const float wscale = l >= 1 ? 0.5f : 1.f;
            const std::string where = (n_nets > 1 ? " of net " + std::to_string(k) : std::string()) + " in layer " + std::to_string(l);
            for (size_t i = 0; i < cnt; ++i) {
                if (!finite_f(w[i])) return fail(c, GPUANN_ERR_INVALID_ARG, f + ": weight " + std::to_string(i) + where + " is not finite");
                if (tensor && overflows(wscale * w[i]))
                    return fail(c, GPUANN_ERR_INVALID_ARG, f + ": weight " + std::to_string(i) + where + " overflows " + type);
            }
            for (int j = 0; j < sizes[l + 1]; ++j) {
                if (!finite_f(b[j])) return fail(c, GPUANN_ERR_INVALID_ARG, f + ": bias " + std::to_string(j) + where + " is not finite");
                if (fused && l == 0 && overflows(b[j]))
                    return fail(c, GPUANN_ERR_INVALID_ARG, f + ": bias " + std::to_string(j) + where + " overflows " + type);
            }
        }
    return GPUANN_OK;
}

// validation + the parameter blocks every path shares (S1-S2 statistics, S4-S7 constants); frees the previous net once
// nothing can refuse the new one any more
static int load_prologue(gpuann_ctx *c, const char *fn, int n_species, int n_layers, const int *sizes, int n_out, int n_nets,
                         const float *const *weights, const float *const *biases, const float *in_mean,
                         const float *in_std, const float *out_mean, const float *out_std, double lambda) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": ctx is NULL");
    if (!sizes || !weights || !biases || !in_mean || !in_std || !out_mean || !out_std)
        return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": NULL argument");
    if (n_species < 1 || n_layers < 1) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": n_species, n_layers must be >= 1");
    if (n_species > GPUANN_MAX_SPECIES || n_layers > GPUANN_MAX_LAYERS)
        return fail(c, GPUANN_ERR_UNSUPPORTED, std::string(fn) + ": n_species > 64 or n_layers > 8");
    if (sizes[0] != n_species + 2 || sizes[n_layers] != n_out)
        return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": sizes[0] must be 2+Ns and sizes[L] must be " + (n_out == 1 ? "1" : "Ns"));
    int maxw = 0;
    for (int l = 0; l <= n_layers; ++l) {
        if (sizes[l] < 1) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": layer width < 1");
        if (sizes[l] > GPUANN_MAX_WIDTH) return fail(c, GPUANN_ERR_UNSUPPORTED, std::string(fn) + ": layer width > 4096");
        maxw = sizes[l] > maxw ? sizes[l] : maxw;
    }
    for (int l = 0; l < n_layers * n_nets; ++l)
        if (!weights[l] || !biases[l]) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": NULL weight or bias pointer");
    for (int j = 0; j < n_species + 2; ++j)
        if (!finite_f(in_mean[j]) || !finite_f(in_std[j]) || !(in_std[j] > 0.f))
            return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": in_mean must be finite and in_std finite and > 0");
    for (int k = 0; k < n_species; ++k)
        if (!finite_f(out_mean[k]) || !finite_f(out_std[k]))
            return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": out_mean / out_std must be finite");
    if (!(lambda >= 0.0) || !std::isfinite(lambda)) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": lambda must be >= 0");
    if (c->thermo_loaded && c->thermo_Ns != n_species)
        return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": n_species differs from the loaded thermo table");

    // Every check that can REFUSE the net runs before the net loaded earlier is freed, so a load that fails with
    // INVALID_ARG or UNSUPPORTED leaves that net in place and usable (include/gpuann.h).  Only ALLOC / CUDA failures
    // further down leave the context without a net.
    {
        const int rc = check_net_supported(c, fn, n_layers, sizes, n_out, n_nets, maxw);
        if (rc != GPUANN_OK) return rc;
        const int rc2 = check_net_values(c, fn, n_layers, sizes, n_out, n_nets, weights, biases);
        if (rc2 != GPUANN_OK) return rc2;
    }

    DeviceGuard g(c->device);
    cudaDeviceSynchronize();
    free_net(c);
    c->Ns = n_species;
    c->L = n_layers;
    for (int l = 0; l <= n_layers; ++l) c->sizes[l] = sizes[l];
    c->max_width = maxw;
    c->lambda = lambda;

    PreParams &pre = c->pre;
    pre = PreParams{};
    pre.n_species = n_species;
    pre.lambda_zero = lambda == 0.0 ? 1 : 0;
    pre.lambda = (float)lambda;
    pre.inv_lambda = lambda == 0.0 ? 0.f : (float)(1.0 / lambda);
    for (int j = 0; j < n_species + 2; ++j) {
        pre.mean[j] = in_mean[j];
        pre.inv_std[j] = (float)(1.0 / (double)in_std[j]);
    }
    PostParams &po = c->post;
    po = PostParams{};
    po.n_species = n_species;
    po.newton_max_iter = c->prm.newton_max_iter;
    po.newton_tol = c->prm.newton_tol;
    po.T_min = c->prm.T_min;
    po.T_max = c->prm.T_max;
    po.lambda = lambda;
    po.lambda_zero = pre.lambda_zero;
    po.inv_lambda = lambda == 0.0 ? 0.0 : 1.0 / lambda;
    po.inv_lambda_int = 0;
    if (lambda > 0.0) {
        const double r = std::round(po.inv_lambda);
        if (r >= 1.0 && r <= 1024.0 && std::fabs(po.inv_lambda - r) < 1e-12 * r) po.inv_lambda_int = (int)r;
    }
    for (int k = 0; k < n_species; ++k) {
        po.out_mean[k] = out_mean[k];
        po.out_std[k] = out_std[k];
    }

    return GPUANN_OK;
}

int gpuann_load_net(gpuann_ctx *c, int n_species, int n_layers, const int *sizes, const float *const *weights,
                    const float *const *biases, const float *in_mean, const float *in_std, const float *out_mean,
                    const float *out_std, double lambda) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_load_net: ctx is NULL");
    {
        const int rc0 = load_prologue(c, "gpuann_load_net", n_species, n_layers, sizes, n_species, 1, weights, biases, in_mean,
                                      in_std, out_mean, out_std, lambda);
        if (rc0 != GPUANN_OK) return rc0;
    }
    DeviceGuard g(c->device);
    PreParams &pre = c->pre;
    PostParams &po = c->post;
    (void)pre;
    (void)po;
    if (c->prm.precision == GPUANN_PRECISION_FP32) {
        size_t wc = 0, bc = 0;
        for (int l = 0; l < n_layers; ++l) {
            wc += (size_t)sizes[l] * sizes[l + 1];
            bc += (size_t)sizes[l + 1];
        }
        c->w32_count = wc;
        c->b32_count = bc;
        int cb = 0;
        fp32_smem_bytes(c, &cb);
        if (cb == 0) return fail(c, GPUANN_ERR_UNSUPPORTED, "gpuann_load_net: layer too wide for the FP32 path (max width 3200)");
        std::vector<float> hw(wc), hb(bc);
        size_t wo = 0, bo = 0;
        for (int l = 0; l < n_layers; ++l) {
            const size_t cnt = (size_t)sizes[l] * sizes[l + 1];
            std::memcpy(hw.data() + wo, weights[l], cnt * sizeof(float));
            std::memcpy(hb.data() + bo, biases[l], (size_t)sizes[l + 1] * sizeof(float));
            wo += cnt;
            bo += sizes[l + 1];
        }
        CU_TRY(c, cudaMalloc(&c->w32, wc * sizeof(float)), "cudaMalloc(weights)");
        CU_TRY(c, cudaMalloc(&c->b32, bc * sizeof(float)), "cudaMalloc(biases)");
        CU_TRY(c, cudaMemcpy(c->w32, hw.data(), wc * sizeof(float), cudaMemcpyHostToDevice), "cudaMemcpy(weights)");
        CU_TRY(c, cudaMemcpy(c->b32, hb.data(), bc * sizeof(float), cudaMemcpyHostToDevice), "cudaMemcpy(biases)");
        c->variant = "fp32";
        c->issued_mac_per_cell = 0;
        c->net_loaded = true;
        return GPUANN_OK;
    }

    // ---- tensor path
    int rc = plan_and_alloc(c, n_species, n_layers, sizes, false);
    if (rc != GPUANN_OK) return rc;
    rc = build_subnet(c, c->net0, n_species, n_layers, sizes, weights, biases, &c->issued_mac_per_cell);
    if (rc != GPUANN_OK) return rc;
    c->cur = &c->net0;
    const bool f16 = c->prm.precision == GPUANN_PRECISION_FP16;
    const bool fused = c->net0.fused.on, tail = c->net0.tail.on;
    c->variant = f16 ? "fp16-fused+tail"
                     : (fused ? (tail ? "bf16-fused+tail" : "bf16-fused") : (tail ? "bf16-layerwise+tail" : "bf16-layerwise"));
    c->net_loaded = true;
    return GPUANN_OK;
}

int gpuann_load_net_ensemble(gpuann_ctx *c, int n_species, int n_layers, const int *sizes, const float *const *weights,
                             const float *const *biases, const float *in_mean, const float *in_std, const float *out_mean,
                             const float *out_std, double lambda) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_load_net_ensemble: ctx is NULL");
    {
        const int rc0 = load_prologue(c, "gpuann_load_net_ensemble", n_species, n_layers, sizes, 1, n_species, weights, biases,
                                      in_mean, in_std, out_mean, out_std, lambda);
        if (rc0 != GPUANN_OK) return rc0;
    }
    if (c->prm.precision == GPUANN_PRECISION_FP32)
        return fail(c, GPUANN_ERR_UNSUPPORTED, "gpuann_load_net_ensemble: tensor path only (BF16 or FP16 context)");
    DeviceGuard g(c->device);
    int rc = plan_and_alloc(c, n_species, n_layers, sizes, true);
    if (rc != GPUANN_OK) return rc;
    c->ens.resize((size_t)n_species);
    int64_t mac_total = 0;
    for (int k = 0; k < n_species; ++k) {
        int64_t mac = 0;
        rc = build_subnet(c, c->ens[(size_t)k], 1, n_layers, sizes, weights + (size_t)k * n_layers, biases + (size_t)k * n_layers, &mac);
        if (rc != GPUANN_OK) return rc;
        mac_total += mac;
        if (!(c->ens[(size_t)k].fused.on && c->ens[(size_t)k].tail.on && n_layers == 4))
            return fail(c, GPUANN_ERR_UNSUPPORTED,
                        "gpuann_load_net_ensemble: every net must run the fused + tail kernels (4 weight matrices, first hidden layer >= 128, last <= 416)");
    }
    c->cur = &c->ens[0];
    c->issued_mac_per_cell = mac_total;
    c->variant = c->prm.precision == GPUANN_PRECISION_FP16 ? "fp16-ensemble" : "bf16-ensemble";
    c->net_loaded = true;
    return GPUANN_OK;
}

int gpuann_load_thermo(gpuann_ctx *c, int n_species, const double *nasa_lo, const double *nasa_hi, const double *T_mid,
                       const double *W) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: ctx is NULL");
    if (!nasa_lo || !W) return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: nasa_lo or W is NULL");
    if (n_species < 1) return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: n_species < 1");
    if (n_species > GPUANN_MAX_SPECIES) return fail(c, GPUANN_ERR_UNSUPPORTED, "gpuann_load_thermo: n_species > 64");
    if (c->net_loaded && c->Ns != n_species)
        return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: n_species differs from the loaded net");
    const bool two = nasa_hi && T_mid;
    ThermoDev *h = new (std::nothrow) ThermoDev();
    if (!h) return fail(c, GPUANN_ERR_ALLOC, "gpuann_load_thermo: host allocation failed");
    std::memset(h, 0, sizeof(ThermoDev));
    h->n_species = n_species;
    h->two_ranges = two ? 1 : 0;
    for (int k = 0; k < n_species; ++k) {
        if (!(W[k] > 0.0) || !std::isfinite(W[k])) {
            delete h;
            return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: W must be finite and > 0");
        }
        const double s = kRu / W[k];
        for (int r = 0; r < 2; ++r) {
            const double *a = (r == 1 && two) ? nasa_hi + 7 * k : nasa_lo + 7 * k;
            for (int j = 0; j < 7; ++j)
                if (!std::isfinite(a[j])) {
                    delete h;
                    return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_load_thermo: non-finite NASA-7 coefficient");
                }
            for (int j = 0; j < 5; ++j) h->cp[k][r][j] = s * a[j];
            h->hh[k][r][0] = s * a[5];
            h->hh[k][r][1] = s * a[0];
            h->hh[k][r][2] = s * a[1] / 2.0;
            h->hh[k][r][3] = s * a[2] / 3.0;
            h->hh[k][r][4] = s * a[3] / 4.0;
            h->hh[k][r][5] = s * a[4] / 5.0;
        }
        h->T_mid[k] = two ? T_mid[k] : 0.0;
        h->inv_W[k] = 1.0 / W[k];
    }
    {
        TailArgs &ta = c->net0.tail.args;  // the tail kernel takes the table by value (first kTailMaxNs species)
        ta.two_ranges = h->two_ranges;
        std::memset(&ta.th, 0, sizeof(ta.th));  // species beyond Ns of the kernel's padded range: all-zero constants
        for (int k = 0; k < kTailMaxNs && k < n_species; ++k) {
            std::memcpy(ta.th.cp[k], h->cp[k], sizeof(ta.th.cp[k]));
            std::memcpy(ta.th.hh[k], h->hh[k], sizeof(ta.th.hh[k]));
            ta.th.T_mid[k] = h->T_mid[k];
        }
        for (int k = 0; k < kTailMaxNs; ++k) ta.invW[k] = k < n_species ? (float)h->inv_W[k] : 0.f;
        std::memset(ta.hhf, 0, sizeof(ta.hhf));
        std::memset(ta.cpf, 0, sizeof(ta.cpf));
        for (int k = 0; k < kTailMaxNs && k < n_species; ++k) {
            for (int m = 0; m < 6; ++m) ta.hhf[k][m] = (float)h->hh[k][0][m];
            for (int m = 0; m < 5; ++m) ta.cpf[k][m] = (float)h->cp[k][0][m];
        }
    }
    DeviceGuard g(c->device);
    cudaDeviceSynchronize();
    cudaError_t e = cudaMemcpy(c->thermo_dev, h, sizeof(ThermoDev), cudaMemcpyHostToDevice);
    delete h;
    if (e != cudaSuccess) return fail_cuda(c, e, "gpuann_load_thermo: cudaMemcpy");
    c->thermo_loaded = true;
    c->thermo_Ns = n_species;
    return GPUANN_OK;
}

}  // extern "C"

// ================================================================ the step
namespace {

int ensure_compaction_scratch(Ctx *c, int64_t n) {
    if (n > c->idx_cap) {
        cudaFree(c->idx);
        c->idx = nullptr;
        c->idx_cap = 0;
        CU_TRY(c, cudaMalloc(&c->idx, (size_t)n * sizeof(int32_t)), "cudaMalloc(idx)");
        c->idx_cap = n;
    }
    const int64_t nb = (n + 2047) / 2048;
    if (nb > c->blk_cap) {
        cudaFree(c->blk_counts);
        c->blk_counts = nullptr;
        c->blk_cap = 0;
        CU_TRY(c, cudaMalloc(&c->blk_counts, (size_t)nb * sizeof(int32_t)), "cudaMalloc(blk_counts)");
        c->blk_cap = nb;
    }
    return GPUANN_OK;
}

// what a pass over one chunk produces: the raw network output (gpuann_debug_forward) or the updated state
struct ChunkOut {
    float *o_raw = nullptr;   // raw mode: o_raw[k * o_stride + local cell]
    int64_t o_stride = 0;
    float *T = nullptr, *Y = nullptr;  // update mode
    const float *h = nullptr;
    double dt = 0.0;
    ExtraOut ex;              // gpuann_chem_step_ex
};

// the tensor path for the chunk [c0, c0+cn): z -> layers -> (raw output | update S4-S8)
int run_chunk_bf16(Ctx *c, int64_t n, int64_t c0, int64_t cn, const float *T, const float *p, const float *Y, bool use_idx,
                   const ChunkOut &out, cudaStream_t s) {
    if (!c->ens.empty()) {
        // per-species ensemble (R24): net k's forward pass (fused kernel + tail kernel in its
        // forward-only mode) writes row k of the raw output; S4-S8 then run in the stand-alone update kernel
        const bool raw_e = out.o_raw != nullptr;
        float *o = raw_e ? out.o_raw : c->o_buf;
        const int64_t stride = raw_e ? out.o_stride : c->chunk;
        for (size_t k = 0; k < c->ens.size(); ++k) {
            c->cur = &c->ens[k];
            CU_TRY(c, launch_fused_l1l2(c, n, c0, cn, T, p, Y, use_idx, s), "fused kernel");
            CU_TRY(c, launch_tail(c, n, c0, cn, nullptr, p, nullptr, nullptr, 1.0, o + (int64_t)k * stride, stride, use_idx, ExtraOut{}, s),
                   "tail kernel");
        }
        if (!raw_e) CU_TRY(c, launch_post(c, n, c0, cn, out.T, out.Y, out.h, c->o_buf, c->chunk, out.dt, use_idx, p, out.ex, s), "update kernel");
        return GPUANN_OK;
    }
    int l0 = 0;
    if (c->cur->fused.on) {
        CU_TRY(c, launch_fused_l1l2(c, n, c0, cn, T, p, Y, use_idx, s), "fused kernel");
        l0 = 2;
    } else {
        CU_TRY(c, launch_pre_bf16(c, n, c0, cn, T, p, Y, use_idx, c->act[0], c->cur->lay[0].Kp, s), "pre kernel");
    }
    const bool raw = out.o_raw != nullptr;
    for (int l = l0; l < c->L; ++l) {
        if (c->cur->tail.on && l == c->L - 2) {
            CU_TRY(c, launch_tail(c, n, c0, cn, out.T, p, out.Y, out.h, out.dt, out.o_raw, out.o_stride, use_idx, out.ex, s), "tail kernel");
            return GPUANN_OK;
        }
        const bool last = l == c->L - 1;
        __nv_bfloat16 *nxt = last ? nullptr : c->act[(l + 1) & 1];
        CU_TRY(c,
               launch_layer_bf16(c, l, cn, &c->cur->lay[l].tmapA, nxt, last ? 0 : c->cur->lay[l + 1].Kp,
                                 last ? (raw ? out.o_raw : c->o_buf) : nullptr, raw ? out.o_stride : c->chunk, c0, use_idx, s),
               "layer kernel");
    }
    if (!raw) CU_TRY(c, launch_post(c, n, c0, cn, out.T, out.Y, out.h, c->o_buf, c->chunk, out.dt, use_idx, p, out.ex, s), "update kernel");
    return GPUANN_OK;
}

int check_step_args(Ctx *c, const char *fn, int64_t n, const void *T, const void *p, const void *Y, const void *h,
                    double dt, bool need_thermo) {
    if (n < 0) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": n_cells < 0");
    if (n > 0 && (!T || !p || !Y || (need_thermo && !h))) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": NULL state pointer");
    if (need_thermo && (!(dt > 0.0) || !std::isfinite(dt))) return fail(c, GPUANN_ERR_INVALID_ARG, std::string(fn) + ": dt must be > 0");
    if (n > 0x7FFFFFFFLL) return fail(c, GPUANN_ERR_UNSUPPORTED, std::string(fn) + ": n_cells >= 2^31");
    if (!c->net_loaded || (need_thermo && !c->thermo_loaded))
        return fail(c, GPUANN_ERR_NOT_READY, std::string(fn) + ": load_net" + (need_thermo ? " and load_thermo" : "") + " first");
    return GPUANN_OK;
}

}  // namespace

extern "C" {

int gpuann_chem_step(gpuann_ctx *c, int64_t n, float *T, const float *p, float *Y, const float *h, double dt,
                     void *stream) {
    return gpuann_chem_step_ex(c, n, T, p, Y, h, dt, nullptr, stream);
}

int gpuann_chem_step_ex(gpuann_ctx *c, int64_t n, float *T, const float *p, float *Y, const float *h, double dt,
                        const gpuann_step_outputs *xo, void *stream) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_chem_step: ctx is NULL");
    int rc = check_step_args(c, "gpuann_chem_step", n, T, p, Y, h, dt, true);
    if (rc != GPUANN_OK) return rc;
    if (n == 0) return GPUANN_OK;
    ExtraOut ex;
    if (xo) {
        ex.rr = xo->rr;
        ex.hrr = xo->hrr;
        ex.cp = xo->cp;
        ex.rho = xo->rho;
        ex.psi = xo->psi;
    }
    DeviceGuard g(c->device);
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    c->last_stream = s;
    if (c->prm.precision == GPUANN_PRECISION_FP32) {
        CU_TRY(c, launch_chem_fp32(c, n, T, p, Y, h, dt, nullptr, false, ex, s), "fp32 kernel");
        return GPUANN_OK;
    }
    const bool use_idx = c->prm.T_active > 0.0;
    if (use_idx) {
        rc = ensure_compaction_scratch(c, n);
        if (rc != GPUANN_OK) return rc;
        CU_TRY(c, launch_compact(c, n, T, (float)c->prm.T_active, s), "compaction kernels");
    } else {
        c->host_active += n;
    }
    ChunkOut out;
    out.T = T;
    out.Y = Y;
    out.h = h;
    out.dt = dt;
    out.ex = ex;
    for (int64_t c0 = 0; c0 < n; c0 += c->chunk) {
        const int64_t cn = (n - c0) < c->chunk ? (n - c0) : c->chunk;
        rc = run_chunk_bf16(c, n, c0, cn, T, p, Y, use_idx, out, s);
        if (rc != GPUANN_OK) return rc;
    }
    return GPUANN_OK;
}

int gpuann_debug_forward(gpuann_ctx *c, int64_t n, const float *T, const float *p, const float *Y, float *o_raw,
                         void *stream) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_debug_forward: ctx is NULL");
    int rc = check_step_args(c, "gpuann_debug_forward", n, T, p, Y, nullptr, 1.0, false);
    if (rc != GPUANN_OK) return rc;
    if (n > 0 && !o_raw) return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_debug_forward: o_raw is NULL");
    if (n == 0) return GPUANN_OK;
    DeviceGuard g(c->device);
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    c->last_stream = s;
    if (c->prm.precision == GPUANN_PRECISION_FP32) {
        CU_TRY(c, launch_chem_fp32(c, n, const_cast<float *>(T), p, const_cast<float *>(Y), nullptr, 1.0, o_raw, true, ExtraOut{}, s),
               "fp32 kernel");
        return GPUANN_OK;
    }
    for (int64_t c0 = 0; c0 < n; c0 += c->chunk) {
        const int64_t cn = (n - c0) < c->chunk ? (n - c0) : c->chunk;
        ChunkOut out;
        out.o_raw = o_raw + c0;
        out.o_stride = n;
        rc = run_chunk_bf16(c, n, c0, cn, T, p, Y, false, out, s);
        if (rc != GPUANN_OK) return rc;
    }
    return GPUANN_OK;
}

int gpuann_chem_step_host(gpuann_ctx *c, int64_t n, float *T, const float *p, float *Y, const float *h, double dt) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_chem_step_host: ctx is NULL");
    int rc = check_step_args(c, "gpuann_chem_step_host", n, T, p, Y, h, dt, true);
    if (rc != GPUANN_OK) return rc;
    if (n == 0) return GPUANN_OK;
    DeviceGuard g(c->device);
    const size_t Ns = (size_t)c->Ns;
    const size_t need = (3 + Ns) * (size_t)n;
    if (need > c->stage_floats) {
        cudaFree(c->stage);
        c->stage = nullptr;
        c->stage_floats = 0;
        CU_TRY(c, cudaMalloc(&c->stage, need * sizeof(float)), "cudaMalloc(staging)");
        c->stage_floats = need;
    }
    float *dT = c->stage, *dp = dT + n, *dh = dp + n, *dY = dh + n;
    cudaStream_t s = c->own_stream;
    const size_t fb = (size_t)n * sizeof(float);
    const bool pipelined = c->prm.precision != GPUANN_PRECISION_FP32 && !(c->prm.T_active > 0.0) && n >= 4 * 128 * (int64_t)c->sm_count;
    if (!pipelined) {
        CU_TRY(c, cudaMemcpyAsync(dT, T, fb, cudaMemcpyHostToDevice, s), "H2D T");
        CU_TRY(c, cudaMemcpyAsync(dp, p, fb, cudaMemcpyHostToDevice, s), "H2D p");
        CU_TRY(c, cudaMemcpyAsync(dh, h, fb, cudaMemcpyHostToDevice, s), "H2D h");
        CU_TRY(c, cudaMemcpyAsync(dY, Y, fb * Ns, cudaMemcpyHostToDevice, s), "H2D Y");
        rc = gpuann_chem_step(c, n, dT, dp, dY, dh, dt, s);
        if (rc != GPUANN_OK) return rc;
        CU_TRY(c, cudaMemcpyAsync(T, dT, fb, cudaMemcpyDeviceToHost, s), "D2H T");
        CU_TRY(c, cudaMemcpyAsync(Y, dY, fb * Ns, cudaMemcpyDeviceToHost, s), "D2H Y");
        CU_TRY(c, cudaStreamSynchronize(s), "cudaStreamSynchronize");
        return GPUANN_OK;
    }
    // Pipelined: the field is cut into slices of whole tiles; slice i+1 is copied in and slice i-1 copied out (on two
    // copy streams) while slice i is computed -- cells are independent, and the kernels take (first cell, count)
    // of a field with row stride n, so a slice needs no repacking.  The step is then PCIe bound or compute bound,
    // whichever is slower, instead of the sum.  INVARIANT: a slice never exceeds the scratch chunk.
    const int64_t unit = 128 * (int64_t)c->sm_count;
    int64_t slice = ((n + 7) / 8 + unit - 1) / unit * unit;
    if (slice > c->chunk) slice = c->chunk;
    const int64_t n_slices = (n + slice - 1) / slice;
    if (!c->copy_in || !c->copy_out) {  // both streams or neither
        cudaStream_t a = nullptr, b = nullptr;
        cudaError_t e = cudaStreamCreateWithFlags(&a, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&b, cudaStreamNonBlocking);
        if (e != cudaSuccess) {
            if (a) cudaStreamDestroy(a);
            if (b) cudaStreamDestroy(b);
            return fail_cuda(c, e, "cudaStreamCreate");
        }
        c->copy_in = a;
        c->copy_out = b;
    }
    while ((int64_t)c->slice_events.size() < 2 * n_slices) {
        cudaEvent_t e;
        CU_TRY(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "cudaEventCreate");
        c->slice_events.push_back(e);
    }
    const size_t pitch = fb;
    c->last_stream = s;
    // any failure inside the loop: wait for the copies already in flight into the caller's buffers, then report
    auto drain = [&]() {
        cudaStreamSynchronize(c->copy_in);
        cudaStreamSynchronize(s);
        cudaStreamSynchronize(c->copy_out);
    };
#define CU_TRY_DRAIN(call, what)                  \
    do {                                          \
        cudaError_t e__ = (call);                 \
        if (e__ != cudaSuccess) {                 \
            drain();                              \
            return fail_cuda(c, e__, what);       \
        }                                         \
    } while (0)
    int64_t i = 0;
    for (int64_t a = 0; a < n; a += slice, ++i) {
        const int64_t len = (n - a) < slice ? (n - a) : slice;
        const size_t lb = (size_t)len * sizeof(float);
        cudaEvent_t e_in = c->slice_events[2 * i], e_done = c->slice_events[2 * i + 1];
        CU_TRY_DRAIN(cudaMemcpyAsync(dT + a, T + a, lb, cudaMemcpyHostToDevice, c->copy_in), "H2D T");
        CU_TRY_DRAIN(cudaMemcpyAsync(dp + a, p + a, lb, cudaMemcpyHostToDevice, c->copy_in), "H2D p");
        CU_TRY_DRAIN(cudaMemcpyAsync(dh + a, h + a, lb, cudaMemcpyHostToDevice, c->copy_in), "H2D h");
        CU_TRY_DRAIN(cudaMemcpy2DAsync(dY + a, pitch, Y + a, pitch, lb, Ns, cudaMemcpyHostToDevice, c->copy_in), "H2D Y");
        CU_TRY_DRAIN(cudaEventRecord(e_in, c->copy_in), "cudaEventRecord");
        CU_TRY_DRAIN(cudaStreamWaitEvent(s, e_in, 0), "cudaStreamWaitEvent");
        ChunkOut out;
        out.T = dT;
        out.Y = dY;
        out.h = dh;
        out.dt = dt;
        rc = run_chunk_bf16(c, n, a, len, dT, dp, dY, false, out, s);
        if (rc != GPUANN_OK) {
            drain();
            return rc;
        }
        CU_TRY_DRAIN(cudaEventRecord(e_done, s), "cudaEventRecord");
        CU_TRY_DRAIN(cudaStreamWaitEvent(c->copy_out, e_done, 0), "cudaStreamWaitEvent");
        CU_TRY_DRAIN(cudaMemcpyAsync(T + a, dT + a, lb, cudaMemcpyDeviceToHost, c->copy_out), "D2H T");
        CU_TRY_DRAIN(cudaMemcpy2DAsync(Y + a, pitch, dY + a, pitch, lb, Ns, cudaMemcpyDeviceToHost, c->copy_out), "D2H Y");
    }
#undef CU_TRY_DRAIN
    c->host_active += n;
    CU_TRY(c, cudaStreamSynchronize(c->copy_out), "cudaStreamSynchronize");
    CU_TRY(c, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    return GPUANN_OK;
}

int gpuann_get_stats(gpuann_ctx *c, int64_t *n_active, int64_t *n_not_converged, int64_t *n_degenerate) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_get_stats: ctx is NULL");
    DeviceGuard g(c->device);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream), "cudaStreamSynchronize");
    Counters h;
    CU_TRY(c, cudaMemcpy(&h, c->counters, sizeof(h), cudaMemcpyDeviceToHost), "cudaMemcpy(counters)");
    if (n_active) *n_active = (int64_t)h.n_active + c->host_active;
    if (n_not_converged) *n_not_converged = (int64_t)h.n_not_converged;
    if (n_degenerate) *n_degenerate = (int64_t)h.n_degenerate;
    return GPUANN_OK;
}

int gpuann_reset_stats(gpuann_ctx *c) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_reset_stats: ctx is NULL");
    DeviceGuard g(c->device);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream), "cudaStreamSynchronize");
    CU_TRY(c, cudaMemset(c->counters, 0, sizeof(Counters)), "cudaMemset(counters)");
    c->host_active = 0;
    return GPUANN_OK;
}

int gpuann_enthalpy(gpuann_ctx *c, int64_t n, const float *T, const float *Y, float *h_out, void *stream) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_enthalpy: ctx is NULL");
    if (n < 0 || (n > 0 && (!T || !Y || !h_out))) return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_enthalpy: bad argument");
    if (!c->thermo_loaded) return fail(c, GPUANN_ERR_NOT_READY, "gpuann_enthalpy: load_thermo first");
    DeviceGuard g(c->device);
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    c->last_stream = s;
    CU_TRY(c, launch_enthalpy(c, n, T, Y, h_out, s), "enthalpy kernel");
    return GPUANN_OK;
}

int gpuann_input_moments(gpuann_ctx *c, int64_t n, int n_species, const float *T, const float *p, const float *Y,
                         double lambda, double *mean_out, double *std_out, void *stream) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_input_moments: ctx is NULL");
    if (n <= 0 || n_species < 1 || n_species > GPUANN_MAX_SPECIES || !T || !p || !Y || !mean_out || !std_out ||
        !(lambda >= 0.0))
        return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_input_moments: bad argument");
    DeviceGuard g(c->device);
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    c->last_stream = s;
    CU_TRY(c, launch_moments(c, n, n_species, T, p, Y, lambda, mean_out, std_out, s), "moments kernel");
    return GPUANN_OK;
}

// gpuann_input_moments for callers that cannot allocate device memory (include/gpuann.h): scratch in a static __device__
// array of k_aux.cu, no cudaMalloc / cudaFree, sizes beyond the array are refused
int gpuann_input_moments_static(gpuann_ctx *c, int64_t n, int n_species, const float *T, const float *p, const float *Y,
                                double lambda, double *mean_out, double *std_out, void *stream) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_input_moments_static: ctx is NULL");
    if (n <= 0 || n_species < 1 || !T || !p || !Y || !mean_out || !std_out || !(lambda >= 0.0))
        return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_input_moments_static: bad argument");
    if (n_species > GPUANN_STATIC_MAX_SPECIES)
        return fail(c, GPUANN_ERR_UNSUPPORTED,
                    "gpuann_input_moments_static: n_species = " + std::to_string(n_species) + " does not fit the static scratch (at most " +
                        std::to_string(GPUANN_STATIC_MAX_SPECIES) + " species, " + std::to_string(GPUANN_STATIC_SCRATCH_BYTES) +
                        " bytes); this entry point never allocates");
    DeviceGuard g(c->device);
    if (!g.ok) return fail(c, GPUANN_ERR_CUDA, "gpuann_input_moments_static: cudaSetDevice failed");
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    c->last_stream = s;
    CU_TRY(c, launch_moments_static(c, n, n_species, T, p, Y, lambda, mean_out, std_out, s), "moments kernels (static scratch)");
    return GPUANN_OK;
}

int64_t gpuann_launch_count(const gpuann_ctx *c) { return c ? c->launches : 0; }

static void recycle_timed(Ctx *c) {
    for (auto &t : c->timed) {
        c->event_pool.push_back(t.e0);
        c->event_pool.push_back(t.e1);
    }
    c->timed.clear();
}

int gpuann_timing_enable(gpuann_ctx *c, int enable) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_timing_enable: ctx is NULL");
    DeviceGuard g(c->device);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream), "cudaStreamSynchronize");
    recycle_timed(c);
    c->timing = enable != 0;
    return GPUANN_OK;
}

int gpuann_timing_read(gpuann_ctx *c, int n_classes, double *ms, int64_t *counts) {
    if (!c) return fail(nullptr, GPUANN_ERR_INVALID_ARG, "gpuann_timing_read: ctx is NULL");
    if (n_classes < 0 || (n_classes > 0 && (!ms || !counts)))
        return fail(c, GPUANN_ERR_INVALID_ARG, "gpuann_timing_read: bad argument");
    DeviceGuard g(c->device);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream), "cudaStreamSynchronize");
    for (int i = 0; i < n_classes; ++i) {
        ms[i] = 0.0;
        counts[i] = 0;
    }
    for (auto &t : c->timed) {
        float dtm = 0.f;
        cudaError_t e = cudaEventElapsedTime(&dtm, t.e0, t.e1);
        if (e != cudaSuccess) return fail_cuda(c, e, "cudaEventElapsedTime");
        if (t.cls >= 0 && t.cls < n_classes) {
            ms[t.cls] += (double)dtm;
            counts[t.cls] += 1;
        }
    }
    recycle_timed(c);
    return GPUANN_OK;
}

int gpuann_timing_num_classes(void) { return kNumKernelClasses; }

const char *gpuann_timing_class_name(int cls) {
    static const char *names[kNumKernelClasses] = {"compact",      "pre_boxcox_norm", "layer0_gemm", "layer1_gemm",
                                                   "layer2_gemm",  "layer3_gemm",     "layer4_gemm", "layer5_gemm",
                                                   "layer6_gemm",  "layer7_gemm",     "post_update_newton",
                                                   "fp32_fused",   "bf16_fused",      "aux",         "bf16_tail"};
    return (cls >= 0 && cls < kNumKernelClasses) ? names[cls] : "";
}

int gpuann_describe(const gpuann_ctx *c, int64_t *issued_mac_per_cell, const char **variant) {
    if (!c) return GPUANN_ERR_INVALID_ARG;
    if (issued_mac_per_cell) *issued_mac_per_cell = c->issued_mac_per_cell;
    if (variant) *variant = c->variant;
    return GPUANN_OK;
}

const char *gpuann_last_error(const gpuann_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }

int gpuann_destroy(gpuann_ctx *c) {
    if (!c) return GPUANN_OK;
    {
        DeviceGuard g(c->device);
        cudaDeviceSynchronize();
        free_net(c);
        cudaFree(c->thermo_dev);
        cudaFree(c->idx);
        cudaFree(c->blk_counts);
        cudaFree(c->n_active_dev);
        cudaFree(c->stage);
        cudaFree(c->counters);
        recycle_timed(c);
        for (cudaEvent_t e : c->event_pool) cudaEventDestroy(e);
        c->event_pool.clear();
        if (c->own_stream) cudaStreamDestroy(c->own_stream);
        if (c->copy_in) cudaStreamDestroy(c->copy_in);
        if (c->copy_out) cudaStreamDestroy(c->copy_out);
        for (cudaEvent_t e : c->slice_events) cudaEventDestroy(e);
        c->slice_events.clear();
        cudaGetLastError();
    }
    delete c;
    return GPUANN_OK;
}

}  // extern "C"
