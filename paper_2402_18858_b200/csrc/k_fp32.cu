// k_fp32.cu -- GPUANN_PRECISION_FP32: the whole step S0-S7 in ONE kernel on the CUDA cores (BASELINE.json
// configs[0]: 4,096 cells, 11-64-64-9).  A block owns CB cells; thread (c, g) = (tid % CB, tid / CB) computes the
// outputs j = g, g+G, ... of every layer for cell c, so a warp reads one weight (broadcast) against CB different
// activations (bank-conflict free: activations are stored [width][CB]).  All weights and biases sit in shared
// memory when they fit (configs[0]: 21.5 KB), else they are read through L1.  FP32 FMA in index order,
// exact-erf GELU (R5); the update S4-S7 in FP64 by the threads g == 0 (post.cuh).
#include "common.cuh"
#include "post.cuh"

namespace gpuann {

constexpr int kFp32Threads = 256;

struct Fp32Net {
    int L;
    int sizes[kMaxLayers + 1];
    int w_off[kMaxLayers];
    int b_off[kMaxLayers];
    int w_count, b_count;
    int max_width;
    int weights_in_smem;
};

__device__ __forceinline__ float gelu_erf(float v) {
    return 0.5f * v * (1.f + erff(v * 0.70710678118654752f));
}

template <int CB>
__global__ void __launch_bounds__(kFp32Threads) k_chem_fp32(int64_t n, float *__restrict__ T, const float *__restrict__ p,
                                                            float *__restrict__ Y, const float *__restrict__ h,
                                                            double dt, float *__restrict__ o_raw, int forward_only,
                                                            float T_active, const float *__restrict__ w_g,
                                                            const float *__restrict__ b_g,
                                                            const ThermoDev *__restrict__ thermo,
                                                            Counters *__restrict__ counters, const Fp32Net net,
                                                            const PreParams pre, const PostParams pp, const ExtraOut ex) {
    extern __shared__ __align__(16) float smem[];
    constexpr int G = kFp32Threads / CB;
    float *act0 = smem;
    float *act1 = act0 + (size_t)net.max_width * CB;
    float *w_s = act1 + (size_t)net.max_width * CB;
    float *b_s = w_s + net.w_count;
    const float *W = w_g, *B = b_g;
    if (net.weights_in_smem) {
        for (int i = threadIdx.x; i < net.w_count; i += kFp32Threads) w_s[i] = w_g[i];
        for (int i = threadIdx.x; i < net.b_count; i += kFp32Threads) b_s[i] = b_g[i];
        W = w_s;
        B = b_s;
    }
    const int c = threadIdx.x % CB, g = threadIdx.x / CB;
    const int64_t cell = (int64_t)blockIdx.x * CB + c;
    const int Ns = pre.n_species, D = Ns + 2;
    const bool in_range = cell < n;
    const float Tin = in_range ? T[cell] : 0.f;
    const bool active = in_range && (forward_only || !(T_active > 0.f && Tin < T_active));  // S0 (R12)

    // S1 + S2: features j = g, g+G, ...
    for (int j = g; j < D; j += G) {
        float x = 0.f;
        if (in_range) {
            if (j == 0) x = Tin;
            else if (j == 1) x = p[cell];
            else {
                const float Yc = fmaxf(Y[(int64_t)(j - 2) * n + cell], 0.f);
                x = boxcox_y(Yc, boxcox_u(Yc, pre.lambda), pre);
            }
            x = (x - pre.mean[j]) * pre.inv_std[j];
        }
        act0[j * CB + c] = x;
    }
    __syncthreads();

    // S3
    float *a = act0, *nx = act1;
    for (int l = 0; l < net.L; ++l) {
        const int n_in = net.sizes[l], n_out = net.sizes[l + 1];
        const float *Wl = W + net.w_off[l];
        const float *Bl = B + net.b_off[l];
        const bool last = (l == net.L - 1);
        for (int j0 = g; j0 < n_out; j0 += 4 * G) {
            // four outputs per pass share the activation loads
            const int j1 = j0 + G, j2 = j0 + 2 * G, j3 = j0 + 3 * G;
            const bool v1 = j1 < n_out, v2 = j2 < n_out, v3 = j3 < n_out;
            const float *r0 = Wl + (size_t)j0 * n_in;
            const float *r1 = Wl + (size_t)(v1 ? j1 : j0) * n_in;
            const float *r2 = Wl + (size_t)(v2 ? j2 : j0) * n_in;
            const float *r3 = Wl + (size_t)(v3 ? j3 : j0) * n_in;
            float s0 = Bl[j0], s1 = v1 ? Bl[j1] : 0.f, s2 = v2 ? Bl[j2] : 0.f, s3 = v3 ? Bl[j3] : 0.f;
#pragma unroll 4
            for (int i = 0; i < n_in; ++i) {
                const float av = a[i * CB + c];
                s0 = fmaf(r0[i], av, s0);
                s1 = fmaf(r1[i], av, s1);
                s2 = fmaf(r2[i], av, s2);
                s3 = fmaf(r3[i], av, s3);
            }
            nx[j0 * CB + c] = last ? s0 : gelu_erf(s0);
            if (v1) nx[j1 * CB + c] = last ? s1 : gelu_erf(s1);
            if (v2) nx[j2 * CB + c] = last ? s2 : gelu_erf(s2);
            if (v3) nx[j3 * CB + c] = last ? s3 : gelu_erf(s3);
        }
        __syncthreads();
        float *t = a;
        a = nx;
        nx = t;
    }
    // a[k*CB + c] = raw output o_k of cell c

    if (forward_only) {
        if (in_range)
            for (int k = g; k < Ns; k += G) o_raw[(int64_t)k * n + cell] = a[k * CB + c];
        return;
    }

    // S4-S7 by the threads of group 0 (one per cell)
    unsigned nact = 0, nconv = 0, ndeg = 0;
    if (g == 0 && active) {
        nact = 1;
        double Yc[kMaxSpecies], Ys[kMaxSpecies];
#pragma unroll 1
        for (int k = 0; k < Ns; ++k) {
            const float yf = fmaxf(Y[(int64_t)k * n + cell], 0.f);
            const float u = boxcox_u(yf, pre.lambda);
            Yc[k] = (double)yf;
            Ys[k] = update_species((double)yf, u, a[k * CB + c], pp.out_std[k], pp.out_mean[k], dt, pp);
        }
        if (renormalise<kMaxSpecies>(Ys, Yc, Ns)) ndeg = 1;
        bool conv;
        const double Tn = thermo->two_ranges ? newton_T<kMaxSpecies>(Ys, Ns, (double)h[cell], (double)Tin, thermo, pp, &conv)
                                             : newton_T_mixture<kMaxSpecies>(Ys, Ns, (double)h[cell], (double)Tin, thermo, pp, &conv);
        if (!conv) nconv = 1;
        if (ex.any()) {
            // gpuann_chem_step_ex (include/gpuann.h; R19-R21), FP64, before the inputs are overwritten
            double inv_w_in = 0.0, inv_w = 0.0, cpm = 0.0, q = 0.0;
#pragma unroll 1
            for (int k = 0; k < Ns; ++k) inv_w_in = fma(Yc[k], thermo->inv_W[k], inv_w_in);
            const double rho_in = (double)p[cell] / (kRu * (double)Tin * inv_w_in);
            const double rate = rho_in / dt;
#pragma unroll 1
            for (int k = 0; k < Ns; ++k) {
                const int r = (thermo->two_ranges && !(Tn < thermo->T_mid[k])) ? 1 : 0;
                const double *cpk = thermo->cp[k][r];
                const double *hh = thermo->hh[k][r];
                const double hk = hh[0] + Tn * (hh[1] + Tn * (hh[2] + Tn * (hh[3] + Tn * (hh[4] + Tn * hh[5]))));
                const double rr = rate * (Ys[k] - (double)Y[(int64_t)k * n + cell]);
                q = fma(-hk, rr, q);
                cpm = fma(Ys[k], cpk[0] + Tn * (cpk[1] + Tn * (cpk[2] + Tn * (cpk[3] + Tn * cpk[4]))), cpm);
                inv_w = fma(Ys[k], thermo->inv_W[k], inv_w);
                if (ex.rr) ex.rr[(int64_t)k * n + cell] = (float)rr;
            }
            const double psi = 1.0 / (kRu * inv_w * Tn);
            if (ex.hrr) ex.hrr[cell] = (float)q;
            if (ex.cp) ex.cp[cell] = (float)cpm;
            if (ex.rho) ex.rho[cell] = (float)((double)p[cell] * psi);
            if (ex.psi) ex.psi[cell] = (float)psi;
        }
#pragma unroll 1
        for (int k = 0; k < Ns; ++k) Y[(int64_t)k * n + cell] = (float)Ys[k];
        T[cell] = (float)Tn;
    }
    if (threadIdx.x < 32) {  // warp 0 holds every g == 0 thread (CB <= 32)
        nact = __reduce_add_sync(0xffffffffu, nact);
        nconv = __reduce_add_sync(0xffffffffu, nconv);
        ndeg = __reduce_add_sync(0xffffffffu, ndeg);
        if (threadIdx.x == 0) {
            if (nact) atomicAdd(&counters->n_active, (unsigned long long)nact);
            if (nconv) atomicAdd(&counters->n_not_converged, (unsigned long long)nconv);
            if (ndeg) atomicAdd(&counters->n_degenerate, (unsigned long long)ndeg);
        }
    }
}

// Shared memory the kernel needs for the loaded net with CB cells per block; picks the largest CB that fits.
// Returns 0 if even CB = 8 does not fit (UNSUPPORTED on the FP32 path).
size_t fp32_smem_bytes(const Ctx *c, int *cells_per_block) {
    const size_t budget = 200 * 1024;
    const size_t wb = (c->w32_count + c->b32_count) * sizeof(float);
    for (int cb : {32, 16, 8}) {
        const size_t act = 2ull * (size_t)c->max_width * cb * sizeof(float);
        if (act > budget) continue;
        *cells_per_block = cb;
        return act + (act + wb <= budget ? wb : 0);
    }
    *cells_per_block = 0;
    return 0;
}

cudaError_t launch_chem_fp32(Ctx *c, int64_t n, float *T, const float *p, float *Y, const float *h, double dt,
                             float *o_raw, bool forward_only, const ExtraOut &ex, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    int cb = 0;
    const size_t smem = fp32_smem_bytes(c, &cb);
    if (cb == 0) return cudaErrorInvalidConfiguration;
    Fp32Net net{};
    net.L = c->L;
    int wo = 0, bo = 0;
    for (int l = 0; l <= c->L; ++l) net.sizes[l] = c->sizes[l];
    for (int l = 0; l < c->L; ++l) {
        net.w_off[l] = wo;
        net.b_off[l] = bo;
        wo += c->sizes[l] * c->sizes[l + 1];
        bo += c->sizes[l + 1];
    }
    net.w_count = (int)c->w32_count;
    net.b_count = (int)c->b32_count;
    net.max_width = c->max_width;
    const size_t act = 2ull * (size_t)c->max_width * cb * sizeof(float);
    net.weights_in_smem = smem > act ? 1 : 0;
    const unsigned blocks = (unsigned)((n + cb - 1) / cb);
    const float Tact = (float)c->prm.T_active;
    cudaError_t e = cudaSuccess;
    LaunchScope ls(c, kClsFp32, s);
#define GPUANN_LAUNCH_FP32(CB)                                                                                       \
    do {                                                                                                             \
        e = cudaFuncSetAttribute(k_chem_fp32<CB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);           \
        if (e == cudaSuccess)                                                                                        \
            k_chem_fp32<CB><<<blocks, kFp32Threads, smem, s>>>(n, T, p, Y, h, dt, o_raw, forward_only ? 1 : 0, Tact, \
                                                               c->w32, c->b32, c->thermo_dev, c->counters, net,     \
                                                               c->pre, c->post, ex);                                 \
    } while (0)
    if (cb == 32) GPUANN_LAUNCH_FP32(32);
    else if (cb == 16) GPUANN_LAUNCH_FP32(16);
    else GPUANN_LAUNCH_FP32(8);
#undef GPUANN_LAUNCH_FP32
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace gpuann
