// k_aux.cu -- the HBM-bound kernels around the MLP: S0 active-cell compaction, S1+S2 (Box-Cox + normalise ->
// BF16 rows for the tensor path), S4-S7 (update + Newton T-solve) as a stand-alone kernel, and the input-recipe
// helpers gpuann_enthalpy / gpuann_input_moments.  All state accesses are along the cell index of the SoA
// fields, i.e. coalesced 128-byte lines per warp.
#include <mutex>

#include "common.cuh"
#include "post.cuh"

namespace gpuann {

// ================================================================ S0: compaction (BASELINE.json configs[4]; R12)
// Order-preserving: idx[] lists the active cells in increasing cell order, so results do not depend on timing.
constexpr int kCompThreads = 256;
constexpr int kCompPerThread = 8;
constexpr int kCompPerBlock = kCompThreads * kCompPerThread;

__device__ __forceinline__ int block_exclusive_scan_256(int v, int *total) {
    __shared__ int warp_sums[kCompThreads / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) warp_sums[w] = incl;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < kCompThreads / 32; ++i) {
        int s = warp_sums[i];
        if (i < w) base += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return base + incl - v;
}

__global__ void __launch_bounds__(kCompThreads) k_compact_count(int64_t n, const float *__restrict__ T, float T_active,
                                                                int32_t *__restrict__ blk_counts) {
    const int64_t base = (int64_t)blockIdx.x * kCompPerBlock + (int64_t)threadIdx.x * kCompPerThread;
    int cnt = 0;
#pragma unroll
    for (int j = 0; j < kCompPerThread; ++j) {
        const int64_t i = base + j;
        if (i < n && !(T[i] < T_active)) ++cnt;
    }
    int total;
    (void)block_exclusive_scan_256(cnt, &total);
    if (threadIdx.x == 0) blk_counts[blockIdx.x] = total;
}

// one block: exclusive scan of the per-block counts in place; total -> *n_active and the statistics counter
__global__ void __launch_bounds__(kCompThreads) k_compact_scan(int nb, int32_t *__restrict__ blk_counts,
                                                               int32_t *__restrict__ n_active,
                                                               Counters *__restrict__ counters) {
    __shared__ int carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += kCompThreads) {
        const int b = b0 + threadIdx.x;
        const int v = b < nb ? blk_counts[b] : 0;
        int total;
        const int ex = block_exclusive_scan_256(v, &total);
        const int carry = carry_s;
        if (b < nb) blk_counts[b] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *n_active = carry_s;
        counters->n_active += (unsigned long long)carry_s;
    }
}

__global__ void __launch_bounds__(kCompThreads) k_compact_scatter(int64_t n, const float *__restrict__ T, float T_active,
                                                                  const int32_t *__restrict__ blk_offsets,
                                                                  int32_t *__restrict__ idx) {
    const int64_t base = (int64_t)blockIdx.x * kCompPerBlock + (int64_t)threadIdx.x * kCompPerThread;
    unsigned mask = 0;
    int cnt = 0;
#pragma unroll
    for (int j = 0; j < kCompPerThread; ++j) {
        const int64_t i = base + j;
        if (i < n && !(T[i] < T_active)) {
            mask |= 1u << j;
            ++cnt;
        }
    }
    int total;
    int pos = blk_offsets[blockIdx.x] + block_exclusive_scan_256(cnt, &total);
#pragma unroll
    for (int j = 0; j < kCompPerThread; ++j)
        if (mask & (1u << j)) idx[pos++] = (int32_t)(base + j);
}

cudaError_t launch_compact(Ctx *c, int64_t n, const float *T, float T_active, cudaStream_t s) {
    const int nb = (int)((n + kCompPerBlock - 1) / kCompPerBlock);
    LaunchScope ls(c, kClsCompact, s, 3);
    k_compact_count<<<nb, kCompThreads, 0, s>>>(n, T, T_active, c->blk_counts);
    k_compact_scan<<<1, kCompThreads, 0, s>>>(nb, c->blk_counts, c->n_active_dev, c->counters);
    k_compact_scatter<<<nb, kCompThreads, 0, s>>>(n, T, T_active, c->blk_counts, c->idx);
    return cudaGetLastError();
}

// ================================================================ S1 + S2 -> BF16 rows (R1, R2, R4)
// One thread per cell of the chunk [c0, c0+cn): z[i][0..Kp) = BF16((x_j - mean_j) * inv_std_j), x = {T, p, y_1..y_Ns},
// zero padded to Kp columns (a multiple of 16, <= 80 here).  Row i of z is 2*Kp bytes, written as 16-byte stores.
__global__ void __launch_bounds__(128) k_pre_bf16(int64_t n, int64_t c0, int64_t cn, const float *__restrict__ T,
                                                  const float *__restrict__ p, const float *__restrict__ Y,
                                                  const int32_t *__restrict__ idx, const int32_t *__restrict__ n_active,
                                                  __nv_bfloat16 *__restrict__ z, int Kp, const PreParams pp) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cn) return;
    int64_t g = c0 + i;
    bool valid = true;
    if (idx) {
        valid = g < (int64_t)*n_active;
        g = valid ? (int64_t)idx[g] : 0;
    }
    uint4 *row = reinterpret_cast<uint4 *>(z + i * Kp);
    const int D = pp.n_species + 2;
    for (int j0 = 0; j0 < Kp; j0 += 8) {
        float v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int j = j0 + q;
            float x = 0.f;
            if (valid && j < D) {
                if (j == 0) x = T[g];
                else if (j == 1) x = p[g];
                else {
                    const float Yc = fmaxf(Y[(int64_t)(j - 2) * n + g], 0.f);
                    x = boxcox_y(Yc, boxcox_u(Yc, pp.lambda), pp);
                }
                x = (x - pp.mean[j]) * pp.inv_std[j];
            }
            v[q] = x;
        }
        uint4 o;
        __nv_bfloat162 t0 = __floats2bfloat162_rn(v[0], v[1]);
        __nv_bfloat162 t1 = __floats2bfloat162_rn(v[2], v[3]);
        __nv_bfloat162 t2 = __floats2bfloat162_rn(v[4], v[5]);
        __nv_bfloat162 t3 = __floats2bfloat162_rn(v[6], v[7]);
        o.x = *reinterpret_cast<uint32_t *>(&t0);
        o.y = *reinterpret_cast<uint32_t *>(&t1);
        o.z = *reinterpret_cast<uint32_t *>(&t2);
        o.w = *reinterpret_cast<uint32_t *>(&t3);
        row[j0 >> 3] = o;
    }
}

cudaError_t launch_pre_bf16(Ctx *c, int64_t n, int64_t c0, int64_t cn, const float *T, const float *p, const float *Y,
                            bool use_idx, __nv_bfloat16 *z, int Kp, cudaStream_t s) {
    if (cn <= 0) return cudaSuccess;
    const int blocks = (int)((cn + 127) / 128);
    LaunchScope ls(c, kClsPre, s);
    k_pre_bf16<<<blocks, 128, 0, s>>>(n, c0, cn, T, p, Y, use_idx ? c->idx : nullptr, c->n_active_dev, z, Kp, c->pre);
    return cudaGetLastError();
}

// ================================================================ S4-S7 as a stand-alone kernel
// FOUR lanes per cell (a "quad"): lane s of the quad owns the species k = s, s + 4, s + 8, ...; the sums over the
// species (renormalisation, Newton residual and slope) are xor-butterfly reductions inside the quad, which give all
// four lanes bit-identical results, so they take the same Newton decisions.  Per-thread state is NSL = ceil(Ns/4)
// doubles: registers, high occupancy.  (One thread per cell with run-time indexed double[64] arrays kept them in
// local memory: 0.47 ms per 1 M cells; fully unrolled over 21 species it needed 128-160 registers: 0.52 ms.)
// o[k*o_stride + i] is the raw network output of local cell i.  Writes Y_new (FP32, in place) and T_new; skipped /
// out-of-range cells are not touched.
__device__ __forceinline__ double quad_sum(double x) {
    x += __shfl_xor_sync(0xffffffffu, x, 1);
    x += __shfl_xor_sync(0xffffffffu, x, 2);
    return x;
}

template <int NSL>
__global__ void __launch_bounds__(128) k_post_q(int64_t n, int64_t c0, int64_t cn, float *__restrict__ T,
                                                float *__restrict__ Y, const float *__restrict__ h,
                                                const float *__restrict__ o, int64_t o_stride, double dt,
                                                const int32_t *__restrict__ idx, const int32_t *__restrict__ n_active,
                                                const ThermoDev *__restrict__ thermo_g, Counters *__restrict__ counters,
                                                float lambda_f, const PostParams pp, const float *__restrict__ p,
                                                const ExtraOut ex) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ThermoDev *th = reinterpret_cast<ThermoDev *>(smem_raw);
    {
        const int words = (int)(sizeof(ThermoDev) / 4);
        const uint32_t *src = reinterpret_cast<const uint32_t *>(thermo_g);
        uint32_t *dst = reinterpret_cast<uint32_t *>(th);
        for (int w = threadIdx.x; w < words; w += blockDim.x) dst[w] = src[w];
    }
    __syncthreads();
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = t >> 2;     // local cell of this quad
    const int s = (int)(t & 3);   // species slice
    const int Ns = pp.n_species;
    bool valid = i < cn;
    int64_t g = c0 + i;
    if (valid && idx) {
        valid = g < (int64_t)*n_active;
        g = valid ? (int64_t)idx[g] : 0;
    }
    if (!valid) g = 0;
    // invalid quads run along on zeros (the shuffles need every lane) and store nothing
    float yin[NSL], oin[NSL];
#pragma unroll
    for (int j = 0; j < NSL; ++j) {  // loads first: 2 NSL independent requests in flight
        const int k = s + 4 * j;
        const bool on = valid && k < Ns;
        yin[j] = on ? Y[(int64_t)k * n + g] : 0.f;
        oin[j] = on ? o[(int64_t)k * o_stride + i] : 0.f;
    }
    const double hc = valid ? (double)h[g] : 0.0, T0 = valid ? (double)T[g] : 300.0;
    double Ys[NSL];
    double S = 0.0, Sc = 0.0;
#pragma unroll
    for (int j = 0; j < NSL; ++j) {
        const int k = s + 4 * j;
        const float yf = fmaxf(yin[j], 0.f);
        Ys[j] = (k < Ns) ? update_species((double)yf, boxcox_u(yf, lambda_f), oin[j], pp.out_std[k < Ns ? k : 0],
                                          pp.out_mean[k < Ns ? k : 0], dt, pp)
                         : 0.0;
        S += Ys[j];
        Sc += (double)yf;
    }
    S = quad_sum(S);
    Sc = quad_sum(Sc);  // (outside the branch below: the shuffles are warp-wide)
    unsigned ndeg = 0, nconv = 0;
    if (S > 0.0) {
        const double rS = 1.0 / S;  // one division per thread; Y* rS differs from Y*/S by <= 1 ulp of FP64
#pragma unroll
        for (int j = 0; j < NSL; ++j) Ys[j] = Ys[j] * rS;
    } else {  // R8: vanishing sum -> max(Y,0)/sum, counted once per cell
        ndeg = (valid && s == 0) ? 1u : 0u;
#pragma unroll
        for (int j = 0; j < NSL; ++j) Ys[j] = (double)fmaxf(yin[j], 0.f) / Sc;
    }
    // S7: Newton on the pre-scaled NASA-7 table (the arithmetic of post.cuh newton_T, species split over the quad)
    double Tn = fmin(fmax(T0, pp.T_min), pp.T_max);
    bool conv = false, done = false;
    const int two = th->two_ranges;
    for (int it = 0; it < pp.newton_max_iter; ++it) {
        double f = 0.0, c = 0.0;
#pragma unroll
        for (int j = 0; j < NSL; ++j) {
            const int k = s + 4 * j;
            if (k < Ns) {
                const int r = (two && !(Tn < th->T_mid[k])) ? 1 : 0;
                const double *cp = th->cp[k][r];
                const double *hh = th->hh[k][r];
                const double cpk = cp[0] + Tn * (cp[1] + Tn * (cp[2] + Tn * (cp[3] + Tn * cp[4])));
                const double hk = hh[0] + Tn * (hh[1] + Tn * (hh[2] + Tn * (hh[3] + Tn * (hh[4] + Tn * hh[5]))));
                f = fma(Ys[j], hk, f);
                c = fma(Ys[j], cpk, c);
            }
        }
        // warp-wide shuffles: quads that have finished keep computing on their frozen state
        f = quad_sum(f) - hc;
        c = quad_sum(c);
        if (!done) {
            if (!(c > 0.0)) {
                done = true;  // R10: stop, not converged
            } else {
                const double dT = -f / c;
                Tn = fmin(fmax(Tn + dT, pp.T_min), pp.T_max);
                if (fabs(dT) < pp.newton_tol) conv = done = true;
            }
        }
        if (__all_sync(0xffffffffu, done)) break;
    }
    if (ex.any()) {
        // gpuann_chem_step_ex (include/gpuann.h; R19-R21), FP64, species split over the quad like everything above; the
        // shuffles are warp-wide, so every lane runs along (ex.any() is uniform)
        double inv_w_in = 0.0, inv_w = 0.0, cpm = 0.0;
#pragma unroll
        for (int j = 0; j < NSL; ++j) {
            const int k = s + 4 * j;
            if (k < Ns) {
                inv_w_in = fma((double)fmaxf(yin[j], 0.f), th->inv_W[k], inv_w_in);
                inv_w = fma(Ys[j], th->inv_W[k], inv_w);
            }
        }
        inv_w_in = quad_sum(inv_w_in);
        inv_w = quad_sum(inv_w);
        const double pin = valid ? (double)p[g] : 101325.0;
        const double rate = valid ? pin / (kRu * T0 * inv_w_in) / dt : 0.0;  // rho of the input state / dt
        double q = 0.0;
#pragma unroll
        for (int j = 0; j < NSL; ++j) {
            const int k = s + 4 * j;
            if (k < Ns) {
                const int r = (two && !(Tn < th->T_mid[k])) ? 1 : 0;
                const double *cp = th->cp[k][r];
                const double *hh = th->hh[k][r];
                const double hk = hh[0] + Tn * (hh[1] + Tn * (hh[2] + Tn * (hh[3] + Tn * (hh[4] + Tn * hh[5]))));
                const double rr = rate * (Ys[j] - (double)yin[j]);
                q = fma(-hk, rr, q);
                cpm = fma(Ys[j], cp[0] + Tn * (cp[1] + Tn * (cp[2] + Tn * (cp[3] + Tn * cp[4]))), cpm);
                if (valid && ex.rr) ex.rr[(int64_t)k * n + g] = (float)rr;
            }
        }
        q = quad_sum(q);
        cpm = quad_sum(cpm);
        if (valid && s == 0) {
            const double psi = 1.0 / (kRu * inv_w * Tn);
            if (ex.hrr) ex.hrr[g] = (float)q;
            if (ex.cp) ex.cp[g] = (float)cpm;
            if (ex.rho) ex.rho[g] = (float)(pin * psi);
            if (ex.psi) ex.psi[g] = (float)psi;
        }
    }
    if (valid) {
        if (!conv && s == 0) nconv = 1u;
#pragma unroll
        for (int j = 0; j < NSL; ++j) {
            const int k = s + 4 * j;
            if (k < Ns) Y[(int64_t)k * n + g] = (float)Ys[j];
        }
        if (s == 0) T[g] = (float)Tn;
    }
    // statistics: one atomic per warp and counter, only when something happened
    nconv = __reduce_add_sync(0xffffffffu, nconv);
    ndeg = __reduce_add_sync(0xffffffffu, ndeg);
    if ((threadIdx.x & 31) == 0) {
        if (nconv) atomicAdd(&counters->n_not_converged, (unsigned long long)nconv);
        if (ndeg) atomicAdd(&counters->n_degenerate, (unsigned long long)ndeg);
    }
}

template <int NSL>
static void launch_post_q(Ctx *c, int64_t n, int64_t c0, int64_t cn, float *T, float *Y, const float *h, const float *o,
                          int64_t o_stride, double dt, const int32_t *ix, const float *p, const ExtraOut &ex, cudaStream_t s) {
    const unsigned blocks = (unsigned)((cn * 4 + 127) / 128);
    k_post_q<NSL><<<blocks, 128, sizeof(ThermoDev), s>>>(n, c0, cn, T, Y, h, o, o_stride, dt, ix, c->n_active_dev,
                                                         c->thermo_dev, c->counters, (float)c->lambda, c->post, p, ex);
}

cudaError_t launch_post(Ctx *c, int64_t n, int64_t c0, int64_t cn, float *T, float *Y, const float *h, const float *o,
                        int64_t o_stride, double dt, bool use_idx, const float *p, const ExtraOut &ex, cudaStream_t s) {
    if (cn <= 0) return cudaSuccess;
    LaunchScope ls(c, kClsPost, s);
    const int32_t *ix = use_idx ? c->idx : nullptr;
    if (c->Ns <= 12) launch_post_q<3>(c, n, c0, cn, T, Y, h, o, o_stride, dt, ix, p, ex, s);
    else if (c->Ns <= 24) launch_post_q<6>(c, n, c0, cn, T, Y, h, o, o_stride, dt, ix, p, ex, s);
    else if (c->Ns <= 40) launch_post_q<10>(c, n, c0, cn, T, Y, h, o, o_stride, dt, ix, p, ex, s);
    else launch_post_q<16>(c, n, c0, cn, T, Y, h, o, o_stride, dt, ix, p, ex, s);
    return cudaGetLastError();
}

// ================================================================ input-recipe helpers (G4, G5)
// G5: h_i = sum_k Y[k][i] h_k(T_i) in FP64 from the FP32 state, rounded to FP32.
__global__ void __launch_bounds__(128) k_enthalpy(int64_t n, const float *__restrict__ T, const float *__restrict__ Y,
                                                  float *__restrict__ h_out, const ThermoDev *__restrict__ th) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double t = (double)T[i];
    const int Ns = th->n_species, two = th->two_ranges;
    double s = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const int r = (two && !(t < th->T_mid[k])) ? 1 : 0;
        const double *hh = th->hh[k][r];
        const double hk = hh[0] + t * (hh[1] + t * (hh[2] + t * (hh[3] + t * (hh[4] + t * hh[5]))));
        s = fma((double)Y[(int64_t)k * n + i], hk, s);
    }
    h_out[i] = (float)s;
}

cudaError_t launch_enthalpy(Ctx *c, int64_t n, const float *T, const float *Y, float *h_out, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    LaunchScope ls(c, kClsAux, s);
    k_enthalpy<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(n, T, Y, h_out, c->thermo_dev);
    return cudaGetLastError();
}

// G4: per-feature sum of (x - shift)^power over the batch, FP64, x = {T, p, F(Y_k)} with the FP64 Box-Cox of
// the FP32 Y.  Per-block partial sums; the host adds them in block order (deterministic).
constexpr int kMomThreads = 256;
__global__ void __launch_bounds__(kMomThreads) k_moment_partial(int64_t n, int D, const float *__restrict__ T,
                                                                const float *__restrict__ p,
                                                                const float *__restrict__ Y, double lambda,
                                                                const double *__restrict__ shift, int square,
                                                                double *__restrict__ partial /* [gridDim.x][D] */) {
    __shared__ double red[kMomThreads / 32];
    for (int j = 0; j < D; ++j) {
        const double sh = shift ? shift[j] : 0.0;
        double acc = 0.0;
        for (int64_t i = (int64_t)blockIdx.x * kMomThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kMomThreads) {
            double x;
            if (j == 0) x = (double)T[i];
            else if (j == 1) x = (double)p[i];
            else {
                double yc = (double)Y[(int64_t)(j - 2) * n + i];
                if (yc < 0.0) yc = 0.0;
                x = lambda != 0.0 ? (pow(yc, lambda) - 1.0) / lambda : log(yc);
            }
            x -= sh;
            acc += square ? x * x : x;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < kMomThreads / 32; ++w) t += red[w];
            partial[(size_t)blockIdx.x * D + j] = t;
        }
        __syncthreads();
    }
}

cudaError_t launch_moments(Ctx *c, int64_t n, int Ns, const float *T, const float *p, const float *Y, double lambda,
                           double *mean_out, double *std_out, cudaStream_t s) {
    const int D = Ns + 2;
    const int blocks = 2 * (c->sm_count > 0 ? c->sm_count : 148);
    double *partial = nullptr, *shift = nullptr;
    cudaError_t e = cudaMalloc(&partial, sizeof(double) * (size_t)blocks * D);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&shift, sizeof(double) * D);
    if (e != cudaSuccess) {
        cudaFree(partial);
        return e;
    }
    std::vector<double> hp((size_t)blocks * D), mean(D);
    for (int pass = 0; pass < 2 && e == cudaSuccess; ++pass) {
        {
            LaunchScope ls(c, kClsAux, s);
            k_moment_partial<<<blocks, kMomThreads, 0, s>>>(n, D, T, p, Y, lambda, pass ? shift : nullptr, pass, partial);
        }
        e = cudaGetLastError();
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(hp.data(), partial, sizeof(double) * hp.size(), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) break;
        for (int j = 0; j < D; ++j) {
            double t = 0.0;
            for (int b = 0; b < blocks; ++b) t += hp[(size_t)b * D + j];
            if (pass == 0) {
                mean[j] = t / (double)n;
                mean_out[j] = mean[j];
            } else {
                std_out[j] = sqrt(t / (double)n);
            }
        }
        if (pass == 0) e = cudaMemcpyAsync(shift, mean.data(), sizeof(double) * D, cudaMemcpyHostToDevice, s);
    }
    cudaStreamSynchronize(s);
    cudaFree(partial);
    cudaFree(shift);
    return e;
}


// ================================================================ gpuann_input_moments_static: the same statistics, NO allocation
// The two-pass moment kernel above needs scratch: one FP64 partial sum per (block, feature) and the D means that pass 2
// subtracts.  launch_moments gets both from cudaMalloc on every call.  This variant is for callers that cannot do that
// while they run (include/gpuann.h says who and why), so its scratch is the file-scope array below: part of the
// library's device image, present on every GPU that loads the library, until the process exits.
//
//   layout (doubles): [kStatMaxBlocks * kStatMaxD] partial sums | [kStatMaxD] mean | [kStatMaxD] std
//   size:             (512 * 66 + 2 * 66) * 8 = 271,392 bytes  (GPUANN_STATIC_SCRATCH_BYTES)
//
// Nothing in it has to start at zero: every word a call reads (partial[b][j] for b < blocks, j < D; mean[j]; std[j]) is
// written earlier in the same call, on the same stream, so whatever the previous call left behind -- more blocks, more
// species -- is never looked at.  The array is shared by all contexts and all streams of a device: two calls that
// overlap on the GPU overwrite each other's sums.
//
// In HOST code `g_moment_scratch` is only a handle of the symbol, not an address a kernel may dereference: the device
// address is looked up once per device with cudaGetSymbolAddress (that device current) and passed to the kernels.
constexpr int kStatMaxBlocks = 512;
constexpr int kStatMaxD = kMaxSpecies + 2;
constexpr int kStatMaxDevices = 64;
constexpr size_t kStatDoubles = (size_t)kStatMaxBlocks * kStatMaxD + 2 * (size_t)kStatMaxD;
static_assert(kStatDoubles * sizeof(double) == GPUANN_STATIC_SCRATCH_BYTES, "gpuann.h states the size of the static scratch");
static_assert(kMaxSpecies == GPUANN_STATIC_MAX_SPECIES, "gpuann.h states the species limit of the static scratch");

static __device__ __align__(256) double g_moment_scratch[kStatDoubles];

static std::mutex g_stat_mu;
static double *g_stat_ptr[kStatMaxDevices] = {};  // device address of g_moment_scratch on device d; nullptr = not looked up

// set-up, once per device; `dev` must be the current device
static cudaError_t moment_scratch_of_device(int dev, double **out) {
    if (dev < 0 || dev >= kStatMaxDevices) return cudaErrorInvalidDevice;
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return e;
    if (cur != dev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_stat_mu);
    if (!g_stat_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_moment_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_stat_ptr[dev] = static_cast<double *>(ptr);
    }
    *out = g_stat_ptr[dev];
    return cudaSuccess;
}

// Adds the per-block partial sums in block order -- the order, the division and the square root of launch_moments' host
// loop, all IEEE FP64 -- so both entry points return the same bits for the same grid.  One thread per feature.
__global__ void __launch_bounds__(128) k_moment_finish(int blocks, int D, int64_t n, int take_sqrt,
                                                       const double *__restrict__ partial, double *__restrict__ result) {
    const int j = threadIdx.x;
    if (j >= D) return;
    double t = 0.0;
    for (int b = 0; b < blocks; ++b) t += partial[(size_t)b * D + j];
    const double q = t / (double)n;
    result[j] = take_sqrt ? sqrt(q) : q;
}

cudaError_t launch_moments_static(Ctx *c, int64_t n, int Ns, const float *T, const float *p, const float *Y, double lambda,
                                  double *mean_out, double *std_out, cudaStream_t s) {
    const int D = Ns + 2;
    if (D > kStatMaxD) return cudaErrorInvalidValue;  // the ABI entry has rejected this with a message already
    int blocks = 2 * (c->sm_count > 0 ? c->sm_count : 148);
    if (blocks > kStatMaxBlocks) blocks = kStatMaxBlocks;
    double *scr = nullptr;
    cudaError_t e = moment_scratch_of_device(c->device, &scr);
    if (e != cudaSuccess) return e;
    double *partial = scr, *mean = scr + (size_t)kStatMaxBlocks * kStatMaxD, *sd = mean + kStatMaxD;
    // (no LaunchScope: with the timing hook on it may create events; these four launches are counted, not timed)
    c->launches += 4;
    k_moment_partial<<<blocks, kMomThreads, 0, s>>>(n, D, T, p, Y, lambda, nullptr, 0, partial);
    k_moment_finish<<<1, 128, 0, s>>>(blocks, D, n, 0, partial, mean);
    k_moment_partial<<<blocks, kMomThreads, 0, s>>>(n, D, T, p, Y, lambda, mean, 1, partial);
    k_moment_finish<<<1, 128, 0, s>>>(blocks, D, n, 1, partial, sd);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(mean_out, mean, sizeof(double) * D, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(std_out, sd, sizeof(double) * D, cudaMemcpyDeviceToHost, s);
    const cudaError_t e2 = cudaStreamSynchronize(s);
    return e != cudaSuccess ? e : e2;
}

}  // namespace gpuann
