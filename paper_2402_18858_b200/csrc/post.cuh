// post.cuh -- per-cell device functions of the steps S1 and S4-S7 (include/gpuann.h), shared by the FP32 kernel,
// the stand-alone update kernel and the fused tensor-path epilogue.  FP64 for everything that decides parity
// (DESIGN.md "Precision of the scalar math"); only Y^lambda is evaluated in FP32.
#pragma once
#include "common.cuh"

namespace gpuann {

// S1 (Eq. 7; R1, R2): u = max(Y,0)^lambda, so that y = (u - 1)/lambda.  u(0) = 0 exactly.
__device__ __forceinline__ float boxcox_u(float Yc, float lambda) {
    return Yc > 0.f ? powf(Yc, lambda) : 0.f;
}

// transformed mass fraction fed to the net: y = (u - 1)/lambda  (log Y when lambda = 0)
__device__ __forceinline__ float boxcox_y(float Yc, float u, const PreParams &pp) {
    return pp.lambda_zero ? logf(Yc) : (u - 1.f) * pp.inv_lambda;
}

__device__ __forceinline__ double powi(double x, int n) {
    double r = 1.0;
    while (n) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}

// S4 + S5 for one species (R3, R7): dy = dt (o sigma_out + mu_out);
// Y* = max(1 + lambda (y + dy), 0)^(1/lambda) = Yc (max(1 + lambda dy / u, 0))^(1/lambda), evaluated in the
// multiplicative form so that the FP32 rounding of u only touches the (small) correction factor.
// Yc = 0 (u = 0): Y* = max(lambda dy, 0)^(1/lambda).  lambda = 0: Y* = Yc exp(dy).
__device__ __forceinline__ double update_species(double Yc, float u, float o, float out_std, float out_mean,
                                                 double dt, const PostParams &pp) {
    const double dy = dt * ((double)o * (double)out_std + (double)out_mean);
    if (pp.lambda_zero) return Yc * exp(dy);
    const double ldy = pp.lambda * dy;
    double base, scale;
    if (u > 0.f) {
        // 1/u: FP32 reciprocal refined by two Newton steps in FP64 (relative error < 1e-15) instead of an FP64 division
        const double ud = (double)u;
        double r = (double)__frcp_rn(u);
        r = r * (2.0 - ud * r);
        r = r * (2.0 - ud * r);
        base = 1.0 + ldy * r;
        scale = Yc;
    } else {
        base = ldy;
        scale = 1.0;
    }
    if (!(base > 0.0)) return 0.0;
    const double pw = pp.inv_lambda_int > 0 ? powi(base, pp.inv_lambda_int) : pow(base, pp.inv_lambda);
    return scale * pw;
}

// S7 (R9-R11): Newton iteration for sum_k Y_k h_k(T) = h on the pre-scaled NASA-7 table `th`
// (shared or global memory).  Y[] holds the renormalised mass fractions.  Returns the last iterate;
// *converged = |dT| < tol was met.
template <int MAXNS>
__device__ __forceinline__ double newton_T(const double (&Y)[MAXNS], int Ns, double h, double T0,
                                           const ThermoDev *__restrict__ th, const PostParams &pp, bool *converged) {
    double T = fmin(fmax(T0, pp.T_min), pp.T_max);
    bool conv = false;
    const int two = th->two_ranges;
    for (int it = 0; it < pp.newton_max_iter; ++it) {
        double f = -h, c = 0.0;
#pragma unroll 1
        for (int k = 0; k < Ns; ++k) {
            const int r = (two && !(T < th->T_mid[k])) ? 1 : 0;
            const double *cp = th->cp[k][r];
            const double *hh = th->hh[k][r];
            const double cpk = cp[0] + T * (cp[1] + T * (cp[2] + T * (cp[3] + T * cp[4])));
            const double hk = hh[0] + T * (hh[1] + T * (hh[2] + T * (hh[3] + T * (hh[4] + T * hh[5]))));
            f = fma(Y[k], hk, f);
            c = fma(Y[k], cpk, c);
        }
        if (!(c > 0.0)) break;
        const double dT = -f / c;
        T = fmin(fmax(T + dT, pp.T_min), pp.T_max);
        if (fabs(dT) < pp.newton_tol) {
            conv = true;
            break;
        }
    }
    *converged = conv;
    return T;
}

// The same solve for a ONE-RANGE table through the mixture polynomials: C_j = sum_k Y_k c_kj once (11 FMAs per species), then
// 11 FMAs per iteration instead of 11 Ns -- the FP64 pipe of this part is slow.  Differs from newton_T
// only by the FP64 rounding of the regrouped sums.
template <int MAXNS>
__device__ __forceinline__ double newton_T_mixture(const double (&Y)[MAXNS], int Ns, double h, double T0,
                                                   const ThermoDev *__restrict__ th, const PostParams &pp, bool *converged) {
    double Ch[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, Cc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll 1
    for (int k = 0; k < Ns; ++k) {
#pragma unroll
        for (int m = 0; m < 6; ++m) Ch[m] = fma(Y[k], th->hh[k][0][m], Ch[m]);
#pragma unroll
        for (int m = 0; m < 5; ++m) Cc[m] = fma(Y[k], th->cp[k][0][m], Cc[m]);
    }
    double T = fmin(fmax(T0, pp.T_min), pp.T_max);
    bool conv = false;
    for (int it = 0; it < pp.newton_max_iter; ++it) {
        const double f = Ch[0] + T * (Ch[1] + T * (Ch[2] + T * (Ch[3] + T * (Ch[4] + T * Ch[5])))) - h;
        const double c = Cc[0] + T * (Cc[1] + T * (Cc[2] + T * (Cc[3] + T * Cc[4])));
        if (!(c > 0.0)) break;
        const double dT = -f / c;
        T = fmin(fmax(T + dT, pp.T_min), pp.T_max);
        if (fabs(dT) < pp.newton_tol) {
            conv = true;
            break;
        }
    }
    *converged = conv;
    return T;
}

// S6: divide by the sum (R8); a vanishing sum falls back to max(Y,0)/sum (counted as degenerate).
// Ys[] in: Y*; out: Y_new.  Yc[] = clamped inputs.  Returns true if degenerate.
template <int MAXNS>
__device__ __forceinline__ bool renormalise(double (&Ys)[MAXNS], const double (&Yc)[MAXNS], int Ns) {
    double S = 0.0;
#pragma unroll 1
    for (int k = 0; k < Ns; ++k) S += Ys[k];
    if (S > 0.0) {
        const double rS = 1.0 / S;  // one division per cell; Y* rS differs from Y*/S by <= 1 ulp of FP64
#pragma unroll 1
        for (int k = 0; k < Ns; ++k) Ys[k] = Ys[k] * rS;
        return false;
    }
    double Sc = 0.0;
#pragma unroll 1
    for (int k = 0; k < Ns; ++k) Sc += Yc[k];
#pragma unroll 1
    for (int k = 0; k < Ns; ++k) Ys[k] = Yc[k] / Sc;
    return true;
}

}  // namespace gpuann
