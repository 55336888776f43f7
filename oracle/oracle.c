/*
 * oracle.c -- plain FP64 CPU oracle for the GPU-ANN chemistry step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and the cpu_baseline / --impl reference legs of bench.py may build, load or call it.
 * It shares no source, header, table or helper with paper_2402_18858_b200/csrc/.
 *
 * What it computes, per cell, in the paper's order (PAPER.md = /root/reference/PAPER.md,
 * arXiv 2402.18858; R<n> = the readings listed in DESIGN.md "Readings of the paper"):
 *
 *   O0  active-cell test (BASELINE.json configs[4]; R12)
 *   O1  Box-Cox transform of the mass fractions        PAPER.md:98-103, Eq. 7 (R1, R2)
 *   O2  input assembly {T, p, F(Y)} and z-score        PAPER.md:98 (R4)
 *   O3  fully connected GELU network                   PAPER.md:103 (R5, R6)
 *   O3' per-species ensemble (n_nets = Ns): o_k = MLP_k(z), one D-...-1 net per species     PAPER.md:103 (R24)
 *   O4  de-normalise the output, scale by dt           PAPER.md:98 (R3)
 *   O5  inverse Box-Cox                                inverse of Eq. 7 (R7)
 *   O6  renormalise so that sum_k Y_k = 1              PAPER.md:92, 108-110 Eq. 9 (R8)
 *   O7  Newton iteration for T on NASA-7 polynomials   PAPER.md:57 (R9, R10, R11)
 *   O8  reaction rates and heat release rate           PAPER.md:112-115 Eq. 10, :142 Fig. 6(b), :148 (R19, R20)
 *   O9  thermal properties of the updated state        PAPER.md:57 (R21)
 * O8 / O9 (round 2) are a separate function, oracle_derived_outputs, that reads the
 * results of O0-O7; nothing in O0-O7 changed when it was added.
 *
 * Everything is scalar double precision; sums run in index order; the only
 * parallelism is an OpenMP "parallel for" over cells (cells are independent).
 * No blocking, fusion or reordering: each function can be checked against the
 * cited passage by eye.
 *
 * Pins (tests/test_oracle_*.py): Eq. 7 end points f(0) = -1/lambda, f(1) = 0
 * (PAPER.md:103), lambda -> 0 limit, round trip; GELU textbook constants and an
 * independent numpy/scipy evaluation; hand-expanded tiny nets; closed-form and
 * brentq Newton roots; sum(Y) = 1; zero-net fixed point; permutation invariance;
 * o_raw from an independently built z (feature order, division by sigma); mu_out != 0;
 * T == 600.0f boundary; vanishing-sum fallback; cp <= 0 stop; clamped Newton start.
 * O8 / O9: density against the ideal-gas law in molar units and a textbook value; sum_k RR_k = rho (1 - sum Y)/dt;
 * HRR dt / rho = integral of cp(T; Y_old) from T_old to T_new (scipy quad); cp = dh/dT by finite differences;
 * rho_new R_mix T_new = p; psi p = rho_new; R_mix = Ru / W for a pure species.
 * Parity unpinned: R3 (what the de-normalised output means) and R5 (erf vs tanh
 * GELU) are choices the paper does not settle; they are fixed by DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* universal gas constant, J/(kmol K) (CODATA 2018, exact since the 2019 SI) */
#define ORACLE_RU 8314.46261815324

/* ---------------------------------------------------------------- O1 / O5 */

/* Eq. 7 as read in R1: f(x) = (x^lambda - 1)/lambda, log(x) when lambda = 0.
 * "[0,1] is mapped to [-1/lambda, 0]" fixes the form. */
double oracle_boxcox(double x, double lambda)
{
    if (lambda != 0.0)
        return (pow(x, lambda) - 1.0) / lambda;
    return log(x);
}

/* inverse of Eq. 7 with the clamp of R7: x = max(1 + lambda*y, 0)^(1/lambda); exp(y) when lambda = 0 */
double oracle_boxcox_inv(double y, double lambda)
{
    if (lambda != 0.0) {
        double q = 1.0 + lambda * y;
        if (q < 0.0) q = 0.0;
        return pow(q, 1.0 / lambda);
    }
    return exp(y);
}

/* ---------------------------------------------------------------- O3 */

/* exact GELU (R5): v * Phi(v) = 0.5 v (1 + erf(v / sqrt 2)) */
double oracle_gelu(double v)
{
    return 0.5 * v * (1.0 + erf(v / sqrt(2.0)));
}

static int max_width(int n_layers, const int *sizes)
{
    int m = 0;
    for (int l = 0; l <= n_layers; ++l)
        if (sizes[l] > m) m = sizes[l];
    return m;
}

static size_t weight_offset(int layer, const int *sizes)
{
    size_t off = 0;
    for (int l = 0; l < layer; ++l)
        off += (size_t)sizes[l] * (size_t)sizes[l + 1];
    return off;
}

static size_t bias_offset(int layer, const int *sizes)
{
    size_t off = 0;
    for (int l = 0; l < layer; ++l)
        off += (size_t)sizes[l + 1];
    return off;
}

/* a_0 = z; a_l = GELU(W_l a_{l-1} + b_l) for l = 1..L-1; o = W_L a_{L-1} + b_L.
 * W_l is row-major [sizes[l]][sizes[l-1]] ("out" by "in"), all layers concatenated in `weights`
 * (FP32 values, promoted); `biases` likewise.  `scratch` holds 2*max_width doubles. */
static void mlp_forward(int n_layers, const int *sizes, const float *weights, const float *biases,
                        const double *z, double *o, double *scratch)
{
    int mw = max_width(n_layers, sizes);
    double *a = scratch, *next = scratch + mw;
    for (int i = 0; i < sizes[0]; ++i) a[i] = z[i];
    for (int l = 1; l <= n_layers; ++l) {
        int n_in = sizes[l - 1], n_out = sizes[l];
        const float *W = weights + weight_offset(l - 1, sizes);
        const float *b = biases + bias_offset(l - 1, sizes);
        for (int r = 0; r < n_out; ++r) {
            double s = (double)b[r];
            for (int c = 0; c < n_in; ++c)
                s += (double)W[(size_t)r * n_in + c] * a[c];
            next[r] = (l < n_layers) ? oracle_gelu(s) : s;
        }
        double *t = a; a = next; next = t;
    }
    for (int r = 0; r < sizes[n_layers]; ++r) o[r] = a[r];
}

/* one input vector through the net; for the brute-force pins on tiny nets */
int oracle_mlp_forward(int n_layers, const int *sizes, const float *weights, const float *biases,
                       const double *z, double *o)
{
    double *scratch = (double *)malloc(sizeof(double) * 2 * (size_t)max_width(n_layers, sizes));
    if (!scratch) return 1;
    mlp_forward(n_layers, sizes, weights, biases, z, o, scratch);
    free(scratch);
    return 0;
}

/* ---------------------------------------------------------------- O7 */

/* NASA-7 polynomials (R9).  a[0..6] = a1..a7 of one temperature range; W in kg/kmol.
 *   cp_k = (Ru/W_k)(a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4)                    J/(kg K)
 *   h_k  = (Ru/W_k)(a1 T + a2 T^2/2 + a3 T^3/3 + a4 T^4/4 + a5 T^5/5 + a6)   J/kg      */
double oracle_species_cp(const double *a, double W, double T)
{
    return (ORACLE_RU / W) * (a[0] + a[1] * T + a[2] * T * T + a[3] * T * T * T + a[4] * T * T * T * T);
}

double oracle_species_h(const double *a, double W, double T)
{
    return (ORACLE_RU / W) * (a[0] * T + a[1] * T * T / 2.0 + a[2] * T * T * T / 3.0
                              + a[3] * T * T * T * T / 4.0 + a[4] * T * T * T * T * T / 5.0 + a[5]);
}

/* low set if T < T_mid,k else high set; nasa_hi == NULL or T_mid == NULL means one range */
static const double *select_range(int k, double T, const double *nasa_lo, const double *nasa_hi, const double *T_mid)
{
    if (nasa_hi == NULL || T_mid == NULL) return nasa_lo + 7 * k;
    return (T < T_mid[k]) ? nasa_lo + 7 * k : nasa_hi + 7 * k;
}

/* mixture enthalpy h(T, Y) = sum_k Y_k h_k(T)  (R11: total mass-specific enthalpy, J/kg) */
double oracle_mixture_h(int Ns, const double *Y, double T, const double *nasa_lo, const double *nasa_hi,
                        const double *T_mid, const double *W)
{
    double s = 0.0;
    for (int k = 0; k < Ns; ++k)
        s += Y[k] * oracle_species_h(select_range(k, T, nasa_lo, nasa_hi, T_mid), W[k], T);
    return s;
}

double oracle_mixture_cp(int Ns, const double *Y, double T, const double *nasa_lo, const double *nasa_hi,
                         const double *T_mid, const double *W)
{
    double s = 0.0;
    for (int k = 0; k < Ns; ++k)
        s += Y[k] * oracle_species_cp(select_range(k, T, nasa_lo, nasa_hi, T_mid), W[k], T);
    return s;
}

static double clampd(double x, double lo, double hi)
{
    if (x < lo) return lo;
    if (x > hi) return hi;
    return x;
}

/* Newton's method for sum_k Y_k h_k(T) = h (R10): start at clamp(T_start), stop when
 * |dT| < tol or after max_iter updates, clamp to [T_min, T_max] after every update, no line search.
 * Returns the last iterate; *iters = number of updates taken; *converged = 1 iff |dT| < tol was met. */
double oracle_newton_T(int Ns, const double *Y, double h, double T_start, const double *nasa_lo,
                       const double *nasa_hi, const double *T_mid, const double *W, double T_min, double T_max,
                       double tol, int max_iter, int *iters, int *converged)
{
    double T = clampd(T_start, T_min, T_max);
    int it = 0, conv = 0;
    while (it < max_iter) {
        double f = oracle_mixture_h(Ns, Y, T, nasa_lo, nasa_hi, T_mid, W) - h;
        double c = oracle_mixture_cp(Ns, Y, T, nasa_lo, nasa_hi, T_mid, W);
        if (!(c > 0.0)) break;
        double dT = -f / c;
        T = clampd(T + dT, T_min, T_max);
        ++it;
        if (fabs(dT) < tol) { conv = 1; break; }
    }
    if (iters) *iters = it;
    if (converged) *converged = conv;
    return T;
}

/* ---------------------------------------------------------------- input-recipe helpers (G4, G5) */

/* G5: h_i = sum_k Y_k,i h_k(T_i) in FP64 from the FP32 state; Y is [Ns][n] species-major */
int oracle_enthalpy_field(int64_t n, int Ns, const float *T, const float *Y, const double *nasa_lo,
                          const double *nasa_hi, const double *T_mid, const double *W, double *h_out)
{
    int fail = 0;
#pragma omp parallel
    {
        double *Yc = (double *)malloc(sizeof(double) * (size_t)Ns);
        if (!Yc) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(static)
            for (int64_t i = 0; i < n; ++i) {
                for (int k = 0; k < Ns; ++k) Yc[k] = (double)Y[(size_t)k * (size_t)n + (size_t)i];
                h_out[i] = oracle_mixture_h(Ns, Yc, (double)T[i], nasa_lo, nasa_hi, T_mid, W);
            }
            free(Yc);
        }
    }
    return fail;
}

/* G4: mean and population standard deviation (ddof = 0) of x = [T, p, F(Y_1)..F(Y_Ns)] over the batch,
 * two passes in FP64, index order.  mean/std have 2+Ns entries. */
int oracle_input_moments(int64_t n, int Ns, const float *T, const float *p, const float *Y, double lambda,
                         double *mean, double *std)
{
    int D = 2 + Ns;
    if (n <= 0) return 1;
    for (int j = 0; j < D; ++j) {
        double s = 0.0;
        for (int64_t i = 0; i < n; ++i) {
            double x;
            if (j == 0) x = (double)T[i];
            else if (j == 1) x = (double)p[i];
            else {
                double yc = (double)Y[(size_t)(j - 2) * (size_t)n + (size_t)i];
                if (yc < 0.0) yc = 0.0;
                x = oracle_boxcox(yc, lambda);
            }
            s += x;
        }
        double m = s / (double)n;
        double v = 0.0;
        for (int64_t i = 0; i < n; ++i) {
            double x;
            if (j == 0) x = (double)T[i];
            else if (j == 1) x = (double)p[i];
            else {
                double yc = (double)Y[(size_t)(j - 2) * (size_t)n + (size_t)i];
                if (yc < 0.0) yc = 0.0;
                x = oracle_boxcox(yc, lambda);
            }
            v += (x - m) * (x - m);
        }
        mean[j] = m;
        std[j] = sqrt(v / (double)n);
    }
    return 0;
}

/* ---------------------------------------------------------------- the whole step */

typedef struct {
    int n_species;       /* Ns */
    int n_layers;        /* L: number of weight matrices */
    const int *sizes;    /* [L+1]: 2+Ns, hidden..., Ns */
    const float *weights;/* concatenated row-major [out][in] per layer */
    const float *biases; /* concatenated */
    const float *in_mean, *in_std;   /* [2+Ns] */
    const float *out_mean, *out_std; /* [Ns], 1/s (R3) */
    double lambda;
    const double *nasa_lo, *nasa_hi, *T_mid, *W; /* [Ns][7], [Ns][7] or NULL, [Ns] or NULL, [Ns] */
    double T_min, T_max, newton_tol;
    int newton_max_iter;
    double T_active;     /* <= 0: every cell active */
    int n_nets;          /* 0 or 1: ONE net with Ns outputs (R6).  Ns: the paper's literal architecture ("Training
                            and prediction are individually performed for each species' mass fraction ... each MLP"; R24):
                            Ns nets of identical shape with sizes[L] = 1; `weights` / `biases` hold net 0, net 1, ... one
                            after the other, each laid out as for a single net; o_k is the output of net k */
} oracle_model;

/* O0..O7 for cell i.  Scratch: Ns*4 + D + 2*max_width doubles. */
static void chem_cell(const oracle_model *m, int64_t n, int64_t i, const float *T, const float *p, const float *Y,
                      const float *h, double dt, double *T_new, double *Y_new, double *o_raw, int32_t *iters,
                      int32_t *flags, double *scratch)
{
    int Ns = m->n_species, D = 2 + Ns;
    double *y = scratch, *Yc = y + Ns, *Ys = Yc + Ns, *o = Ys + Ns, *z = o + Ns, *mlp_scratch = z + D;
    int flag = 0;

    /* O0 (R12): compare the FP32 input temperature with the FP32 threshold; skipped cells pass through */
    if (m->T_active > 0.0 && T[i] < (float)m->T_active) {
        T_new[i] = (double)T[i];
        for (int k = 0; k < Ns; ++k) {
            Y_new[(size_t)k * (size_t)n + (size_t)i] = (double)Y[(size_t)k * (size_t)n + (size_t)i];
            if (o_raw) o_raw[(size_t)k * (size_t)n + (size_t)i] = 0.0;
        }
        if (iters) iters[i] = 0;
        if (flags) flags[i] = 4; /* skipped */
        return;
    }

    /* O1: clamp at 0 (R2) then Eq. 7 */
    for (int k = 0; k < Ns; ++k) {
        double v = (double)Y[(size_t)k * (size_t)n + (size_t)i];
        Yc[k] = (v > 0.0) ? v : 0.0;
        y[k] = oracle_boxcox(Yc[k], m->lambda);
    }
    /* O2: x = [T, p, y_1..y_Ns]; z_j = (x_j - mu_j)/sigma_j */
    z[0] = ((double)T[i] - (double)m->in_mean[0]) / (double)m->in_std[0];
    z[1] = ((double)p[i] - (double)m->in_mean[1]) / (double)m->in_std[1];
    for (int k = 0; k < Ns; ++k)
        z[2 + k] = (y[k] - (double)m->in_mean[2 + k]) / (double)m->in_std[2 + k];
    /* O3 (one net) / O3' (one net per species: the same z feeds every net; net k yields o_k) */
    if (m->n_nets <= 1) {
        mlp_forward(m->n_layers, m->sizes, m->weights, m->biases, z, o, mlp_scratch);
    } else {
        const size_t w_per_net = weight_offset(m->n_layers, m->sizes), b_per_net = bias_offset(m->n_layers, m->sizes);
        for (int k = 0; k < Ns; ++k)
            mlp_forward(m->n_layers, m->sizes, m->weights + (size_t)k * w_per_net, m->biases + (size_t)k * b_per_net, z,
                        &o[k], mlp_scratch);
    }
    /* O4, O5 */
    double S = 0.0;
    for (int k = 0; k < Ns; ++k) {
        double dy = dt * (o[k] * (double)m->out_std[k] + (double)m->out_mean[k]);
        Ys[k] = oracle_boxcox_inv(y[k] + dy, m->lambda);
        S += Ys[k];
    }
    /* O6 */
    if (S > 0.0) {
        for (int k = 0; k < Ns; ++k) Ys[k] = Ys[k] / S;
    } else {
        double Sc = 0.0;
        for (int k = 0; k < Ns; ++k) Sc += Yc[k];
        for (int k = 0; k < Ns; ++k) Ys[k] = Yc[k] / Sc;
        flag |= 2; /* degenerate sum */
    }
    /* O7 */
    int it = 0, conv = 0;
    double Tn = oracle_newton_T(Ns, Ys, (double)h[i], (double)T[i], m->nasa_lo, m->nasa_hi, m->T_mid, m->W,
                                m->T_min, m->T_max, m->newton_tol, m->newton_max_iter, &it, &conv);
    if (!conv) flag |= 1;

    T_new[i] = Tn;
    for (int k = 0; k < Ns; ++k) {
        Y_new[(size_t)k * (size_t)n + (size_t)i] = Ys[k];
        if (o_raw) o_raw[(size_t)k * (size_t)n + (size_t)i] = o[k];
    }
    if (iters) iters[i] = it;
    if (flags) flags[i] = flag;
}

/* State arrays are the FP32 arrays the GPU library receives: T[n], p[n], h[n], Y[Ns][n] (species-major).
 * Outputs are FP64: T_new[n], Y_new[Ns][n], o_raw[Ns][n] (normalised net output before O4; may be NULL),
 * iters[n] (Newton updates; may be NULL), flags[n] (bit0 not converged, bit1 degenerate sum, 4 = skipped;
 * may be NULL).  Returns 0, or 1 on allocation failure / bad arguments. */
int oracle_chem_step(const oracle_model *m, int64_t n, const float *T, const float *p, const float *Y,
                     const float *h, double dt, double *T_new, double *Y_new, double *o_raw, int32_t *iters,
                     int32_t *flags)
{
    if (!m || n < 0 || m->n_layers < 1 || m->sizes[0] != 2 + m->n_species) return 1;
    if (m->n_nets <= 1 && m->sizes[m->n_layers] != m->n_species) return 1;
    if (m->n_nets > 1 && (m->n_nets != m->n_species || m->sizes[m->n_layers] != 1)) return 1;
    int Ns = m->n_species, D = 2 + Ns;
    size_t scratch_len = (size_t)Ns * 4 + (size_t)D + 2 * (size_t)max_width(m->n_layers, m->sizes);
    int fail = 0;
#pragma omp parallel
    {
        double *scratch = (double *)malloc(sizeof(double) * scratch_len);
        if (!scratch) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 16)
            for (int64_t i = 0; i < n; ++i)
                chem_cell(m, n, i, T, p, Y, h, dt, T_new, Y_new, o_raw, iters, flags, scratch);
            free(scratch);
        }
    }
    return fail;
}

/* ---------------------------------------------------------------- O8, O9: derived outputs of a step
 *
 * O8 (R19, R20).  The quantities the solver's combustion model consumes from the chemistry step (PaSR source terms,
 * PAPER.md:148) and the one the paper compares in Fig. 6(b) and trains against in Eq. 10:
 *     rho_i  = p_i / (Ru T_i sum_k Yc_k / W_k)            ideal gas at the INPUT state, Yc = max(Y, 0)      [kg/m3]
 *     RR_k,i = rho_i (Y_new,k,i - Y_k,i) / dt             mass production rate of species k               [kg/(m3 s)]
 *     HRR_i  = - sum_k h_k(T_new,i) RR_k,i                heat release rate, NASA-7 total species enthalpy  [W/m3]
 * O9 (R21).  Thermal properties of the updated state (the transport half needs fits the paper does not give):
 *     cp_i    = sum_k Y_new,k cp_k(T_new)                                                                 [J/(kg K)]
 *     Rmix_i  = Ru sum_k Y_new,k / W_k                                                                    [J/(kg K)]
 *     rho_new = p_i / (Rmix_i T_new,i),   psi_i = 1 / (Rmix_i T_new,i)    (rho = psi p)            [kg/m3], [s2/m2]
 * Skipped cells (flags == 4): RR = 0, HRR = 0; the properties are those of the unchanged state.
 * Inputs: the FP32 state the step received, and its FP64 results.  Any output pointer may be NULL. */
int oracle_derived_outputs(int64_t n, int Ns, const float *T, const float *p, const float *Y, double dt,
                           const double *T_new, const double *Y_new, const int32_t *flags, const double *nasa_lo,
                           const double *nasa_hi, const double *T_mid, const double *W, double *rr, double *hrr,
                           double *cp, double *rmix, double *rho_new, double *psi)
{
    if (n < 0 || Ns < 1 || !T || !p || !Y || !T_new || !Y_new || !nasa_lo || !W || !(dt > 0.0)) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const int skipped = flags && flags[i] == 4;
        /* O8 */
        double inv_w_in = 0.0;
        for (int k = 0; k < Ns; ++k) {
            double yc = (double)Y[(size_t)k * (size_t)n + (size_t)i];
            if (yc < 0.0) yc = 0.0;
            inv_w_in += yc / W[k];
        }
        const double rho_in = (double)p[i] / (ORACLE_RU * (double)T[i] * inv_w_in);
        double q = 0.0;
        for (int k = 0; k < Ns; ++k) {
            const size_t ki = (size_t)k * (size_t)n + (size_t)i;
            const double r = skipped ? 0.0 : rho_in * (Y_new[ki] - (double)Y[ki]) / dt;
            if (rr) rr[ki] = r;
            q -= oracle_species_h(select_range(k, T_new[i], nasa_lo, nasa_hi, T_mid), W[k], T_new[i]) * r;
        }
        if (hrr) hrr[i] = q;
        /* O9 */
        double c = 0.0, inv_w = 0.0;
        for (int k = 0; k < Ns; ++k) {
            const double y = Y_new[(size_t)k * (size_t)n + (size_t)i];
            c += y * oracle_species_cp(select_range(k, T_new[i], nasa_lo, nasa_hi, T_mid), W[k], T_new[i]);
            inv_w += y / W[k];
        }
        const double R = ORACLE_RU * inv_w;
        if (cp) cp[i] = c;
        if (rmix) rmix[i] = R;
        if (rho_new) rho_new[i] = (double)p[i] / (R * T_new[i]);
        if (psi) psi[i] = 1.0 / (R * T_new[i]);
    }
    return 0;
}
