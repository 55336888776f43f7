/*
 * gpuann.h -- C ABI of libgpuann.so: the per-cell ANN chemistry step of the GPU-ANN LES framework
 * (arXiv 2402.18858), written from scratch for NVIDIA B200 (sm_100a).
 *
 * PAPER.md = the paper text; R<n> = the readings listed in DESIGN.md ("Readings of the paper").
 *
 * What one gpuann_chem_step call computes for every cell i (all on the GPU, in this library's kernels):
 *   S0  active-cell test T_i >= T_active                    BASELINE.json configs[4]; R12
 *   S1  Box-Cox transform y_k = (Y_k^lambda - 1)/lambda     PAPER.md:98-103, Eq. 7; R1, R2
 *   S2  x = {T, p, y_1..y_Ns}; z_j = (x_j - mu_j)/sigma_j   PAPER.md:98; R4
 *   S3  fully connected GELU network, o = MLP(z)            PAPER.md:103 (hidden 1600-800-400, GELU),
 *                                                           PAPER.md:56 (half precision inference); R5, R6
 *   S4  dy_k = dt (o_k sigma_out,k + mu_out,k)              PAPER.md:98 ("variation in mass fractions"); R3
 *   S5  Y*_k = max(1 + lambda (y_k + dy_k), 0)^(1/lambda)   inverse of Eq. 7; R7
 *   S6  Y_new,k = Y*_k / sum_j Y*_j                         PAPER.md:92, 108-110 (Eq. 9); R8
 *   S7  Newton iteration for T_new: sum_k Y_new,k h_k(T) = h on NASA-7 polynomials
 *                                                           PAPER.md:57; R9, R10, R11
 *
 * Conventions
 *   - Every entry point returns a gpuann_status; nothing throws or aborts across the ABI.  The message
 *     of the last failure on a context is available from gpuann_last_error.
 *   - "HOST" pointers are read (copied, converted, packed) before the call returns; the caller keeps
 *     ownership and may free them at once.  "DEVICE" pointers are CUDA device memory owned by the
 *     caller; the library never frees or reallocates them.
 *   - The state is structure-of-arrays, FP32: T[n], p[n], h[n], Y[Ns][n] (species-major: the row of
 *     species k starts at Y + k*n_cells) -- one contiguous field per quantity, the layout a finite-volume
 *     solver holds.
 *   - gpuann_chem_step and gpuann_debug_forward only enqueue work on `stream` (a cudaStream_t passed
 *     as void*; NULL = the legacy default stream).  They never synchronise; calls on one stream are
 *     ordered.  A context must not be used from two streams or two host threads at the same time
 *     (its activation scratch is shared).
 *   - Device scratch: one activation buffer of chunk x H2 BF16 (h2, the only activation that crosses HBM; two buffers of
 *     chunk x max width on the fallback path), allocated by gpuann_load_net for chunk = gpuann_params.chunk_cells cells
 *     (default 148 x 128 x 56 = 1,060,864: 1.7 GB for the 23-1600-800-400-21 net; larger fields are processed chunk by
 *     chunk, so the scratch does not grow with n_cells).  Plus, when T_active > 0, an int32 index list of n_cells
 *     entries (grown lazily).
 *   - There is no CPU fallback: without a CUDA device of compute capability 10.x gpuann_create fails
 *     with GPUANN_ERR_UNSUPPORTED.
 */
#ifndef GPUANN_H
#define GPUANN_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gpuann_ctx gpuann_ctx; /* opaque; created by gpuann_create, freed by gpuann_destroy */

typedef enum {
    GPUANN_OK = 0,
    GPUANN_ERR_INVALID_ARG = 1, /* NULL pointer, negative size, inconsistent shapes, sigma <= 0, dt <= 0 */
    GPUANN_ERR_NOT_READY = 2,   /* chem_step before both load_net and load_thermo */
    GPUANN_ERR_UNSUPPORTED = 3, /* no sm_100 device, or a shape outside the limits below */
    GPUANN_ERR_ALLOC = 4,       /* host or device allocation failed */
    GPUANN_ERR_CUDA = 5         /* a CUDA runtime/driver call failed (message has the CUDA error) */
} gpuann_status;

#define GPUANN_MAX_SPECIES 64   /* Ns <= 64 */
#define GPUANN_MAX_LAYERS 8     /* number of weight matrices <= 8 */
#define GPUANN_MAX_WIDTH 4096   /* every layer width <= 4096 */

#define GPUANN_PRECISION_FP32 0 /* CUDA-core FP32 MLP, exact-erf GELU (configs[0]) */
#define GPUANN_PRECISION_BF16 1 /* tcgen05 BF16 x BF16 -> FP32 MLP, activations rounded to BF16 (configs[1..4]) */
#define GPUANN_PRECISION_FP16 2 /* the same kernels with FP16 weights and activations, FP32 accumulate: the half precision
                                   the paper infers in.  Weights are rounded to FP16
                                   after the factor 1/2 that hidden-layer weights are stored with: an FP16-representable
                                   weight is used exactly unless |w| < 2^-13 (w/2 is then subnormal and may lose its last
                                   bit); |w/2| (first layer: |w|, |b|) must stay below 65520 or the load is INVALID_ARG.
                                   Only nets that run the fused + tail kernels (4 weight matrices, Ns <= 48,
                                   last hidden layer <= 416, first hidden layer >= 128): UNSUPPORTED otherwise */

/* Parameters of a context.  gpuann_default_params fills the defaults; passing NULL to gpuann_create
 * is the same as passing the defaults. */
typedef struct {
    int precision;        /* GPUANN_PRECISION_*; default BF16 */
    int newton_max_iter;  /* cap on Newton updates per cell; default 20 (R10) */
    double newton_tol;    /* stop when |dT| < newton_tol [K]; default 1e-6 (R10) */
    double T_min, T_max;  /* clamp applied to the start value and after every update; default 200, 3500 K */
    double T_active;      /* <= 0: every cell is active.  > 0: cells with (float)T < (float)T_active are
                             skipped and their T, Y are not written at all (R12); default 0 */
    int device;           /* CUDA device ordinal, -1 = the current device; default -1 */
    int64_t chunk_cells;  /* cells per internal pass of the BF16 path (activation scratch is sized by it);
                             <= 0 = library default */
} gpuann_params;

void gpuann_default_params(gpuann_params *params);

/* Creates a context on params->device.  *out is NULL on failure.  Errors: INVALID_ARG (out NULL, bad
 * parameter values), UNSUPPORTED (no device of compute capability 10.x), ALLOC, CUDA. */
int gpuann_create(const gpuann_params *params, gpuann_ctx **out);

/* Loads the network of S2-S4.
 *   n_species  Ns (1..GPUANN_MAX_SPECIES)
 *   n_layers   L = number of weight matrices (1..GPUANN_MAX_LAYERS)
 *   sizes      HOST int[L+1]: sizes[0] = 2 + Ns (inputs T, p, y_1..y_Ns in this order),
 *              hidden widths, sizes[L] = Ns
 *   weights    HOST, L pointers; weights[l] is row-major [sizes[l+1]][sizes[l]] ("out" by "in"), FP32.
 *              The BF16 path rounds them to BF16 (round-to-nearest-even); values that are already
 *              BF16-representable are used exactly.
 *   biases     HOST, L pointers; biases[l] is [sizes[l+1]], FP32 (kept in FP32 on both paths)
 *   in_mean, in_std    HOST float[2+Ns]: z-score statistics of {T, p, y_k} (R4); in_std > 0
 *   out_mean, out_std  HOST float[Ns]: de-normalisation of the output, units 1/s (R3)
 *   lambda     Box-Cox exponent (0.1); lambda = 0 selects the log/exp branch of Eq. 7
 * GELU is applied after every layer but the last.  May be called again to replace the net: a load that
 * fails with INVALID_ARG or UNSUPPORTED leaves the net loaded earlier in place and usable; one that fails with ALLOC or
 * CUDA leaves the context without a net (NOT_READY until a load succeeds).  The same holds for gpuann_load_net_ensemble.
 * Errors: INVALID_ARG (NULLs, sizes[0] != 2+Ns, sizes[L] != Ns, width < 1, in_std <= 0 or not finite,
 * lambda < 0, n_species differs from a loaded thermo table, a weight or bias that is not finite or -- on the tensor
 * path -- overflows BF16 / FP16 once stored), UNSUPPORTED (limits above), ALLOC, CUDA. */
int gpuann_load_net(gpuann_ctx *ctx, int n_species, int n_layers, const int *sizes,
                    const float *const *weights, const float *const *biases,
                    const float *in_mean, const float *in_std,
                    const float *out_mean, const float *out_std, double lambda);

/* The paper's literal architecture ("Training and prediction are individually performed for each species'
 * mass fraction ... The architecture of each MLP"; R24): Ns nets of ONE shape with a
 * single output each, all fed by the same z; net k yields o_k, everything after S3 is unchanged.
 *   sizes    HOST int[L+1]: sizes[0] = 2 + Ns, hidden widths, sizes[L] = 1
 *   weights  HOST, Ns*L pointers: layer l of net k at weights[k*L + l], row-major [sizes[l+1]][sizes[l]]; biases likewise
 * Tensor path only (BF16 or FP16 context) and only shapes the fused + tail kernels run (L = 4, first hidden layer >= 128,
 * last hidden layer <= 416): UNSUPPORTED otherwise.  One step is Ns x (fused kernel + tail kernel) + one update kernel.
 * Replaces a net loaded earlier. */
int gpuann_load_net_ensemble(gpuann_ctx *ctx, int n_species, int n_layers, const int *sizes,
                             const float *const *weights, const float *const *biases,
                             const float *in_mean, const float *in_std,
                             const float *out_mean, const float *out_std, double lambda);

/* Loads the thermodynamic table of S7 ("high-order temperature polynomials"; R9).
 *   nasa_lo  HOST double[Ns][7]: a1..a7 of the low-temperature range
 *   nasa_hi  HOST double[Ns][7] or NULL (= one range: nasa_lo is used at every T)
 *   T_mid    HOST double[Ns] or NULL (= one range); species k uses nasa_lo if T < T_mid[k] else nasa_hi
 *   W        HOST double[Ns]: molar masses in kg/kmol (= g/mol), > 0
 *   cp_k = (Ru/W_k)(a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4), h_k = (Ru/W_k)(a1 T + a2 T^2/2 + a3 T^3/3
 *   + a4 T^4/4 + a5 T^5/5 + a6), Ru = 8314.46261815324 J/(kmol K); a7 is not used.
 * Errors: INVALID_ARG (NULLs, W <= 0, n_species differs from a loaded net), UNSUPPORTED, ALLOC, CUDA. */
int gpuann_load_thermo(gpuann_ctx *ctx, int n_species, const double *nasa_lo, const double *nasa_hi,
                       const double *T_mid, const double *W);

/* One chemistry step S0-S7 over n_cells cells, in place, asynchronous on `stream`.
 *   T   DEVICE float[n]      in: T(t) [K]; out: T_new (active cells only)
 *   p   DEVICE float[n]      in: pressure [Pa]; never written
 *   Y   DEVICE float[Ns][n]  in: mass fractions (values < 0 are read as 0, R2); out: Y_new, sum_k = 1
 *                            (active cells only)
 *   h   DEVICE float[n]      in: total (chemical + sensible) mass-specific enthalpy [J/kg], conserved
 *                            over the step (R11); never written
 *   dt  time step [s], > 0 (1e-6)
 * Any alignment and any n_cells are accepted (16-byte aligned pointers with n_cells % 4 == 0 take the
 * vectorised loads).  n_cells == 0 is a no-op.  Newton non-convergence and a vanishing sum of Y* are
 * counted (gpuann_get_stats), not errors; on a vanishing sum Y_new = max(Y,0)/sum.  Results do not depend
 * on n_cells, on the chunking or on the position of a cell, and two runs are bit-identical.
 * Errors: INVALID_ARG, NOT_READY, ALLOC (scratch), CUDA (launch failure). */
int gpuann_chem_step(gpuann_ctx *ctx, int64_t n_cells, float *T, const float *p, float *Y, const float *h,
                     double dt, void *stream);

/* Optional extra outputs of a step; every member is a DEVICE pointer or NULL (= not computed).
 * For an ACTIVE cell i, with T, p, Y the inputs and T_new, Y_new the results of the same step:
 *   rr    float[Ns][n]  RR_k = rho (Y_new,k - Y_k) / dt [kg/(m3 s)], the species source term a PaSR-type combustion model
 *                       consumes; rho = p / (Ru T sum_k max(Y_k,0)/W_k), the ideal-gas density of the INPUT
 *                       state (R19).  Y_k is the input as given (not clamped), so sum_k RR_k = rho (1 - sum_k Y_k) / dt
 *   hrr   float[n]      HRR = - sum_k h_k(T_new) RR_k [W/m3], the heat release rate of PAPER.md:112-115 Eq. 10 and Fig. 6(b)
 *                       (PAPER.md:142), with the NASA-7 total species enthalpies at T_new (R20)
 *   cp    float[n]      sum_k Y_new,k cp_k(T_new) [J/(kg K)]                                   (R21)
 *   rho   float[n]      density of the UPDATED state p / (R_mix T_new), R_mix = Ru sum_k Y_new,k / W_k [kg/m3]
 *   psi   float[n]      compressibility 1 / (R_mix T_new) [s2/m2] (rho = psi p)
 * Cells below T_active are not written (like T and Y).  Transport properties are not provided: the paper gives no fits
 * for them (out of scope). */
typedef struct {
    float *rr;
    float *hrr;
    float *cp;
    float *rho;
    float *psi;
} gpuann_step_outputs;

/* gpuann_chem_step plus the optional outputs above, computed in the same kernels (no extra pass over the state).
 * out == NULL or all members NULL is exactly gpuann_chem_step.  Every path provides them: the tail kernel, the FP32 kernel,
 * and the stand-alone update kernel of nets without a tail kernel and of the per-species ensemble.  Errors as
 * gpuann_chem_step. */
int gpuann_chem_step_ex(gpuann_ctx *ctx, int64_t n_cells, float *T, const float *p, float *Y, const float *h,
                        double dt, const gpuann_step_outputs *out, void *stream);

/* The same step for a caller whose state lives in HOST memory: copies T, p, Y, h to the device
 * (library-owned staging buffers, grown lazily), runs gpuann_chem_step, copies T and Y back and
 * synchronises.  Pinned host memory makes the copies asynchronous.  On the BF16 path without an active-cell
 * threshold and for n_cells >= 4 tiles per SM the field is cut into slices of whole tiles (about eight, never
 * larger than the scratch chunk) and slice i+1 is
 * copied in / slice i-1 copied out on two copy streams while slice i is computed, so the call is bound by the
 * slower of PCIe and compute instead of their sum; the result is bit for bit that of gpuann_chem_step.
 * Arguments as gpuann_chem_step but HOST pointers.  This is the end-to-end entry bench.py times ("e2e"). */
int gpuann_chem_step_host(gpuann_ctx *ctx, int64_t n_cells, float *T, const float *p, float *Y, const float *h,
                          double dt);

/* Test / bench hook: S1-S3 only.  o_raw DEVICE float[Ns][n] receives the normalised network output
 * (before S4) of every cell, skipped or not.  The BF16 tolerance of the task is stated on this quantity. */
int gpuann_debug_forward(gpuann_ctx *ctx, int64_t n_cells, const float *T, const float *p, const float *Y,
                         float *o_raw, void *stream);

/* Counters accumulated since the last gpuann_reset_stats: cells that were active, Newton solves that hit
 * newton_max_iter (or cp <= 0) before |dT| < tol, cells whose sum of Y* vanished.  Synchronises the stream
 * of the last chem_step.  Any out pointer may be NULL. */
int gpuann_get_stats(gpuann_ctx *ctx, int64_t *n_active, int64_t *n_not_converged, int64_t *n_degenerate);
int gpuann_reset_stats(gpuann_ctx *ctx);

/* Input-recipe helpers (G4, G5), so that a caller can build consistent inputs without any CPU
 * implementation of the thermodynamics:
 * gpuann_enthalpy: h_i = sum_k Y[k][i] h_k(T_i) evaluated in FP64, rounded to FP32 (needs load_thermo).
 *   T, Y DEVICE in; h_out DEVICE float[n] out.  Asynchronous on `stream`.
 * gpuann_input_moments: mean and population standard deviation (FP64 accumulation) of the features
 *   {T, p, F(Y_1)..F(Y_Ns)} over the batch, F = Eq. 7 with the given lambda.  T, p, Y DEVICE in;
 *   mean_out, std_out HOST double[2+Ns] out.  Synchronises `stream`. */
int gpuann_enthalpy(gpuann_ctx *ctx, int64_t n_cells, const float *T, const float *Y, float *h_out, void *stream);
int gpuann_input_moments(gpuann_ctx *ctx, int64_t n_cells, int n_species, const float *T, const float *p,
                         const float *Y, double lambda, double *mean_out, double *std_out, void *stream);

/* gpuann_input_moments without any device allocation.
 *
 * gpuann_input_moments takes its scratch (one FP64 partial sum per thread block and feature, plus the means) from
 * cudaMalloc and returns it with cudaFree on every call.  Some users of this library cannot afford that once their run
 * is under way:
 *   - a flow solver that claimed the GPU's memory for its own fields and pools at start-up: a later cudaMalloc, however
 *     small, may simply fail, or it fragments what the solver laid out;
 *   - a time-step loop with other work in flight on the device (halo exchange, the pressure solver on their own
 *     streams): cudaMalloc and cudaFree wait for the whole device, so each call would stall those streams;
 *   - codes run under a "no allocation after initialisation" rule (memory-budget audits, week-long production runs).
 * For them this entry point computes the same statistics with its scratch in a `static __device__` array inside the
 * library: GPUANN_STATIC_SCRATCH_BYTES bytes that every GPU which loads libgpuann.so holds until the process exits,
 * whether or not this function is ever called.  It calls no cudaMalloc, cudaFree or other allocating routine.
 *
 *   Arguments and results as gpuann_input_moments (T, p, Y DEVICE in; mean_out, std_out HOST double[2+Ns] out;
 *   synchronises `stream`).  On the same GPU both functions use the same grid and add in the same order.
 *   Limit: n_species <= GPUANN_STATIC_MAX_SPECIES; anything larger returns GPUANN_ERR_UNSUPPORTED with a message that
 *   names the limit -- it is never served by a hidden allocation.  n_cells is not limited by the scratch.
 *   First call on a device: looks up the array's device address (once per device, kept for later calls), which can make
 *   the CUDA runtime load the library's device code on that GPU.  Make that first call during set-up, before any stream
 *   capture begins.
 *   Sharing: there is ONE array per GPU for all contexts, streams and threads, and it keeps what the last call wrote.
 *   A call overwrites every word before reading it, so nothing has to be cleared in between; but two calls that overlap
 *   on the same GPU (two streams, two host threads, two contexts) race on it and return garbage.  Serialise them.
 *   The timing hook (gpuann_timing_enable) counts this function's four launches but does not time them.
 * Errors: INVALID_ARG (NULLs, n_cells <= 0, n_species < 1, lambda < 0), UNSUPPORTED (limit above), CUDA. */
#define GPUANN_STATIC_MAX_SPECIES 64
#define GPUANN_STATIC_SCRATCH_BYTES 271392 /* (512 blocks x 66 features + 66 means + 66 deviations) x 8 bytes */
int gpuann_input_moments_static(gpuann_ctx *ctx, int64_t n_cells, int n_species, const float *T, const float *p,
                                const float *Y, double lambda, double *mean_out, double *std_out, void *stream);

/* Number of kernel launches this context has enqueued so far (bench.py reports it as gpu_launches). */
int64_t gpuann_launch_count(const gpuann_ctx *ctx);

/* Per-kernel device timing, for the roofline arithmetic of bench.py.  While enabled, every kernel launch of
 * this context is bracketed by two CUDA events on the launching stream (a small host cost per launch, so the
 * headline throughput is measured with timing off).  gpuann_timing_read synchronises the last stream, writes
 * for each kernel class i < n_classes the summed device time ms[i] and the number of launches counts[i]
 * recorded since the last enable/read, and clears the record.  Classes: gpuann_timing_num_classes() of them,
 * named by gpuann_timing_class_name ("layer1_gemm", "post_update_newton", ...; "" if out of range). */
int gpuann_timing_enable(gpuann_ctx *ctx, int enable);
int gpuann_timing_read(gpuann_ctx *ctx, int n_classes, double *ms, int64_t *counts);
int gpuann_timing_num_classes(void);
const char *gpuann_timing_class_name(int cls);

/* Static description of the work one chem_step does, for roofline arithmetic: MACs the tensor path
 * issues per cell including K/N padding (0 on the FP32 path), and the name of the kernel variant chosen
 * for the loaded net: "fp32"; "bf16-fused+tail" (the two-kernel tensor path), "bf16-fused", "bf16-layerwise+tail",
 * "bf16-layerwise" (fallbacks for shapes one or both kernels do not take); "fp16-fused+tail"; "bf16-ensemble" /
 * "fp16-ensemble".  Any out pointer may be NULL. */
int gpuann_describe(const gpuann_ctx *ctx, int64_t *issued_mac_per_cell, const char **variant);

/* Message of the last failure on this context ("" if none).  ctx == NULL returns the message of the last
 * failed gpuann_create on this thread.  The pointer stays valid until the next call on the context. */
const char *gpuann_last_error(const gpuann_ctx *ctx);

/* Frees the context and everything it owns.  NULL is allowed.  Synchronises the device. */
int gpuann_destroy(gpuann_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* GPUANN_H */
