/* df_thermo.h -- C ABI of libdfthermo.so: the per-cell thermochemistry update of
 * arXiv 2312.05800 as hand-written sm_100a CUDA.
 *
 * Citations: "P:n" = /root/reference/PAPER.md line n; "NS" = BASELINE.json north_star;
 * "A#" = the reading of that number in DESIGN.md (where the paper is silent or garbled).
 *
 *   P:34-36  "the entire computational process is executed on GPU, including machine learning
 *            chemistry ... and computation of thermal and transport properties"
 *   P:79     ANN input x = {T, p, F(Y)} (Box-Cox F on mass fractions), output = change of
 *            mass fractions over the step, Z-score normalisation, hidden layers 1600/800/400, GELU
 *   P:62     time step of 1 us; mass fractions must sum to unity (also P:86)
 *   P:44     "Hirschfelder and Curtiss mixture-averaged" transport
 *   NS       names the rules the paper does not print: Newton on NASA-7, Wilke viscosity,
 *            combination-rule conductivity, mixture-averaged diffusivities from binary fits.
 *
 * Conventions
 *   - Symbols: n = n_cells, K = species count, R = 8314.46261815324 J/(kmol K), W kg/kmol,
 *     T K, p Pa, h J/kg, cp J/(kg K), mu Pa s, lambda W/(m K), D m^2/s, omega kg/(m^3 s).
 *   - Field arrays are DEVICE fp32, structure-of-arrays: Y[k*ld + i], species pitch ld >= n,
 *     ld % 4 == 0 and every base pointer 16-byte aligned (float4 access).
 *   - Tables passed to *_create are HOST memory; they are copied and repacked, the caller may
 *     free them on return.  Handles are immutable afterwards: hot calls on different streams
 *     may share them.
 *   - Hot calls validate, enqueue on `stream` (a cudaStream_t passed as void*) and return; they
 *     never synchronise, allocate or touch host memory.  n_cells == 0 is DF_OK and a no-op.
 *   - Unless stated, inputs and outputs must not alias.
 *   - Every function returns DF_OK or an error code; df_last_error() gives the thread-local
 *     message of the last non-OK return.  No exception crosses this boundary.
 *   - There is no CPU fallback: without a CUDA device the create calls return DF_ERR_CUDA.
 */
#ifndef DF_THERMO_H
#define DF_THERMO_H

#if defined(__GNUC__)
#define DF_API __attribute__((visibility("default")))
#else
#define DF_API
#endif

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct df_mech df_mech; /* species tables, opaque */
typedef struct df_ann df_ann;   /* MLP + normalisation tables, opaque */
typedef struct df_ann_mmlp df_ann_mmlp; /* one MLP per species, opaque */
typedef struct df_step_plan df_step_plan; /* one time step captured as a CUDA graph, opaque */
typedef struct df_host_ctx df_host_ctx; /* device staging buffers for df_step_host, opaque */

typedef enum {
    DF_OK = 0,
    DF_ERR_INVALID_ARG = 1, /* NULL, negative size, ld < n, misalignment, K mismatch */
    DF_ERR_UNSUPPORTED = 2, /* shape the kernels are not instantiated for */
    DF_ERR_ALLOC = 3,       /* host or device allocation failed */
    DF_ERR_CUDA = 4         /* a CUDA runtime call or launch failed */
} df_status;

/* ABI version of this header (bumped on any signature change). */
DF_API int df_abi_version(void);
DF_API const char* df_last_error(void);

/* ---- species tables (NS (1),(2); A1, A2, A5) ---------------------------------------------
 * NASA-7, two ranges with one common break T_mid (`hi` applies for T >= T_mid, A2):
 *   cp_k/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
 *   h_k/(R T) = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T        (molar)
 * Pure-species transport fits, L = ln T (A5):
 *   sqrt(mu_k) = T^(1/4) sum_{m<5} visc_fit[k][m] L^m
 *   lambda_k   = T^(1/2) sum_{m<5} cond_fit[k][m] L^m
 *   p D_jk     = T^(3/2) sum_{m<5} bdiff_fit[j][k][m] L^m   (symmetric; diagonal = self-diffusion)
 * Supported: 1 <= K <= 64.  T_low/T_high are informative (evaluation extrapolates, A3). */
DF_API df_status df_mech_create(df_mech** out, int K,
                         const double* W,        /* [K] */
                         const double* nasa_lo,  /* [K][7] */
                         const double* nasa_hi,  /* [K][7] */
                         double T_low, double T_mid, double T_high,
                         const double* visc_fit,  /* [K][5] */
                         const double* cond_fit,  /* [K][5] */
                         const double* bdiff_fit  /* [K][K][5] */);
DF_API df_status df_mech_destroy(df_mech* mech);
DF_API int df_mech_num_species(const df_mech* mech);

/* ---- ANN tables (A8-A11, A13, A14, A16, A19) ------------------------------------------
 * n_layers linear layers, dims[0] = K+2 inputs (T, p, F(Y_0..K-1)), dims[n_layers] = K outputs,
 * GELU after every layer but the last.  W[l] is [dims[l+1]][dims[l]] row-major (y = x W^T + b).
 * precision 0: fp32 FFMA path (any n_layers >= 1, every dims[l] <= 256).
 * precision 1: 16-bit tensor-core path (tcgen05, fp32 accumulate in TMEM).  Weights MUST be bf16-valued (BASELINE's
 *              "bf16 weights": low 16 bits of the fp32 pattern zero, else DF_ERR_INVALID_ARG) and, like the biases,
 *              finite with magnitude <= 65504 (else DF_ERR_UNSUPPORTED): tcgen05 kind::f16 needs both operands in one
 *              format, so the weights are held in fp16 (exact for bf16 values >= 2^-14, within 2^-25 below) and the
 *              activations are rounded to fp16 (A21).  A hidden activation is held as 2 GELU(v) with the factor 1/2 in the
 *              next layer's stored weights (a power of two: same results), so it saturates at |GELU(v)| = 32752.
 *              n_layers == 4, dims[1] % 64 == 0, dims[2] % 32 == 0 with 64 <= dims[2] <= 800,
 *              dims[3] % 16 == 0 with 32 <= dims[3] <= 400, K <= 28.
 * x_mean/x_std [K+2] and u_mean/u_std [K] are the Z-score statistics; the network output
 * o is the z-scored change in Box-Cox space (A9): Delta_k = u_std[k] o_k + u_mean[k].
 * F(y) = (y^lambda - 1)/lambda with lambda = boxcox_lambda > 0 (A10); dt in seconds. */
DF_API df_status df_ann_create(df_ann** out, int n_layers, const int* dims,
                        const float* const* W, const float* const* b, int precision,
                        const double* x_mean, const double* x_std,
                        const double* u_mean, const double* u_std,
                        double boxcox_lambda, double dt);
DF_API df_status df_ann_destroy(df_ann* ann);
/* Device scratch df_chem_ann_source needs for n_cells cells on the CURRENT device (0 on the fp32 path).  The
 * tensor path parks one 128-cell tile of layer-2 activations (fp16) per resident CTA (one per SM), so the value
 * does not grow with n_cells beyond 128 x SM-count cells. */
DF_API size_t df_ann_workspace_bytes(const df_ann* ann, long long n_cells);

/* ---- hot call 1: temperature from enthalpy (NS (1); A3, A4) ------------------------------
 * Solves sum_k Y_k h_k(T)/W_k = h[i] for T by Newton, T <- T - (h(T,Y) - h)/cp(T,Y).
 * T is in/out: on entry the guess (<= 0, NaN or Inf => T_mid), on exit the root.
 * cp (optional) receives cp(T_root, Y).  n_unconverged (optional, device int) is atomically
 * incremented once per cell whose last Newton correction exceeded 1e-2 K. */
DF_API df_status df_thermo_T_from_h(const df_mech* mech, long long n_cells, long long ld,
                             const float* h, const float* Y, float* T, float* cp,
                             int* n_unconverged, void* stream);

/* ---- hot call 2: mixture properties (NS (2); A5-A7) -----------------------------------
 * cp, h = sum Y_k {cp_k, h_k}(T)/W_k; mu by Wilke; lambda = 1/2 (sum X_k lambda_k +
 * 1/sum(X_k/lambda_k)); D[k] = sum_{j!=k} Y_j / sum_{j!=k} X_j/D_jk (self-diffusion D_kk when
 * the denominator is 0).  Any output pointer may be NULL (skipped).  D is [K][ld].
 * Wilke's table B_kj = [8 (1 + W_k/W_j)]^(-1/2) is held as a truncated singular-value factorisation when 7-12 terms
 * reproduce every element to 1e-6 (decided in df_mech_create from the weights; the full table otherwise): the result
 * agrees with the double sum to ~1e-6, inside the 1e-5 the path is held to. */
DF_API df_status df_thermo_properties(const df_mech* mech, long long n_cells, long long ld,
                               const float* T, const float* p, const float* Y,
                               float* cp, float* h, float* mu, float* lambda, float* D,
                               void* stream);

/* ---- hot call 3: ANN chemistry source (NS (3); A8-A12, A17) -----------------
 * features -> MLP -> Delta_k; Y*_k = max(Y_k^lambda + lambda Delta_k, 0)^(1/lambda);
 * Y'_k = Y*_k / sum_j Y*_j; dY_k = Y'_k - Y_k; rho = p Wbar/(R T); omega_k = rho dY_k / dt.
 * omega and dY are [K][ld]; either may be NULL.  workspace: device memory of at least
 * df_ann_workspace_bytes(ann, n_cells) bytes, 1024-byte aligned (may be NULL when that is 0). */
DF_API df_status df_chem_ann_source(const df_ann* ann, const df_mech* mech, long long n_cells, long long ld,
                             const float* T, const float* p, const float* Y,
                             float* omega, float* dY,
                             void* workspace, size_t workspace_bytes, void* stream);

/* ---- hot call 3 without a workspace, for callers that may not allocate device memory --------------------------
 * Same operation, kernel and results as df_chem_ann_source for a precision-1 (tensor path) handle; the kernel's
 * per-CTA scratch is a static device array inside the library instead of a caller-supplied workspace.  The call
 * allocates nothing (no cudaMalloc/cudaFree, no allocating library routine).
 *   - Every GPU that loads the library holds DF_ANN_STATIC_SCRATCH_BYTES of device memory until the process exits.
 *   - DF_ERR_UNSUPPORTED when df_ann_workspace_bytes(ann, n_cells) exceeds that (the 21-1600-800-400-19 network
 *     needs 29.4 MiB at any n_cells on a 148-SM device: it fits), or when the handle is not precision 1 (the fp32
 *     path needs no workspace: df_chem_ann_source with workspace = NULL allocates nothing either).
 *   - All calls on a device share the one array: calls that overlap on the GPU (different streams with no ordering
 *     between them) race on it.  Calls on one stream or ordered by events are safe; nothing in the array has to
 *     start at zero and nothing is carried between calls (every tile writes its chunks before it reads them).
 *   - The first call on a device looks the array's address up (once per device, not capturable); a call with
 *     n_cells = 0 does only that, so a caller can run it ahead of a stream capture. */
#define DF_ANN_STATIC_SCRATCH_BYTES (32u << 20)
DF_API size_t df_ann_static_scratch_bytes(void);
DF_API df_status df_chem_ann_source_static(const df_ann* ann, const df_mech* mech, long long n_cells, long long ld,
                                    const float* T, const float* p, const float* Y,
                                    float* omega, float* dY, void* stream);

/* ---- one MLP per species ("individual training and prediction are carried out for each
 * species mass fraction", "multiple multilayer perceptrons") --------------------------------------------------
 * K independent networks with dims = {K+2, d1, d2, d3, 1} (n_layers = 4, the tensor path's shapes, see df_ann_create
 * precision 1: bf16-valued weights).  W[k*4 + l] / b[k*4 + l] are layer l of species k's network.  All networks
 * share the input vector x = {T, p, F(Y)} and its statistics x_mean/x_std [K+2]; network k's output o^(k) is the
 * z-scored Box-Cox-space change of species k: Delta_k = u_std[k] o^(k) + u_mean[k]; everything after that is the
 * epilogue of df_chem_ann_source.  The hot call runs the K tensor-core chains back to back on `stream`, then one
 * pointwise kernel; workspace (1024-byte aligned) holds the K raw outputs per cell ([K][ld] fp32) and the chain's
 * scratch: df_ann_mmlp_workspace_bytes(m, n_cells, ld) bytes on the current device. */
DF_API df_status df_ann_mmlp_create(df_ann_mmlp** out, int K, int n_layers, const int* dims,
                             const float* const* W, const float* const* b,
                             const double* x_mean, const double* x_std,
                             const double* u_mean, const double* u_std,
                             double boxcox_lambda, double dt);
DF_API df_status df_ann_mmlp_destroy(df_ann_mmlp* m);
DF_API size_t df_ann_mmlp_workspace_bytes(const df_ann_mmlp* m, long long n_cells, long long ld);
DF_API df_status df_chem_ann_source_mmlp(const df_ann_mmlp* m, const df_mech* mech, long long n_cells, long long ld,
                                  const float* T, const float* p, const float* Y,
                                  float* omega, float* dY,
                                  void* workspace, size_t workspace_bytes, void* stream);

/* ---- solver-facing extras of the property pass (reading A22) ------------
 * What a compressible solver with non-unity Lewis numbers needs besides cp, h, mu, lambda, D_k (all per cell, fp32):
 *   rho = p Wbar/(R T);  psi = Wbar/(R T) (= d rho/d p at constant T);  alpha = lambda/cp;  rhoD[k] = rho D_k;
 *   hk[k] = h_k(T)/W_k [J/kg], the species enthalpies of the diffusive enthalpy flux sum_k h_k J_k;
 *   s = sum_k (Y_k/W_k)(s_k(T) - R ln X_k) - (R/Wbar) ln(p/101325 Pa) [J/(kg K)], the ideal-gas mixture entropy
 *   (NASA-7 s_k with a7; X_k = 0 terms drop out).
 * cp, lambda, D are the arrays df_thermo_properties wrote (inputs here; needed only for alpha / rhoD).  rhoD and hk are
 * [K][ld].  Any output may be NULL (skipped). */
DF_API df_status df_thermo_extras(const df_mech* mech, long long n_cells, long long ld,
                           const float* T, const float* p, const float* Y,
                           const float* cp, const float* lambda, const float* D,
                           float* rho, float* psi, float* alpha, float* rhoD, float* hk, float* s, void* stream);

/* ---- PaSR scaling of the source and the temperature gate (reading A23) -----------
 * "the characteristic chemical time is calculated as the slowest formation rate of species and the mixing time
 * scale is calculated as the geometric mean of the Taylor scale and the Kolmogorov scale".  Per cell:
 *   tau_c = max over species with omega_k != 0 of rho Y_k/|omega_k|  (0 if none),  rho = p Wbar/(R T),
 *   tau_mix = sqrt((k_sgs/eps) sqrt(nu/eps)), nu = mu/rho,   kappa = tau_c/(tau_c + tau_mix)  (0 if tau_c = 0),
 *   omega_k <- kappa omega_k, and kappa = 0 where T < T_gate (the ANN saw no state below 500 K).
 * omega [K][ld] is updated in place; kappa [n] (optional) receives the factor. */
DF_API df_status df_chem_pasr_scale(const df_mech* mech, long long n_cells, long long ld,
                             const float* T, const float* p, const float* Y,
                             const float* mu, const float* k_sgs, const float* eps, float T_gate,
                             float* omega, float* kappa, void* stream);

/* ---- single-launch step ("the entire computational process is executed on GPU") -----------
 * A solver calls the update every time step on the same DEVICE arrays.  df_step_plan_create captures the whole step on
 * those arrays -- T <- T_guess (skipped when T_guess is NULL or equal to T: T then holds the guess), df_thermo_T_from_h,
 * df_thermo_properties (outputs that are NULL are skipped; the call is skipped when all are), df_chem_ann_source (when
 * omega is not NULL; workspace as for that call) -- as one CUDA graph; df_thermochem_step replays it on `stream` with a
 * single launch.  The arrays (and the handles) must stay valid and unmoved for the life of the plan; results are those
 * of the three calls made one after the other. */
DF_API df_status df_step_plan_create(df_step_plan** out, const df_mech* mech, const df_ann* ann, long long n_cells, long long ld,
                              const float* h, const float* p, const float* T_guess, const float* Y,
                              float* T, float* cp, float* mu, float* lambda, float* D, float* omega,
                              void* workspace, size_t workspace_bytes);
DF_API df_status df_thermochem_step(df_step_plan* plan, void* stream);
DF_API df_status df_step_plan_destroy(df_step_plan* plan);

/* ---- host-buffer step (bench.py's e2e leg) ----------------------------------------------
 * One pass of the whole path over HOST arrays: copies h, p, T_guess, Y host->device, runs
 * T_from_h -> properties -> ann_source (ann may be NULL: skipped) on the context's stream,
 * copies the requested outputs device->host and synchronises.  The cells are processed in up
 * to 8 slices on three streams (copy-in, kernels, copy-out), so that with pinned host arrays
 * the PCIe transfers in both directions overlap the kernels; with pageable arrays the copies
 * are staged by the driver and the call is still correct.  Pitch of Y, D and omega is ld on
 * both sides.
 * The context owns device staging for up to max_cells cells. */
DF_API df_status df_host_ctx_create(df_host_ctx** out, const df_mech* mech, const df_ann* ann, long long max_cells);
DF_API df_status df_host_ctx_destroy(df_host_ctx* ctx);
DF_API df_status df_step_host(df_host_ctx* ctx, long long n_cells, long long ld,
                       const float* h, const float* p, const float* T_guess, const float* Y,
                       float* T, float* cp, float* mu, float* lambda, float* D, float* omega);

/* ---- measurement helper (not part of the hot path) -------------------------------------------
 * Launches a register-only dependent-FMA kernel on `stream` (blocks x 256 threads, 16 FMAs per thread per iteration):
 * variant 0 = scalar FFMA, 1 = packed FFMA2 (the form the property kernels use).  *flops (host, optional) receives
 * the floating-point operations of the launch (FMA = 2); out (device, optional) receives blocks*256 floats.
 * bench.py times it with CUDA events: the FP32 "alu" roofline peak measured in the same run.
 * variants 2 and 3 are issue-rate probes for the property kernels' pair loops (blocks x 128 threads, out = blocks*128
 * floats): 2 = eight MUFU.RCP (+ eight FADD) per thread and iteration, 3 = the pair loop's mix of 2 MUFU.RCP + 6 FFMA2;
 * for them *flops receives the number of warp-iterations of the launch (iters x blocks x 4). */
DF_API df_status df_probe_fp32_peak(int variant, int blocks, long long iters, float* out, double* flops, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DF_THERMO_H */
