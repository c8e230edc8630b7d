/* tomo.h -- C ABI of libtomo_b200: FFT/Toeplitz MMSE tomographic wave-front reconstruction on one B200.
 *
 * The method is Ono et al., arXiv:1806.07938 (citations below are PAPER.md L<line>, section / equation):
 * solve  M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T zeta = M_s s   (Eq.12, Eq.34) by a fixed
 * number of conjugate-gradient iterations (S2.G L337), every covariance product applied through its 2RBT
 * (block-Toeplitz-Toeplitz-block) structure by zero-padded 2-D FFTs (S2.E L201-270, Eq.18-30), then project
 * phi_hat = M_phi W_phi Sigma_{phi s} W_s^T M_s^T zeta   (Eq.13, Eq.31 L276 / Eq.32, Eq.35).
 *
 * Conventions
 *   - every call returns int: TOMO_OK (0) or a negative error code; tomo_last_error() gives a thread-local
 *     message.  No C++ exception crosses this boundary.  There is NO CPU fallback: every entry point that
 *     computes needs a CUDA device and fails with TOMO_ECUDA without one.
 *   - "host" / "device" in an argument comment says where the pointer must live.  Host arrays are copied
 *     before the call returns.  Device arrays and the stream belong to the caller and must stay valid until
 *     the stream has passed the call; all compute calls are asynchronous on `cuda_stream` (a cudaStream_t
 *     passed as void*, NULL = the legacy default stream) and never synchronise with the host.
 *   - slopes layout (Eq.29):
 *         [frame][wfs][component: x then y][valid subaperture in row-major order of the n x n grid]   fp32
 *     slope unit = phase difference across a subaperture edge pair divided by d (rad/m; reading G6).
 *   - wavefront layout (Eq.35):
 *         [frame][target][valid phase point in row-major order of the (n+1) x (n+1) corner grid]      fp32
 *     radians of phase at the wavelength r0 is given at.
 *   - layered-phase (MCAO) plans, tomo_options.layered != 0 (S2.D L199, S6 L516): "wavefront" is the estimate of every
 *     LAYER on its own square grid, no pupil mask and no modal removal in layer space (reading G31):
 *         [frame][layer k][n_m x n_m grid point, row-major, x fastest]                                fp32
 *     grid point (mx, my) of layer k lies at ((mx, my) - (n_m - 1)/2) gamma_k d in the layer plane, centred on the axis.
 */
#ifndef TOMO_B200_H
#define TOMO_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define TOMO_OK            0
#define TOMO_EINVAL       -1   /* bad sizes, fractions not summing to 1 (1e-9), h_k >= h_gs, n_iter < 0, NULL ...   */
#define TOMO_EUNSUPPORTED -2   /* high-order set mixes NGS/LGS or LGS altitudes (not 2RBT, L158); FFT edge not 2^a3^b5^c */
#define TOMO_ENOTREADY    -3   /* compute call before tomo_plan_upload_kernels                                        */
#define TOMO_ENOMEM       -4
#define TOMO_ECUDA        -5   /* no device, launch or allocation failure                                           */

#define TOMO_HUDGIN 0          /* Eq.47-52 (L584-615), default slope model                                            */
#define TOMO_FRIED  1          /* Eq.54-62 (L630-691)                                                                 */
#define TOMO_FFTMODEL 2        /* Eq.41-46 (L534-572): gradient averaged over the subaperture; the covariances are    */
                               /* Fourier integrals of the von Karman spectrum, evaluated by the builder with 2-D FFTs */
                               /* on a grid of edge >= 512 and pixel d_k/4 (reading G29 of DESIGN.md)                  */

#define TOMO_F32       0       /* fp32 storage and arithmetic (headline path)                                         */
#define TOMO_F32S_F64A 1       /* fp32-stored spectra, fp64 FFT / vectors                                             */
#define TOMO_F64       2       /* everything fp64 (parity gate P-e); the slope / wavefront ABI stays fp32             */

#define TOMO_SOLVER_MULTIKERNEL 0   /* one kernel per phase, whole solve replayed from a CUDA graph                  */
#define TOMO_SOLVER_PERSISTENT  1   /* one cooperative persistent kernel per solve, device-side grid exchanges.      */
                                    /* Where it does not apply (FFT edge not instantiated, non-uniform or 2 x 2      */
                                    /* block noise) tomo_plan_upload_kernels selects the multi-kernel solver instead, */
                                    /* once, and tomo_get_solver reports which one runs and why                      */

typedef struct tomo_plan tomo_plan;          /* opaque; owns every device allocation it makes                        */

typedef struct {
    double ax, ay;        /* direction alpha_j [arcsec] (L41)                                                        */
    double h_gs;          /* guide-star altitude [m]; INFINITY = natural guide star (L158)                           */
    int    n_remove;      /* modes removed from this WFS: 0, 2 (tip/tilt) or 3 (tip/tilt/focus) (L321-329, Eq.36)    */
} tomo_wfs;

typedef struct {
    double D;                          /* pupil diameter [m]                                                         */
    int    n;                          /* subapertures across; d = D/n (Fig.2)                                  */
    double obstruction;                /* central obstruction ratio (0 = none)                                       */
    const unsigned char *subap_mask;   /* host, n*n row-major, non-zero = valid; NULL = centre-inside-pupil rule     */
    int    n_wfs;                      /* high-order WFSs: all NGS, or all LGS at ONE altitude (L158)                */
    const tomo_wfs *wfs;               /* host [n_wfs]                                                               */
    int    n_lo;                       /* low-order NGS sensors: validated only, not part of the CG system (L412)    */
    const tomo_wfs *lo_wfs;            /* host [n_lo] or NULL                                                        */
    int    n_targets;                  /* science directions beta_t (L41, L132)                                      */
    const double *target_xy;           /* host [n_targets][2] arcsec, targets at infinity                            */
} tomo_geometry;

typedef struct {
    int n_layers;                      /* K                                                                          */
    const double *h;                   /* host [K] layer altitudes [m]                                               */
    const double *frac;                /* host [K] Cn2 fractions, sum to 1 (L562)                                    */
} tomo_cn2;

typedef struct {
    const double *sigma2_wfs;          /* host [n_wfs] slope-noise variance (Sigma_eta diagonal, L110, L260) or NULL */
    double noise_frac;                 /* used when sigma2_wfs == NULL: sigma^2 = noise_frac * model slope variance  */
                                       /* of WFS 0, 1/2 [theta_xx(0) + theta_yy(0)]  (reading G15)                   */
    const double *sigma2_subap;        /* optional host [n_wfs][2][n_vs] full diagonal; overrides both; NULL if unused */
    const double *sigma_xy_subap;      /* optional host [n_wfs][n_vs]: covariance between the x- and the y-slope noise of   */
                                       /* one subaperture (elongated LGS spots, L331-333: Sigma_eta becomes 2 x 2 block     */
                                       /* diagonal); needs sigma2_subap; each block must be positive semi-definite          */
                                       /* (EINVAL otherwise).  Solved by the multi-kernel solver.  NULL = diagonal noise    */
} tomo_noise;

typedef struct {
    int slope_model;                   /* TOMO_HUDGIN | TOMO_FRIED | TOMO_FFTMODEL                                   */
    int pad;                           /* FFT edge P for Sigma_ss, 0 = next even 2^a 3^b 5^c >= 2n-1   (L207, G11)    */
    int pad_os;                        /* FFT edge P_os for Sigma_phi-s, 0 = next even 5-smooth >= n'+n-1            */
    int max_batch;                     /* largest n_frames a solve may be given (>= 1)                               */
    int precision;                     /* TOMO_F32 | TOMO_F32S_F64A | TOMO_F64                                       */
    int solver;                        /* TOMO_SOLVER_MULTIKERNEL | TOMO_SOLVER_PERSISTENT                           */
    int build_cos;                     /* 0 = no target projection (tomo_solve then returns zeta-less zeros: EINVAL) */
    int layered;                       /* != 0: estimate the phase of every layer on its meta-pupil grid instead of the    */
                                       /* pupil-plane phase towards targets (L199: the new grid of Eq.16 extended over the  */
                                       /* layer, I'_k removed, layers not summed).  geom->n_targets must be 0.  The grids   */
                                       /* share one edge n_m (reported as n_prime by tomo_get_sizes): the smallest integer  */
                                       /* with the parity of n+1 that is >= max_k (D + 2 h_k fov_radius)/(gamma_k d) + 1    */
    double fov_radius;                 /* [arcsec] field radius the layer grids must cover (layered plans only; 0 = the     */
                                       /* LTAO grid n')                                                                     */
} tomo_options;

/* Validate the problem statement (S2 L41-58; S2.F L297-333), build masks W_s, W_phi (Eq.33-35), modal matrices
 * Z_s, Z_phi and (Z^T Z)^-1 (Eq.36), cone factors gamma_k and the common n' (L158, L179, L295), choose P, P_os and
 * allocate every device buffer.  `opt` may be NULL (defaults: Hudgin, automatic pads, batch 1, fp32,
 * multi-kernel solver, C_os built).  On success *out owns the plan. */
int tomo_plan_create(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0,
                     const tomo_noise *noise, const tomo_options *opt, tomo_plan **out);

/* One-time covariance-kernel builder (L150, L158, L179-197, L265, L295; Eq.50-53).
 *   css_gen: host fp64 [C][C][2n-1][2n-1] generators theta[(i,a),(j,b)](l), index (ly+n-1, lx+n-1), lag = input - output,
 *            C = 2 n_wfs, channel = 2*wfs + component; NULL = build from the von Karman structure function.
 *   cos_gen: host fp64 [T][K'][C][n'+n-1][n'+n-1] generators xi'[t,k,(j,b)](l), l = q - p' in [-(n'-1), n-1]^2,
 *            K' = n_layers (LGS) or 1 (NGS, layers summed); NULL = build.
 * Computes the circular embeddings, their 2-D real DFTs in fp64, folds 1/P^2, keeps the Hermitian half and only
 * blocks (c_out <= c_in), converts to the plan's storage precision and uploads once. */
int tomo_plan_upload_kernels(tomo_plan *plan, const double *css_gen, const double *cos_gen);

/* Full path A1-A8 for one frame: n_iter CG iterations from a cold start, then the projection to every target.
 * slopes: device fp32 [C][n_vs]; wavefront_out: device fp32 [n_targets][n_vphi]. */
int tomo_solve(tomo_plan *plan, const float *slopes, float *wavefront_out, int n_iter, void *cuda_stream);

/* Same for n_frames <= max_batch independent frames; x0 (device fp32 [n_frames][C][n_vs]) is an optional warm
 * start (L428, L506), NULL = cold start (L490). */
int tomo_solve_batch(tomo_plan *plan, const float *slopes, float *wavefront_out, int n_frames, int n_iter,
                     const float *x0, void *cuda_stream);

/* The same path with MINRES instead of CG: the solver the paper keeps for the Toeplitz method (S2.G L337; L426 "MINRES
 * and CG are used for the Toeplitz and sparse methods"; Fig.13: CG does not converge in its noise-free case).
 * Paige-Saunders recurrences (Lanczos vectors v_k, Givens rotations of the tridiagonal, directions w_k) around the same
 * Sigma_ss product kernels, exactly n_iter iterations, no preconditioner, then the projection to every target.
 * Arguments, layouts, ownership and errors as tomo_solve_batch (x0 = optional warm start, NULL = cold start).
 * tomo_get_residuals afterwards returns phibar_k = |b - A x_k|, k = 0..n_iter; tomo_get_zeta the iterate x_{n_iter}.
 * Runs on the solver that runs the plan (tomo_get_solver): inside the persistent kernel -- the same two phases and two grid
 * exchanges per iteration as CG, alpha_k = v_k . A v_k by Parseval where CG takes p.q, beta_{k+1} = |u_k| where CG takes r.r --
 * or as one CUDA graph of the multi-kernel solver. */
int tomo_solve_minres(tomo_plan *plan, const float *slopes, float *wavefront_out, int n_frames, int n_iter,
                      const float *x0, void *cuda_stream);

/* out = M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T v  (Eq.30, Eq.34): one product, for the MVM gate.
 * Computed by the solver that runs the plan's solves (tomo_get_solver): with the persistent solver it is ONE launch of the
 * persistent kernel in its single-product mode (the same phase code, instance and shared-memory layout as a solve), else
 * the multi-kernel product.  v, out: device fp32 [C][n_vs]. */
int tomo_apply_css(tomo_plan *plan, const float *v, float *out, void *cuda_stream);

/* The same product, out = M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T v (Eq.30, Eq.34), for callers that may not
 * allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): this entry point calls no
 * cudaMalloc / cudaFree and no allocating library routine.  It runs the multi-kernel product (projection, row FFTs, per-frequency
 * block product, inverse row FFTs, projection) with ALL its workspace -- the projected input, the product, the two half-spectrum
 * buffers T1 / T2 and the reduction partials -- inside one file-scope device array of TOMO_STATIC_SCRATCH_BYTES, which every GPU
 * that loads the library holds until the process exits.  A plan whose workspace is larger (2 C n_vs + 4 C (P/2+1) n elements of the
 * plan's arithmetic type plus partials; cfg3 / cfg4 in fp32 take 1.6 / 2.1 MB, cfg4 in TOMO_F64 4.2 MB) is refused with
 * TOMO_EINVAL and a message that names both sizes; nothing is launched then.  The array is shared by every plan and every call
 * and keeps the last call's contents: each call clears the part it uses (a memset node on `cuda_stream`) before its kernels.
 * Calls that may overlap on the GPU (different streams, or graphs replayed concurrently) RACE on the array and give wrong
 * results: serialise them, or use tomo_apply_css, whose workspace belongs to the plan.  The array's address is looked up once
 * per device on the first call for that device (make that call outside a capture).  v, out: device fp32 [C][n_vs]; asynchronous
 * on `cuda_stream`; errors as tomo_apply_css. */
#define TOMO_STATIC_SCRATCH_BYTES 4194304
int tomo_apply_css_static(tomo_plan *plan, const float *v, float *out, void *cuda_stream);

/* wavefront_out = M_phi W_phi Sigma_{phi s} W_s^T M_s^T zeta  (Eq.31/32, Eq.35) for every target (A7-A8 only).
 * zeta: device fp32 [C][n_vs]; wavefront_out: device fp32 [n_targets][n_vphi].
 * Layered plans: wavefront_out[k] = Sigma_{phi_k s} W_s^T M_s^T zeta for every layer k, device fp32 [K][n_m][n_m]. */
int tomo_apply_cos(tomo_plan *plan, const float *zeta, float *wavefront_out, void *cuda_stream);

/* One CG iteration (S2.G L337) on caller-held state, for the teacher-forced gate:
 * x, r, p: device fp32 [C][n_vs], updated in place; rho_alpha_beta: device fp64 [3]: in [0] = rho_k = r_k.r_k,
 * out [0] = rho_{k+1}, [1] = alpha_k, [2] = beta_k. */
int tomo_cg_step(tomo_plan *plan, float *x, float *r, float *p, double *rho_alpha_beta, void *cuda_stream);

/* The CG solution zeta of the last solve: device->device copy into zeta_out (device fp32 [n_frames][C][n_vs]). */
int tomo_get_zeta(tomo_plan *plan, float *zeta_out, int n_frames, void *cuda_stream);

/* Measurement aid (bench.py "roofline"): runs n_iter iterations of the multi-kernel loop (A2-A6) on the state the
 * last solve left in the plan, un-graphed, with a CUDA event after every kernel on `cuda_stream`, synchronises the
 * stream and returns the mean device time per launch in ms: ms_out (host fp32 [4]) = rows_fwd, cols, rows_inv,
 * update.  The state of the last solve is overwritten. */
int tomo_time_kernels(tomo_plan *plan, int n_frames, int n_iter, float *ms_out, void *cuda_stream);

/* Measurement aid for the persistent solver: one instrumented solve of n_iter iterations -- CG (minres = 0) from the state
 * the last solve left in the plan, MINRES (minres != 0; TOMO_F32, n_frames = 1) from a cold start on the projected slopes
 * of the last solve; thread 0 of every CTA stamps the SM cycle counter at the phase boundaries.  Synchronises
 * the stream.  us_out (host fp32 [10]), microseconds at the device's nominal SM clock, mean over iterations; work
 * segments are the maximum over CTAs, barrier segments the minimum over CTAs (= pure latency):
 * [0] whole iteration (CTA 0), [1] rho/beta scalars, [2] p~ update, [3] forward y-FFT, [4] block product,
 * [5] inverse y-FFT + T2 write, [6] grid barrier B, [7] alpha/mode scalars (+ first inverse x-FFT), [8] row phase,
 * [9] grid barrier A.  The state of the last solve is overwritten.  If the environment variable TOMO_STAMP_DUMP names a
 * writable file, the raw per-CTA timeline (mean over iterations of every stamp, microseconds from the iteration start, one
 * line per CTA) is also written there; the library reads no other environment variable. */
int tomo_time_phases(tomo_plan *plan, int n_frames, int n_iter, int minres, float *us_out, void *cuda_stream);

/* Measurement aid (bench.py "roofline" with the persistent solver): `reps` launches of the persistent kernel alone
 * (A1-A6: rhs projection + n_iter CG (minres = 0) or MINRES (minres != 0) iterations from a cold start on `slopes`, device fp32 [n_frames][C][n_vs]; no
 * target projection), each bracketed by CUDA events on `cuda_stream`; synchronises the stream and returns the mean
 * device time of one launch in ms (host fp32 [1]). */
int tomo_time_solver(tomo_plan *plan, const float *slopes, int n_frames, int n_iter, int reps, int minres, float *ms_out,
                     void *cuda_stream);

/* Measurement aid (bench.py "l2_roofline", north_star: "... and over L2 bandwidth where the spectra are L2-resident"): the
 * device's L2 -> SM read bandwidth and its plain fp32 FMA rate, measured by two small kernels of this library on
 * `cuda_stream` (synchronises the stream).  The bandwidth kernel sweeps an L2-resident buffer of `l2_bytes` (0 = 64 MiB;
 * keep it under the L2 size) `reps` times with 16-byte `ld.global.cg` loads from 148 x 8 CTAs and returns the best
 * repetition; the FMA kernel runs independent FFMA chains on every SM.  out (host fp32 [2]) = {L2 read GB/s, fp32 TFLOP/s}.
 * Needs no plan.  Returns TOMO_ECUDA without a device. */
int tomo_measure_device(long long l2_bytes, int reps, float *out, void *cuda_stream);

/* Sizes fixed at plan creation; any pointer may be NULL.  Layered plans: n_vphi = n_m * n_m, wavefront_len = K * n_m * n_m,
 * n_prime = n_m. */
int tomo_get_sizes(const tomo_plan *plan, int *n_vs, int *n_vphi, int *slopes_len, int *wavefront_len,
                   int *pad, int *pad_os, int *n_prime);

/* Row-major grid indices of the valid subapertures ([n_vs], host) and valid phase points ([n_vphi], host). */
int tomo_get_valid_index(const tomo_plan *plan, int *subap_idx, int *phase_idx);

/* sigma^2 per WFS actually used (host fp64 [n_wfs]) and the model slope variance of WFS 0 (host fp64 [1]). */
int tomo_get_noise(const tomo_plan *plan, double *sigma2_wfs, double *slope_var);

/* Residual history sqrt(rho_k), k = 0..n_iter of the last solve: host fp64 [n_frames][n_iter+1].  The caller
 * must have synchronised the stream of that solve; this call copies device->host synchronously. */
int tomo_get_residuals(const tomo_plan *plan, double *host_out, int n_frames, int n_iter);

/* The solver that runs this plan's solves, products and CG steps (TOMO_SOLVER_*), decided once by
 * tomo_plan_upload_kernels (TOMO_ENOTREADY before it), and -- when TOMO_SOLVER_PERSISTENT was asked for but does not apply --
 * the reason, copied as a NUL-terminated string into note (host, note_cap bytes; may be NULL).  Never changes afterwards. */
int tomo_get_solver(const tomo_plan *plan, int *solver_in_use, char *note, int note_cap);

/* Bytes of device memory owned by the plan, and the number of kernel launches the last solve enqueued. */
int tomo_get_stats(const tomo_plan *plan, long long *device_bytes, int *launches_last_solve);

/* ---- split low-order path for the NGS tip/tilt sensors of geom->lo_wfs (L321, L412, Table 2; the paper gives no
 * algorithm: reading G30 of DESIGN.md).  Each low-order sensor delivers the mean x- and the mean y-slope over the valid
 * subapertures [rad/m] with white noise of variance sigma2_lo; R_lo = C_tau,g (C_gg + sigma2_lo I)^-1 (Eq.5 L68 on the
 * aperture-mean slope pairs, [2 n_targets][2 n_lo]) is built once on the host (stencil slope models only: EUNSUPPORTED for
 * TOMO_FFTMODEL; EINVAL when n_lo == 0 or the matrix is not positive definite) and uploaded.  *out owns its device memory. */
typedef struct tomo_lo tomo_lo;
int tomo_lo_create(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0, int slope_model, double sigma2_lo,
                   tomo_lo **out);
/* wavefront[frame][target][valid phase point] += tau_x x_p + tau_y y_p, tau = R_lo g_frame, in place on `cuda_stream`
 * (asynchronous).  lo_slopes: DEVICE fp32 [n_frames][n_lo][2 (x, y)]; wavefront: DEVICE fp32 in the layout tomo_solve_batch
 * writes (the tip/tilt-free high-order estimate, Eq.35).  n_frames in [0, 65535]; 0 = no launch (buffers may be NULL). */
int tomo_lo_apply(const tomo_lo *lo, const float *lo_slopes, float *wavefront, int n_frames, void *cuda_stream);
void tomo_lo_destroy(tomo_lo *lo);

void tomo_plan_destroy(tomo_plan *plan);
const char *tomo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TOMO_B200_H */
