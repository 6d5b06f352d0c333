/* wz.h -- C-ABI of the B200 (sm_100a) hot path of arXiv:1005.3276:
 * conjugate-gradient solve of  M^dag M x = b  for the lattice Wess-Zumino
 * fermion matrix with the overlap (Neuberger) operator,
 *
 *   M = Dslash + m P+ + m* P- + 2g phi P+ + 2g* phi* P-,
 *   Dslash = (1 - D2/2)^-1 D1                       (Eq. 2.19)
 *
 * applied as the paper does (Sec. 7): the phi-free part is
 * diagonal in momentum space and is reached by a forward and an inverse 4D FFT
 * with antiperiodic time boundary conditions; the Yukawa
 * part is a site-local multiply in position space.
 *
 * Conventions:
 *  - every data pointer is a DEVICE pointer owned by the caller; the library
 *    allocates only the workspace and tables held by the plan;
 *  - spinor field  = [batch][spin 0..3][x0 = t][x1][x2][x3], x3 fastest,
 *    interleaved (re, im); spin 0,1 = P- (gamma5 = -1), spin 2,3 = P+
 *    (Eq. 2.2);  phi = [x0][x1][x2][x3], shared by the batch;
 *  - element type is complex64 (WZ_C64) or complex128 (WZ_C128), fixed per plan;
 *  - every call is enqueued on the plan's stream and returns without
 *    synchronising, except wz_cg_solve (see there);
 *  - errors are returned, never thrown; there is no CPU fallback.
 */
#ifndef WZ_H_
#define WZ_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wz_plan wz_plan; /* opaque */

typedef enum { WZ_C64 = 0, WZ_C128 = 1 } wz_dtype;

typedef enum {
  WZ_OK = 0,
  WZ_EINVAL = 1,        /* bad argument: null pointer, T odd, extent < 2, nbatch > max_batch,
                           rho outside (0,2), tol <= 0, in == out where not allowed */
  WZ_EUNSUPPORTED = 2,  /* lattice extents this build has no tile kernel for */
  WZ_ENOMEM = 3,        /* device allocation of the plan workspace failed */
  WZ_ECUDA = 4,         /* a CUDA call or launch failed (text via wz_last_error) */
  WZ_ENOTCONVERGED = 5  /* wz_cg_solve: some source hit max_iter */
} wz_status;

const char *wz_status_string(wz_status s);
/* Text of the last CUDA error seen by this thread's calls (empty string if none). */
const char *wz_last_error(void);
/* Library version, "major.minor". */
const char *wz_version(void);

/* Create a plan for a T x L1 x L2 x L3 lattice (T = extent of x0, the antiperiodic
 * time direction; PAPER.md:234 requires T even).  `stream` is a cudaStream_t
 * (0 = legacy default stream) of the CURRENT device: the plan lives on that device, and every call on
 * the plan switches to it for its duration (and back).  The plan owns: twiddle/momentum tables, the
 * matvec temporaries (2 spinors per batch entry) and the CG vectors.  max_batch >= 1.
 * Supported extents: (T,L1) and (L2,L3) pairs listed by wz_supported(). */
wz_status wz_plan_create(wz_plan **plan, int T, int L1, int L2, int L3,
                         wz_dtype dtype, int max_batch, void *stream);
wz_status wz_plan_destroy(wz_plan *plan);
/* 1 if this build has tile kernels for the lattice, else 0. */
int wz_supported(int T, int L1, int L2, int L3, wz_dtype dtype);
/* Bytes of device memory the plan holds. */
unsigned long long wz_plan_workspace_bytes(const wz_plan *plan);

/* 4D DFT of nbatch spinor fields (4 components each).
 * direction +1: forward, kernel exp(-i p.x), unnormalised;
 * direction -1: inverse, kernel exp(+i p.x), times 1/V.
 * antiperiodic_time 0: p0 = 2 pi n0/T;  1: p0 = 2 pi (n0 + 1/2)/T, i.e. the field
 * is multiplied by exp(-i pi x0/T) before the forward transform and by
 * exp(+i pi x0/T) after the inverse one.
 * in == out is allowed. */
wz_status wz_fft4d(wz_plan *plan, int direction, int antiperiodic_time,
                   const void *in, void *out, int nbatch);

/* out = M in (dagger = 0) or M^dag in (dagger = 1), Eq. (2.19); m, g complex as
 * {re, im}; 0 < rho < 2 is the overlap parameter (the paper has rho = 1).
 * in == out is NOT allowed (in is re-read for the Yukawa term): WZ_EINVAL. */
wz_status wz_apply_M(wz_plan *plan, int dagger, const void *phi,
                     const double m[2], const double g[2], double rho,
                     const void *in, void *out, int nbatch);

/* out = M^dag M in. in == out is NOT allowed. */
wz_status wz_apply_MdagM(wz_plan *plan, const void *phi,
                         const double m[2], const double g[2], double rho,
                         const void *in, void *out, int nbatch);

typedef struct {
  int iterations;       /* M^dag M applications inside the CG loop */
  int reliable_updates; /* complex128 residual recomputations (WZ_C64 plans only) */
  int converged;        /* 1 if the stop rule was met */
  double rel_residual_recursive; /* sqrt(rho_k)/||b|| at exit */
  double rel_residual_true;      /* ||b - M^dag M x|| / ||b||, recomputed at exit */
} wz_cg_info;

/* Conjugate gradient on M^dag M x = b, x0 = 0, one
 * independent solve per source; stop when ||r||_2 <= tol ||b||_2.
 *  - b: nbatch spinors of the plan's dtype (device).
 *  - x: nbatch spinors, ALWAYS complex128 (device): WZ_C64 plans iterate in
 *    complex64 with float64 reductions and accumulate the solution in complex128
 *    by reliable updates (reading G9); rounding that solution to
 *    complex64 would by itself lift the true residual above tol.
 *  - info: HOST array of nbatch entries.
 * x must not alias b (WZ_EINVAL).
 * Synchronises the plan's stream before returning.  Returns WZ_ENOTCONVERGED if
 * any source hit max_iter; x then holds the last iterate. */
wz_status wz_cg_solve(wz_plan *plan, const void *phi, const void *b, void *x,
                      const double m[2], const double g[2], double rho,
                      double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Free-inverse preconditioning (Eq. 7.8-7.11) ----
 * M0 = Dslash + m P+ + m* P- is the fermion matrix at g = 0;  M0^-1 = M0^dag / (D_mu^dag D_mu + |m|^2)
 * is diagonal in momentum space (4x4 per momentum).  m != 0 is required.
 * wz_apply_M0inv:   out = M0^-1 in (dagger = 0) or (M0^-1)^dag in (dagger = 1); in == out allowed.
 * wz_apply_MtdagMt: out = Mtilde^dag Mtilde in with Mtilde = M M0^-1 (Eq. 7.10); in != out.
 * wz_cg_solve_pc:   btilde = (M0^-1)^dag b;  CG on Mtilde^dag Mtilde xtilde = btilde from xtilde0 = 0,
 *   stop when ||rtilde|| <= tol ||btilde|| (the preconditioned system's residual; G15);
 *   x = M0^-1 xtilde.  Arguments as wz_cg_solve (x always complex128).  In info,
 *   rel_residual_recursive refers to the preconditioned system, rel_residual_true is
 *   ||b - M^dag M x|| / ||b|| of the ORIGINAL system recomputed at exit. */
wz_status wz_apply_M0inv(wz_plan *plan, int dagger, const double m[2], double rho,
                         const void *in, void *out, int nbatch);
wz_status wz_apply_MtdagMt(wz_plan *plan, const void *phi, const double m[2], const double g[2],
                           double rho, const void *in, void *out, int nbatch);
wz_status wz_cg_solve_pc(wz_plan *plan, const void *phi, const void *b, void *x,
                         const double m[2], const double g[2], double rho,
                         double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Shifted system (Eq. 7.6-7.7; 927-931, Eq. 7.13) ----
 * The partial-fraction terms of the rational approximation need (M^dag M + beta_i) X_i = eta, one
 * conjugate-gradient solve per shift ("solved one at a time").
 * wz_cg_solve_shift: CG on (M^dag M + sigma) x = b, sigma >= 0 real, x0 = 0, stop when
 *   ||b - (M^dag M + sigma) x|| <= tol ||b||.  sigma = 0 is wz_cg_solve.  All other arguments, the
 *   complex128 solution buffer and info as in wz_cg_solve; residuals refer to the shifted system.
 *   sigma < 0 or NaN: WZ_EINVAL. */
wz_status wz_cg_solve_shift(wz_plan *plan, const void *phi, const void *b, void *x,
                            const double m[2], const double g[2], double rho, double sigma,
                            double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Preconditioned shifted system and the rational sum (Eq. 7.14; 877-892 Eq. 7.6-7.7;
 *      948-950 cutoff rule; Table VII) ----
 * wz_cg_solve_shift_pc: with x = M0^-1 xtilde, CG on
 *     (Mtilde^dag Mtilde + sigma (M0^-1)^dag M0^-1) xtilde = btilde,  btilde = (M0^-1)^dag b      (Eq. 7.14)
 *   from xtilde0 = 0, stop rule on THIS system's residual (G15), then x = M0^-1 xtilde.  The sigma
 *   term rides through the same five passes as wz_cg_solve_pc (pass C adds sigma M0^-1 p to what pass D
 *   multiplies by (M0^-1)^dag).  m != 0 and sigma >= 0 required (else WZ_EINVAL); sigma = 0 is
 *   wz_cg_solve_pc.  x: complex128; info.rel_residual_true = ||b - (M^dag M + sigma) x|| / ||b||.
 * wz_rational_apply: out = alpha0 eta + sum_{i < nshift} alphas[i] X_i with (M^dag M + betas[i]) X_i = eta
 *   (Eq. 7.6-7.7), one solve per shift for the whole batch: wz_cg_solve_shift_pc when betas[i] <= pc_cutoff
 *   (the paper uses 100) and m != 0, wz_cg_solve_shift otherwise.  alphas, betas: HOST arrays of nshift
 *   doubles, betas[i] >= 0.  eta: nbatch spinors of the plan's dtype; out: nbatch spinors, ALWAYS
 *   complex128 (device; must not alias eta).  info: HOST array of nshift * nbatch entries, [shift][source].
 *   Returns WZ_ENOTCONVERGED if any solve hit max_iter (out then holds the sum of the last iterates).
 *   Synchronises the stream. */
wz_status wz_cg_solve_shift_pc(wz_plan *plan, const void *phi, const void *b, void *x,
                               const double m[2], const double g[2], double rho, double sigma,
                               double tol, int max_iter, int nbatch, wz_cg_info *info);
wz_status wz_rational_apply(wz_plan *plan, const void *phi, const void *eta, void *out,
                            const double m[2], const double g[2], double rho, double alpha0,
                            const double *alphas, const double *betas, int nshift, double pc_cutoff,
                            double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Multi-shift CG (Eq. 7.6-7.7, 927-931 Eq. 7.13) ----
 * The paper solves the d = 20 systems (M^dag M + beta_i) X_i = eta one at a time.  They share
 * one Krylov space: wz_cg_solve_multishift solves all of them in the iterations of the hardest one (B.
 * Jegerlehner, hep-lat/9612014): CG runs on the system with the smallest shift, the residuals of the others
 * stay collinear with its residual, r_i = zeta_i r, and two site-local updates per shift carry x_i and p_i along.
 *  - sigmas: HOST array of nshift >= 1 shifts, each >= 0, nshift <= 32.
 *  - b: nbatch spinors of the plan's dtype;  x: nshift * nbatch spinors, [shift][source], ALWAYS complex128.
 *  - info: HOST array [shift][source].  iterations = the iteration at which that shift met
 *    |zeta_i| ||r|| <= tol ||b|| (its updates stop there).  WZ_C64 plans iterate in complex64 WITHOUT reliable
 *    updates (a recomputed residual would break the collinearity) and then polish every shift whose true
 *    residual, recomputed in complex128, is above tol: the defect is solved for by wz_cg_solve_shift's loop and
 *    added; iterations then includes the polishing iterations, reliable_updates counts theirs.
 *    rel_residual_true = ||b - (M^dag M + sigma_i) x_i|| / ||b|| recomputed at exit.
 * Synchronises the stream.  WZ_ENOTCONVERGED if any system hit max_iter.
 * wz_rational_apply_multishift: wz_rational_apply with every shift above pc_cutoff (all shifts if pc_cutoff < 0
 *   or m = 0) taken from ONE multi-shift solve; shifts up to pc_cutoff keep the paper's preconditioned solves. */
wz_status wz_cg_solve_multishift(wz_plan *plan, const void *phi, const void *b, void *x,
                                 const double m[2], const double g[2], double rho,
                                 const double *sigmas, int nshift, double tol, int max_iter, int nbatch,
                                 wz_cg_info *info);
wz_status wz_rational_apply_multishift(wz_plan *plan, const void *phi, const void *eta, void *out,
                                       const double m[2], const double g[2], double rho, double alpha0,
                                       const double *alphas, const double *betas, int nshift, double pc_cutoff,
                                       double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Defect correction ("mixed precision conjugate gradient") ----
 * wz_cg_solve_dc (WZ_C64 plans; WZ_EINVAL otherwise): a complex128 outer loop around complex64 inner solves,
 *   X = 0;  repeat:  d = b - M^dag M X  in complex128;  stop if ||d|| <= tol ||b||;
 *                    plain complex64 CG (no reliable updates) on M^dag M e = d to ||r|| <= inner_tol ||d||;  X += e.
 * The other route to double-precision tolerances with complex64 vectors, next to the reliable updates of
 * wz_cg_solve (which keep the search direction across the corrections; this loop restarts the Krylov space).
 * 0 < inner_tol < 1.  info.iterations = inner iterations in total, info.reliable_updates = outer corrections,
 * both residual fields = ||b - M^dag M x|| / ||b|| recomputed in complex128.  x: complex128, must not alias b.
 * Synchronises the stream; WZ_ENOTCONVERGED if the iteration budget max_iter ran out. */
wz_status wz_cg_solve_dc(wz_plan *plan, const void *phi, const void *b, void *x,
                         const double m[2], const double g[2], double rho,
                         double tol, double inner_tol, int max_iter, int nbatch, wz_cg_info *info);

/* wz_cg_solve_dc_half (WZ_C64 plans; lattices with binary16-storage kernels: 8^4, 16^4, 32^4, 48x24^3, else WZ_EUNSUPPORTED):
 * wz_cg_solve_dc with the inner solver's vectors t, chi, r, p STORED as two IEEE binary16 values per complex number
 * (SURVEY.md 8(f) NEXT-3 "half-precision-storage inner solver with defect correction"; oracle O10).  Arithmetic
 * stays float, reductions double, the inner x float, the outer loop complex128; each defect is normalised to unit
 * rms before its inner solve, so no per-vector scales are needed.  10.5u of traffic per inner iteration instead of
 * 18.5u (u = one complex64 spinor).  binary16 carries 11 bits: use inner_tol around 1e-1 ... 1e-2 (each outer
 * correction gains about that factor).  Arguments, info and return values as wz_cg_solve_dc. */
wz_status wz_cg_solve_dc_half(wz_plan *plan, const void *phi, const void *b, void *x,
                              const double m[2], const double g[2], double rho,
                              double tol, double inner_tol, int max_iter, int nbatch, wz_cg_info *info);

/* wz_cg_solve_half (WZ_C64 plans; lattices as wz_cg_solve_dc_half): wz_cg_solve with t, chi, r, p STORED in binary16
 * (oracle O11).  The loop of wz_cg_solve for WZ_C64 plans -- float arithmetic, double reductions, complex128 reliable
 * updates (reading G9), the search direction kept across them -- on the system normalised to unit rms; every
 * reliable update rescales r and p to unit rms again, so the stored values never leave binary16's normal range.
 * 10.5u of traffic per iteration instead of 18.5u.  Arguments, info and return values as wz_cg_solve. */
wz_status wz_cg_solve_half(wz_plan *plan, const void *phi, const void *b, void *x,
                           const double m[2], const double g[2], double rho,
                           double tol, int max_iter, int nbatch, wz_cg_info *info);

/* ---- Locality probe (Eq. 3.9-3.11, Fig. 1) ----
 * wz_apply_Dslash: out = Dslash in = (1 - D2/2)^-1 D1 in (the fermion matrix at m = g = 0); in != out.
 * wz_locality_profile: psi = Dslash eta for a unit point source at the origin in spin component
 *   `spin`; f[r] = max{ ||psi(x)|| over the spinor index : ||x||_1 = r }, taxi-driver distance with the
 *   shorter way round each axis.  f is a HOST array of nf = 1 + sum_mu floor(L_mu / 2) doubles.
 *   Uses plan temporaries; synchronises the stream. */
wz_status wz_apply_Dslash(wz_plan *plan, double rho, const void *in, void *out, int nbatch);
wz_status wz_locality_profile(wz_plan *plan, double rho, int spin, double *f_host, int nf);

/* The kCheck = 8 CG iterations between two looks of the host at the device-resident solver state are 40
 * launches with fixed arguments: by default they are captured once as a CUDA graph (per distinct set of
 * solve arguments) and replayed, so a solve makes no host round trip except that lagged convergence check
 * (BASELINE.json north star (iii)).  wz_plan_set_graph(plan, 0) enqueues the same kernels
 * one by one instead (results are bit-identical; for measurements).  Default: 1. */
wz_status wz_plan_set_graph(wz_plan *plan, int enable);

/* Sources per block of a batched solve.  The sources of a batch are independent solves (one CG state, one
 * set of reductions each): they advance block by block, each block running its 8 iterations between two
 * convergence checks back to back, so that a block's vectors stay in the L2 cache from one pass to the next.
 * 0 = the whole batch in lock step through shared launches.  Results do not depend on it, bit for bit. */
wz_status wz_plan_set_block(wz_plan *plan, int sources_per_block);

/* Residual history of the LAST solve on this plan, as the host saw it at its convergence checks (every 8
 * iterations, one chunk behind the GPU): for `source`, pairs (iteration k, ||r_k|| / ||b||) with the
 * recursive residual (PAPER.md:944 stop rule), the recomputed one right after a reliable update.
 * Copies at most cap pairs into the HOST arrays (either may be NULL to only count); returns the number
 * of pairs recorded, or -1 on a bad argument. */
int wz_plan_cg_history(const wz_plan *plan, int source, int *iterations, double *rel_residual, int cap);

/* ---- M^dag M without a plan and without any device allocation ----
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it).  out = M^dag M in, as wz_apply_MdagM, but the scratch of the matvec (the FFT temporary, chi = M in,
 * the momentum tables) lives in a file-scope device array of WZ_NOALLOC_MAX_BYTES (+ 4 KB) inside the library,
 * which every GPU that loads the library holds until the process exits.  The call makes no cudaMalloc, cudaFree or
 * other allocating CUDA call; it only enqueues kernels on `stream` (the momentum tables are recomputed on the device
 * by a small kernel each call).  Works on the CURRENT device: `stream` (a cudaStream_t, 0 = legacy default stream)
 * and all pointers must belong to it.  The first call on a device also does the one-time set-up (address of the
 * array, upload of the twiddle tables): make that first call outside a stream capture.
 *  - T, L1, L2, L3, dtype: the lattice and element type (no plan); phi, in, out, m, g, rho: as wz_apply_MdagM;
 *    in != out.
 *  - LIMIT: the call needs 2 * nbatch * (4 * T*L1*L2*L3 * sizeof(complex)) bytes of scratch (3 * ... for 64 x 64
 *    (x2,x3) planes); more than WZ_NOALLOC_MAX_BYTES = 8 MiB (e.g. one 16^4 complex128 or one 32x16^3 complex64
 *    source, four 16^4 complex64 sources) returns WZ_EINVAL with the byte counts in wz_last_error().  Unsupported
 *    extents: WZ_EUNSUPPORTED.
 *  - ALL calls share the one array, on every stream: two calls that overlap on the GPU race (serialise them on
 *    one stream or with events).  The array keeps the last call's contents; nothing in it has to start at zero
 *    (every byte a call reads it has written before), so no clearing is needed between calls.
 * Results agree with wz_apply_MdagM to rounding (the tables come from the device's sinpi instead of the host's sin). */
#define WZ_NOALLOC_MAX_BYTES (8u << 20)
wz_status wz_apply_MdagM_noalloc(int T, int L1, int L2, int L3, wz_dtype dtype, const void *phi,
                                 const double m[2], const double g[2], double rho,
                                 const void *in, void *out, int nbatch, void *stream);

/* Number of kernel launches this plan has enqueued so far (for bench.py's
 * gpu_launches), and a reset. */
unsigned long long wz_plan_launch_count(const wz_plan *plan);
void wz_plan_reset_launch_count(wz_plan *plan);

/* Optional per-kernel timing for measurement (bench.py's roofline): while enabled,
 * up to 8192 launches are bracketed by CUDA events on the plan's stream.
 * wz_plan_profile_read synchronises the stream, adds the recorded durations to the
 * per-kind totals, and copies them out: ms[k] = summed milliseconds and count[k] =
 * launches of kind k (arrays of WZ_NKINDS entries, host).  wz_plan_profile(plan, 0)
 * stops recording; wz_plan_profile(plan, 1) clears the totals and starts. */
enum {
  WZ_K_P01_FWD = 0,  /* pass A: twist + DFT axes 0,1 */
  WZ_K_P23_MULT = 1, /* passes B, D: DFT axes 2,3, overlap multiply, inverse DFT axes 2,3 */
  WZ_K_P01_MID = 2,  /* pass C: inverse 0,1 + Yukawa + ||chi||^2 + forward 0,1 */
  WZ_K_P01_END = 3,  /* pass E: inverse 0,1 + Yukawa */
  WZ_K_P23_FFT = 4,  /* stand-alone DFT axes 2,3 */
  WZ_K_P01_INV = 5,  /* stand-alone inverse DFT axes 0,1 */
  WZ_K_P01_FWDCG = 6, /* pass A': x += alpha p, p <- r + beta p, twist + DFT axes 0,1 */
  WZ_K_P01_ENDCG = 7, /* pass E': inverse 0,1 + Yukawa, r -= alpha q, ||r||^2, stop rule */
  WZ_K_OTHER = 8,
  WZ_NKINDS = 9
};
wz_status wz_plan_profile(wz_plan *plan, int enable);
wz_status wz_plan_profile_read(wz_plan *plan, double *ms, unsigned long long *count);
const char *wz_kind_name(int kind);

#ifdef __cplusplus
}
#endif
#endif /* WZ_H_ */
