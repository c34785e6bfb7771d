/* libtm - C ABI of the B200-native coupled T-matrix multiple-scattering solver.
 *
 * Hot path of arXiv 2107.09879 (Appendix I.3-I.4): solve
 *        (I - T A) s = T p                                   (Eqs. I22 + I25)
 * for N scatterers with VSWF truncation lmax, L = 2 lmax (lmax+2) coefficients each, where
 *        A_ji = xi^T(x_j, x_i)  (j != i, same window),  A_jj = 0   (Eq. I21)
 * is the outgoing->regular translation (addition-theorem) operator, built on the fly and never stored
 * (PAPER.md:382-384), T = blockdiag(T_j) are the per-scatterer transition matrices (Eq. I9)
 * and p = a^(0) are the incident-field coefficients (Eq. I12).
 *
 * Conventions (part of the ABI):
 *   - time convention e^{-i w t}, outgoing waves h_l^(1)
 *   - mode (l, m, p), l = 1..lmax, m = -l..l, p in {0 (M-type), 1 (N-type)}
 *     flat index  idx = p*(L/2) + l*(l+1) - 1 + m                                (reading R1)
 *   - normalised associated Legendre functions WITHOUT Condon-Shortley phase     (reading R2)
 *   - every complex array in this API is interleaved double precision (tm_c64), row-major [n_scat][L]
 *   - every data pointer may be a HOST or a DEVICE pointer (resolved with cudaPointerGetAttributes)
 *     unless stated otherwise; the caller owns every buffer it passes; tm_set_* copy what they need.
 *   - all device work is enqueued on the stream given to tm_create; calls that return results to the
 *     caller synchronise that stream before returning.
 *   - return value: TM_OK (0); > 0 soft status (outputs valid); < 0 hard error (context unchanged,
 *     message from tm_last_error).  No exceptions cross the boundary.
 * There is no CPU fallback: every call that computes needs a CUDA device.
 */
#ifndef TM_H_
#define TM_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tm_ctx tm_ctx;
typedef struct { double re, im; } tm_c64;

enum { TM_FP64 = 0, TM_FP32 = 1, TM_MIXED = 2 };         /* internal compute precision of the solver:
   TM_MIXED = GMRES with iterative refinement: Krylov cycles (all-pairs kernel, basis, orthogonalisation) in fp32, the
   iterate, the right-hand side and the TRUE residual of every restart in fp64 - fp64-accurate solutions at close to the
   fp32 kernel's speed; everything outside tm_solve / tm_solve_adjoint runs in fp64 */
enum { TM_OK = 0, TM_NOT_CONVERGED = 1,
       TM_E_INVALID = -1, TM_E_OVERLAP = -2, TM_E_STATE = -3, TM_E_CUDA = -4, TM_E_NOMEM = -5 };
enum { TM_INC_PLANE = 0, TM_INC_GAUSS = 1, TM_INC_COEFFS = 2, TM_INC_JINC = 3 };
enum { TM_FIELD_E_SCA = 0, TM_FIELD_H_SCA = 1, TM_FIELD_E_INC = 2 };   /* H is returned as Z_b * H (reading R10) */
enum { TM_KERNEL_AUTO = 0, TM_KERNEL_GENERAL = 1, TM_KERNEL_COPLANAR = 2, TM_KERNEL_SYM3D = 3, TM_KERNEL_ROT3D = 4 };

/* Plane wave travelling along (beta = polar angle from +z, alpha = azimuth) with amplitude
 * A = A_beta * beta_hat + A_alpha * alpha_hat  (Eqs. II6-II7).
 * Normal incidence, x-polarised, unit amplitude: beta = 0, alpha = 0, A_beta = 1, A_alpha = 0. */
typedef struct { double beta, alpha; tm_c64 A_beta, A_alpha; } tm_plane_desc;

/* Gaussian beam along +z, one focus per window (reading R9 of DESIGN.md: the angular-spectrum machinery of
 * Eqs. II9-II17, with a Gaussian spectral weight).  Transverse field on the focal plane
 * (Ax, Ay) exp(-|x_T - focus_T|^2 / w0^2).  focus: HOST pointer [n_win][3].  n_beta: Gauss-Legendre nodes in
 * the polar angle; 0 -> 400 (reading R9), raised to k_b D_max beta_max / 2 + 40 when the largest source - scatterer
 * distance D_max of a window needs more (beyond ~125 wavelengths for a jinc source); an explicit value is used as given. */
typedef struct { const double *focus; double w0; tm_c64 Ax, Ay; int n_beta; } tm_gauss_desc;

/* Superposition of jinc sources per window - the paper's Nyquist decomposition of a band-limited incident field
 * (Eqs. II1-II17; reading R17).  Source s: flat angular spectrum inside the light cone,
 * centred at src_xyz[s] = (x_0, y_0, z_0), propagating along +z, transverse field on its plane
 * (Ax_s, Ay_s) J_1(k rho)/(k rho); window w owns the sources src_ptr[w] <= s < src_ptr[w+1].
 * amp_is_sample != 0: `amp` holds the SAMPLES (Ex, Ey)(x_s, y_s) of a band-limited field on the lambda/2 grid and the library
 * applies the Nyquist amplitude factor of reading R17 (a sample is carried by a source of amplitude (pi/2) x sample: the
 * ideal disc low-pass of the square lambda/2 lattice); 0: `amp` holds the source amplitudes themselves.
 * All pointers are HOST pointers.  n_beta: Gauss-Legendre nodes on [0, pi/2] (0 -> 400 or more, as in tm_gauss_desc). */
typedef struct { int n_src; const double *src_xyz; const tm_c64 *amp /* [n_src][2] */; const int *src_ptr /* [n_win+1] */;
                 int n_beta; int amp_is_sample; } tm_jinc_desc;

/* Caller-supplied incident coefficients p[n_scat][L] (host or device). */
typedef struct { const tm_c64 *p; } tm_coeffs_desc;

/* GMRES options (reading R13): x0 = 0, restarted GMRES(restart) with CGS2 orthogonalisation on
 * (I - T A) s = T p; stop when ||b - M x|| / ||b|| <= tol per window (true residual, recomputed at every
 * restart and at exit); at most max_iter Arnoldi steps per window. */
typedef struct {
  double tol;
  int    restart;
  int    max_iter;
  int    warm_start;      /* 0: start from x0 = 0.  1: the output array (s_out / lambda_out) holds an initial guess x0 on
                             entry - e.g. the solution of the previous optimisation step (the design
                             changes little between steps); the first residual is b - M x0, the stopping rule still
                             refers to ||b||.  Costs one extra operator application. */
} tm_solve_opts;

/* Per-window report. */
typedef struct {
  int    iterations;      /* Arnoldi steps taken by this window's solve                         */
  int    restarts;        /* restart cycles started                                             */
  int    converged;       /* 1 if rel_residual <= tol                                           */
  int    matvecs;         /* all-pairs operator applications (shared by all windows)            */
  double rel_residual;    /* true ||b - M x||_2 / ||b||_2 at exit                               */
  double seconds;         /* device time of the whole solve (CUDA events), same for all windows */
} tm_solve_info;

/* Create a context (scatterers at x_i with non-intersecting enclosing spheres).
 *   pos_xyz   [n_scat][3] doubles (host or device), units such that k_b * |x| is the phase
 *   win_ptr   HOST pointer [n_win+1], monotone, win_ptr[0] = 0, win_ptr[n_win] = n_scat; NULL (with
 *             n_win = 1) => one window.  Scatterers interact only inside their window (reading R16;
 *             independent Nyquist windows batched on one GPU).
 *   lmax      1..6 (generated kernels: coplanar when all z are equal, rotation-based 3-D otherwise)
 *   k_b       background wavenumber (wavelength 1 => 2 pi)
 *   precision TM_FP64 or TM_FP32 (API data stays fp64)
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the default stream
 * Errors: TM_E_INVALID (bad sizes, non-finite or coincident positions), TM_E_CUDA, TM_E_NOMEM. */
int tm_create(tm_ctx **out, int n_scat, const double *pos_xyz, int n_win, const int *win_ptr,
              int lmax, double k_b, int precision, void *cuda_stream);

/* Per-scatterer transition matrices s = T a (Eq. I9), given per type.
 *   diag_only != 0: T [n_types][L] (diagonal, e.g. Mie spheres); else T [n_types][L][L] row-major.
 *   type_of   [n_scat] ints (host or device), values in [0, n_types)
 *   r_enclosing  HOST [n_types] radii or NULL; when given, overlapping enclosing spheres inside a window
 *             => TM_E_OVERLAP (the paper's assumption).  O(N^2) check on the device. */
int tm_set_tmatrices(tm_ctx *ctx, int n_types, int diag_only, const tm_c64 *T, const int *type_of,
                     const double *r_enclosing);

/* Incident field -> coefficients p_j = a^(0)_j of every scatterer, computed on the device
 * (Eq. I12; kind selects tm_plane_desc / tm_gauss_desc / tm_coeffs_desc / tm_jinc_desc). */
int tm_set_incident(tm_ctx *ctx, int kind, const void *desc);

/* Copy the current incident coefficients p [n_scat][L] out (host or device). */
int tm_get_incident(tm_ctx *ctx, tm_c64 *p_out);

/* Forward solve (I - T A) s = T p by device-resident restarted GMRES.
 *   s_out [n_scat][L] (host or device); info: HOST [n_win] or NULL.
 * Returns TM_OK, TM_NOT_CONVERGED (best iterate returned), or an error.  TM_E_STATE before
 * tm_set_tmatrices / tm_set_incident. */
int tm_solve(tm_ctx *ctx, const tm_solve_opts *opts, tm_c64 *s_out, tm_solve_info *info);

/* Adjoint (plain transpose, Eq. IV9): (I - T A)^T lambda = w, with the same all-pairs kernel
 * through the identity A^T = P A P, P = (m -> -m) permutation (structural identity S3). */
int tm_solve_adjoint(tm_ctx *ctx, const tm_c64 *w, const tm_solve_opts *opts, tm_c64 *lambda_out,
                     tm_solve_info *info);

/* Several right-hand sides on ONE geometry - both polarisations of a plane wave, many sources on one layout
 * (PAPER.md:31-37); SURVEY.md 8(f) NEXT-3.  adjoint = 0: rhs [n_rhs][n_scat][L] are INCIDENT coefficients p_r, solved is
 * (I - T A) s_r = T p_r; adjoint = 1: rhs are weight vectors w_r, solved is (I - T A)^T lambda_r = w_r.  out [n_rhs][n_scat][L];
 * info: HOST [n_rhs][n_win] or NULL; rhs and out host or device.  The right-hand sides are solved TOGETHER: the geometry is
 * replicated as one set of windows per right-hand side on an auxiliary context (created at the first call for this n_rhs and kept,
 * n_rhs times the memory of ctx), every right-hand side keeps its own Krylov scalars and convergence mask, and every launch of
 * the batched solver is shared.  Same solutions as n_rhs separate solves (same iteration counts, 1e-15); measured gain on one
 * B200: 1.15x / 1.21x for n_rhs = 2 / 4 on a 32x32 lattice at lmax 3 (latency-bound), 1.00x / 1.04x on 56x56 at lmax 6
 * (all-pairs-bound) - DESIGN.md section 9.  The incident field of ctx itself (tm_set_incident) is not touched.
 * 1 <= n_rhs <= 64.  Returns as tm_solve (TM_NOT_CONVERGED if any right-hand side of any window did not converge). */
int tm_solve_multi(tm_ctx *ctx, int adjoint, int n_rhs, const tm_c64 *rhs, const tm_solve_opts *opts, tm_c64 *out,
                   tm_solve_info *info);

/* One operator application: y = (I - T A) x (transpose = 0) or y = (I - T A)^T x (transpose = 1).
 * transpose = 2: y = A x (bare all-pairs translation matvec, Eq. I21; no T needed).  Parity and throughput. */
int tm_matvec(tm_ctx *ctx, int transpose, const tm_c64 *x, tm_c64 *y);

/* Scattered fields at detector points (Eqs. I13/I24):
 *   E_sca(x) = sum_i sum_{lmp} s_{lmp;i} Phi_{lmp}(k_b (x - x_i)),  Z_b H_sca = -i sum s Phi_{l,m,1-p} (reading R10).
 *   pts [n_pts][3] doubles, s [n_scat][L], out [n_pts][3] Cartesian complex; all windows are summed
 *   (the paper sums the sub-region fields).  The outgoing waves of a scatterer are singular at its own centre:
 *   for a point that coincides with a centre that scatterer's term is left out (the field of all the others is returned).
 *   TM_FIELD_E_INC: the incident E field of the last tm_set_incident (plane wave, Gaussian beams or jinc sources; all
 *   sources of all windows summed; s is ignored and may be NULL; TM_E_STATE after TM_INC_COEFFS or before tm_set_incident),
 *   so that E_total = E_INC + E_SCA. */
int tm_fields(tm_ctx *ctx, int n_pts, const double *pts, const tm_c64 *s, int which, tm_c64 *out);

/* The same scattered fields through an entry point that ALLOCATES NOTHING - for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  No context: the caller passes inputs and outputs as
 * DEVICE pointers (pos_dev [n_scat][3], s_dev [n_scat][L], pts_dev [n_pts][3], out_dev [n_pts][3]; host pointers are refused,
 * nothing is copied), the kernels are enqueued on cuda_stream and the call returns WITHOUT synchronising (results are ready in
 * stream order).  The per-source-chunk partial sums - the scratch tm_fields takes from its context - live in a file-scope static
 * device array of 8 MiB that every GPU loading the library holds until exit.  Limits and rules:
 *   - n_pts <= 65536 per call (lmax 1..6, n_scat >= 1); larger point sets are REJECTED with TM_E_INVALID and a message from
 *     tm_fields_static_error() - split them or use tm_fields; there is no fallback allocation;
 *   - all calls on a device share the one array: calls that OVERLAP on the GPU (two streams, two host threads, graphs replayed
 *     concurrently) race on it and must be serialised by the caller; back-to-back calls on one stream are safe;
 *   - the array keeps the last call's contents; nothing needs clearing (every partial sum read is written first by the same call);
 *   - tm_fields_static_setup() resolves the array's device address for the CURRENT device (cudaGetSymbolAddress, once per
 *     device); tm_fields_static does it lazily, so call the set-up once per device before a stream capture begins.
 * Output equals tm_fields' (same kernels; bit-identical when both use the same number of source chunks).
 * which: TM_FIELD_E_SCA or TM_FIELD_H_SCA.  Returns TM_OK, TM_E_INVALID or TM_E_CUDA. */
int tm_fields_static_setup(void);
int tm_fields_static(int lmax, double k_b, int n_scat, const double *pos_dev, const tm_c64 *s_dev, int n_pts,
                     const double *pts_dev, int which, tm_c64 *out_dev, void *cuda_stream);
const char *tm_fields_static_error(void);      /* message of the calling thread's last failed tm_fields_static* call */

/* Device scratch.  tm_workspace_bytes: bytes tm_solve / tm_solve_adjoint need for these options (Krylov
 * basis etc.).  tm_set_workspace: hand in caller-allocated DEVICE memory (e.g. a torch tensor), 256-byte
 * aligned, which must outlive its use; without it the library allocates (and caches) its own. */
size_t tm_workspace_bytes(const tm_ctx *ctx, const tm_solve_opts *opts);
int tm_set_workspace(tm_ctx *ctx, void *dev_ptr, size_t bytes);

/* Force the all-pairs kernel variant (TM_KERNEL_*):
 *   COPLANAR  generated code, all z equal (refused with TM_E_INVALID otherwise); two parity halves for lmax <= 3,
 *             four mirror sectors with shared-memory accumulators for lmax 4..6
 *   ROT3D     generated code, arbitrary 3-D positions, every lmax: rotation - axial translation - rotation with the polar
 *             rotation as constant frame change - phase rotation - constant frame change (O(L^1.5) work per pair);
 *             lmax 4..6: warp-split organisation (register accumulators, instruction stream shared by the warps)
 *   SYM3D     generated code, arbitrary 3-D positions, lmax <= 3 (refused otherwise): direct pair-frame operator
 *   GENERAL   table-driven, arbitrary positions, lmax <= 6 (correct-by-table reference)
 * Default AUTO = COPLANAR if all z are equal, else ROT3D. */
int tm_set_kernel(tm_ctx *ctx, int kernel);
/* Which variant is active (TM_KERNEL_GENERAL, TM_KERNEL_COPLANAR, TM_KERNEL_SYM3D or TM_KERNEL_ROT3D). */
int tm_get_kernel(const tm_ctx *ctx);

/* Device time (ms, CUDA events on the context's stream) of the all-pairs kernel launches since the last
 * call with reset > 0, and their count: lets a caller attribute time without a profiler.  reset > 0 (re)starts TIMING MODE:
 * an event pair around every all-pairs launch; in timing mode a restart cycle is issued launch by launch.  reset < 0
 * leaves timing mode (the default) and zeroes the launch counters: the solvers then replay each full restart cycle of a window-sized problem as one CUDA
 * graph (windows of ~31^2 scatterers are launch-bound), and only the launch counts are maintained. */
int tm_kernel_time(tm_ctx *ctx, int reset, double *allpairs_ms, long long *allpairs_launches,
                   long long *total_launches);

/* Geometry sensitivities through one adjoint solve (Appendix IV, Eqs. IV7-IV9).  For the bilinear
 * functional J = w^T s (Eq. IV3/IV4) and lambda from tm_solve_adjoint(w), a geometry parameter p of scatterer j changes
 * only T_j, and   dJ/dp = lambda_j^T (dT_j/dp) T_j^{-1} s_j = lambda_j^T (dT_j/dp) (p_j + (A s)_j).
 *   dT      derivative of every TYPE's T-matrix with respect to its parameter, same layout as T in tm_set_tmatrices
 *   lambda, s  [n_scat][L] (host or device): adjoint and forward solutions
 *   out     [n_scat] complex: out[j] = lambda_j^T dT_{type(j)} (p_j + (A s)_j); for a parameter shared by a type, sum
 *           out over the sites of the type.  One all-pairs matvec + one small kernel.  Needs T and the incident field. */
int tm_grad_tmatrix(tm_ctx *ctx, const tm_c64 *dT, const tm_c64 *lambda, const tm_c64 *s, tm_c64 *out);

/* Position sensitivities through the same adjoint solve (Eqs. IV3-IV6, IV9):
 *   out[j][alpha] = lambda^T T (dA/dx_{j,alpha}) s  (+ lambda_j^T T_j dp_j/dx_{j,alpha} when dp is given)
 * = dJ/dx_{j,alpha} for J = w^T s at fixed w (the explicit term of Eq. IV6 - the detector overlap of the moved
 * scatterer's own waves - is the caller's, it does not involve the solver).  Identity S3 folds the row-block and
 * column-block parts of dA/dx_j into two all-pairs products with the DERIVATIVE of the translation operator,
 *   G_j = mu_j^T (d_alpha A s)_j + (P s_j)^T (d_alpha A P mu)_j ,  mu = T^T lambda,
 * and d_alpha A is ANALYTIC ("can be computed analytically"): differentiating the addition theorem with
 * respect to the destination centre gives  dA(d)/dd_alpha = k_b D^alpha A^ext(d),  A^ext = the translation operator with
 * destination rows up to lmax + 1 and D^alpha three constant sparse matrices (the gradient ladder of the regular
 * wavefunctions, generated at build time).  Cost: TWO all-pairs products at lmax + 1 for all 3 n_scat derivatives, on an
 * auxiliary context created at the first call and kept; planar layouts stay on the coplanar kernels (the z-derivative
 * sits in the constant matrix).  Every lmax of the API (1..6), any layout, every precision.
 *   lambda, s [n_scat][L]; dp [n_scat][3][L] or NULL (plane wave: dp = i k_alpha p); out [n_scat][3] complex. */
int tm_grad_positions(tm_ctx *ctx, const tm_c64 *lambda, const tm_c64 *s, const tm_c64 *dp, tm_c64 *out);

/* Host helper: d(diag T)/dR of the Mie T-matrix of tm_mie_tmatrix (Richardson-extrapolated central differences of the
 * closed form with the RELATIVE step 1e-3 R, so the accuracy - about 1e-10 relative - does not depend on the length
 * unit), out[L]. */
int tm_mie_tmatrix_dR(int lmax, double k_b, double radius, tm_c64 eps_r, tm_c64 *out);

/* Executed floating-point work of the active all-pairs kernel per ORDERED pair:
 * fp_instructions = FMA/MUL/ADD issue slots on the FP64 (or FP32) pipe, flop with FMA = 2.  Counted from the
 * generated straight-line code (coplanar kernel; per-pair geometry excluded, so rooflines are conservative) or
 * from the term table (general kernel). */
int tm_pair_cost(const tm_ctx *ctx, double *fp_instructions, double *flop);

/* Register-resident FMA microbenchmark on the current device (no memory traffic, 8 independent chains per
 * thread): the measured peak of the plain FP64 / FP32 pipe that the all-pairs kernel is bounded by.
 * precision TM_FP64 / TM_FP32, or TM_PEAK_FP64_TENSOR: chains of FP64 tensor-core instructions (DMMA m8n8k4), the bound a
 * dense-block multi-right-hand-side route would have; result in TFLOP/s (FMA = 2 flop).  Needs a CUDA device. */
enum { TM_PEAK_FP64_TENSOR = 3 };
int tm_measure_fma_peak(int precision, double *tflops, void *cuda_stream);

/* Host helper: diagonal of the Lorenz-Mie T-matrix of a homogeneous sphere (reading R11; closed form,
 * T_{l,p=0} = -b_l, T_{l,p=1} = -a_l), out[L] in flat mode order.  eps_r complex relative permittivity. */
int tm_mie_tmatrix(int lmax, double k_b, double radius, tm_c64 eps_r, tm_c64 *out);

/* Null-field (extended boundary condition) transition matrix of homogeneous, non-magnetic bodies of revolution about z
 * (the paper's meta-atoms are cylinders, Eqs. I10-I11), computed on the device:
 *     T = - B_rg B_out^{-1} ,
 *     B_{nu,mu} = int_S [ RPhi_{l'm'p'}(k_s x) x Psi_{l,-m,1-p}(k_b x) + (k_s/k_b) RPhi_{l'm'1-p'}(k_s x) x Psi_{l,-m,p}(k_b x) ] . n dS ,
 * Psi = RPhi for B_rg and the outgoing Phi for B_out, k_s = k_b sqrt(eps_r) (principal root).  Readings: R18 - Eq. I10 prints a
 * minus between the two terms, they add; R19 - the matrix built with the outgoing function (printed as P, Eq. I10a) is the
 * one inverted.  Both are fixed by the Lorenz-Mie limit (a sphere reproduces tm_mie_tmatrix) and the displaced sphere.
 * The surface is r = r(theta) (star-shaped about the origin), handed over discretised - the paper's "numerical
 * discretization" of the surface integrals: per shape n_nodes quadrature nodes theta[i] in (0, pi), r[i] > 0,
 * dr_dtheta[i] and the quadrature weight[i] in theta (e.g. Gauss-Legendre per smooth panel of the generatrix; the phi
 * integral is done analytically: T is block diagonal in m).  All four arrays [n_shapes][n_nodes], host or device.
 *   lmax_internal  truncation of the field expansions INSIDE the method (surface-field and test functions): the block
 *              systems are built and solved with l <= lmax_internal and the rows / columns with l <= lmax are returned.
 *              0 or lmax = the paper's setting (everything at lmax = 6); up to 12.  For the paper's tall
 *              silicon cylinders the lmax-6 result is far from converged near resonances
 *   eps_r      complex relative permittivity of the scatterer against the background, as in tm_mie_tmatrix (time convention
 *              e^{-i omega t}: Im eps_r >= 0 is a lossy medium; negative real eps_r and Im eps_r < 0 are refused)
 *   T_out      [n_shapes][L][L] row-major, s = T a, flat mode order R1 - the `T` of tm_set_tmatrices(diag_only = 0);
 *              host or device, fully written (zeros outside the m = m' blocks)
 * One launch for all shapes (a library of radii / heights is one call); synchronises cuda_stream before returning.
 * Errors: TM_E_INVALID (sizes, lmax > 6, lmax_internal not 0 and outside [lmax, 12], eps_r = 0 / negative real / Im < 0, r <= 0, theta outside (0, pi)), TM_E_CUDA, TM_E_NOMEM. */
int tm_nullfield_tmatrix(int lmax, int lmax_internal, double k_b, tm_c64 eps_r, int n_shapes, int n_nodes, const double *theta, const double *r,
                         const double *dr_dtheta, const double *weight, tm_c64 *T_out, void *cuda_stream);

/* d T / d(shape parameter) of the null-field T-matrix ("T_j depends on the geometry parameters of scatterer
 * j"; the `dT` of tm_grad_tmatrix).  The caller hands over, per shape, FOUR generatrices - the surface at parameter values
 * p + h, p - h, p + h/2, p - h/2, in this order - laid out [n_shapes][4][n_nodes]; the library computes the four T-matrices in
 * the same launch as tm_nullfield_tmatrix and combines them on the device into the Richardson-extrapolated central
 * difference (4 D(h/2) - D(h)) / 3, D(h) = (T(p+h) - T(p-h)) / 2h  (error O(h^4)).  A stated deviation from an analytic
 * dT/dp, like tm_mie_tmatrix_dR.  dT_out [n_shapes][L][L], host or device.  Errors as tm_nullfield_tmatrix, and h <= 0. */
int tm_nullfield_dtmatrix(int lmax, int lmax_internal, double k_b, tm_c64 eps_r, int n_shapes, int n_nodes, const double *theta, const double *r,
                          const double *dr_dtheta, const double *weight, double h, tm_c64 *dT_out, void *cuda_stream);

/* T-matrix look-up table ("we are setting up a lookup table for the transition matrices and interpolating between
 * them, this derivative can be numerically approximated using the same lookup table"; Fig. 2c).
 * Given the T-matrices of a scatterer family at n_tab >= 4 values p_tab[0] < p_tab[1] < ... of one geometry parameter (a radius;
 * the nodes need not be equidistant) - T_tab [n_tab][n_entry], n_entry = L (diagonal T) or L*L (full T), e.g. from
 * tm_mie_tmatrix / tm_nullfield_tmatrix - computes on the device, for n_out parameter values p[j],
 *     T_out[j][e]  = sum_{a=0..3} w_a(p[j])  T_tab[i0 + a][e]          (cubic Lagrange polynomial through the four nodes
 *     dT_out[j][e] = sum_{a=0..3} w_a'(p[j]) T_tab[i0 + a][e]           i0 .. i0+3 around the interval that holds p[j])
 * with i0 = clamp(i - 1, 0, n_tab - 4) for p_tab[i] <= p[j] < p_tab[i+1] (last interval closed on the right): reading R20 of
 * DESIGN.md; dT_out is the exact derivative of the interpolant, so gradients are consistent with the interpolated forward model.
 * T_out [n_out][n_entry] is what tm_set_tmatrices takes with type_of[j] = j, dT_out what tm_grad_tmatrix takes; dT_out may be NULL.
 * Every pointer may be host or device memory (device arrays are used in place, host arrays are staged); the call returns after
 * the work on cuda_stream has finished.  Errors: TM_E_INVALID (n_tab < 4, nodes not finite / not strictly increasing, any p[j]
 * outside [p_tab[0], p_tab[n_tab-1]] or NaN - nothing is extrapolated; the outputs are then unspecified), TM_E_NOMEM, TM_E_CUDA. */
int tm_ttable_interp(int n_tab, const double *p_tab, long long n_entry, const tm_c64 *T_tab, int n_out, const double *p, tm_c64 *T_out,
                     tm_c64 *dT_out, void *cuda_stream);

/* Memory (the solver state is what limits the problem size on one GPU).  All device memory of the
 * library comes from the current device's stream-ordered pool (cudaMallocAsync) with the release threshold raised, so a
 * context created and destroyed once per optimisation step re-uses the same physical memory.  This call hands the cached,
 * unused memory back to the driver (e.g. before another library needs it); live contexts are not affected.
 * Returns TM_OK or TM_E_CUDA. */
int tm_release_cached_memory(void);

/* Debug aid: guard bands around every INTERNAL device buffer (a stand-in for compute-sanitizer's memcheck where that tool cannot
 * run).  enable = 1: every device block the library allocates FROM NOW ON (contexts created afterwards, their scratch, tables,
 * Krylov state) carries a 4 KiB margin of sentinel bytes on each side; enable = 0: new blocks are plain again (blocks already
 * guarded stay so until freed); enable < 0: query only.  Every call synchronises the device, compares the margins of all live
 * guarded blocks and returns the number of damaged margins found so far, including those of blocks freed in the meantime
 * (0 = no kernel wrote outside an internal buffer); *n_blocks (may be NULL) receives how many guarded blocks have been handed
 * out.  Costs 8 KiB per block and nothing when off (the default).  Not thread-safe against concurrent compute calls on other host
 * threads.  Returns a count >= 0 or TM_E_CUDA. */
long long tm_debug_guards(int enable, long long *n_blocks);

int tm_num_modes(int lmax);                    /* L = 2 lmax (lmax + 2) */
const char *tm_last_error(const tm_ctx *ctx);  /* ctx may be NULL: last error of tm_create */
void tm_destroy(tm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* TM_H_ */
