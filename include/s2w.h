/* s2w.h -- C ABI of the B200-native scale-discretised directional wavelet transform
 * on the sphere S^2 and the ball B^3 (hot path of arXiv:2402.01282).
 *
 * "P:n" = line n of PAPER.md (the paper text this library was written from).
 * Every transform entry point runs hand-written sm_100a CUDA kernels in fp64; there is
 * no CPU fallback.  Calls that need a device fail with S2W_ECUDA when none is present;
 * the kernel-build calls (s2wav_kernels, s2ball_kernels, s2ball_radial_nodes) are pure
 * host code and work without a GPU.
 *
 * Conventions:
 *   MW sampling at band-limit L: theta_t = pi(2t+1)/(2L-1), t = 0..L-1;
 *   phi_p = 2 pi p/(2L-1), p = 0..2L-2; gamma_g = 2 pi g/(2N-1), g = 0..2N-2.
 *   Y_lm = sqrt((2l+1)/4pi) d^l_{m0}(theta) e^{i m phi};  D^l_mn = e^{-i m alpha} d^l_mn(beta) e^{-i n gamma}
 *   (Eq. 47), d^l_mn(beta) = <l m| exp(-i beta J_y) |l n>.
 *   Scales j = J0..J, J = smallest integer with lambda^J >= L; kappa^j(l) = kappa_lambda(l / lambda^j)
 *   (Eq. A5); L_j = min(ceil(lambda^{j+1}), L) with multiresolution (Eq. 38), else L;
 *   scaling band-limit L_s = min(ceil(lambda^{J0}), L) with multiresolution, else L.
 *
 * Layouts: C row-major.  Signals [batch][theta][phi]; sphere coefficients per signal: the scaling block
 * [L_s][2L_s-1] first, then the scales ascending, each [2N-1 gamma][L_j beta][2L_j-1 alpha]
 * (s2w_plan_scale_shape gives shapes and offsets); consecutive signals of a batch are
 * s2w_plan_coeff_elems() apart.  With S2W_REAL elements are double, otherwise interleaved
 * complex128 (re, im).  Ball: signal [P shells][L][2L-1]; coefficients: scaling block [P][L][2L-1],
 * then scales ordered j' (radial) outer, j (angular) inner, each [P_j'][2N-1][L_j][2L_j-1].
 *
 * Ownership: the caller owns every signal, coefficient and workspace buffer (device memory);
 * a plan owns only its own tables and is immutable after creation.
 * Errors: every call returns 0 (S2W_OK) or a negative code; nothing throws across the ABI;
 * s2w_last_error() returns a thread-local message.
 */
#ifndef S2W_H
#define S2W_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct s2w_plan s2w_plan;

enum { S2W_OK = 0, S2W_EINVAL = -1, S2W_ENOMEM = -2, S2W_ECUDA = -3, S2W_EUNSUPPORTED = -4 };
enum { S2W_REAL = 1, S2W_PRECOMPUTE = 2, S2W_DH = 4, S2W_RECURSION = 8 };

/* ---- kernel-build calls (host only; Appendix A; "calculated and cached") ---- */

/* Number of wavelet scales: writes J (top scale index) for band-limit L and dilation lambda. */
int s2w_scale_count(int L, double lambda, int *J);

/* Sphere filters.  psi: host [J-J0+1][L][2N-1] complex (re,im interleaved), Psi^j_{l n} at
 * [j-J0][l][n+N-1] = sqrt((2l+1)/8pi^2) kappa^j(l) zeta_{l n} (Eq. A9 without p; zeta: Eq. A6);
 * phi: host [L], Phi_{l 0} = sqrt((2l+1)/4pi) sqrt(k_lambda(l/lambda^J0)) (Eq. A10).
 * Either pointer may be NULL.  EINVAL if L<1, N<1, N>L, lambda<=1, J0<0 or J0>J. */
int s2wav_kernels(double *psi, double *phi, int L, int N, double lambda, int J0);

/* Ball filters, stored separably (Eq. A9): kappa_l [J-J0+1][L] = kappa^j(l), kappa_p [J'-J0+1][P] =
 * kappa^{j'}(p) = kappa_nu(p/nu^{j'}), zeta [L][2N-1] complex, phi [P][L] = Phi_{l 0 p} =
 * sqrt((2l+1)/4pi) sqrt(a+b-ab), a = k_lambda(l/lambda^J0), b = k_nu(p/nu^J0)  (Eq. A10; reading R9).
 * J0 is used for both the angular and the radial lowest scale (reading R10). */
int s2ball_kernels(double *kappa_l, double *kappa_p, double *zeta, double *phi,
                   int L, int P, int N, double lambda_l, double lambda_p, int J0);

/* Gauss-Laguerre radial nodes (generalised, alpha = 2, reading R8): r [P] = tau x_i with L_P^(2)(x_i) = 0,
 * and q [P] = tau^3 w_i e^{x_i}, the weight that multiplies f(r_i) K_p(r_i) in the quadrature of Eq. 7. */
int s2ball_radial_nodes(double *r, double *q, int P, double tau);

/* ---- plans: the cached precomputed components ---- */

/* Sampling: by default every function on the sphere is sampled on the McEwen-Wiaux grid of its band-limit Lg: theta_t =
 * pi (2t+1)/(2Lg-1), t < Lg, phi_p = 2 pi p/(2Lg-1).  With S2W_DH ("sampling agnostic"; reading R19) sphere
 * plans use the Driscoll-Healy grid instead: 2Lg rings theta_t = pi (2t+1)/(4Lg), the same 2Lg-1 samples in phi / alpha;
 * signals are then [batch][2L][2L-1], coefficient blocks [2N-1][2L_j][2L_j-1] (s2w_plan_scale_shape reports n_theta =
 * 2L_j), and the theta quadrature is the diagonal Driscoll-Healy rule instead of the reweighting operator.  Scalar
 * (spin-0) sphere plans up to L = 1024; ball plans, spin plans and the adjoint calls return S2W_EUNSUPPORTED with it.
 * flags: S2W_REAL (signal and coefficients real); S2W_PRECOMPUTE: the Wigner-d values of every theta grid of the plan
 * are tabulated in device memory at creation ("simply precomputed"; 8 B per (ring, m >= 0, l, n): 21.5 GB at
 * L = 1024, N = 5) and the contractions stream that table through the FP64 tensor pipe instead of running the
 * recursion; S2W_ENOMEM if the table does not fit.  On McEwen-Wiaux grids with L_j <= 256 the table of the rings -> harmonic
 * direction carries the theta quadrature as well ((R d^l_mn)(theta_t), R the real symmetric reweighting operator of step
 * a2), so that step a2 is a plain transposing copy there.  Ball plans with L <= 256 take S2W_PRECOMPUTE by default (tens
 * of MB of tables shared by hundreds of shell columns); S2W_RECURSION: never precompute (on-the-fly recursion).
 * batch = number of independent signals per call (>= 1).  device = CUDA device ordinal.
 * Creation allocates device tables, runs set-up kernels and synchronises. */
int s2wav_plan_create(s2w_plan **out, int L, int N, double lambda, int J0, int multiresolution,
                      int flags, int batch, int device);
/* The same for a spin-s signal (spin fields: Eq. 1, Eq. 12; the formula of sY_lm is reading R2, Goldberg et al. 1967 convention -- the paper prints none): the signal and the scaling coefficients are expanded
 * in spin-weighted harmonics sY_lm = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi} (f_lm = 0 below l = |s|),
 * the wavelet coefficients on SO(3) are as in the scalar case.  spin != 0 needs a complex plan and |spin| < L
 * (S2W_EINVAL otherwise); spin = 0 is s2wav_plan_create. */
int s2wav_plan_create_spin(s2w_plan **out, int L, int N, double lambda, int J0, int multiresolution,
                           int flags, int batch, int device, int spin);
int s2ball_plan_create(s2w_plan **out, int L, int P, int N, double lambda_l, double lambda_p, int J0,
                       double tau, int flags, int device);
int s2w_plan_destroy(s2w_plan *plan);

/* Scale ranges: angular j = J0..J and (ball) radial j' = J0p..Jp (sphere: J0p = Jp = 0). */
int s2w_plan_scales(const s2w_plan *plan, int *J0, int *J, int *J0p, int *Jp);
/* Shape and element offset (within one signal's coefficient block) of scale (j, jp); j = -1 is the scaling block
 * (n_gamma = 1).  n_r is the number of radial shells (1 on the sphere). */
int s2w_plan_scale_shape(const s2w_plan *plan, int j, int jp, int *n_r, int *n_gamma, int *n_theta, int *n_phi,
                         size_t *offset_elems);
/* Elements (double or complex128) of one signal's coefficient block / of one signal. */
size_t s2w_plan_coeff_elems(const s2w_plan *plan);
size_t s2w_plan_signal_elems(const s2w_plan *plan);
/* Bytes of device scratch the plan-level transforms need (caller allocates, 256-byte aligned). */
size_t s2w_plan_workspace_bytes(const s2w_plan *plan);

/* ---- transforms on an explicit plan: asynchronous on `stream`, no allocation, no host sync ---- */
/* Analysis, Alg. 1 / Alg. 2: in = signal(s), out = coefficients. */
int s2w_plan_forward(const s2w_plan *plan, const void *in_dev, void *out_dev, void *work_dev, void *stream);
/* Synthesis, Alg. 1 / Alg. 2: in = coefficients, out = signal(s). */
int s2w_plan_inverse(const s2w_plan *plan, const void *in_dev, void *out_dev, void *work_dev, void *stream);

/* Adjoint transforms (the "differentiable" half of the paper, P:9: the maps are linear, so a
 * vector-Jacobian product is the adjoint map applied to the cotangent).  With <u, v> = sum conj(u_i) v_i over the stored
 * samples (pixels / coefficient samples, no quadrature weights):
 *   <A f, y> = <f, A^H y>    s2w_plan_forward_adjoint: in = coefficient-shaped y, out = signal-shaped A^H y;
 *   <S w, g> = <w, S^H g>    s2w_plan_inverse_adjoint: in = signal-shaped g,      out = coefficient-shaped S^H g,
 * A = s2w_plan_forward, S = s2w_plan_inverse.  Same buffers, layouts, workspace and stream semantics as those.
 * Sphere and ball plans, real or complex (on an S2W_REAL plan cotangents and results are real: the adjoint is the
 * transpose of the real matrix). */
int s2w_plan_forward_adjoint(const s2w_plan *plan, const void *in_dev, void *out_dev, void *work_dev, void *stream);
int s2w_plan_inverse_adjoint(const s2w_plan *plan, const void *in_dev, void *out_dev, void *work_dev, void *stream);

/* Harmonic-space taps used by the parity tests: forward spherical harmonic transform of the plan's signal(s)
 * (steps a1-a3 of DESIGN.md) writing flm [batch][L][2L-1] complex128 at [l][m+L-1] (ball: [P][L][2L-1], after the
 * radial transform: f_{lmp}), and its inverse. */
int s2w_plan_harmonic_forward(const s2w_plan *plan, const void *f_dev, void *flm_dev, void *work_dev, void *stream);
int s2w_plan_harmonic_inverse(const s2w_plan *plan, const void *flm_dev, void *f_dev, void *work_dev, void *stream);

/* s2w_plan_harmonic_forward for callers that cannot allocate device memory (code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): the same forward spherical harmonic transform (steps a1-a3; Eq. 2 / Eq. 13,
 * P:49 / P:116, by the separation of variables of P:378-384), same kernels, same f_dev / flm_dev layouts, but the scratch
 * (f_lm accumulator, ring spectra F, reweighted columns Ft) lives in a static device array of
 * S2W_STATIC_SCRATCH_BYTES inside the library instead of a caller workspace.  Every GPU that loads the library holds
 * that array until the process exits.  The call allocates nothing: no cudaMalloc / cudaFree, no stream, event or graph
 * creation (the first call on a device resolves the array's device address with cudaGetSymbolAddress).
 * Sphere plans only (S2W_EUNSUPPORTED for ball plans, and while s2w_timing_enable(1) is in force: the timers create
 * events).  S2W_EINVAL, with the sizes in s2w_last_error(), if the plan needs more scratch than the array holds:
 * 16 B x batch x (M L + 2 N M L), M = L (S2W_REAL) or 2L-1 (the F buffers are sized for the plan's largest stage, the N
 * rows of a top wavelet scale; each term rounded up to 16 elements) -- at batch = 1: L <= 836 (real, N = 1), 547 (real,
 * N = 3), 591 (complex, N = 1), 387 (complex, N = 3); use s2w_plan_harmonic_forward with a caller workspace beyond that.
 * All calls on a device share the one array, which keeps the previous call's contents; what must start at zero (the
 * f_lm accumulator) is cleared by the call itself on `stream`.  Two calls that overlap on the GPU (different streams,
 * or different host threads without stream ordering between them) RACE on the array: order them on one stream or
 * with events.  Asynchronous on `stream`; plan and buffers must belong to the current device. */
#define S2W_STATIC_SCRATCH_BYTES (32u << 20)
int s2w_plan_harmonic_forward_static(const s2w_plan *plan, const void *f_dev, void *flm_dev, void *stream);

/* ---- the transforms named by the problem statement: explicit arguments, device pointers.
 * The plan and its workspace are looked up in an internal cache keyed on the arguments (the first call builds them
 * and synchronises; later calls are asynchronous on `stream`). ---- */
int s2wav_forward(const void *f_dev, void *w_dev, int L, int N, double lambda, int J0, int multiresolution,
                  int flags, int batch, void *stream);
int s2wav_inverse(const void *w_dev, void *f_dev, int L, int N, double lambda, int J0, int multiresolution,
                  int flags, int batch, void *stream);
int s2ball_forward(const void *f_dev, void *w_dev, int L, int P, int N, double lambda_l, double lambda_p,
                   int J0, double tau, int flags, void *stream);
int s2ball_inverse(const void *w_dev, void *f_dev, int L, int P, int N, double lambda_l, double lambda_p,
                   int J0, double tau, int flags, void *stream);

/* Same, with HOST buffers: copies in, transforms, copies out, synchronises (the end-to-end path bench.py times). */
int s2wav_forward_host(const void *f_host, void *w_host, int L, int N, double lambda, int J0, int multiresolution,
                       int flags, int batch);
int s2wav_inverse_host(const void *w_host, void *f_host, int L, int N, double lambda, int J0, int multiresolution,
                       int flags, int batch);

int s2ball_forward_host(const void *f_host, void *w_host, int L, int P, int N, double lambda_l, double lambda_p,
                        int J0, double tau, int flags);
int s2ball_inverse_host(const void *w_host, void *f_host, int L, int P, int N, double lambda_l, double lambda_p,
                        int J0, double tau, int flags);

/* Drop every cached plan and workspace. */
/* ---- the generalised Fourier transforms on B^3 and H^4 as stand-alone calls ----
 * Z = K Y, the spherical-Laguerre transform (Eqs. 9-11): f [P][L][2L-1] samples on the P Gauss-Laguerre shells
 * r_i = tau x_i (s2ball_radial_nodes) x the MW grid  <->  f_{lmp} [P][L][2L-1] at [p][l][m+L-1]; double with S2W_REAL
 * in flags (the coefficients are complex128 either way), complex128 otherwise.
 * Q = K D, the Wigner-Laguerre transform on H^4 = R+ x SO(3) (Eqs. 24-25; "Q = K D"; reading R18: the
 * basis function is Q^l_{mnp} = K_p(r) D^l_{mn}(rho) with Eq. 4 unconjugated and Eq. 5 conjugated, as printed there):
 *   forward  f^l_{mnp} = int f(h) K_p(r) D^l_{mn}(rho) r^2 dr dOmega(rho)
 *   inverse  f(h) = sum_{l,m,n,p} (2l+1)/(8 pi^2) f^l_{mnp} K_p(r) D^{l*}_{mn}(rho)
 * f [P][2N-1][L][2L-1] complex128 = f(r_i, gamma_g, beta_t, alpha_a), gamma_g = 2 pi g/(2N-1), (beta_t, alpha_a) the MW
 * grid; fhat [2N-1][P][L][2L-1] complex128 at [n+N-1][p][l][m+L-1], |n| <= min(N-1, l), |m| <= l.  Exact for functions
 * band-limited at (L, N, P).  All pointers are device pointers owned by the caller; the calls are asynchronous on
 * `stream` after the first call with given parameters (which builds and caches the plan; calls that share a cached plan
 * are serialised).  Errors: S2W_EINVAL for L < 1, N < 1, N > L, N > 32, P < 1, tau <= 0, null pointers. */
int s2ball_z_forward(const void *f_dev, void *flmp_dev, int L, int P, double tau, int flags, void *stream);
int s2ball_z_inverse(const void *flmp_dev, void *f_dev, int L, int P, double tau, int flags, void *stream);
int s2ball_q_forward(const void *f_dev, void *fhat_dev, int L, int P, int N, double tau, void *stream);
int s2ball_q_inverse(const void *fhat_dev, void *f_dev, int L, int P, int N, double tau, void *stream);

int s2w_cache_clear(void);

/* FP64 pipe probe: runs a register-resident DFMA chain (kind 0) or an mma.sync m8n8k4 f64 chain (kind 1) on
 * `device` and writes the achieved TFLOP/s.  Used by bench.py to report the measured ALU peak. */
int s2w_probe_fp64(int kind, int device, double *tflops);

/* Per-class device timers (bench.py's roofline and step breakdown).  While enabled, every kernel launch of the
 * library is bracketed by a cudaEvent pair on its stream (no host synchronisation is added).  s2w_timing_read
 * synchronises on the recorded events, writes the summed device milliseconds and the launch count of each class
 * since the previous read into ms[nclass] / launches[nclass] (host arrays), and clears the record.  Classes:
 * 0 inverse Wigner contraction (a5, a7), 1 forward Wigner contraction (a3, a6), 2 ring FFT (a1), 3 (alpha, gamma)
 * FFT (a8), 4 theta reweighting (a2), 5 radial Laguerre contraction (a10), 6 everything else; classes >= nclass
 * are folded into the last one. */
#define S2W_TIMING_CLASSES 7
int s2w_timing_enable(int on);
int s2w_timing_read(double *ms, unsigned long long *launches, int nclass);

/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
unsigned long long s2w_launch_count(void);

const char *s2w_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
