// kernels.h -- host-callable launchers of the CUDA kernels (ring_fft.cu, wigner.cu, radial.cu).
#pragma once
#include <cuda_runtime.h>

#include "../../include/s2w.h"
#include "common.cuh"

namespace s2w {

#define S2W_MAX_N 32                 // directionality limit: 2N-1 <= 63 gamma samples
#define S2W_MAX_ROWS (2 * S2W_MAX_N)  // rows n handled by one launch

struct FftTab;
struct RwTab;

// rows (values of n) one SO(3) FFT launch works on
struct So3Args {
    int N;                       // directionality: 2N-1 gamma samples
    int nn;                      // number of rows
    int nrows;                   // rows per signal in the F array
    int n_val[S2W_MAX_ROWS];     // n
    int n_row[S2W_MAX_ROWS];     // row index of n in F
    int n_rowm[S2W_MAX_ROWS];    // row index of -n in F
    const size_t *sig_off;       // device array [batch]: element offset of signal b's coefficient block, or null:
                                 // b * sig_stride (the ball's stacked shells of all radial scales j' are not equidistant)
    int f_transposed;            // synthesis side only, where so3_fwd_writes_transposed() says so: F is written as
                                 // [b][row][m][t] (the forward contraction's input layout) instead of [b][row][t][m]
};
// element offset of signal b's block in the pixel-side array
__host__ __device__ inline size_t so3_base(const So3Args &A, int b, size_t sig_stride)
{
    return A.sig_off ? A.sig_off[b] : (size_t)b * sig_stride;
}

struct RwArgs {
    int nn, nrows, Md, isReal;
    int n_val[S2W_MAX_ROWS];
    int n_row[S2W_MAX_ROWS];
};

// one launch of the on-the-fly Wigner contraction (steps a3, a5, a6, a7)
//
// Rings are handled in GROUPS of 32 (one warp lane each): the rings of each hemisphere are sorted by |cos beta|
// (equator first); group 2j holds north rings 32j..32j+31 of that order, group 2j+1 the south ones.  All rings of a
// group start the recursion at the same degree gstart (monotone non-decreasing in j), with seeds stored at that degree.
struct WigArgs {
    int Lg;        // band-limit of the theta grid (|m| < Lg, l < Lg)
    int nt;        // rings of the grid, t = 0..nt-1: Lg (McEwen-Wiaux) or 2 Lg (Driscoll-Healy)
    int Lfull;     // band-limit of the plan (l-stride of flmT, extent of the coefficient table)
    int B;         // signals
    int isReal;    // harmonic arrays hold m >= 0 only
    int nn;        // number of n values
    int nrows;     // rows per signal in F
    int lmin;      // first l with a non-zero filter entry
    int G;         // ring groups (even)
    int n_val[S2W_MAX_ROWS], n_tab[S2W_MAX_ROWS], n_row[S2W_MAX_ROWS], n_rowm[S2W_MAX_ROWS], n_filtm[S2W_MAX_ROWS];
    size_t tri;                 // entries per n in the coefficient table: Lfull (Lfull+1)/2
    const double *coef;         // [ntab][tri][4]: (alpha, gamma, e_N, e_S) of the step l -> l+1 at packed (m, l)
    const int *gstart;          // [ntab][Lg (m)][G]: first degree at which group g is active
    const double2 *dseed;       // [ntab][Lg (m)][32 G]: (d~^{gstart}, u~_{gstart-1}) per ring slot
    const double *yv;           // [32 G] 1 - |cos beta| per ring slot (0 for empty slots)
    const int *ring;            // [32 G] ring index t of the slot, -1 if empty
    const double *dtab;         // precomputed-kernel variant: [ntab][tri_g][32 G] d^l_mn(beta) per ring slot, else null
    size_t tri_g;               // Lg (Lg + 1) / 2
    int dense;                  // forward direction, dtab = the quadrature-folded table (launch_wigner_table_fold): every ring
                                // group is active from l = max(m, |n|) on (no group starts), the input is F transposed, NOT reweighted
    const cplx *filt;           // [nn][Lg] filter applied to row q at degree l
    // two scales sharing one recursion (same grid, same rows n; at most 2 complex columns): the second scale's filter,
    // support start (>= lmin) and array; null / unused otherwise
    const cplx *filt2;
    int lmin2;
    cplx *F2;
    cplx *flmT;                 // [B][Mfull][Lfull]  f_{l m} stored m-major; Mfull = Lfull (real) or 2 Lfull - 1
    cplx *F;                    // inverse direction: output [B][nrows][Lg][Md], Md = Lg (real) or 2 Lg - 1;
                                // forward direction: input, transposed [B][nrows][Md][Lg]
};

void set_error(const std::string &msg);

// S2W_PRECOMPUTE on small grids: fold the theta quadrature (the reweighting operator R_sigma of DESIGN.md 6.3, real and
// symmetric) into the table of one n: X[l][t][m] = d^l_mn(theta_t) (gather), Y = R X per column by the reweighting kernels,
// dtab_rw = Y in the table's layout (scatter).  sum_t d(theta_t) (R F)(theta_t) = sum_t (R d)(theta_t) F(theta_t).
int launch_wigner_table_gather(const double *dtab, size_t tri_g, int tab, int n, int Lg, int nt, int G, const int *ring, cplx *X,
                               cudaStream_t st);
int launch_wigner_table_scatter(const cplx *Y, double *dtab_rw, size_t tri_g, int tab, int n, int Lg, int nt, int G,
                                const int *ring, cudaStream_t st);
int launch_twiddles(cplx *tw, int Mtab, cudaStream_t st);
int launch_fft_tables(const FftTab &T, cplx *chirp, cplx *rw_in1, cplx *rw_out1, cplx *rw_in3, cplx *rw_out3,
                      cplx *bhat_m, cplx *bhat_p, cplx *what, cudaStream_t st);
// pixel-side arrays: signal b starts sig_stride elements after signal b-1; rows of Lg rings each
int launch_ring_fwd(bool real, const void *in, cplx *out, int B, int Lg, size_t sig_stride, const FftTab &T,
                    cudaStream_t st);
int launch_ring_inv(bool real, const cplx *in, void *out, int B, int Lg, size_t sig_stride, const FftTab &T,
                    cudaStream_t st);
int launch_so3_inv(bool real, const cplx *F, void *W, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st);
// whether launch_so3_fwd honours So3Args::f_transposed for these arguments (only the prime-factor kernels of the 255-sample
// grids do: the quadrature-folded table path of small grids then needs no transposing copy at all)
bool so3_fwd_writes_transposed(bool real, const So3Args &A, const FftTab &T);
int launch_so3_fwd(bool real, const void *W, size_t sig_stride, cplx *F, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st);
// a2: reads F[b][row][t][mi], writes the reweighted columns TRANSPOSED, Ft[b][row][mi][t] (what the forward Wigner
// contraction reads: ring data of one m contiguous)
int launch_reweight(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const FftTab &T, cudaStream_t st);
// dst[b][c][r] = w[r] src[b][r][c] (w = null: 1): layout change between F[n][t][m] and Ft[n][m][t]; with the Driscoll-Healy
// quadrature weights w[t] it is step a2 on a Driscoll-Healy grid
int launch_transpose(const cplx *src, cplx *dst, int R, int C, int nb, cudaStream_t st, const double *w = 0);
int launch_reweight_th(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const RwTab &R, cudaStream_t st);   // L >= 8, L <= 2048
int launch_fft_forward(cplx *data, const FftTab &T, cudaStream_t st);   // plan-time, in place, digit-reversed out
// the radix-16 core (fft16_kernels.cu), lengths 1024 / 2048 / 4096
int launch_fft16_forward(cplx *data, int M, cudaStream_t st);           // plan-time, in place, the core's own order out
int launch_fft16_spectrum(cplx *khat, int kind, int n, int M, cudaStream_t st);  // Bluestein kernel spectra (kind 0: -, 1: +)
int launch_so3_pair16(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch,
                      const FftTab &T, cudaStream_t st);                // a8, real signals, 2N-1 <= 9
int launch_reweight16(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const RwTab &R, cudaStream_t st);  // a2
int launch_ring16(bool fwd, bool real, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T,
                  cudaStream_t st);                                     // a1, M = 256 ... 4096
bool so3_c16_supported(const So3Args &A, const FftTab &T);            // a8, complex signals, <= 3 rows, M = 256 ... 1024
int launch_so3_c16(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st);
// a8, complex signals, <= 3 rows, 2 L_j - 1 = 255 = 3 x 5 x 17: prime-factor transform without twiddles (pfa255_kernels.cu)
bool so3_pfa255_supported(const So3Args &A, const FftTab &T);
int launch_so3_pfa255(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                      cudaStream_t st);

// a8, real signals, 2N-1 <= 9, 2 L_j - 1 = 4095 = 9 x 5 x 7 x 13: prime-factor transform without twiddles (pfa4095_kernels.cu)
bool so3_pfa4095_supported(const So3Args &A, const FftTab &T);
int launch_so3_pfa4095(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                       cudaStream_t st);

// plan creation on the grid of L_j = 1024 (2047 = 23 x 89 samples): fills the device table of the Rader spectra the
// prime-factor kernels of that grid use; until it has run on a device the grid stays on the Bluestein kernels there
int pfa2047_init(cudaStream_t st);
bool ring_pfa255_supported(bool real, const FftTab &T);              // a1, complex signals, the 255-sample grid
int launch_ring_pfa255(bool fwd, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T, cudaStream_t st);
bool ring_pfa4095_supported(bool real, const FftTab &T);             // a1, real signals, the 4095-sample grid
int launch_ring_pfa4095(bool fwd, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T, cudaStream_t st);

// plan-time: group start degrees and seeds from the range-extended values d^{l0}_{mn}(beta_t) = mant 2^expo ([ntab][Lg m][Lg t])
int launch_wigner_seeds(const double *mant, const int *expo, const double *coef, size_t tri, int Lfull, int Lg, int nt, int G,
                        const int *n_vals, int ntab, const double *yv, const int *ring, int *gstart, double2 *dseed,
                        cudaStream_t st);
int launch_wigner_seed_floor(const double *coef, size_t tri, int Lfull, int Lg, int G, int ntab, const double *yv,
                             const int *gstart, const double2 *dseed, int lfloor, int *gstart_f, double2 *dseed_f,
                             cudaStream_t st);
int launch_wigner_table(const double *coef, size_t tri, int Lfull, int Lg, int G, const int *n_vals, int ntab,
                        const double *yv, const int *gstart, const double2 *dseed, double *dtab, size_t tri_g,
                        cudaStream_t st);
// krange: device array, one [kbeg, kend) per 64-row tile of A (block-sparse stacked matrices), or null
int launch_radial(const double *A, int R, int K, const cplx *in, cplx *out, size_t cols, int Lfull, const double *win,
                  const double *wout, bool accumulate, cudaStream_t st, const int2 *krange = 0);
int launch_wigner_inverse(const WigArgs &A, cudaStream_t st);   // harmonic -> rings   (a5, a7)
int launch_wigner_forward(const WigArgs &A, cudaStream_t st);   // rings -> harmonic   (a3, a6), accumulates

int launch_flm_pack(const cplx *flm_user, cplx *flmT, int B, int L, bool real, cudaStream_t st);
int launch_flm_unpack(const cplx *flmT, cplx *flm_user, int B, int L, bool real, cudaStream_t st);
int launch_flm_pack_pm(const cplx *pos, const cplx *neg, cplx *flmT, int B, int L, cudaStream_t st);
int launch_flm_unpack_pm(const cplx *flmT, cplx *pos, cplx *neg, int B, int L, cudaStream_t st);

int probe_fp64(int kind, double *tflops);

}  // namespace s2w
