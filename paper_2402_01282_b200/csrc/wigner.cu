// wigner.cu -- on-the-fly Wigner-d recursion fused with the l-contraction and the filter multiply
// (steps a3-a7 of DESIGN.md; "dominated by the Wigner transforms").
//
//   inverse direction (a5, a7):  F_mn(beta_t) = sum_l d^l_mn(beta_t) G_n(l) f_lm                     (Eq. 5/47)
//   forward direction (a3, a6):  f_lm += G'_n(l) sum_t d^l_mn(beta_t) h_mn(beta_t)                   (Eq. 4/48)
//
// d^l_mn(beta) follows the three-term recursion in l (Varshalovich et al., cited P:434)
//   d^{l+1} = (alpha_l cos(beta) - beta_l) d^l - gamma_l d^{l-1},
//   alpha_l = (l+1)(2l+1)/sqrt(((l+1)^2-m^2)((l+1)^2-n^2)),  beta_l = alpha_l m n/(l(l+1)),
//   gamma_l = alpha_l sqrt((l^2-m^2)(l^2-n^2))/(l(2l+1)),
// evaluated in DIFFERENCE FORM.  Near the poles consecutive d^l are nearly equal (north) or nearly opposite (south),
// and the plain recursion doubles-integrates its rounding errors (error ~ l^1.5 eps: 1e-11 at l = 1000).
// With y = 1 - |cos beta| and, for southern rings, the mirrored sequence d~^l = (-1)^l d^l (which obeys the same
// recursion with cos(beta) -> -cos(beta), beta_l -> -beta_l):
//   u_l = gamma_l u_{l-1} + (e - alpha_l y) d~^l,      d~^{l+1} = d~^l + u_l,
//   e = e_N = alpha_l - gamma_l - 1 - beta_l (north),  e = e_S = alpha_l - gamma_l - 1 + beta_l (south),
// where e_N, e_S are tabulated from long double (they vanish exactly where d is constant in l) and y carries the
// angle with full relative precision.  4 FP64 operations per step, shared by all columns of the block.
//
// Rings are processed in groups of 32 (a warp, one lane per ring): each hemisphere's rings sorted by |cos beta|,
// group 2j = north rings 32j.., group 2j+1 = south rings 32j...  A group starts at the first degree at which any of
// its rings has reached |d| >= 2^-70 (the exponentially small start of the recursion is neither computed nor able to
// underflow); the start is warp-uniform and monotone in j, so a warp that owns groups j0 < j1 < ... runs phases with
// 1, 2, ... active groups and no per-step checks.  Even warps own north groups, odd warps south groups.
//
// Inverse direction: DFMA, accumulators in registers.  Forward direction: the sum over rings is done by the FP64
// tensor pipe (mma.sync.m8n8k4.f64: D[col][l] += h^T[col][ring] d[ring][l]), the d values of an l-octet passing
// through a warp-private shared-memory transpose.
#include <climits>
#include <cstdlib>

#include "kernels.h"
#include "smem_attr.cuh"

namespace s2w {

namespace {

#define WIG_TL 64   // l-tile of the inverse kernels (the recursion kernel uses 256 on grids with several groups per warp)
#define FWD_TILE(R) ((R) == 1 ? 64 : 256)  // l-tile of the forward kernel: short on small grids, long on large ones
#define RAMP_THRESHOLD_EXP (-70)

__device__ __forceinline__ size_t tri_off(int m, int Lfull) { return (size_t)m * Lfull - ((size_t)m * (m - 1)) / 2 - m; }

struct NList {
    int v[S2W_MAX_ROWS];
};

// one recursion step l -> l+1 (see the header): ag = (alpha_l, gamma_l), e = e_N or e_S
__device__ __forceinline__ void wig_step(double &d, double &u, double y, double alpha, double gamma, double e)
{
    const double eps = fma(-alpha, y, e);
    u = fma(gamma, u, eps * d);
    d += u;
}

// ---------------------------------------------------------------------------------------------------------------
// plan-time: group start degrees and seeds.  One warp per (group, m, table n); lane = ring slot.
//   pass 0: every ring runs the range-extended recursion from its seed d^{l0} = mant 2^expo until |d| >= 2^-70;
//           the group start is the minimum over the warp.
//   fix   : suffix minimum over the groups of a hemisphere (monotone starts).
//   pass 1: every ring runs to the group start and stores (d~, u~) there.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) wigner_seed_kernel(const double *__restrict__ mant, const int *__restrict__ expo,
                                                        const double *__restrict__ coef, size_t tri, int Lfull, int Lg,
                                                        int nt, int G, NList nl, const double *__restrict__ yv,
                                                        const int *__restrict__ ring, int *__restrict__ gstart,
                                                        double2 *__restrict__ dseed, int pass)
{
    const int g = blockIdx.x, m = blockIdx.y, tab = blockIdx.z, lane = threadIdx.x;
    const int k = g * 32 + lane;
    const int t = ring[k];
    const int n = nl.v[tab], an = n < 0 ? -n : n;
    const int l0 = m > an ? m : an;
    const bool south = (g & 1) != 0;
    const size_t gidx = ((size_t)tab * Lg + m) * G + g;
    const int target = pass == 0 ? Lg : gstart[gidx];
    double d = 0.0, u = 0.0;
    int e = 0, l = l0;
    if (t >= 0 && l0 < Lg) {
        const size_t idx = ((size_t)tab * Lg + m) * nt + t;
        d = mant[idx];
        if (south && (l0 & 1)) d = -d;
        u = d;
        e = expo[idx];
    }
    int ls = Lg;
    if (d != 0.0) {
        const double *c = coef + ((size_t)tab * tri + tri_off(m, Lfull)) * 4;
        const double y = yv[k];
        while (l < target) {
            if (pass == 0 && e + ilogb(d) >= RAMP_THRESHOLD_EXP) break;
            const double4 q = *reinterpret_cast<const double4 *>(c + 4 * (size_t)l);
            wig_step(d, u, y, q.x, q.y, south ? q.w : q.z);
            ++l;
            if (fabs(d) > 0x1p300 || fabs(u) > 0x1p300) {
                d *= 0x1p-300;
                u *= 0x1p-300;
                e += 300;
            }
        }
        if (d != 0.0) ls = l;
    }
    if (pass == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const int other = __shfl_xor_sync(0xffffffffu, ls, o);
            ls = other < ls ? other : ls;
        }
        if (lane == 0) gstart[gidx] = ls;
    } else {
        double2 s = make_double2(0.0, 0.0);
        if (target < Lg && d != 0.0) s = make_double2(ldexp(d, e), ldexp(u, e));
        dseed[((size_t)tab * Lg + m) * (size_t)(32 * G) + k] = s;
    }
}

// plan-time: start degrees and seeds of a stage whose filter support begins at lfloor > 0.  The recursion of a group
// that would start below lfloor has nothing to contribute there, so it is run once, here, from the group start to
// lfloor (the same steps the transform kernels would take) and the state is stored as that stage's seed.
__global__ void __launch_bounds__(32) wigner_seed_floor_kernel(const double *__restrict__ coef, size_t tri, int Lfull, int Lg,
                                                              int G, const double *__restrict__ yv,
                                                              const int *__restrict__ gstart,
                                                              const double2 *__restrict__ dseed, int lfloor,
                                                              int *__restrict__ gstart_f, double2 *__restrict__ dseed_f)
{
    const int g = blockIdx.x, m = blockIdx.y, tab = blockIdx.z, lane = threadIdx.x;
    const int k = g * 32 + lane;
    const size_t gidx = ((size_t)tab * Lg + m) * G + g;
    const size_t sidx = ((size_t)tab * Lg + m) * (size_t)(32 * G) + k;
    const int gs = gstart[gidx];
    int target = gs;
    if (gs < Lg && gs < lfloor) target = lfloor < Lg ? lfloor : Lg;
    double2 s = dseed[sidx];
    if (target > gs) {
        const double *c = coef + ((size_t)tab * tri + tri_off(m, Lfull)) * 4;
        const double y = yv[k];
        const bool south = (g & 1) != 0;
        double d = s.x, u = s.y;
        for (int l = gs; l < target; ++l) {
            const double4 q = *reinterpret_cast<const double4 *>(c + 4 * (size_t)l);
            wig_step(d, u, y, q.x, q.y, south ? q.w : q.z);
        }
        s = make_double2(d, u);
    }
    dseed_f[sidx] = s;
    if (lane == 0) gstart_f[gidx] = target;
}

__global__ void wigner_start_fix_kernel(int *__restrict__ gstart, int G, int count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    int *gs = gstart + (size_t)i * G;
    for (int hemi = 0; hemi < 2; ++hemi) {
        int run = INT_MAX;
        for (int j = G / 2 - 1; j >= 0; --j) {
            const int v = gs[2 * j + hemi];
            run = v < run ? v : run;
            gs[2 * j + hemi] = run;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// column bookkeeping shared by both directions
// ---------------------------------------------------------------------------------------------------------------
struct ColInfo {
    int b;       // signal
    int minus;   // 1: the (-m,-n) column of a complex signal
    bool valid;
};
__device__ __forceinline__ ColInfo col_info(const WigArgs &A, int cc)
{
    ColInfo c;
    const int CT = A.isReal ? A.B : 2 * A.B;
    c.valid = cc < CT;
    c.b = A.isReal ? cc : (cc >> 1);
    c.minus = A.isReal ? 0 : (cc & 1);
    return c;
}

// stage the recursion coefficients of degrees lt..lt+TL-1 of row (m, tab): s_ag = (alpha, gamma), s_e = (e_N, e_S)
template <int TL>
__device__ __forceinline__ void stage_coef(const double *__restrict__ crow, int lt, int l0, int Lg, double2 *s_ag,
                                           double2 *s_e)
{
    for (int i = threadIdx.x; i < TL; i += blockDim.x) {
        const int l = lt + i;
        double4 q = make_double4(0.0, 0.0, 0.0, 0.0);
        if (l >= l0 && l < Lg) q = *reinterpret_cast<const double4 *>(crow + 4 * (size_t)l);
        s_ag[i] = make_double2(q.x, q.y);
        s_e[i] = make_double2(q.z, q.w);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// inverse direction: one block per (m >= 0, column chunk) covering all rings; warp w owns groups w, w+W, w+2W, ...
// (slot r = group r W + w), lane = ring.  Loops over the n of the launch.
// ---------------------------------------------------------------------------------------------------------------
// NCT columns in shared memory per degree, the first NACC of them accumulated (0: recursion only)
template <int NCT, int R, int RA, int NACC>
__device__ __forceinline__ void inv_range(int la, int lb, int lt, int hemi, const double2 *s_ag, const double2 *s_e,
                                          const double *s_X, const double (&y)[R], double (&d)[R], double (&u)[R],
                                          double (&acc)[R][NCT])
{
    const double *se = reinterpret_cast<const double *>(s_e) + hemi;
    for (int l = la; l < lb; ++l) {
        const int i = l - lt;
        const double2 ag = s_ag[i];
        const double e = se[2 * i];
        double xv[NACC > 0 ? NACC : 1];
#pragma unroll
        for (int c = 0; c < NACC; ++c) xv[c] = s_X[i * NCT + c];
#pragma unroll
        for (int r = 0; r < RA; ++r) {
#pragma unroll
            for (int c = 0; c < NACC; ++c) acc[r][c] = fma(d[r], xv[c], acc[r][c]);
            wig_step(d[r], u[r], y[r], ag.x, ag.y, e);
        }
    }
}

template <int NCT, int R, int NACC>
__device__ __forceinline__ void inv_dispatch(int ra, int la, int lb, int lt, int hemi, const double2 *s_ag,
                                             const double2 *s_e, const double *s_X, const double (&y)[R],
                                             double (&d)[R], double (&u)[R], double (&acc)[R][NCT])
{
    if (R >= 4 && ra == 4) return inv_range<NCT, R, (R >= 4 ? 4 : R), NACC>(la, lb, lt, hemi, s_ag, s_e, s_X, y, d, u, acc);
    if (R >= 3 && ra == 3) return inv_range<NCT, R, (R >= 3 ? 3 : R), NACC>(la, lb, lt, hemi, s_ag, s_e, s_X, y, d, u, acc);
    if (R >= 2 && ra == 2) return inv_range<NCT, R, (R >= 2 ? 2 : R), NACC>(la, lb, lt, hemi, s_ag, s_e, s_X, y, d, u, acc);
    if (ra >= 1) return inv_range<NCT, R, 1, NACC>(la, lb, lt, hemi, s_ag, s_e, s_X, y, d, u, acc);
}

// NS = 2 (batches of at most 2 complex columns): two wavelet scales that live on the same theta grid with the same rows
// n -- the two top scales of a multiresolution transform -- share ONE recursion: NC columns of scale A (filter A.filt,
// support from A.lmin, output A.F) and NC columns of scale B (A.filt2, A.lmin2 >= A.lmin, A.F2).  With few columns the
// recursion (4 FP64 instructions per step) outweighs the accumulation (NC), so sharing it is worth up to a third.
template <int NC, int R, int MAXT, int NS>
__global__ void __launch_bounds__(MAXT, (MAXT <= 256 ? 2 : 1)) wigner_inverse_kernel(WigArgs A)
{
    constexpr int NCT = NC * NS;
    constexpr int TL = R == 1 ? 64 : 256;  // l-tile: long tiles (fewer barriers) on the large grids, short on small ones
    __shared__ double2 s_ag[TL];
    __shared__ double2 s_e[TL];
    __shared__ double s_X[2][TL * NCT];  // [0]: X_l, [1]: (-1)^l X_l (southern warps)

    const int m = blockIdx.x, chunk = blockIdx.y;
    const int Lg = A.Lg, Lfull = A.Lfull, G = A.G;
    const int Md = A.isReal ? Lg : 2 * Lg - 1;
    const int Mfull = A.isReal ? Lfull : 2 * Lfull - 1;
    const int T = blockDim.x, W = T >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, hemi = warp & 1;

    int tr[R];
    double y[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int g = r * W + warp;
        tr[r] = g < G ? A.ring[g * 32 + lane] : -1;
        y[r] = g < G ? A.yv[g * 32 + lane] : 0.0;
    }

    for (int q = 0; q < A.nn; ++q) {
        const int n = A.n_val[q], an = n < 0 ? -n : n;
        const int l0 = m > an ? m : an;
        if (l0 >= Lg) continue;
        const int tab = A.n_tab[q];
        const double *crow = A.coef + ((size_t)tab * A.tri + tri_off(m, Lfull)) * 4;
        const int *gsrow = A.gstart + ((size_t)tab * Lg + m) * G;
        const double2 *seedrow = A.dseed + ((size_t)tab * Lg + m) * (size_t)(32 * G);
        const double sgn = ((m + n) & 1) ? -1.0 : 1.0;
        const int lacc = l0 > A.lmin ? l0 : A.lmin;                        // first l that contributes (scale A)
        const int lacc2 = NS > 1 ? (l0 > A.lmin2 ? l0 : A.lmin2) : lacc;    // ... to scale B

        int gs[R + 1];
        double d[R], u[R], acc[R][NCT];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int g = r * W + warp;
            gs[r] = g < G ? gsrow[g] : INT_MAX;
            d[r] = 0.0;
            u[r] = 0.0;
#pragma unroll
            for (int c = 0; c < NCT; ++c) acc[r][c] = 0.0;
        }
        gs[R] = INT_MAX;
        // first degree any group of the block needs: groups 0 and 1 start first
        int bmin = gsrow[0];
        if (G > 1 && gsrow[1] < bmin) bmin = gsrow[1];
        if (bmin < l0) bmin = l0;

        for (int lt = bmin & ~(TL - 1); lt < Lg; lt += TL) {
            __syncthreads();
            stage_coef<TL>(crow, lt, l0, Lg, s_ag, s_e);
            for (int i = threadIdx.x; i < TL * (NCT / 2); i += T) {
                const int k = i / TL, ll = i % TL;  // consecutive threads -> consecutive l (coalesced)
                const int sc = k / (NC / 2), kk = k - sc * (NC / 2);
                const int l = lt + ll;
                const ColInfo ci = col_info(A, chunk * (NC / 2) + kk);
                cplx X = cmake(0.0, 0.0);
                if (l >= (sc ? lacc2 : lacc) && l < Lg && ci.valid) {
                    const int mi = A.isReal ? m : (ci.minus ? Lfull - 1 - m : Lfull - 1 + m);
                    const cplx f = A.flmT[((size_t)ci.b * Mfull + mi) * Lfull + l];
                    const cplx Gf = (sc ? A.filt2 : A.filt)[(size_t)(ci.minus ? A.n_filtm[q] : q) * Lg + l];
                    X = cmul(Gf, f);
                    if (ci.minus) X = cscale(X, sgn);
                }
                const double alt = (l & 1) ? -1.0 : 1.0;
                s_X[0][ll * NCT + 2 * k] = X.x;
                s_X[0][ll * NCT + 2 * k + 1] = X.y;
                s_X[1][ll * NCT + 2 * k] = alt * X.x;
                s_X[1][ll * NCT + 2 * k + 1] = alt * X.y;
            }
            __syncthreads();

            const int lb = (lt + TL) < Lg ? (lt + TL) : Lg;
            int l = lt > gs[0] ? lt : gs[0];
            while (l < lb) {
                int ra = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (gs[r] <= l) ++ra;
                    if (gs[r] == l) {  // group r starts here (warp-uniform)
                        const double2 s = seedrow[(r * W + warp) * 32 + lane];
                        d[r] = s.x;
                        u[r] = s.y;
                    }
                }
                int le = lb;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (gs[r] > l && gs[r] < le) le = gs[r];
                // recursion only below the filter support of scale A, scale A alone up to the support of scale B
                if (lacc > l && lacc < le) le = lacc;
                if (lacc2 > l && lacc2 < le) le = lacc2;
                if (l < lacc)
                    inv_dispatch<NCT, R, 0>(ra, l, le, lt, hemi, s_ag, s_e, s_X[hemi], y, d, u, acc);
                else if (NS > 1 && l < lacc2)
                    inv_dispatch<NCT, R, NC>(ra, l, le, lt, hemi, s_ag, s_e, s_X[hemi], y, d, u, acc);
                else
                    inv_dispatch<NCT, R, NCT>(ra, l, le, lt, hemi, s_ag, s_e, s_X[hemi], y, d, u, acc);
                l = le;
            }
        }

        // store F_{m,n}(t) and (complex signals) F_{-m,-n}(t)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (tr[r] < 0) continue;
#pragma unroll
            for (int k = 0; k < NCT / 2; ++k) {
                const int sc = k / (NC / 2), kk = k - sc * (NC / 2);
                const ColInfo ci = col_info(A, chunk * (NC / 2) + kk);
                if (!ci.valid) continue;
                if (ci.minus && m == 0) continue;  // (0,-n) is the plus column of another n
                const int row = ci.minus ? A.n_rowm[q] : A.n_row[q];
                const int mi = A.isReal ? m : (ci.minus ? Lg - 1 - m : Lg - 1 + m);
                (sc ? A.F2 : A.F)[(((size_t)ci.b * A.nrows + row) * A.nt + tr[r]) * Md + mi] =
                    cmake(acc[r][2 * k], acc[r][2 * k + 1]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// forward direction: one block per (m >= 0, chunk of 4 complex = 8 real columns) covering ALL rings.
// Per l-octet every active group (warp, slot) runs 8 recursion steps, writing d~ into a warp-private shared-memory
// tile laid out as eight 4-ring x 8-degree B-fragments; the tensor pipe then accumulates
//     D[col][l] += sum_{ring} hT[col][ring] d~[ring][l]          (mma.sync.m8n8k4.f64, 8 per group and octet)
// with hT (the ring data, constant over l) held in registers as A-fragments.  Per l-tile the warps' partial sums meet
// in shared memory (southern warps with the sign (-1)^l that turns d~ back into d), are multiplied by the output
// filter and added to f_lm with one red.global.add.f64 per value (each address is touched once per launch).
// ---------------------------------------------------------------------------------------------------------------
#define FWD_QS 36                 // doubles per 4-ring fragment row block (32 + 4 pad: conflict-free transposed stores)
#define FWD_GT (8 * FWD_QS)       // doubles per group tile

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// one l-octet of RA active groups (all started before the octet): 8 recursion steps of RA independent chains with the
// d~ values stored as B-fragments, then (if the octet has outputs) 8 RA tensor-pipe accumulations.
template <int R, int RA>
__device__ __forceinline__ void fwd_octet(const double2 *s_ag8, const double *se8, double *dst, const double *src,
                                          bool mm, const double (&y)[R], double (&d)[R], double (&u)[R],
                                          const double (&hA)[R][8], double &c0, double &c1, double &c2, double &c3)
{
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const double2 ag = s_ag8[s];
        const double e = se8[2 * s];
#pragma unroll
        for (int r = 0; r < RA; ++r) {
            dst[r * FWD_GT + 4 * s] = d[r];
            wig_step(d[r], u[r], y[r], ag.x, ag.y, e);
        }
    }
    if (mm) {
        __syncwarp();
#pragma unroll
        for (int r = 0; r < RA; ++r) {
#pragma unroll
            for (int qd = 0; qd < 8; qd += 2) {
                dmma884(c0, c1, hA[r][qd], src[r * FWD_GT + qd * FWD_QS]);
                dmma884(c2, c3, hA[r][qd + 1], src[r * FWD_GT + (qd + 1) * FWD_QS]);
            }
        }
        __syncwarp();
    }
}

// ---- few columns (CF = 2 or 4 real columns per recursion): plain FP64 instead of the tensor pipe ---------------------
// A DMMA consumes 32 d~ values whatever the number of columns, i.e. 8 DFMA-equivalents per (ring, degree) -- for one
// complex column 6 of the 8 tile rows are idle (L = 2048, batch 1: 9 useful flops of the 24 issued per tuple).  Here a
// lane first sums its OWN R rings, p_c(l) = sum_r d~_r(l) h_r[c] (R CF DFMA per degree), and only the CF partial sums per
// degree are transposed through shared memory (P[degree s][c][lane]) and summed over the 32 lanes: 32 R + 8 CF (R + 1)
// FP64 instructions per warp and octet instead of 96 R, and CF instead of R shared-memory round trips per degree.
#define FWD_PS 33  // doubles per row of P (32 lanes + 1: a lane walks along its row with immediate offsets, conflict-free)
template <int R, int RA, int CF, bool MM>
__device__ __forceinline__ void fwd_octet_dfma(const double2 *s_ag8, const double *se8, double *pw,
                                               const double (&y)[R], double (&d)[R], double (&u)[R],
                                               const double (&h)[R][CF > 0 ? CF : 1])
{
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const double2 ag = s_ag8[s];
        const double e = se8[2 * s];
        double p[CF > 0 ? CF : 1];
#pragma unroll
        for (int r = 0; r < RA; ++r) {
            if (MM) {
#pragma unroll
                for (int c = 0; c < CF; ++c) p[c] = r ? fma(d[r], h[r][c], p[c]) : d[r] * h[r][c];
            }
            wig_step(d[r], u[r], y[r], ag.x, ag.y, e);
        }
        if (MM) {
#pragma unroll
            for (int c = 0; c < CF; ++c) pw[(s * CF + c) * FWD_PS] = p[c];
        }
    }
}

template <int R, int CF>
__device__ __forceinline__ void fwd_octet_dfma_ra(int ra, bool mm, const double2 *ag8, const double *se8, double *pw,
                                                  const double (&y)[R], double (&d)[R], double (&u)[R],
                                                  const double (&h)[R][CF > 0 ? CF : 1])
{
#define S2W_OCT(RA_)                                                            \
    {                                                                           \
        if (mm)                                                                 \
            fwd_octet_dfma<R, (R >= RA_ ? RA_ : R), CF, true>(ag8, se8, pw, y, d, u, h);  \
        else                                                                    \
            fwd_octet_dfma<R, (R >= RA_ ? RA_ : R), CF, false>(ag8, se8, pw, y, d, u, h); \
        return;                                                                 \
    }
    if (R >= 4 && ra == 4) S2W_OCT(4)
    if (R >= 3 && ra == 3) S2W_OCT(3)
    if (R >= 2 && ra == 2) S2W_OCT(2)
    S2W_OCT(1)
#undef S2W_OCT
}

// sum over the 32 lanes of the 8 CF partial sums of an octet: row o = s CF + c of P holds one value per lane.  Lane
// (o, half) adds 32 / (32 / K) of them; rows are FWD_PS = 33 doubles apart, so the 16 lanes of a half-warp hit 16 banks.
template <int CF>
__device__ __forceinline__ double fwd_octet_reduce(const double *P, int lane)
{
    constexpr int K = 8 * CF, NH = 32 / K, CNT = 32 / NH;  // K = 16: two lanes per output, 16 addends each
    const int o = lane % K, half = lane / K;
    const double *row = P + o * FWD_PS + half * CNT;
    double v0 = row[0], v1 = row[1], v2 = row[2], v3 = row[3];
#pragma unroll
    for (int i = 4; i < CNT; i += 4) {
        v0 += row[i];
        v1 += row[i + 1];
        v2 += row[i + 2];
        v3 += row[i + 3];
    }
    double v = (v0 + v1) + (v2 + v3);
    if (NH == 2) v += __shfl_xor_sync(0xffffffffu, v, 16);
    return v;
}

// NCH = 2 (table kernel on grids with one ring group per warp and many columns: the stacked shells of a ball plan): a
// block owns two chunks of 4 complex columns, so that one gathered B-fragment of the table feeds two DMMAs (the gathers,
// eight 32-byte runs per 8-byte load instruction, are what the L1 pipe of these launches is busy with)
template <int R, int MAXT, bool PRE, bool FUSE, int CF = 0, int NCH = 1>
__global__ void __launch_bounds__(MAXT, (MAXT <= 256 ? 2 : 1)) wigner_forward_kernel(WigArgs A)
{
    static_assert(CF == 0 || (!PRE && (CF == 2 || CF == 4)), "CF: 0 (tensor pipe), 2 or 4 real columns (FP64 pipe)");
    static_assert(NCH == 1 || (NCH == 2 && PRE && !FUSE && CF == 0), "NCH = 2: table kernel only");
    constexpr int NC = 8;
    constexpr int TLF = FWD_TILE(R);
    __shared__ double2 s_ag[TLF];
    __shared__ double2 s_e[TLF];
    // per-tile sums over all warps (shared-memory atomics), true sign: (degree ll, column c) at SRED(ll, c) -- degree
    // pairs 20 doubles apart, so that the 16 lanes of a half-warp (4 degree pairs x 4 columns of a D fragment) hit 16
    // different bank pairs (with rows of 8 the four degree pairs shared one: 4-way conflicts on the load and the CAS)
#define SRED(ll, c) ((((ll) >> 1) * 20) + (((ll) & 1) * 8) + (c))
    __shared__ double s_red[(TLF / 2) * 20];
    __shared__ double s_red2[NCH == 2 ? (TLF / 2) * 20 : 1];  // the second chunk's sums
    extern __shared__ double s_dt[];   // the B-fragment tiles [W][R][FWD_GT]

    const int m = blockIdx.x, chunk = blockIdx.y * NCH;
    const int Lg = A.Lg, Lfull = A.Lfull, G = A.G;
    const int Md = A.isReal ? Lg : 2 * Lg - 1;
    const int Mfull = A.isReal ? Lfull : 2 * Lfull - 1;
    const int T = blockDim.x, W = T >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, hemi = warp & 1;
    // per warp: R B-fragment tiles, or (CF > 0) the 8 CF x 32 partial sums of an octet
    constexpr int DT_WARP = R * FWD_GT > 8 * CF * FWD_PS ? R * FWD_GT : 8 * CF * FWD_PS;
    double *dt = s_dt + (size_t)warp * DT_WARP;
    // gridDim.z > 1: the ring groups of the grid are dealt out to gridDim.z blocks per (m, chunk), 8 warps each, instead
    // of one block of 16 warps (grids with more than 32 groups): two blocks per SM, so that one block's barriers and
    // epilogue overlap the other's recursion.  Slot r of warp w is group (r gridDim.z + blockIdx.z) W + w; each block
    // adds its partial sums into f_lm with the atomics the epilogue uses anyway.
    const int gz = gridDim.z, bz = blockIdx.z;
#define FWD_GRP(r) (((r) * gz + bz) * W + warp)
    const int wr_off = (lane >> 2) * FWD_QS + (lane & 3);  // + 4 * (l & 7): store slot of this lane's ring

    double y[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int g = FWD_GRP(r);
        y[r] = g < G ? A.yv[g * 32 + lane] : 0.0;
    }
    // A-fragment coordinates of this lane: column c = lane / 4, ring quad member lane % 4
    const int fc = lane >> 2, fk = lane & 3;
    // A.F2 set (at most 2 complex columns): the tile rows 4..7, idle otherwise, carry a second scale that shares the
    // recursion (same grid, same rows n): rows 0..3 = columns of scale A (A.F, A.filt), rows 4..7 = scale B (A.F2, A.filt2)
    constexpr bool fuse = FUSE;
    const ColInfo fci = col_info(A, fuse ? ((fc & 3) >> 1) : chunk * (NC / 2) + (fc >> 1));
    const ColInfo fci2 = col_info(A, (chunk + 1) * (NC / 2) + (fc >> 1));  // NCH = 2
    const cplx *Fsrc = (fuse && fc >= 4) ? A.F2 : A.F;

    for (int q = 0; q < A.nn; ++q) {
        const int n = A.n_val[q], an = n < 0 ? -n : n;
        const int l0 = m > an ? m : an;
        if (l0 >= Lg) continue;
        const int tab = A.n_tab[q];
        const double *crow = A.coef + ((size_t)tab * A.tri + tri_off(m, Lfull)) * 4;
        const int *gsrow = A.gstart + ((size_t)tab * Lg + m) * G;
        const double2 *seedrow = A.dseed + ((size_t)tab * Lg + m) * (size_t)(32 * G);
        const double sgn = ((m + n) & 1) ? -1.0 : 1.0;
        const int lacc = l0 > A.lmin ? l0 : A.lmin;

        // ring data as A-fragments: hA[r][quad] = h[ring (r, quad, fk)][column fc]
        int gs[R];
        double d[R], u[R], hA[R][8], h[R][CF > 0 ? CF : 1];  // hA: tensor-pipe path, h: CF > 0
        double hA2[R][NCH == 2 ? 8 : 1];                     // second chunk (NCH = 2)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int g = FWD_GRP(r);
            gs[r] = g < G ? ((PRE && A.dense) ? l0 : gsrow[g]) : INT_MAX;
            d[r] = 0.0;
            u[r] = 0.0;
            if constexpr (CF > 0) {
                // ring data of this lane's own ring: (re, im) of complex column k (not fused: CF / 2 columns of A.F;
                // fused: column 0 of scale A, then of scale B), zero for padding slots
                const int t = g < G ? A.ring[g * 32 + lane] : -1;
#pragma unroll
                for (int k = 0; k < CF / 2; ++k) {
                    const ColInfo ci = col_info(A, FUSE ? 0 : k);
                    const int row = ci.minus ? A.n_rowm[q] : A.n_row[q];
                    const int mi = A.isReal ? m : (ci.minus ? Lg - 1 - m : Lg - 1 + m);
                    const bool ok = t >= 0 && ci.valid;
                    const cplx *src = ((FUSE && k) ? A.F2 : A.F) +
                                      (((size_t)(ci.valid ? ci.b : 0) * A.nrows + row) * Md + mi) * A.nt + (ok ? t : 0);
                    const cplx v = *src;
                    const double keep = ok ? (ci.minus ? sgn : 1.0) : 0.0;
                    h[r][2 * k] = ok ? v.x * keep : 0.0;
                    h[r][2 * k + 1] = ok ? v.y * keep : 0.0;
                }
                continue;
            }
            // branch-free, so that the 8 ring indices and then the 8 values are loaded together (one latency each,
            // not one per value): invalid rings / columns read element 0 of a valid column and are zeroed afterwards
            const int row = fci.minus ? A.n_rowm[q] : A.n_row[q];
            const int mi = A.isReal ? m : (fci.minus ? Lg - 1 - m : Lg - 1 + m);
            const double *hcol = reinterpret_cast<const double *>(
                                     Fsrc + (((size_t)(fci.valid ? fci.b : 0) * A.nrows + row) * Md + mi) * A.nt) + (fc & 1);
            const int *ringp = A.ring + (g < G ? g : 0) * 32 + fk;
            int tq[8];
#pragma unroll
            for (int qd = 0; qd < 8; ++qd) tq[qd] = ringp[qd * 4];
            const double keep = fci.valid ? (fci.minus ? sgn : 1.0) : 0.0;
#pragma unroll
            for (int qd = 0; qd < 8; ++qd) {
                const bool ok = g < G && tq[qd] >= 0;
                const double v = hcol[2 * (size_t)(ok ? tq[qd] : 0)];
                hA[r][qd] = ok ? v * keep : 0.0;
            }
            if constexpr (NCH == 2) {
                const int row2 = fci2.minus ? A.n_rowm[q] : A.n_row[q];
                const int mi2 = A.isReal ? m : (fci2.minus ? Lg - 1 - m : Lg - 1 + m);
                const double *hcol2 = reinterpret_cast<const double *>(
                                          A.F + (((size_t)(fci2.valid ? fci2.b : 0) * A.nrows + row2) * Md + mi2) * A.nt) + (fc & 1);
                const double keep2 = fci2.valid ? (fci2.minus ? sgn : 1.0) : 0.0;
#pragma unroll
                for (int qd = 0; qd < 8; ++qd) {
                    const bool ok = g < G && tq[qd] >= 0;
                    const double v = hcol2[2 * (size_t)(ok ? tq[qd] : 0)];
                    hA2[r][qd] = ok ? v * keep2 : 0.0;
                }
            }
        }
        // tiles start at the first group start; tiles wholly below the filter support run the recursion only
        int first = gsrow[0];
        if (G > 1 && gsrow[1] < first) first = gsrow[1];
        if (first < l0 || (PRE && A.dense)) first = l0;

        for (int lt = first & ~(TLF - 1); lt < Lg; lt += TLF) {
            __syncthreads();
            for (int i = threadIdx.x; i < (TLF / 2) * 20; i += T) {
                s_red[i] = 0.0;
                if (NCH == 2) s_red2[i] = 0.0;
            }
            if (!PRE) stage_coef<TLF>(crow, lt, l0, Lg, s_ag, s_e);
            __syncthreads();
            const bool want = lt + TLF > lacc;  // this tile has outputs
            const double *se = reinterpret_cast<const double *>(s_e) + hemi;
#pragma unroll 1
            for (int oc = 0; oc < TLF / 8; ++oc) {
                const int lo = lt + 8 * oc;
                double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
                double e0 = 0.0, e1 = 0.0, e2 = 0.0, e3 = 0.0;  // second chunk (NCH = 2)
                bool contributed = false;
                if (PRE) {
                    // precomputed-kernel variant (a9): B-fragments straight from the d-table in HBM
                    if (gs[0] < lo + 8 && lo < Lg && want && lo + 8 > lacc) {
                        contributed = true;
                        const int lrow = lo + (lane >> 2);
                        const bool ok = lrow >= l0 && lrow < Lg;
                        const double *trow = A.dtab + ((size_t)tab * A.tri_g + tri_off(m, Lg) + (ok ? lrow : l0)) *
                                                          (size_t)(32 * G) + (lane & 3);
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            if (gs[r] >= lo + 8) continue;
                            const double *src = trow + FWD_GRP(r) * 32;
                            double bv[8];
#pragma unroll
                            for (int qd = 0; qd < 8; ++qd) bv[qd] = ok ? __ldg(src + 4 * qd) : 0.0;
#pragma unroll
                            for (int qd = 0; qd < 8; qd += 2) {
                                dmma884(c0, c1, hA[r][qd], bv[qd]);
                                dmma884(c2, c3, hA[r][qd + 1], bv[qd + 1]);
                                if constexpr (NCH == 2) {
                                    dmma884(e0, e1, hA2[r][qd], bv[qd]);
                                    dmma884(e2, e3, hA2[r][qd + 1], bv[qd + 1]);
                                }
                            }
                        }
                    }
                } else if (gs[0] < lo + 8 && lo < Lg) {
                    const bool mm = want && (lo + 8 > lacc);
                    contributed = mm;
                    int ra = 0;
                    bool starting = false;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (gs[r] < lo + 8) {
                            ++ra;
                            if (gs[r] >= lo) starting = true;
                        }
                    }
                    double *dst = dt + wr_off;
                    const double *src = dt + lane;
                    if (CF > 0) {
                        double *pw = dt + lane;
                        if (!starting) {
                            fwd_octet_dfma_ra<R, CF>(ra, mm, s_ag + 8 * oc, se + 16 * oc, pw, y, d, u, h);
                        } else {
#pragma unroll 1
                            for (int s = 0; s < 8; ++s) {
                                const double2 ag = s_ag[8 * oc + s];
                                const double e = se[2 * (8 * oc + s)];
                                double pp[CF > 0 ? CF : 1];
#pragma unroll
                                for (int c = 0; c < CF; ++c) pp[c] = 0.0;
#pragma unroll
                                for (int r = 0; r < R; ++r) {
                                    if (r < ra) {
                                        if (gs[r] == lo + s) {  // the group starts here (warp-uniform)
                                            const double2 sd = seedrow[FWD_GRP(r) * 32 + lane];
                                            d[r] = sd.x;
                                            u[r] = sd.y;
                                        }
#pragma unroll
                                        for (int c = 0; c < CF; ++c) pp[c] = fma(d[r], h[r][c], pp[c]);
                                        wig_step(d[r], u[r], y[r], ag.x, ag.y, e);
                                    }
                                }
#pragma unroll
                                for (int c = 0; c < CF; ++c) pw[(s * CF + c) * FWD_PS] = pp[c];
                            }
                        }
                        if (mm) {
                            __syncwarp();
                            double v = fwd_octet_reduce<(CF > 0 ? CF : 2)>(dt, lane);
                            constexpr int K = 8 * (CF > 0 ? CF : 2);
                            if (lane < K) {
                                const int sdeg = lane / (CF > 0 ? CF : 2);
                                // southern warps: d = (-1)^l d~, and the octet starts at an even degree
                                if (hemi && (sdeg & 1)) v = -v;
                                // CF > 0 layout of s_red: [degree][CF], the K lanes hit K consecutive doubles (the SRED
                                // layout of the tensor-pipe path would put them four to a bank)
                                atomicAdd(&s_red[(8 * oc) * (CF > 0 ? CF : 2) + lane], v);
                            }
                            __syncwarp();
                        }
                        contributed = false;  // the sums of this octet are in s_red already
                    } else if (!starting) {
                        const double2 *ag8 = s_ag + 8 * oc;
                        const double *se8 = se + 16 * oc;
                        if (R >= 4 && ra == 4)
                            fwd_octet<R, (R >= 4 ? 4 : R)>(ag8, se8, dst, src, mm, y, d, u, hA, c0, c1, c2, c3);
                        else if (R >= 3 && ra == 3)
                            fwd_octet<R, (R >= 3 ? 3 : R)>(ag8, se8, dst, src, mm, y, d, u, hA, c0, c1, c2, c3);
                        else if (R >= 2 && ra == 2)
                            fwd_octet<R, (R >= 2 ? 2 : R)>(ag8, se8, dst, src, mm, y, d, u, hA, c0, c1, c2, c3);
                        else
                            fwd_octet<R, 1>(ag8, se8, dst, src, mm, y, d, u, hA, c0, c1, c2, c3);
                    } else {
#pragma unroll 1
                        for (int s = 0; s < 8; ++s) {
                            const double2 ag = s_ag[8 * oc + s];
                            const double e = se[2 * (8 * oc + s)];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                if (r < ra) {
                                    if (gs[r] == lo + s) {  // the group starts here (warp-uniform)
                                        const double2 sd = seedrow[FWD_GRP(r) * 32 + lane];
                                        d[r] = sd.x;
                                        u[r] = sd.y;
                                    }
                                    dst[r * FWD_GT + 4 * s] = d[r];
                                    wig_step(d[r], u[r], y[r], ag.x, ag.y, e);
                                }
                            }
                        }
                        if (mm) {
                            __syncwarp();
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                if (r >= ra) continue;
#pragma unroll
                                for (int qd = 0; qd < 8; qd += 2) {
                                    dmma884(c0, c1, hA[r][qd], src[r * FWD_GT + qd * FWD_QS]);
                                    dmma884(c2, c3, hA[r][qd + 1], src[r * FWD_GT + (qd + 1) * FWD_QS]);
                                }
                            }
                            __syncwarp();
                        }
                    }
                }
                // D fragment: row (column index) lane / 4, degrees 2 (lane % 4) + {0, 1} of the octet
                // (southern warps: d = (-1)^l d~, and the octet starts at an even degree)
                if (contributed) {
                    const double v0 = c0 + c2, v1 = c1 + c3;
                    atomicAdd(&s_red[SRED(8 * oc + 2 * fk, fc)], v0);
                    atomicAdd(&s_red[SRED(8 * oc + 2 * fk + 1, fc)], (!PRE && hemi) ? -v1 : v1);
                    if constexpr (NCH == 2) {
                        atomicAdd(&s_red2[SRED(8 * oc + 2 * fk, fc)], e0 + e2);
                        atomicAdd(&s_red2[SRED(8 * oc + 2 * fk + 1, fc)], e1 + e3);
                    }
                }
            }
            if (!want) continue;
            __syncthreads();
            // cross-warp sum, output filter, accumulate into f_lm
            for (int i = threadIdx.x; i < TLF * (NC / 2) * NCH; i += T) {
                const int ch = i / (TLF * (NC / 2)), k = (i / TLF) % (NC / 2), ll = i % TLF;
                const double *sred = (NCH == 2 && ch) ? s_red2 : s_red;
                const int l = lt + ll;
                if (fuse && k >= 2) continue;  // fused: k = complex column, both scales summed below
                const ColInfo ci = col_info(A, fuse ? k : (chunk + ch) * (NC / 2) + k);
                if (l < lacc || l >= Lg || !ci.valid) continue;
                if (ci.minus && m == 0) continue;
                cplx val = cmake(0.0, 0.0);
                for (int sc = 0; sc < (fuse ? 2 : 1); ++sc) {
                    const int c0i = 2 * k + 4 * sc;
                    const int cp = FUSE ? 2 * sc : 2 * k;  // CF > 0: column pair of (scale sc | complex column k)
                    const double re = CF > 0 ? s_red[ll * (CF > 0 ? CF : 2) + cp] : sred[SRED(ll, c0i)];
                    const double im = CF > 0 ? s_red[ll * (CF > 0 ? CF : 2) + cp + 1] : sred[SRED(ll, c0i + 1)];
                    const cplx Gf = (sc ? A.filt2 : A.filt)[(size_t)(ci.minus ? A.n_filtm[q] : q) * Lg + l];
                    val = cadd(val, cmul(Gf, cmake(re, im)));
                }
                const int mi = A.isReal ? m : (ci.minus ? Lfull - 1 - m : Lfull - 1 + m);
                double *dst = reinterpret_cast<double *>(&A.flmT[((size_t)ci.b * Mfull + mi) * Lfull + l]);
                atomicAdd(dst, val.x);
                atomicAdd(dst + 1, val.y);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// precomputed-kernel variant (step a9; "simply precomputed"; O(N L^3) memory)
//
// dtab[tab][packed (m, l >= m) of the grid][32 G ring slots] holds d^l_mn(beta) itself (southern rings with their true
// sign), zero below the group start.  One warp per (group, m, n) fills its rows by the recursion above.  The
// contraction kernels then only stream the table: both directions are batched small-N GEMMs on the FP64 tensor pipe
// (mma.sync.m8n8k4.f64), HBM-bound at 8 B per (ring, m, l, n) tuple for up to 4 complex columns.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) wigner_table_kernel(const double *__restrict__ coef, size_t tri, int Lfull, int Lg,
                                                         int G, NList nl, const double *__restrict__ yv,
                                                         const int *__restrict__ gstart,
                                                         const double2 *__restrict__ dseed, double *__restrict__ dtab,
                                                         size_t tri_g)
{
    const int g = blockIdx.x, m = blockIdx.y, tab = blockIdx.z, lane = threadIdx.x;
    const int k = g * 32 + lane;
    const bool south = (g & 1) != 0;
    const int gs = gstart[((size_t)tab * Lg + m) * G + g];
    if (gs >= Lg) return;
    const double2 sd = dseed[((size_t)tab * Lg + m) * (size_t)(32 * G) + k];
    double d = sd.x, u = sd.y;
    const double y = yv[k];
    const double *c = coef + ((size_t)tab * tri + tri_off(m, Lfull)) * 4;
    double *out = dtab + ((size_t)tab * tri_g + tri_off(m, Lg)) * (size_t)(32 * G) + k;
    for (int l = gs; l < Lg; ++l) {
        out[(size_t)l * (32 * G)] = (south && (l & 1)) ? -d : d;
        const double4 q = *reinterpret_cast<const double4 *>(c + 4 * (size_t)l);
        wig_step(d, u, y, q.x, q.y, south ? q.w : q.z);
    }
}

// the table of one n as reweighting input X[l][t][m] (complex, imaginary part zero) and back (kernels.h)
__global__ void wigner_table_gather_kernel(const double *__restrict__ dtab, size_t tri_g, int tab, int n, int Lg, int nt,
                                           int G, const int *__restrict__ ring, cplx *__restrict__ X)
{
    const int l = blockIdx.x, m = blockIdx.y;
    const int an = n < 0 ? -n : n;
    const bool in = l >= m && l >= an;
    const double *row = dtab + ((size_t)tab * tri_g + tri_off(m, Lg) + (in ? l : m)) * (size_t)(32 * G);
    for (int k = threadIdx.x; k < 32 * G; k += blockDim.x) {
        const int t = ring[k];
        if (t >= 0 && t < nt) X[((size_t)l * nt + t) * Lg + m] = cmake(in ? row[k] : 0.0, 0.0);
    }
}

__global__ void wigner_table_scatter_kernel(const cplx *__restrict__ Y, double *__restrict__ dtab_rw, size_t tri_g, int tab,
                                            int n, int Lg, int nt, int G, const int *__restrict__ ring)
{
    const int l = blockIdx.x, m = blockIdx.y;
    const int an = n < 0 ? -n : n;
    if (l < m || l < an) return;
    double *row = dtab_rw + ((size_t)tab * tri_g + tri_off(m, Lg) + l) * (size_t)(32 * G);
    for (int k = threadIdx.x; k < 32 * G; k += blockDim.x) {
        const int t = ring[k];
        row[k] = (t >= 0 && t < nt) ? Y[((size_t)l * Lg + m) * nt + t].x : 0.0;
    }
}

// inverse direction from the table: D[ring][col] += A[ring][l] B[l][col], A-fragments (8 rings x 4 degrees) gathered
// from the table, B = filter x f_lm from shared memory, accumulators 8 rings x 8 columns per ring octet.
// NCH > 1 (small grids with many columns: the stacked shells of a ball plan): a block owns NCH chunks of 4 complex columns,
// so that one gathered A-fragment (an 8-byte load per lane over four 64-byte runs of the table; knocking these loads out
// took 0.6 of the 2.0 ms of the class at C5) feeds NCH DMMAs.  Rows of s_X are NCB + 4 doubles apart: the B-fragment reads
// (degree lane % 4, column lane / 4) of a half-warp then fall into 16 different banks.
template <int R, int MAXT, int NCH = 1>
__global__ void __launch_bounds__(MAXT) precomp_inverse_kernel(WigArgs A)
{
    constexpr int NC = 8;
    constexpr int NCB = NC * NCH;                 // real columns of the block
    constexpr int XS = NCB + 4;                   // row stride of s_X
    __shared__ double s_X[WIG_TL * XS];

    const int m = blockIdx.x, chunk = blockIdx.y * NCH;
    const int Lg = A.Lg, Lfull = A.Lfull, G = A.G;
    const int Md = A.isReal ? Lg : 2 * Lg - 1;
    const int Mfull = A.isReal ? Lfull : 2 * Lfull - 1;
    const int T = blockDim.x, W = T >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int fr = lane >> 2, fk = lane & 3;  // A: ring fr of the octet, degree fk of the quad; B: degree fk, column fr

    for (int q = 0; q < A.nn; ++q) {
        const int n = A.n_val[q], an = n < 0 ? -n : n;
        const int l0 = m > an ? m : an;
        if (l0 >= Lg) continue;
        const int tab = A.n_tab[q];
        const int *gsrow = A.gstart + ((size_t)tab * Lg + m) * G;
        const double sgn = ((m + n) & 1) ? -1.0 : 1.0;
        const int lacc = l0 > A.lmin ? l0 : A.lmin;
        const double *tbase = A.dtab + ((size_t)tab * A.tri_g + tri_off(m, Lg)) * (size_t)(32 * G);

        int gs[R];
        double acc[R][NCH][4][2];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int g = r * W + warp;
            gs[r] = g < G ? gsrow[g] : INT_MAX;
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
                for (int o = 0; o < 4; ++o) acc[r][ch][o][0] = acc[r][ch][o][1] = 0.0;
        }
        int first = gsrow[0];
        if (G > 1 && gsrow[1] < first) first = gsrow[1];
        if (first < lacc) first = lacc;

        for (int lt = first & ~(WIG_TL - 1); lt < Lg; lt += WIG_TL) {
            __syncthreads();
            for (int i = threadIdx.x; i < WIG_TL * (NCB / 2); i += T) {
                const int k = i / WIG_TL, ll = i % WIG_TL;
                const int l = lt + ll;
                const ColInfo ci = col_info(A, chunk * (NC / 2) + k);
                cplx X = cmake(0.0, 0.0);
                if (l >= lacc && l < Lg && ci.valid) {
                    const int mi = A.isReal ? m : (ci.minus ? Lfull - 1 - m : Lfull - 1 + m);
                    const cplx f = A.flmT[((size_t)ci.b * Mfull + mi) * Lfull + l];
                    const cplx Gf = A.filt[(size_t)(ci.minus ? A.n_filtm[q] : q) * Lg + l];
                    X = cmul(Gf, f);
                    if (ci.minus) X = cscale(X, sgn);
                }
                s_X[ll * XS + 2 * k] = X.x;
                s_X[ll * XS + 2 * k + 1] = X.y;
            }
            __syncthreads();
#pragma unroll 2
            for (int lq = 0; lq < WIG_TL; lq += 4) {
                const int lo = lt + lq;
                if (lo + 4 <= lacc || lo >= Lg || gs[0] >= lo + 4) continue;
                double bv[NCH];
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) bv[ch] = s_X[(lq + fk) * XS + ch * NC + fr];
                const int lrow = lo + fk;
                const bool ok = lrow >= l0 && lrow < Lg;
                const double *trow = tbase + (size_t)(ok ? lrow : l0) * (32 * G) + fr;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (gs[r] >= lo + 4) continue;
                    const double *src = trow + (r * W + warp) * 32;
                    double av[4];
#pragma unroll
                    for (int o = 0; o < 4; ++o) av[o] = ok ? __ldg(src + 8 * o) : 0.0;
#pragma unroll
                    for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
                        for (int o = 0; o < 4; ++o) dmma884(acc[r][ch][o][0], acc[r][ch][o][1], av[o], bv[ch]);
                }
            }
        }

        // D fragment: ring lane / 4 of the octet, real columns 2 (lane % 4) + {0, 1} = complex column lane % 4
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            const ColInfo ci = col_info(A, (chunk + ch) * (NC / 2) + fk);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int g = r * W + warp;
                if (g >= G || !ci.valid) continue;
                if (ci.minus && m == 0) continue;
                const int row = ci.minus ? A.n_rowm[q] : A.n_row[q];
                const int mi = A.isReal ? m : (ci.minus ? Lg - 1 - m : Lg - 1 + m);
#pragma unroll
                for (int o = 0; o < 4; ++o) {
                    const int t = A.ring[g * 32 + o * 8 + fr];
                    if (t < 0) continue;
                    A.F[(((size_t)ci.b * A.nrows + row) * A.nt + t) * Md + mi] = cmake(acc[r][ch][o][0], acc[r][ch][o][1]);
                }
            }
        }
    }
}

// ---- bulk-asynchronous (TMA) staging of the table: cp.async.bulk global -> shared with mbarrier completion ----------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D bulk copy (bytes: a multiple of 16, both addresses 16-byte aligned); completes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// The inverse direction from the table with TMA-staged tiles (north_star: "batched dense contraction on the fp64 tensor
// pipe (DMMA), with TMA-staged tiles").  Same contraction as precomp_inverse_kernel, but the A operand --
// 4 degrees x 32 ring slots of each of the warp's R groups per step, 256-byte runs of the table -- reaches shared memory
// by cp.async.bulk (SASS UBLKCP) into a ring of PRE_STAGES stages PER WARP, completion signalled on a per-stage
// mbarrier, PRE_STAGES - 1 steps ahead of the DMMA that consumes it.  A warp produces and consumes only its own
// stages (its lane 0 issues the copies after __syncwarp), so there is no cross-warp synchronisation on the table stream;
// the per-lane 8-byte __ldg gathers of the plain kernel kept at most 4 loads per lane in flight (0.56 of the HBM roof).
// A warp owns R CONTIGUOUS groups here (ring slots 32 R warp ...), so a degree's row for the warp is one contiguous run
// of up to 256 R bytes: one bulk copy per degree.  Stage layout: [degree of the quad][32 R ring slots + 4 pad doubles],
// so that the A-fragment reads (ring lane/4 of an octet, degree lane%4) of a half-warp fall into 16 different bank pairs.
template <int R>
struct PreStage {
    static constexpr int row = 32 * R + 4;        // one degree: the warp's R contiguous groups + 4 pad doubles
    static constexpr int doubles = 4 * row;
};
template <int R, int MAXT, int STAGES>
__global__ void __launch_bounds__(MAXT, (MAXT <= 256 ? 2 : 1)) precomp_inverse_tma_kernel(WigArgs A)
{
    constexpr int NC = 8;
    constexpr int XS = NC + 4;  // row stride of s_X: conflict-free B-fragment reads (see precomp_inverse_kernel)
    __shared__ double s_X[WIG_TL * XS];
    extern __shared__ __align__(16) double s_dyn[];   // [W][STAGES][4 degrees][32 R + 4] then the mbarriers [W][STAGES]

    const int m = blockIdx.x, chunk = blockIdx.y;
    const int Lg = A.Lg, Lfull = A.Lfull, G = A.G;
    const int Md = A.isReal ? Lg : 2 * Lg - 1;
    const int Mfull = A.isReal ? Lfull : 2 * Lfull - 1;
    const int T = blockDim.x, W = T >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int fr = lane >> 2, fk = lane & 3;
    double *wst = s_dyn + (size_t)warp * STAGES * PreStage<R>::doubles;
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(s_dyn + (size_t)W * STAGES * PreStage<R>::doubles) +
                               warp * STAGES;
    if (lane == 0) {
#pragma unroll
        for (int sgi = 0; sgi < STAGES; ++sgi) mbar_init(&bars[sgi], 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the barriers are visible to the async proxy
    }
    __syncwarp();
    unsigned it_prod = 0, it_cons = 0;  // steps issued / consumed by this warp since kernel start (stage and parity)

    for (int q = 0; q < A.nn; ++q) {
        const int n = A.n_val[q], an = n < 0 ? -n : n;
        const int l0 = m > an ? m : an;
        if (l0 >= Lg) continue;
        const int tab = A.n_tab[q];
        const int *gsrow = A.gstart + ((size_t)tab * Lg + m) * G;
        const double sgn = ((m + n) & 1) ? -1.0 : 1.0;
        const int lacc = l0 > A.lmin ? l0 : A.lmin;
        const double *tbase = A.dtab + ((size_t)tab * A.tri_g + tri_off(m, Lg)) * (size_t)(32 * G);

        int gs[R];
        double acc[R][4][2];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int g = warp * R + r;
            gs[r] = g < G ? gsrow[g] : INT_MAX;
#pragma unroll
            for (int o = 0; o < 4; ++o) acc[r][o][0] = acc[r][o][1] = 0.0;
        }
        int first = gsrow[0];
        if (G > 1 && gsrow[1] < first) first = gsrow[1];
        if (first < lacc) first = lacc;
        const int lt0 = first & ~(WIG_TL - 1);

        // a step = one degree quad lo..lo+3; `live` steps are those the plain kernel does not skip
        auto live = [&](int lo) { return !(lo + 4 <= lacc || lo >= Lg || gs[0] >= lo + 4); };
        auto issue = [&](int lo) {  // lane 0: bulk copies of the quad's rows for the warp's started groups
            const unsigned sgi = it_prod % STAGES;
            double *dst = wst + (size_t)sgi * PreStage<R>::doubles;
            unsigned bytes = 0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (gs[r] >= lo + 4) continue;
                bytes = (r + 1) * 256;
            }
            {
                int rows = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (lo + k >= l0 && lo + k < Lg) ++rows;
                bytes *= rows;
            }
            mbar_arrive_expect_tx(&bars[sgi], bytes);
            // the warp's started groups are a prefix of its R contiguous groups (starts are monotone within a hemisphere
            // and the two hemispheres of a pair start together or the northern one first): one copy per degree
            int nact = 0;
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (gs[r] < lo + 4) nact = r + 1;
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (lo + k >= l0 && lo + k < Lg)
                    bulk_g2s(dst + k * PreStage<R>::row, tbase + (size_t)(lo + k) * (32 * G) + (size_t)warp * R * 32, nact * 256,
                             &bars[sgi]);
            ++it_prod;
        };
        // prologue: up to STAGES - 1 live steps ahead
        int lo_prod = lt0;
        {
            int ahead = 0;
            while (lo_prod < Lg && ahead < STAGES - 1) {
                if (live(lo_prod)) {
                    if (lane == 0) issue(lo_prod);
                    ++ahead;
                }
                lo_prod += 4;
            }
        }
        it_prod = __shfl_sync(0xffffffffu, it_prod, 0);

        for (int lt = lt0; lt < Lg; lt += WIG_TL) {
            __syncthreads();
            for (int i = threadIdx.x; i < WIG_TL * (NC / 2); i += T) {
                const int k = i / WIG_TL, ll = i % WIG_TL;
                const int l = lt + ll;
                const ColInfo ci = col_info(A, chunk * (NC / 2) + k);
                cplx X = cmake(0.0, 0.0);
                if (l >= lacc && l < Lg && ci.valid) {
                    const int mi = A.isReal ? m : (ci.minus ? Lfull - 1 - m : Lfull - 1 + m);
                    const cplx f = A.flmT[((size_t)ci.b * Mfull + mi) * Lfull + l];
                    const cplx Gf = A.filt[(size_t)(ci.minus ? A.n_filtm[q] : q) * Lg + l];
                    X = cmul(Gf, f);
                    if (ci.minus) X = cscale(X, sgn);
                }
                s_X[ll * XS + 2 * k] = X.x;
                s_X[ll * XS + 2 * k + 1] = X.y;
            }
            __syncthreads();
            for (int lq = 0; lq < WIG_TL; lq += 4) {
                const int lo = lt + lq;
                if (!live(lo)) continue;
                // keep the pipeline full: the next live step not yet issued (its stage was released by the __syncwarp
                // that ended the step STAGES - 1 steps ago)
                while (lo_prod < Lg && !live(lo_prod)) lo_prod += 4;
                if (lo_prod < Lg) {
                    if (lane == 0) issue(lo_prod);
                    it_prod = __shfl_sync(0xffffffffu, it_prod, 0);
                    lo_prod += 4;
                }
                const unsigned sgi = it_cons % STAGES;
                mbar_wait(&bars[sgi], (it_cons / STAGES) & 1);
                ++it_cons;
                const double *src = wst + (size_t)sgi * PreStage<R>::doubles + fk * PreStage<R>::row + fr;
                const double bv = s_X[(lq + fk) * XS + fr];
                const int lrow = lo + fk;
                const bool ok = lrow >= l0 && lrow < Lg;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (gs[r] >= lo + 4) continue;
                    double av[4];
#pragma unroll
                    for (int o = 0; o < 4; ++o) av[o] = ok ? src[r * 32 + 8 * o] : 0.0;
#pragma unroll
                    for (int o = 0; o < 4; ++o) dmma884(acc[r][o][0], acc[r][o][1], av[o], bv);
                }
                __syncwarp();  // every lane has read the stage before lane 0 refills it
            }
        }

        const ColInfo ci = col_info(A, chunk * (NC / 2) + fk);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int g = warp * R + r;
            if (g >= G || !ci.valid) continue;
            if (ci.minus && m == 0) continue;
            const int row = ci.minus ? A.n_rowm[q] : A.n_row[q];
            const int mi = A.isReal ? m : (ci.minus ? Lg - 1 - m : Lg - 1 + m);
#pragma unroll
            for (int o = 0; o < 4; ++o) {
                const int t = A.ring[g * 32 + o * 8 + fr];
                if (t < 0) continue;
                A.F[(((size_t)ci.b * A.nrows + row) * A.nt + t) * Md + mi] = cmake(acc[r][o][0], acc[r][o][1]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// layout conversion between the user's flm[b][l][m+L-1] and the internal m-major flmT[b][mi][l]
// ---------------------------------------------------------------------------------------------------------------
__global__ void flm_pack_kernel(const cplx *__restrict__ flm, cplx *__restrict__ flmT, int L, int real)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x, mi = blockIdx.y, b = blockIdx.z;
    if (l >= L) return;
    const int Mfull = real ? L : 2 * L - 1;
    const int m = real ? mi : mi - (L - 1);
    const int am = m < 0 ? -m : m;
    cplx v = cmake(0.0, 0.0);
    if (am <= l) v = flm[((size_t)b * L + l) * (2 * L - 1) + (m + L - 1)];
    flmT[((size_t)b * Mfull + mi) * L + l] = v;
}

__global__ void flm_unpack_kernel(const cplx *__restrict__ flmT, cplx *__restrict__ flm, int L, int real)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x, mi = blockIdx.y, b = blockIdx.z;  // mi over 2L-1
    if (l >= L) return;
    const int m = mi - (L - 1);
    const int am = m < 0 ? -m : m;
    cplx v = cmake(0.0, 0.0);
    if (am <= l) {
        if (real) {
            v = flmT[((size_t)b * L + am) * L + l];
            if (m < 0) {
                v = cconj(v);
                if (am & 1) v = cscale(v, -1.0);
            }
        } else {
            v = flmT[((size_t)b * (2 * L - 1) + mi) * L + l];
        }
    }
    flm[((size_t)b * L + l) * (2 * L - 1) + mi] = v;
}

__global__ void flm_pack_pm_kernel(const cplx *__restrict__ pos, const cplx *__restrict__ neg, cplx *__restrict__ flmT, int L)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x, mi = blockIdx.y, b = blockIdx.z;
    if (l >= L) return;
    const int m = mi - (L - 1), am = m < 0 ? -m : m;
    cplx v = cmake(0.0, 0.0);
    if (am <= l) v = (m >= 0 ? pos : neg)[((size_t)b * L + l) * (2 * L - 1) + mi];
    flmT[((size_t)b * (2 * L - 1) + mi) * L + l] = v;
}

__global__ void flm_unpack_pm_kernel(const cplx *__restrict__ flmT, cplx *__restrict__ pos, cplx *__restrict__ neg, int L)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x, mi = blockIdx.y, b = blockIdx.z;
    if (l >= L) return;
    const int m = mi - (L - 1), am = m < 0 ? -m : m;
    const cplx v = am <= l ? flmT[((size_t)b * (2 * L - 1) + mi) * L + l] : cmake(0.0, 0.0);
    (m >= 0 ? pos : neg)[((size_t)b * L + l) * (2 * L - 1) + mi] = v;
}

// ---------------------------------------------------------------------------------------------------------------
// FP64 pipe probes
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_probe_kernel(double *out, int iters, double a, double b)
{
    double v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = (double)(threadIdx.x + i) * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = fma(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) dmma_probe_kernel(double *out, int iters, double a, double b)
{
    double c[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        c[i][0] = 0.0;
        c[i][1] = 0.0;
    }
    double fa = a + threadIdx.x * 1e-9, fb = b;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i) dmma884(c[i][0], c[i][1], fa, fb);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

// block shape for a grid with G ring groups: W warps (even), R groups per warp
struct WigCfg {
    int R, W, MAXT;
};
bool wig_cfg(int G, WigCfg &c)
{
    if (G < 2 || (G & 1) || G > 64) return false;
    c.W = G <= 8 ? G : (G <= 32 ? 8 : 16);
    c.R = (G + c.W - 1) / c.W;
    c.MAXT = c.W <= 8 ? 256 : 512;
    return c.R <= 4;
}

template <int NC, int R, int MAXT, int NS>
void launch_inv_t(const WigArgs &A, int T, int chunks, cudaStream_t st)
{
    dim3 grid(A.Lg, chunks);
    S2W_LAUNCH_C(S2W_K_WIGNER_INV, (wigner_inverse_kernel<NC, R, MAXT, NS>), grid, T, 0, st, A);
}

template <int R, int MAXT, bool PRE, bool FUSE, int CF = 0, int NCH = 1>
int launch_fwd_t(const WigArgs &A, int T, int chunks, cudaStream_t st, int gz = 1)
{
    // per warp: R B-fragment tiles (tensor pipe) or the 8 CF x 32 partial sums of an octet (CF > 0)
    constexpr size_t per_warp = ((size_t)R * FWD_GT > (size_t)8 * CF * FWD_PS ? (size_t)R * FWD_GT : (size_t)8 * CF * FWD_PS) * sizeof(double);
    const size_t smem = PRE ? 0 : (size_t)(T / 32) * per_warp;
    // the attribute is per device and per function: query and raise it when needed (smem_attr.cuh), no per-process flag
    {
        const int rc = set_smem(wigner_forward_kernel<R, MAXT, PRE, FUSE, CF, NCH>, (size_t)(MAXT / 32) * per_warp);
        if (rc) return rc;
    }
    dim3 grid(A.Lg, chunks, gz);
    S2W_LAUNCH_C(S2W_K_WIGNER_FWD, (wigner_forward_kernel<R, MAXT, PRE, FUSE, CF, NCH>), grid, T, smem, st, A);
    return S2W_OK;
}

template <int NC, int NS>
int dispatch_inv(const WigArgs &A, const WigCfg &c, int chunks, cudaStream_t st)
{
#define S2W_WIG_CASE(RR, MT)                              \
    if (c.R == RR && c.MAXT == MT) {                      \
        launch_inv_t<NC, RR, MT, NS>(A, 32 * c.W, chunks, st); \
        return S2W_OK;                                    \
    }
    S2W_WIG_CASE(1, 256)
    S2W_WIG_CASE(2, 256)
    S2W_WIG_CASE(3, 256)
    S2W_WIG_CASE(4, 256)
    S2W_WIG_CASE(3, 512)
    S2W_WIG_CASE(4, 512)
#undef S2W_WIG_CASE
    return S2W_EINVAL;
}

static bool split_on()
{
    static const bool split = [] {
        const char *e = getenv("S2W_FWD_SPLIT");
        return !(e && e[0] == '0');
    }();
    return split;
}

int dispatch_fwd(const WigArgs &A, const WigCfg &c, int chunks, cudaStream_t st)
{
    // grids with more than 32 ring groups (L_j > 1024): two 8-warp blocks per (m, chunk), each with half of the groups
    // (wigner_forward_kernel, gridDim.z), instead of one 16-warp block
    const bool split = split_on();
    // few columns: the FP64-pipe variant (fwd_octet_dfma).  CF = real columns per recursion: 2 CT, twice that when two
    // scales share the recursion.  S2W_FWD_DFMA = 0: never, 2: only CF = 2, 4 (default): CF = 2 and CF = 4
    static const int dfma_max = [] {
        const char *e = getenv("S2W_FWD_DFMA");
        return e ? atoi(e) : 4;
    }();
    static const int pre_nch = [] {
        const char *e = getenv("S2W_PRE_NCH");
        return e ? atoi(e) : 2;
    }();
    // table kernel, one ring group per warp, many columns: two column chunks per block (wigner_forward_kernel, NCH)
    if (A.dtab && c.R == 1 && chunks >= 8 && pre_nch > 1)
        return launch_fwd_t<1, 256, true, false, 0, 2>(A, 32 * c.W, (chunks + 1) / 2, st);
    const int CT = A.isReal ? A.B : 2 * A.B;
    const int cf = (A.F2 ? 4 : 2) * CT;
    const int gz = (split_on() && c.W == 16) ? 2 : 1;
    // CF = 4 pays from three ring groups per warp on (FP64 instructions per warp and octet: 64 R + 32 against 96 R)
    static const int dfma4_minR = [] {
        const char *e = getenv("S2W_FWD_DFMA4_MINR");
        return e ? atoi(e) : 3;
    }();
    if (!A.dtab && cf <= dfma_max && (cf == 2 || c.R >= dfma4_minR) && (c.MAXT == 256 || gz == 2)) {
#define S2W_WIG_CASE(RR)                                                                                   \
    if (c.R == RR) {                                                                                       \
        if (A.F2) return launch_fwd_t<RR, 256, false, true, 4>(A, gz == 2 ? 256 : 32 * c.W, 1, st, gz);    \
        return cf == 2 ? launch_fwd_t<RR, 256, false, false, 2>(A, gz == 2 ? 256 : 32 * c.W, 1, st, gz)    \
                       : launch_fwd_t<RR, 256, false, false, 4>(A, gz == 2 ? 256 : 32 * c.W, 1, st, gz);   \
    }
        S2W_WIG_CASE(1)
        S2W_WIG_CASE(2)
        S2W_WIG_CASE(3)
        S2W_WIG_CASE(4)
#undef S2W_WIG_CASE
    }
    if (split && c.W == 16) {
#define S2W_WIG_CASE(RR)                                                                \
    if (c.R == RR)                                                                      \
        return A.dtab ? launch_fwd_t<RR, 256, true, false>(A, 256, chunks, st, 2)       \
                      : (A.F2 ? launch_fwd_t<RR, 256, false, true>(A, 256, chunks, st, 2) \
                              : launch_fwd_t<RR, 256, false, false>(A, 256, chunks, st, 2));
        S2W_WIG_CASE(3)
        S2W_WIG_CASE(4)
#undef S2W_WIG_CASE
    }
#define S2W_WIG_CASE(RR, MT)                                                              \
    if (c.R == RR && c.MAXT == MT)                                                        \
        return A.dtab ? launch_fwd_t<RR, MT, true, false>(A, 32 * c.W, chunks, st)        \
                      : (A.F2 ? launch_fwd_t<RR, MT, false, true>(A, 32 * c.W, chunks, st) \
                              : launch_fwd_t<RR, MT, false, false>(A, 32 * c.W, chunks, st));
    S2W_WIG_CASE(1, 256)
    S2W_WIG_CASE(2, 256)
    S2W_WIG_CASE(3, 256)
    S2W_WIG_CASE(4, 256)
    S2W_WIG_CASE(3, 512)
    S2W_WIG_CASE(4, 512)
#undef S2W_WIG_CASE
    return S2W_EINVAL;
}

// the TMA-staged inverse kernel: 3 stages per warp at 8 warps (two blocks per SM), 2 at 16 warps
template <int R, int MAXT>
int launch_inv_pre_tma(const WigArgs &A, int T, int chunks, cudaStream_t st)
{
    constexpr int STAGES = MAXT <= 256 ? 3 : 2;
    const size_t smem = (size_t)(MAXT / 32) * STAGES * (PreStage<R>::doubles * sizeof(double) + sizeof(unsigned long long));
    int rc = set_smem(precomp_inverse_tma_kernel<R, MAXT, STAGES>, smem);
    if (rc) return rc;
    dim3 grid(A.Lg, chunks);
    S2W_LAUNCH_C(S2W_K_WIGNER_INV, (precomp_inverse_tma_kernel<R, MAXT, STAGES>), grid, T, smem, st, A);
    return S2W_OK;
}

int dispatch_inv_pre(const WigArgs &A, const WigCfg &c, int chunks, cudaStream_t st)
{
    static const bool tma = [] {
        const char *e = getenv("S2W_PRE_TMA");
        return !(e && e[0] == '0');
    }();
    // small grids (one ring group per warp: L_j <= 256) keep the __ldg kernel: their 256-byte copies cost more than
    // they hide (ball, L = P = 128, precompute: 3.15 ms with TMA against 1.99 ms)
    if (tma && c.R >= 2) {
#define S2W_WIG_CASE(RR, MT) \
    if (c.R == RR && c.MAXT == MT) return launch_inv_pre_tma<RR, MT>(A, 32 * c.W, chunks, st);
        S2W_WIG_CASE(2, 256)
        S2W_WIG_CASE(3, 256)
        S2W_WIG_CASE(4, 256)
        S2W_WIG_CASE(3, 512)
        S2W_WIG_CASE(4, 512)
#undef S2W_WIG_CASE
    }
    static const int pre_nch = [] {
        const char *e = getenv("S2W_PRE_NCH");
        return e ? atoi(e) : 2;
    }();
    if (c.R == 1 && chunks >= 8 && pre_nch > 1) {  // one ring group per warp, many columns: several chunks per block
        if (pre_nch == 2) {
            dim3 grid(A.Lg, (chunks + 1) / 2);
            S2W_LAUNCH_C(S2W_K_WIGNER_INV, (precomp_inverse_kernel<1, 256, 2>), grid, 32 * c.W, 0, st, A);
        } else {
            dim3 grid(A.Lg, (chunks + 3) / 4);
            S2W_LAUNCH_C(S2W_K_WIGNER_INV, (precomp_inverse_kernel<1, 256, 4>), grid, 32 * c.W, 0, st, A);
        }
        return S2W_OK;
    }
#define S2W_WIG_CASE(RR, MT)                                                                                  \
    if (c.R == RR && c.MAXT == MT) {                                                                          \
        dim3 grid(A.Lg, chunks);                                                                              \
        S2W_LAUNCH_C(S2W_K_WIGNER_INV, (precomp_inverse_kernel<RR, MT>), grid, 32 * c.W, 0, st, A);            \
        return S2W_OK;                                                                                        \
    }
    S2W_WIG_CASE(1, 256)
    S2W_WIG_CASE(2, 256)
    S2W_WIG_CASE(3, 256)
    S2W_WIG_CASE(4, 256)
    S2W_WIG_CASE(3, 512)
    S2W_WIG_CASE(4, 512)
#undef S2W_WIG_CASE
    return S2W_EINVAL;
}

int launch_wigner(bool fwd, const WigArgs &A, cudaStream_t st)
{
    if (A.nn <= 0 || A.Lg <= 0) return S2W_OK;
    WigCfg c;
    if (!wig_cfg(A.G, c)) {
        set_error("band-limits above 2048 are not supported by the on-the-fly Wigner kernels");
        return S2W_EUNSUPPORTED;
    }
    const int CT = A.isReal ? A.B : 2 * A.B;
    if (fwd) return dispatch_fwd(A, c, (CT + 3) / 4, st);
    if (A.dtab) return dispatch_inv_pre(A, c, (CT + 3) / 4, st);
    if (A.F2) {  // two scales, one recursion: batches of at most two complex columns
        if (CT > 2) return S2W_EINVAL;
        return CT == 2 ? dispatch_inv<4, 2>(A, c, 1, st) : dispatch_inv<2, 2>(A, c, 1, st);
    }
    if (CT >= 3) return dispatch_inv<8, 1>(A, c, (CT + 3) / 4, st);
    if (CT == 2) return dispatch_inv<4, 1>(A, c, 1, st);
    return dispatch_inv<2, 1>(A, c, 1, st);
}

}  // namespace

int launch_wigner_seeds(const double *mant, const int *expo, const double *coef, size_t tri, int Lfull, int Lg, int nt, int G,
                        const int *n_vals, int ntab, const double *yv, const int *ring, int *gstart, double2 *dseed,
                        cudaStream_t st)
{
    NList nl;
    for (int i = 0; i < ntab; ++i) nl.v[i] = n_vals[i];
    dim3 grid(G, Lg, ntab);
    S2W_LAUNCH(wigner_seed_kernel, grid, 32, 0, st, mant, expo, coef, tri, Lfull, Lg, nt, G, nl, yv, ring, gstart, dseed, 0);
    const int count = Lg * ntab;
    S2W_LAUNCH(wigner_start_fix_kernel, (count + 127) / 128, 128, 0, st, gstart, G, count);
    S2W_LAUNCH(wigner_seed_kernel, grid, 32, 0, st, mant, expo, coef, tri, Lfull, Lg, nt, G, nl, yv, ring, gstart, dseed, 1);
    return S2W_OK;
}

int launch_wigner_seed_floor(const double *coef, size_t tri, int Lfull, int Lg, int G, int ntab, const double *yv,
                             const int *gstart, const double2 *dseed, int lfloor, int *gstart_f, double2 *dseed_f,
                             cudaStream_t st)
{
    dim3 grid(G, Lg, ntab);
    S2W_LAUNCH(wigner_seed_floor_kernel, grid, 32, 0, st, coef, tri, Lfull, Lg, G, yv, gstart, dseed, lfloor, gstart_f,
               dseed_f);
    return S2W_OK;
}

int launch_wigner_table(const double *coef, size_t tri, int Lfull, int Lg, int G, const int *n_vals, int ntab,
                        const double *yv, const int *gstart, const double2 *dseed, double *dtab, size_t tri_g,
                        cudaStream_t st)
{
    NList nl;
    for (int i = 0; i < ntab; ++i) nl.v[i] = n_vals[i];
    dim3 grid(G, Lg, ntab);
    S2W_LAUNCH(wigner_table_kernel, grid, 32, 0, st, coef, tri, Lfull, Lg, G, nl, yv, gstart, dseed, dtab, tri_g);
    return S2W_OK;
}

int launch_wigner_table_gather(const double *dtab, size_t tri_g, int tab, int n, int Lg, int nt, int G, const int *ring, cplx *X,
                               cudaStream_t st)
{
    dim3 grid(Lg, Lg);
    S2W_LAUNCH(wigner_table_gather_kernel, grid, 128, 0, st, dtab, tri_g, tab, n, Lg, nt, G, ring, X);
    return S2W_OK;
}

int launch_wigner_table_scatter(const cplx *Y, double *dtab_rw, size_t tri_g, int tab, int n, int Lg, int nt, int G,
                                const int *ring, cudaStream_t st)
{
    dim3 grid(Lg, Lg);
    S2W_LAUNCH(wigner_table_scatter_kernel, grid, 128, 0, st, Y, dtab_rw, tri_g, tab, n, Lg, nt, G, ring);
    return S2W_OK;
}

int launch_wigner_inverse(const WigArgs &A, cudaStream_t st) { return launch_wigner(false, A, st); }
int launch_wigner_forward(const WigArgs &A, cudaStream_t st) { return launch_wigner(true, A, st); }

// Wigner-Laguerre transform: the internal array of the signed row n holds f_{m,n} for m >= 0 and f_{m,-n} for m < 0 (the
// contraction kernels pair the column (m, n) with (-m, -n)); pos / neg are the user arrays [b][l][m+L-1] of n and -n.
int launch_flm_pack_pm(const cplx *pos, const cplx *neg, cplx *flmT, int B, int L, cudaStream_t st)
{
    dim3 grid((L + 127) / 128, 2 * L - 1, B);
    S2W_LAUNCH(flm_pack_pm_kernel, grid, 128, 0, st, pos, neg, flmT, L);
    return S2W_OK;
}
int launch_flm_unpack_pm(const cplx *flmT, cplx *pos, cplx *neg, int B, int L, cudaStream_t st)
{
    dim3 grid((L + 127) / 128, 2 * L - 1, B);
    S2W_LAUNCH(flm_unpack_pm_kernel, grid, 128, 0, st, flmT, pos, neg, L);
    return S2W_OK;
}

int launch_flm_pack(const cplx *flm_user, cplx *flmT, int B, int L, bool real, cudaStream_t st)
{
    dim3 grid((L + 127) / 128, real ? L : 2 * L - 1, B);
    S2W_LAUNCH(flm_pack_kernel, grid, 128, 0, st, flm_user, flmT, L, real ? 1 : 0);
    return S2W_OK;
}

int launch_flm_unpack(const cplx *flmT, cplx *flm_user, int B, int L, bool real, cudaStream_t st)
{
    dim3 grid((L + 127) / 128, 2 * L - 1, B);
    S2W_LAUNCH(flm_unpack_kernel, grid, 128, 0, st, flmT, flm_user, L, real ? 1 : 0);
    return S2W_OK;
}

int probe_fp64(int kind, double *tflops)
{
    double *d = 0;
    S2W_CUDA_CHECK(cudaMalloc(&d, 8));
    cudaDeviceProp prop;
    int dev = 0;
    S2W_CUDA_CHECK(cudaGetDevice(&dev));
    S2W_CUDA_CHECK(cudaGetDeviceProperties(&prop, dev));
    const int blocks = prop.multiProcessorCount * 8, iters = 20000;
    cudaEvent_t e0, e1;
    S2W_CUDA_CHECK(cudaEventCreate(&e0));
    S2W_CUDA_CHECK(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        S2W_CUDA_CHECK(cudaEventRecord(e0));
        if (kind == 0) {
            S2W_LAUNCH(dfma_probe_kernel, blocks, 256, 0, 0, d, iters, 0.999999, 1e-7);
        } else {
            S2W_LAUNCH(dmma_probe_kernel, blocks, 256, 0, 0, d, iters, 0.999999, 1e-7);
        }
        S2W_CUDA_CHECK(cudaEventRecord(e1));
        S2W_CUDA_CHECK(cudaEventSynchronize(e1));
        float ms = 0;
        S2W_CUDA_CHECK(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    S2W_CUDA_CHECK(cudaGetLastError());
    double flops;
    if (kind == 0)
        flops = (double)blocks * 256.0 * iters * 16.0 * 2.0;
    else
        flops = (double)blocks * 8.0 * iters * 4.0 * (2.0 * 8 * 8 * 4);
    *tflops = flops / (best * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    return S2W_OK;
}

}  // namespace s2w
