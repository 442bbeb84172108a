// plan.cu -- plans (cached tables) and the transform drivers behind the C ABI of include/s2w.h.
//
// Sphere analysis (Alg. 1), with the step names of DESIGN.md:
//   a1 ring DFT -> a2 reweight -> a3 forward SHT contraction  (f_lm, kept m-major on the device)
//   scaling: a7-type contraction at L_s with filter Phi_l0 -> a1 inverse                   (Eq. 29/41)
//   each j : a4+a5 filter x inverse Wigner contraction at L_j -> a8 (alpha, gamma) DFT       (Eq. 27/40)
// Sphere synthesis (Alg. 1) runs the mirror image and accumulates into f_lm     (Eq. 42).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "fft_core.cuh"
#include "host_math.h"
#include "kernels.h"

namespace s2w {

static thread_local std::string g_err;
static unsigned long long g_launches = 0;
void set_error(const std::string &msg) { g_err = msg; }
void count_launch() { ++g_launches; }
void debug_launch(const char *name)
{
    static const char *env = getenv("S2W_DEBUG_LAUNCH");
    if (!env) return;
    static bool reported = false;
    // "2": wait for the kernel, so that a fault is attributed to the launch that caused it (never under stream capture)
    const cudaError_t e = env[0] == '2' ? cudaDeviceSynchronize() : cudaPeekAtLastError();
    if (e != cudaSuccess && !reported) {
        reported = true;
        fprintf(stderr, "[s2w] launch of %s left the error: %s\n", name, cudaGetErrorString(e));
    }
}

// ---- per-class device timers: cudaEvent pairs around every launch while enabled (s2w_timing_enable/read) ----
namespace {
struct TimedLaunch {
    cudaEvent_t a, b;
    int cls;
};
bool g_timing = false;
std::vector<TimedLaunch> g_timed;     // recorded since the last read
std::vector<TimedLaunch> g_ev_free;   // recycled event pairs
std::mutex g_timing_mu;
}  // namespace
void timing_begin(int cls, cudaStream_t st)
{
    if (!g_timing) return;
    std::lock_guard<std::mutex> lock(g_timing_mu);
    TimedLaunch t;
    if (!g_ev_free.empty()) {
        t = g_ev_free.back();
        g_ev_free.pop_back();
    } else {
        if (cudaEventCreate(&t.a) != cudaSuccess || cudaEventCreate(&t.b) != cudaSuccess) return;
    }
    t.cls = cls;
    cudaEventRecord(t.a, st);
    g_timed.push_back(t);
}
void timing_end(cudaStream_t st)
{
    if (!g_timing) return;
    std::lock_guard<std::mutex> lock(g_timing_mu);
    if (!g_timed.empty()) cudaEventRecord(g_timed.back().b, st);
}

namespace {

typedef long double ld;
const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

struct DevPool {  // owns device allocations of a plan
    std::vector<void *> ptrs;
    template <typename T>
    int alloc(T **p, size_t count)
    {
        void *q = 0;
        cudaError_t e = cudaMalloc(&q, std::max<size_t>(count, 1) * sizeof(T));
        if (e != cudaSuccess) {
            set_error(std::string("cudaMalloc: ") + cudaGetErrorString(e));
            cudaGetLastError();
            return e == cudaErrorMemoryAllocation ? S2W_ENOMEM : S2W_ECUDA;
        }
        ptrs.push_back(q);
        *p = (T *)q;
        return S2W_OK;
    }
    template <typename T>
    int upload(T **p, const std::vector<T> &h)
    {
        int rc = alloc(p, h.size());
        if (rc) return rc;
        if (!h.empty()) S2W_CUDA_CHECK(cudaMemcpy(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
        return S2W_OK;
    }
    void release()
    {
        for (void *p : ptrs) cudaFree(p);
        ptrs.clear();
    }
};

struct GridTab {  // everything that depends on the theta/phi grid of band-limit Lg
    int Lg;
    FftTab fft;
    RwTab rw;        // Toeplitz/Hankel reweighting tables (rw.L = 0 on tiny grids)
    int nt;          // rings: Lg (McEwen-Wiaux) or 2 Lg (Driscoll-Healy)
    double *dhw;     // Driscoll-Healy: [nt] (2 Lg - 1) q_t, the quadrature weights in the normalisation of the contraction
                     // stages' filters (which carry 1/(2 Lg - 1)); null on McEwen-Wiaux grids
    int G;           // ring groups of 32 (even): 2j north, 2j+1 south, each hemisphere sorted by |cos beta|
    double *yv;      // [32 G] 1 - |cos beta_t| of the ring in each slot
    int *ring;       // [32 G] ring index t, -1 for an empty slot
    int *gstart;     // [ntab][Lg][G]
    double2 *dseed;  // [ntab][Lg][32 G]
    double *dtab;    // S2W_PRECOMPUTE: [ntab][Lg (Lg+1)/2][32 G] d^l_mn(beta) per ring slot (else null)
    double *dtab_rw; // S2W_PRECOMPUTE, McEwen-Wiaux grids with Lg <= S2W_FOLD_MAX_L: the same table with the theta quadrature
                     // folded in, (R_sigma d^l_mn)(theta_t): the rings -> harmonic contraction then takes F transposed, and
                     // the reweighting step (a2) disappears from the transform (else null)
};

struct Stage {  // one Wigner contraction launch: rows, filters
    int grid;   // index into plan->grids
    int Lg;
    int lmin;
    int nn, nrows;
    int n_val[S2W_MAX_ROWS], n_tab[S2W_MAX_ROWS], n_row[S2W_MAX_ROWS], n_rowm[S2W_MAX_ROWS], n_filtm[S2W_MAX_ROWS];
    cplx *filt_ana;  // [nn][Lg]  harmonic -> rings
    cplx *filt_syn;  // [nn][Lg]  rings -> harmonic
    // adjoint transforms: c conj(filt_ana) for the rings -> harmonic contraction that is the adjoint
    // of this stage's harmonic -> rings one, conj(filt_syn) / c for the other direction; c = number of (alpha, gamma)
    // or phi samples per ring, the factor between the unnormalised inverse DFT and the adjoint of the normalised one
    cplx *filt_ana_adj;
    cplx *filt_syn_adj;
    // start degrees and seeds of the recursion advanced to lmin (0: the grid's own tables): a stage whose filter
    // support begins at lmin does not re-run the recursion from each group's start up to lmin at every transform
    int *gstart_f;
    double2 *dseed_f;
};

struct Scale {
    int j, jp;
    int Lj, Pj;
    size_t offset;  // element offset in one signal's coefficient block
    Stage st;
    double *Kinv;   // ball: [Pj nodes][Pj p]   K_p(r_i) kappa^{j'}(p) on the Pj-node grid       (analysis)
    double *Kfwd;   // ball: [Pj p][Pj nodes]   q_i K_p(r_i) kappa^{j'}(p)                       (synthesis)
    double *KinvT, *KfwdT;  // their transposes (adjoint transforms)
};

}  // namespace
}  // namespace s2w

using namespace s2w;

#define S2W_LANES 4  // most lanes a captured sphere transform uses (workspace is sized for them)
#define S2W_BALL_LANES 2  // streams the angular scales of a stacked ball transform are dealt to

struct s2w_plan {
    int kind;  // 0 sphere, 1 ball
    int L, N, P, J0, J, J0p, Jp, multires, flags, batch, device;
    double lambda, nu, tau;
    bool real;
    DevPool pool;
    std::vector<GridTab> grids;
    int spin;               // spin number s of the signal (spin fields: Eq. 1): the SHT stages contract with d^l_{m,-s}
    std::vector<int> tabn;  // table values of n: script-N united with {-spin, +spin}
    double *coef;
    size_t tri;
    cplx *tw;
    int Mtab;
    Stage sht;       // plain spherical harmonic transform at L (filters c_l and (2 pi/n) c_l)
    Stage scaling;   // scaling coefficients at L_s
    int Ls;
    size_t scaling_offset;
    std::vector<Scale> scales;
    size_t coeff_elems, signal_elems;
    size_t ws_flm_elems, ws_F_elems, ws_bytes;
    // ball
    double *Kfull_fwd;  // [P p][P nodes]  q_i K_p(r_i)
    double *Kfull_inv;  // [P nodes][P p]  K_p(r_i)
    double *Kfull_fwdT, *Kfull_invT;  // their transposes (adjoint transforms)
    double *phi_ball;   // [P][L] sqrt(4pi/(2l+1)) Phi_{l0p}
    size_t ws_shell_elems;  // ball: elements of one [P][Mfull][L] harmonic array
    // ball, stacked shells: for a fixed angular scale j the radial scales j' differ only in their shell count P_j' and
    // share grid, filters and tables, so the shells of ALL j' are stacked (PS = sum_j' P_j') and every step of a scale j
    // is ONE launch over PS shells instead of one per (j, j') (Alg. 2)
    // kind 2: Wigner-Laguerre plan (Q = K D on H^4 = R+ x SO(3), Eqs. 24-25): one single-row stage per signed n whose
    // mirror columns land in the row of -n, and a stage listing all rows for the (alpha, gamma) FFT and the reweighting
    std::vector<Stage> qst;
    Stage qall;
    int dh;                       // S2W_DH: Driscoll-Healy sampling (2 L_j rings per grid), sphere plans only
    int PS;                       // stacked shells
    std::vector<Scale> ang;       // the angular stage of each j (Pj = PS)
    std::vector<size_t *> ang_off;  // device [PS]: element offset of stacked shell b's block of scale j in a coefficient array
    double *Kstk_inv;             // [PS nodes][P p]   rows of scale j': K_p(r_i) kappa^{j'}(p), zero for p >= P_j'
    double *Kstk_fwd;             // [P p][PS nodes]   q_i K_p(r_i) kappa^{j'}(p)
    int2 *krange_inv, *krange_fwd;  // per 64-row tile of the two matrices: the k range that holds non-zeros
    size_t ws_stk_elems, ws_stkF_elems, ws_stk_off;  // stacked harmonic array, one F buffer, offset of this part (elements)
    // CUDA graphs of whole transforms (s2w_plan_forward / s2w_plan_inverse), keyed by direction and buffer addresses:
    // a transform is 40 (sphere) to 900 (ball) small launches, replayed as one graph launch after its first call.
    // The only mutable state of a plan; guarded by graph_mu.
    struct GraphEntry {
        int dir;
        const void *in;
        void *out, *work;
        cudaGraphExec_t exec;
        unsigned long long launches;
    };
    mutable std::vector<GraphEntry> graphs;
    mutable cudaStream_t capture_stream;
    mutable std::mutex graph_mu;
    // lanes of a captured sphere transform (sphere_forward / sphere_inverse): the scales are independent, so they are
    // dealt to S2W_LANES streams of the graph, each with its own F buffers (largest scale first, to the lane with the
    // least work so far)
    mutable cudaStream_t lane_stream[S2W_LANES - 1];
    mutable cudaEvent_t lane_fork, lane_join[S2W_LANES - 1];
    mutable bool lanes_on;  // set by run_transform while it captures
};

namespace s2w {
namespace {

int find_tab(const s2w_plan *p, int n)
{
    for (size_t i = 0; i < p->tabn.size(); ++i)
        if (p->tabn[i] == n) return (int)i;
    return -1;
}

int grid_index(s2w_plan *p, int Lg)
{
    for (size_t i = 0; i < p->grids.size(); ++i)
        if (p->grids[i].Lg == Lg) return (int)i;
    return -1;
}

int ceil_log2(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

// Range-extended seeds d^{l0}_{mn}(beta_t), l0 = max(m,|n|), m >= 0, as mantissa * 2^expo (long double arithmetic):
//   d^m_{mn} = sqrt((2m)!/((m+n)!(m-n)!)) cos^{m+n}(beta/2) (-sin(beta/2))^{m-n}   for m >= |n|,
// built by the one-term recursion in m, and for m < |n| from d^l_{mn} = (-1)^{m-n} d^l_{nm} = d^l_{-n,-m}.
// rings beta_t, t < nt: McEwen-Wiaux pi (2t+1)/(2 Lg - 1), nt = Lg; Driscoll-Healy pi (2t+1)/(4 Lg), nt = 2 Lg
void host_seeds(int Lg, int nt, bool dh, const std::vector<int> &tabn, std::vector<double> &mant, std::vector<int> &expo,
                std::vector<double> &yv, std::vector<int> &ring, int &G)
{
    const size_t per = (size_t)Lg * nt;
    mant.assign(tabn.size() * per, 0.0);
    expo.assign(tabn.size() * per, 0);
    std::vector<ld> ch(nt), sh(nt);
    // ring groups: each hemisphere sorted by |cos beta| ascending, y = 1 - |cos beta| = 2 sin^2(beta/2) or 2 cos^2(beta/2)
    std::vector<std::pair<ld, int> > hemi[2];
    for (int t = 0; t < nt; ++t) {
        ld beta = dh ? PI_L * (ld)(2 * t + 1) / (ld)(4 * Lg) : PI_L * (ld)(2 * t + 1) / (ld)(2 * Lg - 1);
        ch[t] = cosl(beta / 2);
        sh[t] = sinl(beta / 2);
        const bool south = dh ? t >= Lg : 4 * t + 2 > 2 * Lg - 1;  // beta > pi/2
        const ld y = south ? 2 * ch[t] * ch[t] : 2 * sh[t] * sh[t];
        hemi[south ? 1 : 0].push_back(std::make_pair(-y, t));  // |cos| ascending = y descending
    }
    std::sort(hemi[0].begin(), hemi[0].end());
    std::sort(hemi[1].begin(), hemi[1].end());
    const size_t most = std::max(hemi[0].size(), hemi[1].size());
    G = 2 * (int)std::max<size_t>(1, (most + 31) / 32);
    yv.assign((size_t)32 * G, 0.0);
    ring.assign((size_t)32 * G, -1);
    for (int h = 0; h < 2; ++h)
        for (size_t i = 0; i < hemi[h].size(); ++i) {
            const size_t slot = ((i / 32) * 2 + h) * 32 + i % 32;
            yv[slot] = (double)(-hemi[h][i].first);
            ring[slot] = hemi[h][i].second;
        }
    auto put = [&](size_t idx, ld v) {
        int e = 0;
        ld mnt = frexpl(v, &e);
        mant[idx] = (double)mnt;
        expo[idx] = e;
    };
    // S(l0, q) at ring t by direct product (only used for l0 = |n| <= N-1)
    auto S_direct = [&](int l0, int q, int t) -> ld {
        int a = l0 + q, b = l0 - q;
        ld v = 1;
        for (int i = 1; i <= b; ++i) v *= sqrtl((ld)(a + i) / (ld)i) * (-sh[t]);
        for (int i = 1; i <= a; ++i) v *= ch[t];
        return v;
    };
    std::vector<ld> ratio(Lg + 1);
    for (size_t tab = 0; tab < tabn.size(); ++tab) {
        const int n = tabn[tab], an = n < 0 ? -n : n;
        if (an >= Lg) continue;
        for (int m = an; m + 1 < Lg; ++m)
            ratio[m] = sqrtl((ld)(2 * m + 2) * (ld)(2 * m + 1) / ((ld)(m + 1 + n) * (ld)(m + 1 - n)));
        for (int t = 0; t < nt; ++t) {
            // m < |n|
            for (int m = 0; m < an; ++m) {
                ld v;
                if (n > 0)
                    v = (((an - m) & 1) ? -1 : 1) * S_direct(an, m, t);
                else
                    v = S_direct(an, -m, t);
                put((tab * Lg + m) * (size_t)nt + t, v);
            }
            // m >= |n|
            ld s = 1;
            if (n >= 0)
                for (int i = 0; i < 2 * an; ++i) s *= ch[t];
            else
                for (int i = 0; i < 2 * an; ++i) s *= sh[t];
            const ld cs = -ch[t] * sh[t];
            for (int m = an; m < Lg; ++m) {
                put((tab * Lg + m) * (size_t)nt + t, s);
                if (m + 1 < Lg) s *= ratio[m] * cs;
            }
        }
    }
}

// Recursion coefficients of the step l -> l+1 in difference form (wigner.cu), packed rows l = m..L-1 for every m >= 0
// and every table value of n: (alpha_l, gamma_l, e_N, e_S), e_N/S = alpha_l - gamma_l - 1 -/+ beta_l, formed in long
// double so that the cancellation in e leaves a correctly rounded double.  Entries with l < |n| are zero.
void host_coef(int L, const std::vector<int> &tabn, std::vector<double> &coef)
{
    const size_t tri = (size_t)L * (L + 1) / 2;
    coef.assign(tabn.size() * tri * 4, 0.0);
    for (size_t tab = 0; tab < tabn.size(); ++tab) {
        const int n = tabn[tab], an = n < 0 ? -n : n;
        size_t o = tab * tri * 4;
        for (int m = 0; m < L; ++m)
            for (int l = m; l < L; ++l, o += 4) {
                if (l < an) continue;
                ld a = 1, b = 0, g = 0;
                if (l > 0) {
                    const ld lp = l + 1, lq = l, md = m, nd = n;
                    a = lp * (2 * lq + 1) / sqrtl((lp * lp - md * md) * (lp * lp - nd * nd));
                    b = a * md * nd / (lq * lp);
                    g = a * sqrtl((lq * lq - md * md) * (lq * lq - nd * nd)) / (lq * (2 * lq + 1));
                }
                coef[o] = (double)a;
                coef[o + 1] = (double)g;
                coef[o + 2] = (double)(a - g - 1 - b);
                coef[o + 3] = (double)(a - g - 1 + b);
            }
    }
}

// Tables of the Toeplitz/Hankel reweighting (ring_fft.cu, reweight_th_kernel) for band-limit L >= 8, in long double.
// With n = 2L-1 and theta_t = pi (2t+1)/n, K[t,s] = sum_{|k|,|k'| < L} w(k+k') e^{-i(k theta_s + k' theta_t)},
// w(q) = int_0^pi e^{i q theta} sin(theta) dtheta (reading R3), one finds K[t,s] = (-1)^{t-s} (c_t - c_s)/sin(pi (t-s)/n)
// off the diagonal; c_t (with c_0 = 0) is read off the first column, the diagonal is summed directly.
struct RwHost {
    std::vector<double> delta, dsum, vpole, rpole, kT, kG;
    int M2, logM2;
};
void host_rw_tables(int L, RwHost &H)
{
    const int n = 2 * L - 1, Lm = L - 1;
    std::vector<ld> cs(2 * n), sn(2 * n);
    for (int j = 0; j < 2 * n; ++j) {
        cs[j] = cosl(PI_L * (ld)j / (ld)n);
        sn[j] = sinl(PI_L * (ld)j / (ld)n);
    }
    auto idx = [&](long long a) {  // a mod 2n
        long long r = a % (2LL * n);
        return (int)(r < 0 ? r + 2LL * n : r);
    };
    // G0(k') = sum_k w(k+k') e^{-i k theta_0};  w even q: 2/(1-q^2) real, q = +-1: +-i pi/2
    std::vector<ld> g0r(n), g0i(n);
    for (int kp = -(L - 1); kp <= L - 1; ++kp) {
        ld ar = 0, ai = 0;
        for (int k = -(L - 1); k <= L - 1; ++k) {
            const int q = k + kp;
            const int J = idx(k);  // e^{-i k theta_0} = cs[J] - i sn[J]
            if ((q & 1) == 0) {
                const ld w = 2 / (1 - (ld)q * (ld)q);
                ar += w * cs[J];
                ai -= w * sn[J];
            } else if (q == 1 || q == -1) {
                const ld w = (q == 1 ? 1 : -1) * PI_L / 2;  // i w (cs - i sn) = w sn + i w cs
                ar += w * sn[J];
                ai += w * cs[J];
            }
        }
        g0r[kp + L - 1] = ar;
        g0i[kp + L - 1] = ai;
    }
    std::vector<ld> c(n), kd(n);
    for (int t = 0; t < n; ++t) {
        ld re = 0;
        for (int kp = -(L - 1); kp <= L - 1; ++kp) {
            const int J = idx((long long)kp * (2 * t + 1));  // e^{-i k' theta_t}
            re += g0r[kp + L - 1] * cs[J] + g0i[kp + L - 1] * sn[J];
        }
        c[t] = ((t & 1) ? -1 : 1) * re * sn[t];
        // diagonal: sum_q w(q) (n - |q|) e^{-i q theta_t}
        ld d = 2 * (ld)n + PI_L * (ld)(n - 1) * sn[idx(2 * t + 1)];
        for (int q = 2; q <= 2 * L - 2; q += 2)
            d += 2 * (2 / (1 - (ld)q * (ld)q)) * (ld)(n - q) * cs[idx((long long)q * (2 * t + 1))];
        kd[t] = d;
    }
    auto K = [&](int t, int s) -> ld {
        if (t == s) return kd[t];
        const int d = t - s;
        const ld sd = d > 0 ? sn[d] : -sn[-d];
        return ((d & 1) ? -1 : 1) * (c[t] - c[s]) / sd;
    };
    H.delta.assign(L, 0.0);
    H.dsum.assign(L, 0.0);
    H.vpole.assign(2 * (size_t)L, 0.0);
    H.rpole.assign(2 * (size_t)L, 0.0);
    for (int t = 0; t < Lm; ++t) {
        H.delta[t] = (double)(c[t] - c[n - 1 - t]);
        H.dsum[t] = (double)((kd[t] + kd[n - 1 - t]) / n);
        for (int par = 0; par < 2; ++par) {
            const ld sg = par ? -1 : 1;
            H.vpole[(size_t)par * L + t] = (double)((K(t, L - 1) + sg * K(n - 1 - t, L - 1)) / n);
            H.rpole[(size_t)par * L + t] = (double)((K(L - 1, t) + sg * K(L - 1, n - 1 - t)) / n);
        }
    }
    H.rpole[L - 1] = H.rpole[(size_t)L + L - 1] = (double)(kd[L - 1] / n);
    H.logM2 = std::max(1, ceil_log2(2 * Lm - 1));
    H.M2 = 1 << H.logM2;
    H.kT.assign(H.M2, 0.0);
    H.kG.assign(H.M2, 0.0);
    const ld scale = 1 / ((ld)n * (ld)H.M2);
    for (int d = -(Lm - 1); d <= Lm - 1; ++d) {
        const int slot = d < 0 ? d + H.M2 : d;
        if (d != 0) H.kT[slot] = (double)(scale / (d > 0 ? sn[d] : -sn[-d]));
        H.kG[slot] = (double)(scale / sn[d + Lm]);
    }
}

int build_rw(s2w_plan *p, GridTab &g)
{
    const int L = g.Lg;
    memset(&g.rw, 0, sizeof(g.rw));
    if (L < 8) return S2W_OK;
    RwHost H;
    host_rw_tables(L, H);
    const int M2 = H.M2, Lm = L - 1;
    FftTab &T = g.rw.fft;
    T.n = 0;
    T.L = L;
    T.logM = H.logM2;
    T.M = M2;
    T.tw = p->tw;
    T.twmul = p->Mtab / M2;
    T.twmask = p->Mtab - 1;
    T.twlo = std::min(6, ceil_log2(p->Mtab));
    // spectra in the transform's own (digit-reversed) order, and that order itself from the transform of e_1
    std::vector<cplx> hbuf((size_t)3 * M2, cmake(0.0, 0.0));
    for (int i = 0; i < M2; ++i) {
        hbuf[i] = cmake(H.kT[i], 0.0);
        hbuf[(size_t)M2 + i] = cmake(H.kG[i], 0.0);
    }
    hbuf[(size_t)2 * M2 + 1] = cmake(1.0, 0.0);
    cplx *dbuf;
    int rc;
    if ((rc = p->pool.upload(&dbuf, hbuf))) return rc;
    for (int a = 0; a < 3; ++a)
        if ((rc = launch_fft_forward(dbuf + (size_t)a * M2, T, 0))) return rc;
    S2W_CUDA_CHECK(cudaMemcpy(hbuf.data(), dbuf, hbuf.size() * sizeof(cplx), cudaMemcpyDeviceToHost));
    std::vector<int> kof(M2), pos(M2, -1), negpos(M2);
    for (int q = 0; q < M2; ++q) {
        const cplx v = hbuf[(size_t)2 * M2 + q];  // exp(-2 pi i k / M2)
        long long k = llround(-std::atan2(v.y, v.x) * (double)M2 / (2.0 * pi_d()));
        k %= M2;
        if (k < 0) k += M2;
        kof[q] = (int)k;
        pos[k] = q;
    }
    for (int k = 0; k < M2; ++k)
        if (pos[k] < 0) {
            set_error("internal error: transform order is not a permutation");
            return S2W_ECUDA;
        }
    for (int q = 0; q < M2; ++q) {
        negpos[q] = pos[(M2 - kof[q]) % M2];
        // reversal phase of the Hankel part: exp(-2 pi i k (Lm - 1) / M2)
        const long long j = ((long long)kof[q] * (Lm - 1)) % M2;
        const ld ang = -2 * PI_L * (ld)j / (ld)M2;
        const ld pr = cosl(ang), pi_ = sinl(ang);
        const cplx gq = hbuf[(size_t)M2 + q];
        hbuf[(size_t)M2 + q] = cmake((double)(gq.x * pr - gq.y * pi_), (double)(gq.x * pi_ + gq.y * pr));
    }
    std::vector<int2> pairs;
    std::vector<cplx> tg;
    for (int q = 0; q < M2; ++q) {
        const int qn = negpos[q];
        if (qn < q) continue;
        pairs.push_back(make_int2(q, qn));
        tg.push_back(hbuf[q]);
        tg.push_back(hbuf[(size_t)M2 + q]);
        tg.push_back(hbuf[qn]);
        tg.push_back(hbuf[(size_t)M2 + qn]);
    }
    int2 *dpairs;
    cplx *dtg;
    double *dd, *ds, *dv, *dr;
    if ((rc = p->pool.upload(&dpairs, pairs))) return rc;
    if ((rc = p->pool.upload(&dtg, tg))) return rc;
    g.rw.npairs = (int)pairs.size();
    g.rw.pairs = dpairs;
    g.rw.TG = dtg;
    if ((rc = p->pool.upload(&dd, H.delta))) return rc;
    if ((rc = p->pool.upload(&ds, H.dsum))) return rc;
    if ((rc = p->pool.upload(&dv, H.vpole))) return rc;
    if ((rc = p->pool.upload(&dr, H.rpole))) return rc;
    g.rw.delta = dd;
    g.rw.dsum = ds;
    g.rw.vpole = dv;
    g.rw.rpole = dr;
    g.rw.L = L;
    if (M2 == 4096 || M2 == 2048 || M2 == 1024 || M2 == 512 || M2 == 256) {
        // the same two spectra in the order of the radix-16 core (fft16_core.cuh), which is read off the transform of e_1
        std::vector<cplx> h16((size_t)3 * M2, cmake(0.0, 0.0));
        for (int i = 0; i < M2; ++i) {
            h16[i] = cmake(H.kT[i], 0.0);
            h16[(size_t)M2 + i] = cmake(H.kG[i], 0.0);
        }
        h16[(size_t)2 * M2 + 1] = cmake(1.0, 0.0);
        cplx *d16;
        if ((rc = p->pool.upload(&d16, h16))) return rc;
        for (int a = 0; a < 3; ++a)
            if ((rc = launch_fft16_forward(d16 + (size_t)a * M2, M2, 0))) return rc;
        S2W_CUDA_CHECK(cudaMemcpy(h16.data(), d16, h16.size() * sizeof(cplx), cudaMemcpyDeviceToHost));
        std::vector<cplx> tg16((size_t)2 * M2);
        const int R1 = M2 / 256;
        for (int q = 0; q < M2; ++q) {
            const cplx v = h16[(size_t)2 * M2 + q];  // exp(-2 pi i k / M2)
            long long k = llround(-std::atan2(v.y, v.x) * (double)M2 / (2.0 * pi_d()));
            k %= M2;
            if (k < 0) k += M2;
            // launch_fft16_forward stores position p = j1 256 + j2 16 + j3 (frequency j1 + R1 (j2 + 16 j3)) at
            // q = j1 256 + j3 16 + j2 (F16_TPOS)
            if (k != (q >> 8) + R1 * ((q & 15) + 16 * ((q >> 4) & 15))) {
                set_error("internal error: the radix-16 transform's order is not the documented one");
                return S2W_ECUDA;
            }
            const long long j = (k * (Lm - 1)) % M2;  // reversal phase of the Hankel part
            const ld ang = -2 * PI_L * (ld)j / (ld)M2;
            const ld pr = cosl(ang), pi_ = sinl(ang);
            const cplx gq = h16[(size_t)M2 + q];
            tg16[q] = h16[q];
            tg16[(size_t)M2 + q] = cmake((double)(gq.x * pr - gq.y * pi_), (double)(gq.x * pi_ + gq.y * pr));
        }
        cplx *dtg16;
        if ((rc = p->pool.upload(&dtg16, tg16))) return rc;
        g.rw.TG16 = dtg16;
    }
    return S2W_OK;
}

// largest band-limit of a grid whose precomputed table also gets the quadrature-folded copy (GridTab::dtab_rw): small
// grids, where the reweighting kernels cost more than the contraction saves by skipping the rings below a group start
static int fold_max_l()
{
    static const int v = [] {
        const char *e = getenv("S2W_FOLD_MAX_L");
        return e ? atoi(e) : 256;
    }();
    return v;
}

int build_grid(s2w_plan *p, int Lg)
{
    if (grid_index(p, Lg) >= 0) return S2W_OK;
    GridTab g;
    memset(&g, 0, sizeof(g));
    g.Lg = Lg;
    FftTab &T = g.fft;
    T.n = 2 * Lg - 1;
    T.L = Lg;
    T.logM = std::max(1, ceil_log2(2 * T.n - 1));
    T.M = 1 << T.logM;
    T.tw = p->tw;
    T.twmul = p->Mtab / T.M;
    T.twmask = p->Mtab - 1;
    T.twlo = std::min(6, ceil_log2(p->Mtab));
    cplx *chirp, *i1, *o1, *i3, *o3, *bm, *bp, *wh;
    int rc;
    if ((rc = p->pool.alloc(&chirp, T.n))) return rc;
    if ((rc = p->pool.alloc(&i1, T.n))) return rc;
    if ((rc = p->pool.alloc(&o1, T.n))) return rc;
    if ((rc = p->pool.alloc(&i3, T.n))) return rc;
    if ((rc = p->pool.alloc(&o3, T.n))) return rc;
    if ((rc = p->pool.alloc(&bm, T.M))) return rc;
    if ((rc = p->pool.alloc(&bp, T.M))) return rc;
    if ((rc = p->pool.alloc(&wh, T.M))) return rc;
    T.chirp = chirp;
    T.rw_in1 = i1;
    T.rw_out1 = o1;
    T.rw_in3 = i3;
    T.rw_out3 = o3;
    T.bhat_m = bm;
    T.bhat_p = bp;
    T.what = wh;
    if ((rc = launch_fft_tables(T, chirp, i1, o1, i3, o3, bm, bp, wh, 0))) return rc;
    if (f16_supported(T.M)) {  // the Bluestein spectra in the order of the radix-16 core
        cplx *bm16, *bp16;
        if ((rc = p->pool.alloc(&bm16, T.M))) return rc;
        if ((rc = p->pool.alloc(&bp16, T.M))) return rc;
        if ((rc = launch_fft16_spectrum(bm16, 0, T.n, T.M, 0))) return rc;
        if ((rc = launch_fft16_spectrum(bp16, 1, T.n, T.M, 0))) return rc;
        T.bhat16_m = bm16;
        T.bhat16_p = bp16;
    }
    g.nt = p->dh ? 2 * Lg : Lg;
    T.nt = g.nt;
    if (Lg == 1024 && !p->dh && (rc = pfa2047_init(0))) return rc;  // Rader spectra of the 2047-sample prime-factor kernels
    if (p->dh) {
        // Driscoll-Healy quadrature (their Theorem 3): q_t = (2/L) sin(theta_t) sum_{k<L} sin((2k+1) theta_t)/(2k+1)
        memset(&g.rw, 0, sizeof(g.rw));
        std::vector<double> w(g.nt);
        for (int t = 0; t < g.nt; ++t) {
            const ld th = PI_L * (ld)(2 * t + 1) / (ld)(4 * Lg);
            ld acc = 0;
            for (int k = 0; k < Lg; ++k) acc += sinl((ld)(2 * k + 1) * th) / (ld)(2 * k + 1);
            w[t] = (double)((ld)(2 * Lg - 1) * 2 / (ld)Lg * sinl(th) * acc);
        }
        if ((rc = p->pool.upload(&g.dhw, w))) return rc;
    } else if ((rc = build_rw(p, g)))
        return rc;

    std::vector<double> mant, yv;
    std::vector<int> expo, ring;
    host_seeds(Lg, g.nt, p->dh != 0, p->tabn, mant, expo, yv, ring, g.G);
    double *dmant;
    int *dexpo;
    if ((rc = p->pool.upload(&g.yv, yv))) return rc;
    if ((rc = p->pool.upload(&g.ring, ring))) return rc;
    // temporaries (freed after the seed kernels)
    const size_t cnt = mant.size();
    const size_t ntab = p->tabn.size();
    S2W_CUDA_CHECK(cudaMalloc((void **)&dmant, std::max<size_t>(cnt, 1) * sizeof(double)));
    S2W_CUDA_CHECK(cudaMalloc((void **)&dexpo, std::max<size_t>(cnt, 1) * sizeof(int)));
    S2W_CUDA_CHECK(cudaMemcpy(dmant, mant.data(), cnt * sizeof(double), cudaMemcpyHostToDevice));
    S2W_CUDA_CHECK(cudaMemcpy(dexpo, expo.data(), cnt * sizeof(int), cudaMemcpyHostToDevice));
    if ((rc = p->pool.alloc(&g.gstart, ntab * Lg * g.G))) return rc;
    if ((rc = p->pool.alloc(&g.dseed, ntab * Lg * (size_t)32 * g.G))) return rc;
    rc = launch_wigner_seeds(dmant, dexpo, p->coef, p->tri, p->L, Lg, g.nt, g.G, p->tabn.data(), (int)ntab, g.yv, g.ring,
                             g.gstart, g.dseed, 0);
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(dmant);
    cudaFree(dexpo);
    if (rc) return rc;
    if (e != cudaSuccess) {
        set_error(std::string("plan set-up kernels: ") + cudaGetErrorString(e));
        return S2W_ECUDA;
    }
    if (p->flags & S2W_PRECOMPUTE) {
        const size_t tri_g = (size_t)Lg * (Lg + 1) / 2;
        const size_t elems = ntab * tri_g * (size_t)32 * g.G;
        if ((rc = p->pool.alloc(&g.dtab, elems))) {
            if (rc == S2W_ENOMEM) set_error("the precomputed Wigner-d table does not fit in device memory");
            return rc;
        }
        S2W_CUDA_CHECK(cudaMemsetAsync(g.dtab, 0, elems * sizeof(double), 0));
        if ((rc = launch_wigner_table(p->coef, p->tri, p->L, Lg, g.G, p->tabn.data(), (int)ntab, g.yv, g.gstart, g.dseed,
                                      g.dtab, tri_g, 0)))
            return rc;
        S2W_CUDA_CHECK(cudaDeviceSynchronize());
        if (!p->dh && g.rw.L && Lg <= fold_max_l()) {
            // sum_t d(theta_t) (R F)(theta_t) = sum_t (R d)(theta_t) F(theta_t), R real symmetric: run the
            // reweighting kernels once over the table's columns (ring index t at fixed (l, m, n)) instead of over every
            // transform's columns
            if ((rc = p->pool.alloc(&g.dtab_rw, elems))) return rc;
            S2W_CUDA_CHECK(cudaMemsetAsync(g.dtab_rw, 0, elems * sizeof(double), 0));
            cplx *X = 0, *Y = 0;
            const size_t slab = (size_t)Lg * g.nt * Lg;
            if (cudaMalloc((void **)&X, slab * sizeof(cplx)) != cudaSuccess || cudaMalloc((void **)&Y, slab * sizeof(cplx)) != cudaSuccess) {
                cudaFree(X);
                cudaGetLastError();
                set_error("no device memory for the set-up buffers of the quadrature-folded table");
                return S2W_ENOMEM;
            }
            for (size_t tab = 0; tab < ntab && !rc; ++tab) {
                RwArgs R;
                memset(&R, 0, sizeof(R));
                R.nn = 1;
                R.nrows = 1;
                R.Md = Lg;
                R.isReal = 1;
                R.n_val[0] = p->tabn[tab];
                R.n_row[0] = 0;
                rc = launch_wigner_table_gather(g.dtab, tri_g, (int)tab, p->tabn[tab], Lg, g.nt, g.G, g.ring, X, 0);
                if (!rc) rc = launch_reweight_th(X, Y, R, Lg, g.rw, 0);
                if (!rc) rc = launch_wigner_table_scatter(Y, g.dtab_rw, tri_g, (int)tab, p->tabn[tab], Lg, g.nt, g.G, g.ring, 0);
            }
            const cudaError_t ce = cudaDeviceSynchronize();
            cudaFree(X);
            cudaFree(Y);
            if (rc) return rc;
            if (ce != cudaSuccess) {
                set_error(std::string("quadrature-folded table: ") + cudaGetErrorString(ce));
                return S2W_ECUDA;
            }
        }
    }
    p->grids.push_back(g);
    return S2W_OK;
}

// rows of a stage from a list of n values (all |n| < Lg), in the F layout with `nrows` rows per signal where row(n) is
// given by row_of(n)
int fill_stage_rows(s2w_plan *p, Stage &st, const std::vector<int> &ns, const std::vector<int> &rows, int nrows)
{
    st.nn = (int)ns.size();
    st.nrows = nrows;
    if (st.nn > S2W_MAX_ROWS) return S2W_EINVAL;
    for (int q = 0; q < st.nn; ++q) {
        st.n_val[q] = ns[q];
        st.n_tab[q] = find_tab(p, ns[q]);
        st.n_row[q] = rows[q];
        st.n_rowm[q] = rows[q];
        st.n_filtm[q] = q;
        for (int q2 = 0; q2 < st.nn; ++q2)
            if (ns[q2] == -ns[q]) {
                st.n_rowm[q] = rows[q2];
                st.n_filtm[q] = q2;
            }
        if (st.n_tab[q] < 0) return S2W_EINVAL;
    }
    return S2W_OK;
}

void fill_wig_args(const s2w_plan *p, const Stage &st, bool synthesis, int B, cplx *flmT, cplx *F, WigArgs &A)
{
    const GridTab &g = p->grids[st.grid];
    A.Lg = st.Lg;
    A.nt = g.nt;
    A.Lfull = p->L;
    A.B = B;
    A.isReal = p->real ? 1 : 0;
    A.nn = st.nn;
    A.nrows = st.nrows;
    A.lmin = st.lmin;
    for (int q = 0; q < st.nn; ++q) {
        A.n_val[q] = st.n_val[q];
        A.n_tab[q] = st.n_tab[q];
        A.n_row[q] = st.n_row[q];
        A.n_rowm[q] = st.n_rowm[q];
        A.n_filtm[q] = st.n_filtm[q];
    }
    A.tri = p->tri;
    A.coef = p->coef;
    A.G = g.G;
    A.gstart = st.gstart_f ? st.gstart_f : g.gstart;
    A.dseed = st.dseed_f ? st.dseed_f : g.dseed;
    A.yv = g.yv;
    A.ring = g.ring;
    A.dtab = g.dtab;
    A.dense = 0;
    A.tri_g = (size_t)st.Lg * (st.Lg + 1) / 2;
    A.filt = synthesis ? st.filt_syn : st.filt_ana;
    A.filt2 = 0;
    A.lmin2 = st.lmin;
    A.F2 = 0;
    A.flmT = flmT;
    A.F = F;
}

void fill_so3_args(const s2w_plan *p, const Stage &st, So3Args &A)
{
    A.f_transposed = 0;
    A.sig_off = 0;
    A.N = p->N;
    A.nn = st.nn;
    A.nrows = st.nrows;
    for (int q = 0; q < st.nn; ++q) {
        A.n_val[q] = st.n_val[q];
        A.n_row[q] = st.n_row[q];
        A.n_rowm[q] = st.n_rowm[q];
    }
}

void fill_rw_args(const s2w_plan *p, const Stage &st, RwArgs &A)
{
    A.nn = st.nn;
    A.nrows = st.nrows;
    A.isReal = p->real ? 1 : 0;
    A.Md = p->real ? st.Lg : 2 * st.Lg - 1;
    for (int q = 0; q < st.nn; ++q) {
        A.n_val[q] = st.n_val[q];
        A.n_row[q] = st.n_row[q];
    }
}

int check_params(int L, int N, double lambda, int J0)
{
    if (L < 1 || N < 1 || N > L || !(lambda > 1.0) || J0 < 0) {
        set_error("invalid argument: need L >= 1, 1 <= N <= L, lambda > 1, J0 >= 0");
        return S2W_EINVAL;
    }
    if (N > S2W_MAX_N) {
        set_error("N above S2W_MAX_N");
        return S2W_EUNSUPPORTED;
    }
    if (J0 > scale_count(L, lambda)) {
        set_error("invalid argument: J0 > J");
        return S2W_EINVAL;
    }
    return S2W_OK;
}

// common part of plan creation: tables that depend on (L, N) only
int plan_common(s2w_plan *p)
{
    int rc;
    p->tabn.clear();
    for (int n = -(p->N - 1); n <= p->N - 1; n += (p->kind == 2 ? 1 : 2)) p->tabn.push_back(n);
    if (find_tab(p, -p->spin) < 0) p->tabn.push_back(-p->spin);
    if (find_tab(p, p->spin) < 0) p->tabn.push_back(p->spin);  // the mirror columns (-m, -s) run the recursion of +s
    p->tri = (size_t)p->L * (p->L + 1) / 2;
    {
        std::vector<double> coef;
        host_coef(p->L, p->tabn, coef);
        if ((rc = p->pool.upload(&p->coef, coef))) return rc;
    }
    p->Mtab = 1 << std::max(1, ceil_log2(2 * (2 * p->L - 1) - 1));
    if ((rc = p->pool.alloc(&p->tw, p->Mtab))) return rc;
    if ((rc = launch_twiddles(p->tw, p->Mtab, 0))) return rc;
    S2W_CUDA_CHECK(cudaDeviceSynchronize());
    return S2W_OK;
}

int make_stage_filters(s2w_plan *p, Stage &st, const std::vector<cplx> &ana, const std::vector<cplx> &syn, double c)
{
    int rc;
    if ((rc = p->pool.upload(&st.filt_ana, ana))) return rc;
    if ((rc = p->pool.upload(&st.filt_syn, syn))) return rc;
    std::vector<cplx> aa(ana.size()), sa(syn.size());
    for (size_t i = 0; i < ana.size(); ++i) aa[i] = cmake(c * ana[i].x, -c * ana[i].y);
    for (size_t i = 0; i < syn.size(); ++i) sa[i] = cmake(syn[i].x / c, -syn[i].y / c);
    if ((rc = p->pool.upload(&st.filt_ana_adj, aa))) return rc;
    if ((rc = p->pool.upload(&st.filt_syn_adj, sa))) return rc;
    return S2W_OK;
}

// SHT stage at band-limit Lg with analysis-direction filter a(l) (harmonic -> rings) and synthesis filter s(l)
int make_n0_stage(s2w_plan *p, Stage &st, int Lg, const std::vector<double> &a, const std::vector<double> &s)
{
    int rc;
    if ((rc = build_grid(p, Lg))) return rc;
    memset(&st, 0, sizeof(st));
    st.grid = grid_index(p, Lg);
    st.Lg = Lg;
    st.lmin = 0;
    // spin-s harmonics sY_lm = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi} (reading R2, Goldberg convention): the row n = -s, zero
    // below l = |s| (the contraction kernels start at max(|m|, |n|)); no row at all when the band-limit is <= |s|.
    // The kernels pair the column (m, n) with (-m, -n) (one recursion serves both), so for s != 0 the stage carries
    // the recursions of n = -s (columns m >= 0 of row 0) and n = +s (whose mirror columns are (-m, -s): the m < 0 half of
    // row 0); the other halves land in / are read from a second, scratch row that the FFT side keeps at zero.
    const int nspin = -p->spin;
    std::vector<int> ns, rows;
    if (std::abs(nspin) < Lg) {
        ns.push_back(nspin);
        rows.push_back(0);
        if (nspin != 0) {
            ns.push_back(-nspin);
            rows.push_back(1);
        }
    }
    if ((rc = fill_stage_rows(p, st, ns, rows, nspin != 0 ? 2 : 1))) return rc;
    const double sgn = (p->spin & 1) ? -1.0 : 1.0;
    std::vector<cplx> fa((size_t)std::max(1, st.nn) * Lg), fs((size_t)std::max(1, st.nn) * Lg);
    for (int q = 0; q < std::max(1, st.nn); ++q)
        for (int l = 0; l < Lg; ++l) {
            fa[(size_t)q * Lg + l] = cmake(sgn * a[l], 0.0);
            fs[(size_t)q * Lg + l] = cmake(sgn * s[l], 0.0);
        }
    return make_stage_filters(p, st, fa, fs, 2.0 * Lg - 1.0);
}

// wavelet stage of angular scale j at band-limit sc.Lj: rows n of script-N inside the band-limit, filters
// conj(Psi^j_{ln}) (analysis, Eq. 40) and Psi^j_{ln} (2pi)^2/(2L_j-1) (synthesis, Eq. 42), with
// Psi^j_{ln} = sqrt((2l+1)/8pi^2) kappa^j(l) zeta_{ln} (Eq. A9).  kj = kappa^j(l), l < L.
int make_scale_stage(s2w_plan *p, Scale &sc, const double *kj, const std::vector<double> &zeta)
{
    const int N = p->N, nn = 2 * N - 1;
    const double pi = pi_d();
    int rc;
    if ((rc = build_grid(p, sc.Lj))) return rc;
    Stage &st = sc.st;
    st.grid = grid_index(p, sc.Lj);
    st.Lg = sc.Lj;
    st.lmin = sc.Lj;
    for (int l = 0; l < sc.Lj; ++l)
        if (kj[l] != 0.0) {
            st.lmin = l;
            break;
        }
    std::vector<int> ns, rows;
    if (st.lmin < sc.Lj)
        for (int ni = 0; ni < N; ++ni) {
            int n = -(N - 1) + 2 * ni;
            if (std::abs(n) < sc.Lj) {
                ns.push_back(n);
                rows.push_back(ni);
            }
        }
    if ((rc = fill_stage_rows(p, st, ns, rows, N))) return rc;
    if (st.nn > 0 && st.lmin > 0 && !(p->flags & S2W_PRECOMPUTE)) {
        const GridTab &g = p->grids[st.grid];
        const size_t ntab = p->tabn.size();
        if ((rc = p->pool.alloc(&st.gstart_f, ntab * sc.Lj * g.G))) return rc;
        if ((rc = p->pool.alloc(&st.dseed_f, ntab * sc.Lj * (size_t)32 * g.G))) return rc;
        if ((rc = launch_wigner_seed_floor(p->coef, p->tri, p->L, sc.Lj, g.G, (int)ntab, g.yv, g.gstart, g.dseed, st.lmin,
                                           st.gstart_f, st.dseed_f, 0)))
            return rc;
    }
    std::vector<cplx> fa((size_t)st.nn * sc.Lj), fs((size_t)st.nn * sc.Lj);
    const double syn_norm = 4.0 * pi * pi / (2.0 * sc.Lj - 1.0);
    for (int q = 0; q < st.nn; ++q)
        for (int l = 0; l < sc.Lj; ++l) {
            const double pre = std::sqrt((2.0 * l + 1.0) / (8.0 * pi * pi)) * kj[l];
            const size_t zo = ((size_t)l * nn + (st.n_val[q] + N - 1)) * 2;
            const double re = pre * zeta[zo], im = pre * zeta[zo + 1];
            fa[(size_t)q * sc.Lj + l] = cmake(re, -im);
            fs[(size_t)q * sc.Lj + l] = cmake(re * syn_norm, im * syn_norm);
        }
    return make_stage_filters(p, st, fa, fs, (2.0 * sc.Lj - 1.0) * nn);
}

}  // namespace

// ---- transform drivers (sphere) ---------------------------------------------------------------------------------

struct Work {
    cplx *flmT;
    cplx *F;    // [B][n][t][m]
    cplx *Ft;   // [B][n][m][t]: reweighted columns, input of the forward contraction
    cplx *Ft2;  // the same for the second of two scales that share one recursion
};

static Work carve(const s2w_plan *p, void *work)
{
    Work w;
    w.flmT = (cplx *)work;
    w.F = w.flmT + ((p->ws_flm_elems + 15) / 16) * 16;
    w.Ft = w.F + ((p->ws_F_elems + 15) / 16) * 16;
    w.Ft2 = w.Ft + ((p->ws_F_elems + 15) / 16) * 16;
    return w;
}

// The lanes of a captured transform: lane 0 is the capture stream with the caller's buffers, lane i > 0 has a stream
// of the plan and two more F-sized buffers of the workspace.  Only under run_transform's capture (lanes_on):
// streams and events belong to the plan, and the capture holds the plan's graph mutex.
struct Lanes {
    int n;
    cudaStream_t s[S2W_LANES];
    Work w[S2W_LANES];
    double load[S2W_LANES];
    int pick(double cost)  // the lane with the least work so far
    {
        int best = 0;
        for (int i = 1; i < n; ++i)
            if (load[i] < load[best]) best = i;
        load[best] += cost;
        return best;
    }
};

static int lanes_fork(const s2w_plan *p, const Work &w, cplx *spare, cudaStream_t s, bool allow, Lanes *ln,
                      size_t Fsz_override = 0, int max_lanes = S2W_LANES)
{
    ln->n = 1;
    ln->s[0] = s;
    ln->w[0] = w;
    for (int i = 0; i < S2W_LANES; ++i) ln->load[i] = 0.0;
    static const int nl = [] {
        const char *e = getenv("S2W_LANES");
        const int v = e ? atoi(e) : S2W_LANES;
        return v < 1 ? 1 : (v > S2W_LANES ? S2W_LANES : v);
    }();
    const int nuse = nl < max_lanes ? nl : max_lanes;
    if (!allow || !p->lanes_on || nuse == 1) return S2W_OK;
    const size_t Fsz = Fsz_override ? Fsz_override : ((p->ws_F_elems + 15) / 16) * 16;
    if (!p->lane_fork) S2W_CUDA_CHECK(cudaEventCreateWithFlags(&p->lane_fork, cudaEventDisableTiming));
    S2W_CUDA_CHECK(cudaEventRecord(p->lane_fork, s));
    for (int i = 1; i < nuse; ++i) {
        if (!p->lane_stream[i - 1]) {
            S2W_CUDA_CHECK(cudaStreamCreateWithFlags(&p->lane_stream[i - 1], cudaStreamNonBlocking));
            S2W_CUDA_CHECK(cudaEventCreateWithFlags(&p->lane_join[i - 1], cudaEventDisableTiming));
        }
        S2W_CUDA_CHECK(cudaStreamWaitEvent(p->lane_stream[i - 1], p->lane_fork, 0));
        ln->s[i] = p->lane_stream[i - 1];
        ln->w[i] = w;
        ln->w[i].F = spare + (size_t)(2 * i - 2) * Fsz;  // `spare`: 2 (S2W_LANES - 1) F-sized buffers
        ln->w[i].Ft = ln->w[i].F + Fsz;
        ln->w[i].Ft2 = 0;
    }
    ln->n = nuse;
    return S2W_OK;
}

static int lanes_join(const s2w_plan *p, const Lanes &ln)
{
    for (int i = 1; i < ln.n; ++i) {
        S2W_CUDA_CHECK(cudaEventRecord(p->lane_join[i - 1], ln.s[i]));
        S2W_CUDA_CHECK(cudaStreamWaitEvent(ln.s[0], p->lane_join[i - 1], 0));
    }
    return S2W_OK;
}

static double scale_cost(const Scale &sc) { return (double)sc.Lj * sc.Lj * sc.Lj * (sc.st.nn + 0.01); }

// Step a2 on the grid of a stage: F[b][row][t][mi] -> Ft[b][row][mi][t] with the theta quadrature applied.  McEwen-Wiaux:
// the reweighting operator of reading R3 (Toeplitz/Hankel form, or the Bluestein kernel on tiny grids); Driscoll-Healy:
// the diagonal quadrature weights q_t, applied by the transposing copy.
// `folded`: the caller contracts with the quadrature-folded table (GridTab::dtab_rw, see use_folded): transposing copy only.
static int stage_reweight(const s2w_plan *p, const Stage &st, const cplx *F, cplx *Ft, int B, cudaStream_t s,
                          bool folded = false)
{
    const GridTab &g = p->grids[st.grid];
    if (folded) return launch_transpose(F, Ft, g.nt, p->real ? st.Lg : 2 * st.Lg - 1, B * st.nrows, s, 0);
    if (g.dhw) return launch_transpose(F, Ft, g.nt, p->real ? st.Lg : 2 * st.Lg - 1, B * st.nrows, s, g.dhw);
    RwArgs R;
    fill_rw_args(p, st, R);
    return g.rw.L ? launch_reweight_th(F, Ft, R, B, g.rw, s) : launch_reweight(F, Ft, R, B, g.fft, s);
}

// rings -> harmonic contraction of a stage with the quadrature-folded table (transforms only; the adjoint calls and the
// stand-alone Q transform keep the plain table and the explicit reweighting)
static bool use_folded(const s2w_plan *p, const Stage &st, WigArgs *A)
{
    const GridTab &g = p->grids[st.grid];
    if (!g.dtab_rw) return false;
    if (A) {
        A->dtab = g.dtab_rw;
        A->dense = 1;
    }
    return true;
}

// pixels of one signal on the grid of band-limit Lg: rings x (2 Lg - 1)
static size_t grid_pixels(const s2w_plan *p, int Lg) { return (size_t)(p->dh ? 2 * Lg : Lg) * (2 * Lg - 1); }

// Ring FFTs of an SHT stage (a1).  A spin stage has two rows per signal in F (the second one scratch, kept at zero on
// the way to the forward contraction), so its signals are transformed one by one into / out of row 0.
static int stage_ring_fwd(const s2w_plan *p, const Stage &st, const void *f, size_t sig_stride, int B, cplx *F,
                          cudaStream_t s)
{
    const FftTab &T = p->grids[st.grid].fft;
    if (st.nrows == 1) return launch_ring_fwd(p->real, f, F, B, st.Lg, sig_stride, T, s);
    const size_t per = (size_t)st.nrows * grid_pixels(p, st.Lg);
    S2W_CUDA_CHECK(cudaMemsetAsync(F, 0, (size_t)B * per * sizeof(cplx), s));
    for (int b = 0; b < B; ++b) {
        int rc = launch_ring_fwd(false, (const cplx *)f + (size_t)b * sig_stride, F + (size_t)b * per, 1, st.Lg, sig_stride, T, s);
        if (rc) return rc;
    }
    return S2W_OK;
}

static int stage_ring_inv(const s2w_plan *p, const Stage &st, const cplx *F, void *f, size_t sig_stride, int B,
                          cudaStream_t s)
{
    const FftTab &T = p->grids[st.grid].fft;
    if (st.nrows == 1) return launch_ring_inv(p->real, F, f, B, st.Lg, sig_stride, T, s);
    const size_t per = (size_t)st.nrows * grid_pixels(p, st.Lg);
    for (int b = 0; b < B; ++b) {
        int rc = launch_ring_inv(false, F + (size_t)b * per, (cplx *)f + (size_t)b * sig_stride, 1, st.Lg, sig_stride, T, s);
        if (rc) return rc;
    }
    return S2W_OK;
}

// pixels [B][L][2L-1] -> flmT
static int sht_forward_dev(const s2w_plan *p, const Stage &st, const void *f, size_t sig_stride, int B, const Work &w,
                           bool zero_first, cudaStream_t s)
{
    const GridTab &g = p->grids[st.grid];
    int rc;
    if (st.nn == 0) {  // band-limit <= |spin|: nothing to project onto
        if (zero_first)
            S2W_CUDA_CHECK(cudaMemsetAsync(w.flmT, 0, (size_t)B * (p->real ? p->L : 2 * p->L - 1) * p->L * sizeof(cplx), s));
        return S2W_OK;
    }
    if ((rc = stage_ring_fwd(p, st, f, sig_stride, B, w.F, s))) return rc;
    if ((rc = stage_reweight(p, st, w.F, w.Ft, B, s, use_folded(p, st, 0)))) return rc;
    if (zero_first) {
        const size_t Mfull = p->real ? p->L : 2 * p->L - 1;
        S2W_CUDA_CHECK(cudaMemsetAsync(w.flmT, 0, (size_t)B * Mfull * p->L * sizeof(cplx), s));
    }
    WigArgs A;
    fill_wig_args(p, st, true, B, w.flmT, w.Ft, A);
    use_folded(p, st, &A);
    return launch_wigner_forward(A, s);
}

// flmT -> pixels
static int sht_inverse_dev(const s2w_plan *p, const Stage &st, void *f, size_t sig_stride, int B, const Work &w,
                           cudaStream_t s)
{
    const GridTab &g = p->grids[st.grid];
    if (st.nn == 0) {
        const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
        for (int b = 0; b < B; ++b)
            S2W_CUDA_CHECK(cudaMemsetAsync((char *)f + (size_t)b * sig_stride * esz, 0,
                                           grid_pixels(p, st.Lg) * esz, s));
        return S2W_OK;
    }
    WigArgs A;
    fill_wig_args(p, st, false, B, w.flmT, w.F, A);
    int rc;
    if ((rc = launch_wigner_inverse(A, s))) return rc;
    return stage_ring_inv(p, st, w.F, f, sig_stride, B, s);
}

// a4 + a5 + a8 for one scale: filter x inverse Wigner contraction at L_j, then the (alpha, gamma) DFT.  B signals whose
// coefficient blocks are sig_stride elements apart.
static int scale_analysis(const s2w_plan *p, const Scale &sc, int B, const Work &w, void *dst, size_t sig_stride,
                          cudaStream_t s, const size_t *sig_off = 0)
{
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    if (sc.st.nn == 0) {
        for (int b = 0; b < B; ++b)
            S2W_CUDA_CHECK(cudaMemsetAsync((char *)dst + (size_t)b * sig_stride * esz, 0,
                                           (size_t)(2 * p->N - 1) * grid_pixels(p, sc.Lj) * esz, s));
        return S2W_OK;
    }
    int rc;
    WigArgs A;
    fill_wig_args(p, sc.st, false, B, w.flmT, w.F, A);
    if ((rc = launch_wigner_inverse(A, s))) return rc;
    So3Args S;
    fill_so3_args(p, sc.st, S);
    S.sig_off = sig_off;
    return launch_so3_inv(p->real, w.F, dst, sig_stride, S, B, p->grids[sc.st.grid].fft, s);
}

// a8 + a2 + a6 + a4 for one scale: (alpha, gamma) DFT, reweighting, forward Wigner contraction accumulating into flmT.
static int scale_synthesis(const s2w_plan *p, const Scale &sc, int B, const Work &w, const void *src, size_t sig_stride,
                           cudaStream_t s, const size_t *sig_off = 0)
{
    if (sc.st.nn == 0) return S2W_OK;
    const GridTab &g = p->grids[sc.st.grid];
    int rc;
    So3Args S;
    fill_so3_args(p, sc.st, S);
    S.sig_off = sig_off;
    if (use_folded(p, sc.st, 0) && so3_fwd_writes_transposed(p->real, S, g.fft)) {
        S.f_transposed = 1;  // folded quadrature: a2 would be a transposing copy; the (alpha, gamma) kernel writes Ft itself
        if ((rc = launch_so3_fwd(p->real, src, sig_stride, w.Ft, S, B, g.fft, s))) return rc;
    } else {
        if ((rc = launch_so3_fwd(p->real, src, sig_stride, w.F, S, B, g.fft, s))) return rc;
        if ((rc = stage_reweight(p, sc.st, w.F, w.Ft, B, s, use_folded(p, sc.st, 0)))) return rc;
    }
    WigArgs A;
    fill_wig_args(p, sc.st, true, B, w.flmT, w.Ft, A);
    use_folded(p, sc.st, &A);
    return launch_wigner_forward(A, s);
}

// Host-buffer pipelining of the sphere transforms (s2wav_*_host): coefficient blocks cross PCIe on a second stream while
// other scales are being computed.  Analysis: each block is copied out as soon as its kernels are done; synthesis: all
// blocks are copied in up front, in the order of use, and each scale waits only for its own block.  Blocks are visited
// largest scale first, so that the copies of the two big top scales overlap the computation of the rest.
struct HostPipe {
    cudaStream_t copy;
    char *host;   // coefficient buffer on the host, [batch][coeff_elems]
    char *dev;    // the same on the device
    size_t pitch; // bytes between consecutive signals
    int B;
    std::vector<cudaEvent_t> evs;
    int next_event(cudaEvent_t *e)
    {
        cudaEvent_t ev;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) return S2W_ECUDA;
        evs.push_back(ev);
        *e = ev;
        return S2W_OK;
    }
    int block_out(size_t off_bytes, size_t bytes, cudaStream_t s)  // computed on s -> host
    {
        cudaEvent_t ev;
        if (next_event(&ev)) return S2W_ECUDA;
        S2W_CUDA_CHECK(cudaEventRecord(ev, s));
        S2W_CUDA_CHECK(cudaStreamWaitEvent(copy, ev, 0));
        S2W_CUDA_CHECK(cudaMemcpy2DAsync(host + off_bytes, pitch, dev + off_bytes, pitch, bytes, B, cudaMemcpyDeviceToHost, copy));
        return S2W_OK;
    }
    int block_in(size_t off_bytes, size_t bytes, cudaEvent_t *ready)  // host -> device, event when it has arrived
    {
        S2W_CUDA_CHECK(cudaMemcpy2DAsync(dev + off_bytes, pitch, host + off_bytes, pitch, bytes, B, cudaMemcpyHostToDevice, copy));
        if (next_event(ready)) return S2W_ECUDA;
        S2W_CUDA_CHECK(cudaEventRecord(*ready, copy));
        return S2W_OK;
    }
    void release()
    {
        for (cudaEvent_t e : evs) cudaEventDestroy(e);
        evs.clear();
    }
};

// Two scales can share one recursion (wigner.cu: NS = 2 inverse kernel, fused tile rows of the forward kernel) when
// they live on the same grid with the same rows n and the batch has at most two complex columns; `a` is the one whose
// filter support starts first.  On-the-fly plans only.
static bool scales_fusable(const s2w_plan *p, const Scale &a, const Scale &b, int B)
{
    if ((p->flags & S2W_PRECOMPUTE) || (p->real ? B : 2 * B) > 2) return false;
    if (a.st.grid != b.st.grid || a.st.nn != b.st.nn || a.st.nn == 0 || a.st.lmin > b.st.lmin) return false;
    for (int q = 0; q < a.st.nn; ++q)
        if (a.st.n_val[q] != b.st.n_val[q] || a.st.n_row[q] != b.st.n_row[q]) return false;
    return true;
}

// a4 + a5 for two fusable scales in one launch (outputs w.F and w.Ft), then a8 for each
static int scale_pair_analysis(const s2w_plan *p, const Scale &a, const Scale &b, int B, const Work &w, void *dst_a,
                               void *dst_b, size_t sig_stride, cudaStream_t s)
{
    int rc;
    WigArgs A;
    fill_wig_args(p, a.st, false, B, w.flmT, w.F, A);
    A.filt2 = b.st.filt_ana;
    A.lmin2 = b.st.lmin;
    A.F2 = w.Ft;
    if ((rc = launch_wigner_inverse(A, s))) return rc;
    So3Args S;
    fill_so3_args(p, a.st, S);
    const FftTab &T = p->grids[a.st.grid].fft;
    if ((rc = launch_so3_inv(p->real, w.F, dst_a, sig_stride, S, B, T, s))) return rc;
    return launch_so3_inv(p->real, w.Ft, dst_b, sig_stride, S, B, T, s);
}

// a8 + a2 for each of two fusable scales (into w.Ft and w.Ft2), then a6 + a4 for both in one launch
static int scale_pair_synthesis(const s2w_plan *p, const Scale &a, const Scale &b, int B, const Work &w, const void *src_a,
                                const void *src_b, size_t sig_stride, cudaStream_t s)
{
    const GridTab &g = p->grids[a.st.grid];
    int rc;
    So3Args S;
    fill_so3_args(p, a.st, S);
    RwArgs R;
    fill_rw_args(p, a.st, R);
    for (int k = 0; k < 2; ++k) {
        cplx *Ft = k ? w.Ft2 : w.Ft;
        if ((rc = launch_so3_fwd(p->real, k ? src_b : src_a, sig_stride, w.F, S, B, g.fft, s))) return rc;
        if ((rc = stage_reweight(p, a.st, w.F, Ft, B, s))) return rc;
    }
    WigArgs A;
    fill_wig_args(p, a.st, true, B, w.flmT, w.Ft, A);
    A.filt2 = b.st.filt_syn;
    A.lmin2 = b.st.lmin;
    A.F2 = w.Ft2;
    return launch_wigner_forward(A, s);
}

static int sphere_forward(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s, HostPipe *hp = 0)
{
    const Work w = carve(p, work);
    const int B = p->batch;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t nn = 2 * p->N - 1;
    int rc;
    if ((rc = sht_forward_dev(p, p->sht, in, p->signal_elems, B, w, true, s))) return rc;
    const int ns = (int)p->scales.size();
    Lanes ln;
    if ((rc = lanes_fork(p, w, w.Ft2 + ((p->ws_F_elems + 15) / 16) * 16, s, !hp, &ln))) return rc;
    const bool lanes = ln.n > 1;
    // the two top scales share one recursion when they can; they go first (their blocks are the big host copies)
    int rest = ns;
    if (ns >= 2 && scales_fusable(p, p->scales[ns - 2], p->scales[ns - 1], B)) {
        const Scale &a = p->scales[ns - 2], &b = p->scales[ns - 1];
        if ((rc = scale_pair_analysis(p, a, b, B, w, (char *)out + a.offset * esz, (char *)out + b.offset * esz,
                                      p->coeff_elems, s)))
            return rc;
        if (hp && (rc = hp->block_out(b.offset * esz, nn * grid_pixels(p, b.Lj) * esz, s))) return rc;
        if (hp && (rc = hp->block_out(a.offset * esz, nn * grid_pixels(p, a.Lj) * esz, s))) return rc;
        rest = ns - 2;
        ln.load[0] += scale_cost(a) + scale_cost(b);  // the pair ran on lane 0 (the only one with an Ft2 buffer)
    }
    for (int k = 0; k < rest; ++k) {  // largest first when pipelined: the lanes (or the host copies) stay balanced
        const Scale &sc = p->scales[(hp || lanes) ? rest - 1 - k : k];
        const int l = ln.pick(scale_cost(sc));
        if ((rc = scale_analysis(p, sc, B, ln.w[l], (char *)out + sc.offset * esz, p->coeff_elems, ln.s[l]))) return rc;
        if (hp && (rc = hp->block_out(sc.offset * esz, nn * grid_pixels(p, sc.Lj) * esz, s))) return rc;
    }
    // scaling coefficients
    const int l = ln.pick(0.0);
    if ((rc = sht_inverse_dev(p, p->scaling, (char *)out + p->scaling_offset * esz, p->coeff_elems, B, ln.w[l], ln.s[l])))
        return rc;
    if (hp && (rc = hp->block_out(p->scaling_offset * esz, grid_pixels(p, p->Ls) * esz, s))) return rc;
    if ((rc = lanes_join(p, ln))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

static int sphere_inverse(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s, HostPipe *hp = 0)
{
    const Work w = carve(p, work);
    const int B = p->batch;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t nn = 2 * p->N - 1;
    const int ns = (int)p->scales.size();
    int rc;
    std::vector<cudaEvent_t> ready(ns + 1);
    if (hp) {
        if ((rc = hp->block_in(p->scaling_offset * esz, grid_pixels(p, p->Ls) * esz, &ready[ns]))) return rc;
        for (int k = 0; k < ns; ++k) {
            const Scale &sc = p->scales[ns - 1 - k];
            if ((rc = hp->block_in(sc.offset * esz, nn * grid_pixels(p, sc.Lj) * esz, &ready[ns - 1 - k]))) return rc;
        }
        S2W_CUDA_CHECK(cudaStreamWaitEvent(s, ready[ns], 0));
    }
    if ((rc = sht_forward_dev(p, p->scaling, (const char *)in + p->scaling_offset * esz, p->coeff_elems, B, w, true,
                              s)))
        return rc;
    Lanes ln;
    if ((rc = lanes_fork(p, w, w.Ft2 + ((p->ws_F_elems + 15) / 16) * 16, s, !hp, &ln))) return rc;
    const bool lanes = ln.n > 1;
    int rest = ns;
    if (ns >= 2 && scales_fusable(p, p->scales[ns - 2], p->scales[ns - 1], B)) {
        const Scale &a = p->scales[ns - 2], &b = p->scales[ns - 1];
        if (hp) {
            S2W_CUDA_CHECK(cudaStreamWaitEvent(s, ready[ns - 1], 0));
            S2W_CUDA_CHECK(cudaStreamWaitEvent(s, ready[ns - 2], 0));
        }
        if ((rc = scale_pair_synthesis(p, a, b, B, w, (const char *)in + a.offset * esz, (const char *)in + b.offset * esz,
                                       p->coeff_elems, s)))
            return rc;
        rest = ns - 2;
        ln.load[0] += scale_cost(a) + scale_cost(b);
    }
    for (int k = 0; k < rest; ++k) {  // the forward contractions of all scales accumulate into flmT by atomics
        const int i = (hp || lanes) ? rest - 1 - k : k;
        const Scale &sc = p->scales[i];
        if (hp) S2W_CUDA_CHECK(cudaStreamWaitEvent(s, ready[i], 0));
        const int l = ln.pick(scale_cost(sc));
        if ((rc = scale_synthesis(p, sc, B, ln.w[l], (const char *)in + sc.offset * esz, p->coeff_elems, ln.s[l])))
            return rc;
    }
    if ((rc = lanes_join(p, ln))) return rc;
    if ((rc = sht_inverse_dev(p, p->sht, out, p->signal_elems, B, w, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- adjoint transforms (sphere, real and complex signals) ---------------------------
// With <u, v> = sum conj(u) v over the stored samples, the adjoint of a chain is the reversed chain of adjoints:
//   (inverse DFT E)^H = n x (normalised forward DFT),   (normalised forward DFT E^H / n)^H = E / n,
//   (harmonic -> rings contraction D diag(a))^H = diag(conj a) D^T  = the rings -> harmonic contraction, no quadrature,
//   (rings -> harmonic contraction diag(s) D^T R)^H = R D diag(conj s): the reweighting operator R = E_x^T K E_x
//   (extension, the real symmetric kernel K of section 6.3, fold) is its own adjoint.
// The same kernels in the other order; the constants live in filt_ana_adj / filt_syn_adj, and transpose_kernel stands
// in where the reweighting kernel's transposed output is missing (or has to be undone).

// w.F [B][nrows][t][m]  ->  flmT += c conj(a_l) sum_t d^l_{mn}(theta_t) F
static int adj_rings_to_harmonic(const s2w_plan *p, const Stage &st, int B, const Work &w, cudaStream_t s)
{
    const int Md = p->real ? st.Lg : 2 * st.Lg - 1;
    int rc;
    if (st.nn == 0) return S2W_OK;
    if ((rc = launch_transpose(w.F, w.Ft, st.Lg, Md, B * st.nrows, s))) return rc;
    WigArgs A;
    fill_wig_args(p, st, true, B, w.flmT, w.Ft, A);
    A.filt = st.filt_ana_adj;
    return launch_wigner_forward(A, s);
}

// flmT  ->  w.F [B][nrows][t][m] = R sum_l d^l_{mn}(theta_t) conj(s_l) / c flm
static int adj_harmonic_to_rings(const s2w_plan *p, const Stage &st, int B, const Work &w, cudaStream_t s)
{
    const GridTab &g = p->grids[st.grid];
    const int Md = p->real ? st.Lg : 2 * st.Lg - 1;
    int rc;
    if (st.nn == 0) {
        S2W_CUDA_CHECK(cudaMemsetAsync(w.F, 0, (size_t)B * st.nrows * st.Lg * Md * sizeof(cplx), s));
        return S2W_OK;
    }
    WigArgs A;
    fill_wig_args(p, st, false, B, w.flmT, w.F, A);
    A.filt = st.filt_syn_adj;
    if ((rc = launch_wigner_inverse(A, s))) return rc;
    RwArgs R;
    fill_rw_args(p, st, R);
    if ((rc = g.rw.L ? launch_reweight_th(w.F, w.Ft, R, B, g.rw, s) : launch_reweight(w.F, w.Ft, R, B, g.fft, s))) return rc;
    return launch_transpose(w.Ft, w.F, Md, st.Lg, B * st.nrows, s);
}

// adjoint of the analysis: coefficients -> signal
static int sphere_forward_adjoint(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const Work w = carve(p, work);
    const int B = p->batch;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const char *y = (const char *)in;
    int rc;
    S2W_CUDA_CHECK(cudaMemsetAsync(w.flmT, 0, (size_t)B * (p->real ? p->L : 2 * p->L - 1) * p->L * sizeof(cplx), s));
    Lanes ln;  // every block accumulates into flmT by atomics: the blocks are dealt to the lanes, largest first
    if ((rc = lanes_fork(p, w, w.Ft2 + ((p->ws_F_elems + 15) / 16) * 16, s, true, &ln))) return rc;
    for (size_t k = p->scales.size(); k-- > 0;) {
        const Scale &sc = p->scales[k];
        if (sc.st.nn == 0) continue;
        const int l = ln.pick(scale_cost(sc));
        So3Args S;
        fill_so3_args(p, sc.st, S);
        if ((rc = launch_so3_fwd(p->real, y + sc.offset * esz, p->coeff_elems, ln.w[l].F, S, B, p->grids[sc.st.grid].fft, ln.s[l])))
            return rc;
        if ((rc = adj_rings_to_harmonic(p, sc.st, B, ln.w[l], ln.s[l]))) return rc;
    }
    {
        const int l = ln.pick(0.0);
        if ((rc = stage_ring_fwd(p, p->scaling, y + p->scaling_offset * esz, p->coeff_elems, B, ln.w[l].F, ln.s[l])))
            return rc;
        if ((rc = adj_rings_to_harmonic(p, p->scaling, B, ln.w[l], ln.s[l]))) return rc;
    }
    if ((rc = lanes_join(p, ln))) return rc;
    if ((rc = adj_harmonic_to_rings(p, p->sht, B, w, s))) return rc;
    if ((rc = stage_ring_inv(p, p->sht, w.F, out, p->signal_elems, B, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// adjoint of the synthesis: signal -> coefficients
static int sphere_inverse_adjoint(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const Work w = carve(p, work);
    const int B = p->batch;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    char *y = (char *)out;
    int rc;
    S2W_CUDA_CHECK(cudaMemsetAsync(w.flmT, 0, (size_t)B * (p->real ? p->L : 2 * p->L - 1) * p->L * sizeof(cplx), s));
    if ((rc = stage_ring_fwd(p, p->sht, in, p->signal_elems, B, w.F, s))) return rc;
    if ((rc = adj_rings_to_harmonic(p, p->sht, B, w, s))) return rc;
    Lanes ln;  // every block reads the same flmT
    if ((rc = lanes_fork(p, w, w.Ft2 + ((p->ws_F_elems + 15) / 16) * 16, s, true, &ln))) return rc;
    for (size_t k = p->scales.size(); k-- > 0;) {
        const Scale &sc = p->scales[k];
        if (sc.st.nn == 0) {
            for (int b = 0; b < B; ++b)
                S2W_CUDA_CHECK(cudaMemsetAsync(y + ((size_t)b * p->coeff_elems + sc.offset) * esz, 0,
                                               (size_t)(2 * p->N - 1) * grid_pixels(p, sc.Lj) * esz, s));
            continue;
        }
        const int l = ln.pick(scale_cost(sc));
        if ((rc = adj_harmonic_to_rings(p, sc.st, B, ln.w[l], ln.s[l]))) return rc;
        So3Args S;
        fill_so3_args(p, sc.st, S);
        if ((rc = launch_so3_inv(p->real, ln.w[l].F, y + sc.offset * esz, p->coeff_elems, S, B, p->grids[sc.st.grid].fft, ln.s[l])))
            return rc;
    }
    {
        const int l = ln.pick(0.0);
        if ((rc = adj_harmonic_to_rings(p, p->scaling, B, ln.w[l], ln.s[l]))) return rc;
        if ((rc = stage_ring_inv(p, p->scaling, ln.w[l].F, y + p->scaling_offset * esz, p->coeff_elems, B, ln.s[l])))
            return rc;
    }
    if ((rc = lanes_join(p, ln))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- transform drivers (ball, Alg. 2) -----------------------------------------------------------------
// workspace: flm_sh [P][Mfull][L] (per-shell harmonic coefficients), flmp [P][Mfull][L] (f_{lmp}), F.
struct BallWork {
    cplx *flm_sh, *flmp, *F, *Ft;
};
static BallWork carve_ball(const s2w_plan *p, void *work)
{
    BallWork w;
    const size_t sh = ((p->ws_shell_elems + 15) / 16) * 16;
    w.flm_sh = (cplx *)work;
    w.flmp = w.flm_sh + sh;
    w.F = w.flmp + sh;
    w.Ft = w.F + ((p->ws_F_elems + 15) / 16) * 16;
    return w;
}

static int ball_forward(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const BallWork bw = carve_ball(p, work);
    Work w;
    w.flmT = bw.flm_sh;
    w.F = bw.F;
    w.Ft = bw.Ft;
    w.Ft2 = 0;
    cplx *spare = bw.Ft + ((p->ws_F_elems + 15) / 16) * 16;
    const int P = p->P, L = p->L;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t cols = (size_t)(p->real ? L : 2 * L - 1) * L;
    const size_t shell = (size_t)L * (2 * L - 1);
    int rc;
    // Z: per-shell spherical harmonic transform, then the radial quadrature (Eq. 10)
    if ((rc = sht_forward_dev(p, p->sht, in, shell, P, w, true, s))) return rc;
    if ((rc = launch_radial(p->Kfull_fwd, P, P, bw.flm_sh, bw.flmp, cols, L, 0, 0, false, s))) return rc;
    // scaling coefficients: Phi f, Z^-1 at full resolution (Eq. 35; R9)
    if ((rc = launch_radial(p->Kfull_inv, P, P, bw.flmp, bw.flm_sh, cols, L, p->phi_ball, 0, false, s))) return rc;
    if ((rc = sht_inverse_dev(p, p->sht, (char *)out + p->scaling_offset * esz, shell, P, w, s))) return rc;
    // wavelet coefficients (Eqs. 33, 43-44), stacked shells: ONE inverse Laguerre contraction onto the
    // node grids of all radial scales j' (stacked matrix, kappa^{j'}(p) folded in), then for every angular scale j the
    // sphere's scale stage a4 + a5 + a8 over all PS = sum_j' P_j' shells in one launch each
    static const bool stacked = getenv("S2W_BALL_UNSTACKED") == 0;
    if (stacked) {
        cplx *stk = (cplx *)work + p->ws_stk_off;
        cplx *Fs = stk + p->ws_stk_elems;
        if ((rc = launch_radial(p->Kstk_inv, p->PS, P, bw.flmp, stk, cols, L, 0, 0, false, s, p->krange_inv))) return rc;
        Work ws = w;
        ws.flmT = stk;
        ws.F = Fs;
        ws.Ft = Fs + p->ws_stkF_elems;
        Lanes ln;
        if ((rc = lanes_fork(p, ws, Fs + 2 * p->ws_stkF_elems, s, true, &ln, p->ws_stkF_elems, S2W_BALL_LANES))) return rc;
        const size_t nj = p->ang.size();
        for (size_t k = nj; k-- > 0;) {
            const Scale &sc = p->ang[k];
            if (sc.st.nn == 0) {  // empty angular scale: its blocks of every j' are zero
                for (size_t a = k; a < p->scales.size(); a += nj) {
                    const Scale &q = p->scales[a];
                    S2W_CUDA_CHECK(cudaMemsetAsync((char *)out + q.offset * esz, 0,
                                                   (size_t)q.Pj * (2 * p->N - 1) * q.Lj * (2 * q.Lj - 1) * esz, s));
                }
                continue;
            }
            const int l = ln.pick(scale_cost(sc));
            if ((rc = scale_analysis(p, sc, p->PS, ln.w[l], out, 0, ln.s[l], p->ang_off[k]))) return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        S2W_CUDA_CHECK(cudaPeekAtLastError());
        return S2W_OK;
    }
    size_t i = 0;
    while (i < p->scales.size()) {
        const Scale &first = p->scales[i];
        if ((rc = launch_radial(first.Kinv, first.Pj, first.Pj, bw.flmp, bw.flm_sh, cols, L, 0, 0, false, s))) return rc;
        size_t e = i;
        while (e < p->scales.size() && p->scales[e].jp == first.jp) ++e;
        Lanes ln;  // the angular scales of one j' read the same flm_sh: dealt to the lanes, largest first
        if ((rc = lanes_fork(p, w, spare, s, true, &ln))) return rc;
        for (size_t k = e; k-- > i;) {
            const Scale &sc = p->scales[k];
            const size_t stride = (size_t)(2 * p->N - 1) * sc.Lj * (2 * sc.Lj - 1);
            const int l = ln.pick(scale_cost(sc));
            if ((rc = scale_analysis(p, sc, sc.Pj, ln.w[l], (char *)out + sc.offset * esz, stride, ln.s[l]))) return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        i = e;
    }
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

static int ball_inverse(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const BallWork bw = carve_ball(p, work);
    Work w;
    w.flmT = bw.flm_sh;
    w.F = bw.F;
    w.Ft = bw.Ft;
    w.Ft2 = 0;
    cplx *spare = bw.Ft + ((p->ws_F_elems + 15) / 16) * 16;
    const int P = p->P, L = p->L;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t Mfull = p->real ? L : 2 * L - 1;
    const size_t cols = Mfull * L;
    const size_t shell = (size_t)L * (2 * L - 1);
    int rc;
    // scaling part: Z W^Phi, times Phi (Eq. 46)
    if ((rc = sht_forward_dev(p, p->sht, (const char *)in + p->scaling_offset * esz, shell, P, w, true, s))) return rc;
    if ((rc = launch_radial(p->Kfull_fwd, P, P, bw.flm_sh, bw.flmp, cols, L, 0, p->phi_ball, false, s))) return rc;
    // wavelet part, stacked shells: every angular scale j adds its PS shells into the stacked harmonic array (one launch
    // per step and scale), then ONE radial quadrature with the stacked matrix
    static const bool stacked = getenv("S2W_BALL_UNSTACKED") == 0;
    if (stacked) {
        cplx *stk = (cplx *)work + p->ws_stk_off;
        cplx *Fs = stk + p->ws_stk_elems;
        S2W_CUDA_CHECK(cudaMemsetAsync(stk, 0, (size_t)p->PS * cols * sizeof(cplx), s));
        Work ws = w;
        ws.flmT = stk;
        ws.F = Fs;
        ws.Ft = Fs + p->ws_stkF_elems;
        Lanes ln;
        if ((rc = lanes_fork(p, ws, Fs + 2 * p->ws_stkF_elems, s, true, &ln, p->ws_stkF_elems, S2W_BALL_LANES))) return rc;
        for (size_t k = p->ang.size(); k-- > 0;) {
            const Scale &sc = p->ang[k];
            const int l = ln.pick(scale_cost(sc));
            if ((rc = scale_synthesis(p, sc, p->PS, ln.w[l], in, 0, ln.s[l], p->ang_off[k]))) return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        if ((rc = launch_radial(p->Kstk_fwd, P, p->PS, stk, bw.flmp, cols, L, 0, 0, true, s, p->krange_fwd))) return rc;
        if ((rc = launch_radial(p->Kfull_inv, P, P, bw.flmp, bw.flm_sh, cols, L, 0, 0, false, s))) return rc;
        if ((rc = sht_inverse_dev(p, p->sht, out, shell, P, w, s))) return rc;
        S2W_CUDA_CHECK(cudaPeekAtLastError());
        return S2W_OK;
    }
    size_t i = 0;
    while (i < p->scales.size()) {
        const Scale &first = p->scales[i];
        S2W_CUDA_CHECK(cudaMemsetAsync(bw.flm_sh, 0, (size_t)first.Pj * cols * sizeof(cplx), s));
        size_t e = i;
        while (e < p->scales.size() && p->scales[e].jp == first.jp) ++e;
        Lanes ln;  // the angular scales of one j' accumulate into the same flm_sh by atomics
        if ((rc = lanes_fork(p, w, spare, s, true, &ln))) return rc;
        for (size_t k = e; k-- > i;) {
            const Scale &sc = p->scales[k];
            const size_t stride = (size_t)(2 * p->N - 1) * sc.Lj * (2 * sc.Lj - 1);
            const int l = ln.pick(scale_cost(sc));
            if ((rc = scale_synthesis(p, sc, sc.Pj, ln.w[l], (const char *)in + sc.offset * esz, stride, ln.s[l])))
                return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        i = e;
        if ((rc = launch_radial(first.Kfwd, first.Pj, first.Pj, bw.flm_sh, bw.flmp, cols, L, 0, 0, true, s))) return rc;
    }
    // Z^-1
    if ((rc = launch_radial(p->Kfull_inv, P, P, bw.flmp, bw.flm_sh, cols, L, 0, 0, false, s))) return rc;
    if ((rc = sht_inverse_dev(p, p->sht, out, shell, P, w, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- adjoint transforms (ball): the chains of ball_forward / ball_inverse reversed, radial matrices transposed ------
static int ball_forward_adjoint(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const BallWork bw = carve_ball(p, work);
    Work w;
    w.flmT = bw.flm_sh;
    w.F = bw.F;
    w.Ft = bw.Ft;
    w.Ft2 = 0;
    cplx *spare = bw.Ft + ((p->ws_F_elems + 15) / 16) * 16;
    const int P = p->P, L = p->L;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t cols = (size_t)(p->real ? L : 2 * L - 1) * L;
    const size_t shell = (size_t)L * (2 * L - 1);
    const char *y = (const char *)in;
    int rc;
    S2W_CUDA_CHECK(cudaMemsetAsync(bw.flmp, 0, (size_t)P * cols * sizeof(cplx), s));
    // wavelet blocks: per j' the adjoint scale stages accumulate into flm_sh, then K_inv^T onto f_{lmp}
    size_t i = 0;
    while (i < p->scales.size()) {
        const Scale &first = p->scales[i];
        S2W_CUDA_CHECK(cudaMemsetAsync(bw.flm_sh, 0, (size_t)first.Pj * cols * sizeof(cplx), s));
        size_t e = i;
        while (e < p->scales.size() && p->scales[e].jp == first.jp) ++e;
        Lanes ln;
        if ((rc = lanes_fork(p, w, spare, s, true, &ln))) return rc;
        for (size_t k = e; k-- > i;) {
            const Scale &sc = p->scales[k];
            if (sc.st.nn == 0) continue;
            const size_t stride = (size_t)(2 * p->N - 1) * sc.Lj * (2 * sc.Lj - 1);
            const int l = ln.pick(scale_cost(sc));
            So3Args S;
            fill_so3_args(p, sc.st, S);
            if ((rc = launch_so3_fwd(p->real, y + sc.offset * esz, stride, ln.w[l].F, S, sc.Pj, p->grids[sc.st.grid].fft, ln.s[l])))
                return rc;
            if ((rc = adj_rings_to_harmonic(p, sc.st, sc.Pj, ln.w[l], ln.s[l]))) return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        i = e;
        if ((rc = launch_radial(first.KinvT, first.Pj, first.Pj, bw.flm_sh, bw.flmp, cols, L, 0, 0, true, s))) return rc;
    }
    // scaling block: (Y^-1)^H per shell, then Phi K_inv^T
    S2W_CUDA_CHECK(cudaMemsetAsync(bw.flm_sh, 0, (size_t)P * cols * sizeof(cplx), s));
    if ((rc = launch_ring_fwd(p->real, y + p->scaling_offset * esz, w.F, P, L, shell, p->grids[p->sht.grid].fft, s))) return rc;
    if ((rc = adj_rings_to_harmonic(p, p->sht, P, w, s))) return rc;
    if ((rc = launch_radial(p->Kfull_invT, P, P, bw.flm_sh, bw.flmp, cols, L, 0, p->phi_ball, true, s))) return rc;
    // Z^H: K_fwd^T, then Y^H per shell
    if ((rc = launch_radial(p->Kfull_fwdT, P, P, bw.flmp, bw.flm_sh, cols, L, 0, 0, false, s))) return rc;
    if ((rc = adj_harmonic_to_rings(p, p->sht, P, w, s))) return rc;
    if ((rc = launch_ring_inv(p->real, w.F, out, P, L, shell, p->grids[p->sht.grid].fft, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

static int ball_inverse_adjoint(const s2w_plan *p, const void *in, void *out, void *work, cudaStream_t s)
{
    const BallWork bw = carve_ball(p, work);
    Work w;
    w.flmT = bw.flm_sh;
    w.F = bw.F;
    w.Ft = bw.Ft;
    w.Ft2 = 0;
    cplx *spare = bw.Ft + ((p->ws_F_elems + 15) / 16) * 16;
    const int P = p->P, L = p->L;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t cols = (size_t)(p->real ? L : 2 * L - 1) * L;
    const size_t shell = (size_t)L * (2 * L - 1);
    char *y = (char *)out;
    int rc;
    // (Z^-1)^H: (Y^-1)^H per shell, then K_inv^T
    S2W_CUDA_CHECK(cudaMemsetAsync(bw.flm_sh, 0, (size_t)P * cols * sizeof(cplx), s));
    if ((rc = launch_ring_fwd(p->real, in, w.F, P, L, shell, p->grids[p->sht.grid].fft, s))) return rc;
    if ((rc = adj_rings_to_harmonic(p, p->sht, P, w, s))) return rc;
    if ((rc = launch_radial(p->Kfull_invT, P, P, bw.flm_sh, bw.flmp, cols, L, 0, 0, false, s))) return rc;
    // wavelet blocks: K_fwd^T onto the P_j' grid, then the adjoint scale stages
    size_t i = 0;
    while (i < p->scales.size()) {
        const Scale &first = p->scales[i];
        if ((rc = launch_radial(first.KfwdT, first.Pj, first.Pj, bw.flmp, bw.flm_sh, cols, L, 0, 0, false, s))) return rc;
        size_t e = i;
        while (e < p->scales.size() && p->scales[e].jp == first.jp) ++e;
        Lanes ln;
        if ((rc = lanes_fork(p, w, spare, s, true, &ln))) return rc;
        for (size_t k = e; k-- > i;) {
            const Scale &sc = p->scales[k];
            const size_t stride = (size_t)(2 * p->N - 1) * sc.Lj * (2 * sc.Lj - 1);
            if (sc.st.nn == 0) {
                S2W_CUDA_CHECK(cudaMemsetAsync(y + sc.offset * esz, 0, (size_t)sc.Pj * stride * esz, s));
                continue;
            }
            const int l = ln.pick(scale_cost(sc));
            if ((rc = adj_harmonic_to_rings(p, sc.st, sc.Pj, ln.w[l], ln.s[l]))) return rc;
            So3Args S;
            fill_so3_args(p, sc.st, S);
            if ((rc = launch_so3_inv(p->real, ln.w[l].F, y + sc.offset * esz, stride, S, sc.Pj, p->grids[sc.st.grid].fft, ln.s[l])))
                return rc;
        }
        if ((rc = lanes_join(p, ln))) return rc;
        i = e;
    }
    // scaling block: K_fwd^T Phi, then Y^H per shell
    if ((rc = launch_radial(p->Kfull_fwdT, P, P, bw.flmp, bw.flm_sh, cols, L, p->phi_ball, 0, false, s))) return rc;
    if ((rc = adj_harmonic_to_rings(p, p->sht, P, w, s))) return rc;
    if ((rc = launch_ring_inv(p->real, w.F, y + p->scaling_offset * esz, P, L, shell, p->grids[p->sht.grid].fft, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

}  // namespace s2w

// =================================================================================================================
// C ABI
// =================================================================================================================
extern "C" {

const char *s2w_last_error(void) { return g_err.c_str(); }
unsigned long long s2w_launch_count(void) { return g_launches; }

int s2w_scale_count(int L, double lambda, int *J)
{
    if (L < 1 || !(lambda > 1.0) || !J) {
        set_error("invalid argument");
        return S2W_EINVAL;
    }
    *J = scale_count(L, lambda);
    return S2W_OK;
}

int s2wav_kernels(double *psi, double *phi, int L, int N, double lambda, int J0)
{
    int rc = check_params(L, N, lambda, J0);
    if (rc) return rc;
    const int J = scale_count(L, lambda);
    std::vector<double> kappa, ksc, zeta;
    kappa_profiles(L, lambda, J0, J, kappa, ksc);
    zeta_tiling(L, N, zeta);
    const double pi = pi_d();
    const int nn = 2 * N - 1;
    if (psi)
        for (int j = J0; j <= J; ++j)
            for (int l = 0; l < L; ++l) {
                const double pre = std::sqrt((2.0 * l + 1.0) / (8.0 * pi * pi)) * kappa[(size_t)(j - J0) * L + l];
                for (int ni = 0; ni < nn; ++ni) {
                    const size_t o = (((size_t)(j - J0) * L + l) * nn + ni) * 2;
                    psi[o] = pre * zeta[((size_t)l * nn + ni) * 2];
                    psi[o + 1] = pre * zeta[((size_t)l * nn + ni) * 2 + 1];
                }
            }
    if (phi)
        for (int l = 0; l < L; ++l) phi[l] = std::sqrt((2.0 * l + 1.0) / (4.0 * pi)) * std::sqrt(ksc[l]);
    return S2W_OK;
}

int s2ball_kernels(double *kappa_l, double *kappa_p, double *zeta, double *phi, int L, int P, int N, double lambda_l,
                   double lambda_p, int J0)
{
    int rc = check_params(L, N, lambda_l, J0);
    if (rc) return rc;
    if (P < 1 || !(lambda_p > 1.0) || J0 > scale_count(P, lambda_p)) {
        set_error("invalid argument: need P >= 1, lambda_p > 1, J0 <= J'");
        return S2W_EINVAL;
    }
    const int J = scale_count(L, lambda_l), Jp = scale_count(P, lambda_p);
    std::vector<double> kl, kscl, kp, kscp, z;
    kappa_profiles(L, lambda_l, J0, J, kl, kscl);
    kappa_profiles(P, lambda_p, J0, Jp, kp, kscp);
    zeta_tiling(L, N, z);
    if (kappa_l) std::copy(kl.begin(), kl.end(), kappa_l);
    if (kappa_p) std::copy(kp.begin(), kp.end(), kappa_p);
    if (zeta) std::copy(z.begin(), z.end(), zeta);
    const double pi = pi_d();
    if (phi)
        for (int p = 0; p < P; ++p)
            for (int l = 0; l < L; ++l) {
                const double a = kscl[l], b = kscp[p];
                phi[(size_t)p * L + l] = std::sqrt((2.0 * l + 1.0) / (4.0 * pi)) * std::sqrt(a + b - a * b);
            }
    return S2W_OK;
}

int s2ball_radial_nodes(double *r, double *q, int P, double tau)
{
    if (P < 1 || !(tau > 0.0) || !r || !q) {
        set_error("invalid argument: need P >= 1, tau > 0");
        return S2W_EINVAL;
    }
    std::vector<double> x, w;
    gauss_laguerre2(P, x, w);
    if ((int)x.size() != P) {
        set_error("Gauss-Laguerre root search failed");
        return S2W_EUNSUPPORTED;
    }
    for (int i = 0; i < P; ++i) {
        r[i] = tau * x[i];
        q[i] = tau * tau * tau * w[i];
    }
    return S2W_OK;
}

int s2wav_plan_create(s2w_plan **out, int L, int N, double lambda, int J0, int multiresolution, int flags, int batch,
                      int device)
{
    return s2wav_plan_create_spin(out, L, N, lambda, J0, multiresolution, flags, batch, device, 0);
}

int s2wav_plan_create_spin(s2w_plan **out, int L, int N, double lambda, int J0, int multiresolution, int flags, int batch,
                           int device, int spin)
{
    if (!out) {
        set_error("null plan pointer");
        return S2W_EINVAL;
    }
    *out = 0;
    int rc = check_params(L, N, lambda, J0);
    if (rc) return rc;
    if (spin != 0 && ((flags & S2W_REAL) || std::abs(spin) >= L)) {
        set_error("invalid argument: a spin signal is complex and needs |spin| < L");
        return S2W_EINVAL;
    }
    if (batch < 1) {
        set_error("invalid argument: batch < 1");
        return S2W_EINVAL;
    }
    if (L > 2048) {
        set_error("L > 2048 is not supported");
        return S2W_EUNSUPPORTED;
    }
    if ((flags & S2W_DH) && (spin != 0 || L > 1024)) {
        set_error("Driscoll-Healy sampling: scalar signals (spin 0) up to L = 1024 (2L rings = 64 ring groups)");
        return S2W_EUNSUPPORTED;
    }
    S2W_CUDA_CHECK(cudaSetDevice(device));
    s2w_plan *p = new s2w_plan();
    p->kind = 0;
    p->dh = (flags & S2W_DH) ? 1 : 0;
    p->spin = spin;
    p->capture_stream = 0;
    for (int i = 0; i < S2W_LANES - 1; ++i) {
        p->lane_stream[i] = 0;
        p->lane_join[i] = 0;
    }
    p->lane_fork = 0;
    p->lanes_on = false;
    p->L = L;
    p->N = N;
    p->P = 1;
    p->lambda = lambda;
    p->nu = 0;
    p->tau = 1;
    p->J0 = J0;
    p->J = scale_count(L, lambda);
    p->J0p = p->Jp = 0;
    p->multires = multiresolution ? 1 : 0;
    p->flags = flags;
    p->batch = batch;
    p->device = device;
    p->real = (flags & S2W_REAL) != 0;
    p->Kfull_fwd = p->Kfull_inv = 0;
    p->Kfull_fwdT = p->Kfull_invT = 0;
    p->phi_ball = 0;
#define S2W_PLAN_TRY(expr)          \
    do {                            \
        rc = (expr);                \
        if (rc) {                   \
            s2w_plan_destroy(p);    \
            return rc;              \
        }                           \
    } while (0)
    S2W_PLAN_TRY(plan_common(p));

    const double pi = pi_d();
    std::vector<double> kappa, ksc, zeta;
    kappa_profiles(L, lambda, J0, p->J, kappa, ksc);
    zeta_tiling(L, N, zeta);
    const int nn = 2 * N - 1;

    // plain SHT at L: harmonic -> rings uses c_l, rings -> harmonic uses (2 pi / n) c_l   (Eqs. 2-3)
    {
        std::vector<double> a(L), s(L);
        for (int l = 0; l < L; ++l) {
            a[l] = std::sqrt((2.0 * l + 1.0) / (4.0 * pi));
            s[l] = a[l] * 2.0 * pi / (2.0 * L - 1.0);
        }
        S2W_PLAN_TRY(make_n0_stage(p, p->sht, L, a, s));
    }
    // scaling coefficients at L_s: c_l sqrt(4pi/(2l+1)) Phi_l0 = Phi_l0   (Eq. 29)
    p->Ls = scaling_bandlimit(L, lambda, J0, p->multires);
    {
        std::vector<double> a(p->Ls), s(p->Ls);
        for (int l = 0; l < p->Ls; ++l) {
            a[l] = std::sqrt((2.0 * l + 1.0) / (4.0 * pi)) * std::sqrt(ksc[l]);
            s[l] = a[l] * 2.0 * pi / (2.0 * p->Ls - 1.0);
        }
        S2W_PLAN_TRY(make_n0_stage(p, p->scaling, p->Ls, a, s));
    }
    size_t off = 0;
    p->scaling_offset = 0;
    const size_t rf = p->dh ? 2 : 1;  // rings per band-limit: Driscoll-Healy grids have 2 L_j rings
    off += grid_pixels(p, p->Ls);
    size_t maxF = (size_t)(p->spin ? 2 : 1) * rf * L * (p->real ? L : 2 * L - 1);
    for (int j = J0; j <= p->J; ++j) {
        Scale sc;
        memset(&sc, 0, sizeof(sc));
        sc.j = j;
        sc.jp = 0;
        sc.Pj = 1;
        sc.Lj = scale_bandlimit(j, L, lambda, p->multires);
        sc.offset = off;
        off += (size_t)nn * grid_pixels(p, sc.Lj);
        S2W_PLAN_TRY(make_scale_stage(p, sc, &kappa[(size_t)(j - J0) * L], zeta));
        maxF = std::max(maxF, (size_t)N * rf * sc.Lj * (p->real ? sc.Lj : 2 * sc.Lj - 1));
        p->scales.push_back(sc);
    }
    p->coeff_elems = off;
    p->signal_elems = grid_pixels(p, L);
    p->ws_flm_elems = (size_t)batch * (p->real ? L : 2 * L - 1) * L;
    p->ws_F_elems = (size_t)batch * maxF;
    p->ws_bytes = (((p->ws_flm_elems + 15) / 16) * 16 + (3 + 2 * (S2W_LANES - 1)) * (((p->ws_F_elems + 15) / 16) * 16)) * sizeof(cplx) + 256;
    S2W_PLAN_TRY(cudaDeviceSynchronize() == cudaSuccess ? S2W_OK : S2W_ECUDA);
    *out = p;
    return S2W_OK;
}

static int ball_plan_create(s2w_plan **out, int L, int P, int N, double lambda_l, double lambda_p, int J0, double tau,
                            int flags, int device);

int s2ball_plan_create(s2w_plan **out, int L, int P, int N, double lambda_l, double lambda_p, int J0, double tau,
                       int flags, int device)
{
    int rc = ball_plan_create(out, L, P, N, lambda_l, lambda_p, J0, tau, flags, device);
    // the precomputed tables are a default here, not a request: without room for them the plan runs the recursion
    if (rc == S2W_ENOMEM && !(flags & (S2W_PRECOMPUTE | S2W_RECURSION))) {
        cudaGetLastError();
        rc = ball_plan_create(out, L, P, N, lambda_l, lambda_p, J0, tau, flags | S2W_RECURSION, device);
    }
    return rc;
}

static int ball_plan_create(s2w_plan **out, int L, int P, int N, double lambda_l, double lambda_p, int J0, double tau,
                            int flags, int device)
{
    if (!out) {
        set_error("null plan pointer");
        return S2W_EINVAL;
    }
    *out = 0;
    int rc = check_params(L, N, lambda_l, J0);
    if (!rc && (flags & S2W_DH)) {
        set_error("Driscoll-Healy sampling is available for sphere plans only");
        return S2W_EUNSUPPORTED;
    }
    if (rc) return rc;
    if (P < 1 || !(lambda_p > 1.0) || !(tau > 0.0) || J0 > scale_count(P, lambda_p)) {
        set_error("invalid argument: need P >= 1, lambda_p > 1, tau > 0, J0 <= J'");
        return S2W_EINVAL;
    }
    if (L > 2048) {
        set_error("L > 2048 is not supported");
        return S2W_EUNSUPPORTED;
    }
    // Small angular band-limits: a ball plan contracts hundreds of columns (shells x signed columns) with every Wigner-d
    // value, and the tables of all its grids are a few tens of MB (L2-resident): the precomputed-kernel variant with the
    // theta quadrature folded into the table (GridTab::dtab_rw) is the default there ("simply precomputed" below
    // L ~ 256); S2W_RECURSION keeps the on-the-fly recursion.
    if (!(flags & (S2W_PRECOMPUTE | S2W_RECURSION)) && L <= fold_max_l()) flags |= S2W_PRECOMPUTE;
    S2W_CUDA_CHECK(cudaSetDevice(device));
    s2w_plan *p = new s2w_plan();
    p->kind = 1;
    p->spin = 0;
    p->capture_stream = 0;
    for (int i = 0; i < S2W_LANES - 1; ++i) {
        p->lane_stream[i] = 0;
        p->lane_join[i] = 0;
    }
    p->lane_fork = 0;
    p->lanes_on = false;
    p->L = L;
    p->N = N;
    p->P = P;
    p->lambda = lambda_l;
    p->nu = lambda_p;
    p->tau = tau;
    p->J0 = J0;
    p->J = scale_count(L, lambda_l);
    p->J0p = J0;
    p->Jp = scale_count(P, lambda_p);
    p->multires = 1;
    p->flags = flags;
    p->batch = 1;
    p->device = device;
    p->real = (flags & S2W_REAL) != 0;
    p->Kfull_fwd = p->Kfull_inv = 0;
    p->Kfull_fwdT = p->Kfull_invT = 0;
    p->phi_ball = 0;
    p->dh = 0;
    S2W_PLAN_TRY(plan_common(p));

    const double pi = pi_d();
    std::vector<double> kl, kscl, kp, kscp, zeta;
    kappa_profiles(L, lambda_l, J0, p->J, kl, kscl);
    kappa_profiles(P, lambda_p, J0, p->Jp, kp, kscp);
    zeta_tiling(L, N, zeta);
    const int nn = 2 * N - 1;
    {
        std::vector<double> a(L), s(L);
        for (int l = 0; l < L; ++l) {
            a[l] = std::sqrt((2.0 * l + 1.0) / (4.0 * pi));
            s[l] = a[l] * 2.0 * pi / (2.0 * L - 1.0);
        }
        S2W_PLAN_TRY(make_n0_stage(p, p->sht, L, a, s));
    }
    p->scaling = p->sht;
    p->Ls = L;  // the scaling function is non-zero on the cross {l small} u {p small}: full resolution (R9)
    // radial matrices on the full P-node grid
    {
        std::vector<double> x, qw, K;
        gauss_laguerre2(P, x, qw);
        if ((int)x.size() != P) {
            set_error("Gauss-Laguerre root search failed");
            s2w_plan_destroy(p);
            return S2W_EUNSUPPORTED;
        }
        laguerre_basis(P, x, tau, K);  // K[p][i]
        const double t3 = tau * tau * tau;
        std::vector<double> fwd((size_t)P * P), inv((size_t)P * P), phi((size_t)P * L);
        for (int pp = 0; pp < P; ++pp)
            for (int i = 0; i < P; ++i) {
                fwd[(size_t)pp * P + i] = t3 * qw[i] * K[(size_t)pp * P + i];
                inv[(size_t)i * P + pp] = K[(size_t)pp * P + i];
            }
        for (int pp = 0; pp < P; ++pp)
            for (int l = 0; l < L; ++l) {
                const double a = kscl[l], b = kscp[pp];
                phi[(size_t)pp * L + l] = std::sqrt(a + b - a * b);  // sqrt(4pi/(2l+1)) Phi_{l0p}
            }
        S2W_PLAN_TRY(p->pool.upload(&p->Kfull_fwd, fwd));
        S2W_PLAN_TRY(p->pool.upload(&p->Kfull_inv, inv));
        {
            std::vector<double> fwdT((size_t)P * P), invT((size_t)P * P);
            for (int a = 0; a < P; ++a)
                for (int b = 0; b < P; ++b) {
                    fwdT[(size_t)b * P + a] = fwd[(size_t)a * P + b];
                    invT[(size_t)b * P + a] = inv[(size_t)a * P + b];
                }
            S2W_PLAN_TRY(p->pool.upload(&p->Kfull_fwdT, fwdT));
            S2W_PLAN_TRY(p->pool.upload(&p->Kfull_invT, invT));
        }
        S2W_PLAN_TRY(p->pool.upload(&p->phi_ball, phi));
    }
    size_t off = 0;
    p->scaling_offset = 0;
    off += (size_t)P * L * (2 * L - 1);
    size_t maxF = (size_t)L * (p->real ? L : 2 * L - 1);
    // angular stages, one per j (shared by all j')
    std::vector<Scale> ang;
    for (int j = J0; j <= p->J; ++j) {
        Scale sc;
        memset(&sc, 0, sizeof(sc));
        sc.j = j;
        sc.Lj = scale_bandlimit(j, L, lambda_l, true);
        S2W_PLAN_TRY(make_scale_stage(p, sc, &kl[(size_t)(j - J0) * L], zeta));
        maxF = std::max(maxF, (size_t)N * sc.Lj * (p->real ? sc.Lj : 2 * sc.Lj - 1));
        ang.push_back(sc);
    }
    for (int jp = p->J0p; jp <= p->Jp; ++jp) {
        const int Pj = scale_bandlimit(jp, P, lambda_p, true);
        std::vector<double> x, qw, K;
        gauss_laguerre2(Pj, x, qw);
        if ((int)x.size() != Pj) {
            set_error("Gauss-Laguerre root search failed");
            s2w_plan_destroy(p);
            return S2W_EUNSUPPORTED;
        }
        laguerre_basis(Pj, x, tau, K);  // K[p][i], p < Pj, on the Pj-node grid
        const double t3 = tau * tau * tau;
        const double *kj = &kp[(size_t)(jp - p->J0p) * P];
        std::vector<double> kinv((size_t)Pj * Pj), kfwd((size_t)Pj * Pj);
        for (int pp = 0; pp < Pj; ++pp)
            for (int i = 0; i < Pj; ++i) {
                kinv[(size_t)i * Pj + pp] = K[(size_t)pp * Pj + i] * kj[pp];
                kfwd[(size_t)pp * Pj + i] = t3 * qw[i] * K[(size_t)pp * Pj + i] * kj[pp];
            }
        double *dKinv, *dKfwd, *dKinvT, *dKfwdT;
        S2W_PLAN_TRY(p->pool.upload(&dKinv, kinv));
        S2W_PLAN_TRY(p->pool.upload(&dKfwd, kfwd));
        {
            std::vector<double> kinvT((size_t)Pj * Pj), kfwdT((size_t)Pj * Pj);
            for (int a = 0; a < Pj; ++a)
                for (int b = 0; b < Pj; ++b) {
                    kinvT[(size_t)b * Pj + a] = kinv[(size_t)a * Pj + b];
                    kfwdT[(size_t)b * Pj + a] = kfwd[(size_t)a * Pj + b];
                }
            S2W_PLAN_TRY(p->pool.upload(&dKinvT, kinvT));
            S2W_PLAN_TRY(p->pool.upload(&dKfwdT, kfwdT));
        }
        for (size_t a = 0; a < ang.size(); ++a) {
            Scale sc = ang[a];
            sc.jp = jp;
            sc.Pj = Pj;
            sc.Kinv = dKinv;
            sc.Kfwd = dKfwd;
            sc.KinvT = dKinvT;
            sc.KfwdT = dKfwdT;
            sc.offset = off;
            off += (size_t)Pj * nn * sc.Lj * (2 * sc.Lj - 1);
            p->scales.push_back(sc);
        }
    }
    p->coeff_elems = off;
    p->signal_elems = (size_t)P * L * (2 * L - 1);
    p->ws_shell_elems = (size_t)P * (p->real ? L : 2 * L - 1) * L;
    p->ws_flm_elems = 2 * (((p->ws_shell_elems + 15) / 16) * 16);
    p->ws_F_elems = (size_t)P * maxF;
    // stacked shells (see the plan's fields): matrices, k ranges per 64-row tile, per-j offset tables
    {
        const int njp = p->Jp - p->J0p + 1, nj = (int)ang.size();
        std::vector<int> base(njp + 1, 0), Pjs(njp);
        for (int a = 0; a < njp; ++a) {
            Pjs[a] = p->scales[(size_t)a * nj].Pj;
            base[a + 1] = base[a] + Pjs[a];
        }
        const int PS = base[njp];
        p->PS = PS;
        std::vector<double> kinv((size_t)PS * P, 0.0), kfwd((size_t)P * PS, 0.0);
        for (int a = 0; a < njp; ++a) {
            const int Pj = Pjs[a];
            std::vector<double> hi((size_t)Pj * Pj), hf((size_t)Pj * Pj);
            const Scale &sc = p->scales[(size_t)a * nj];
            S2W_PLAN_TRY(cudaMemcpy(hi.data(), sc.Kinv, hi.size() * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess ? S2W_OK : S2W_ECUDA);
            S2W_PLAN_TRY(cudaMemcpy(hf.data(), sc.Kfwd, hf.size() * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess ? S2W_OK : S2W_ECUDA);
            for (int i = 0; i < Pj; ++i)
                for (int pp = 0; pp < Pj; ++pp) {
                    kinv[(size_t)(base[a] + i) * P + pp] = hi[(size_t)i * Pj + pp];
                    kfwd[(size_t)pp * PS + base[a] + i] = hf[(size_t)pp * Pj + i];
                }
        }
        S2W_PLAN_TRY(p->pool.upload(&p->Kstk_inv, kinv));
        S2W_PLAN_TRY(p->pool.upload(&p->Kstk_fwd, kfwd));
        std::vector<int2> kri((PS + 63) / 64), krf((P + 63) / 64);
        for (size_t t = 0; t < kri.size(); ++t) {  // rows = stacked nodes, ascending P_j': the last row's P_j' bounds k
            const int rlast = std::min(PS - 1, (int)t * 64 + 63);
            int a = 0;
            while (base[a + 1] <= rlast) ++a;
            kri[t] = make_int2(0, Pjs[a]);
        }
        for (size_t t = 0; t < krf.size(); ++t) {  // rows = p: nodes of the scales with P_j' > first p of the tile
            int a = 0;
            while (a < njp - 1 && Pjs[a] <= (int)t * 64) ++a;
            krf[t] = make_int2(base[a], PS);
        }
        S2W_PLAN_TRY(p->pool.upload(&p->krange_inv, kri));
        S2W_PLAN_TRY(p->pool.upload(&p->krange_fwd, krf));
        for (int j = 0; j < nj; ++j) {
            Scale sc = ang[j];
            sc.Pj = PS;
            sc.jp = -1;
            p->ang.push_back(sc);
            std::vector<size_t> offs(PS);
            for (int a = 0; a < njp; ++a) {
                const Scale &q = p->scales[(size_t)a * nj + j];
                const size_t stride = (size_t)nn * q.Lj * (2 * q.Lj - 1);
                for (int i = 0; i < Pjs[a]; ++i) offs[base[a] + i] = q.offset + (size_t)i * stride;
            }
            size_t *doff;
            S2W_PLAN_TRY(p->pool.upload(&doff, offs));
            p->ang_off.push_back(doff);
        }
        p->ws_stk_elems = (((size_t)PS * (p->real ? L : 2 * L - 1) * L + 15) / 16) * 16;
        p->ws_stkF_elems = (((size_t)PS * maxF + 15) / 16) * 16;
    }
    p->ws_stk_off = p->ws_flm_elems + (2 + 2 * (S2W_LANES - 1)) * (((p->ws_F_elems + 15) / 16) * 16);
    p->ws_bytes = (p->ws_stk_off + p->ws_stk_elems + 2 * S2W_BALL_LANES * p->ws_stkF_elems) * sizeof(cplx) + 256;
    S2W_PLAN_TRY(cudaDeviceSynchronize() == cudaSuccess ? S2W_OK : S2W_ECUDA);
    *out = p;
    return S2W_OK;
}

int s2w_plan_destroy(s2w_plan *p)
{
    if (!p) return S2W_OK;
    for (auto &g : p->graphs) cudaGraphExecDestroy(g.exec);
    if (p->capture_stream) cudaStreamDestroy(p->capture_stream);
    for (int i = 0; i < S2W_LANES - 1; ++i) {
        if (p->lane_stream[i]) cudaStreamDestroy(p->lane_stream[i]);
        if (p->lane_join[i]) cudaEventDestroy(p->lane_join[i]);
    }
    if (p->lane_fork) cudaEventDestroy(p->lane_fork);
    p->pool.release();
    delete p;
    return S2W_OK;
}

int s2w_plan_scales(const s2w_plan *p, int *J0, int *J, int *J0p, int *Jp)
{
    if (!p) return S2W_EINVAL;
    if (J0) *J0 = p->J0;
    if (J) *J = p->J;
    if (J0p) *J0p = p->J0p;
    if (Jp) *Jp = p->Jp;
    return S2W_OK;
}

int s2w_plan_scale_shape(const s2w_plan *p, int j, int jp, int *n_r, int *n_gamma, int *n_theta, int *n_phi,
                         size_t *offset_elems)
{
    if (!p) return S2W_EINVAL;
    int nr = 1, ngam = 1, nt = 0, np = 0;
    size_t off = 0;
    if (j < 0) {
        nr = p->kind == 1 ? p->P : 1;
        nt = (p->dh ? 2 : 1) * p->Ls;
        np = 2 * p->Ls - 1;
        off = p->scaling_offset;
    } else {
        const Scale *sc = 0;
        for (size_t i = 0; i < p->scales.size(); ++i)
            if (p->scales[i].j == j && p->scales[i].jp == jp) sc = &p->scales[i];
        if (!sc) {
            set_error("no such scale");
            return S2W_EINVAL;
        }
        nr = sc->Pj;
        ngam = 2 * p->N - 1;
        nt = (p->dh ? 2 : 1) * sc->Lj;
        np = 2 * sc->Lj - 1;
        off = sc->offset;
    }
    if (n_r) *n_r = nr;
    if (n_gamma) *n_gamma = ngam;
    if (n_theta) *n_theta = nt;
    if (n_phi) *n_phi = np;
    if (offset_elems) *offset_elems = off;
    return S2W_OK;
}

size_t s2w_plan_coeff_elems(const s2w_plan *p) { return p ? p->coeff_elems : 0; }
size_t s2w_plan_signal_elems(const s2w_plan *p) { return p ? p->signal_elems : 0; }
size_t s2w_plan_workspace_bytes(const s2w_plan *p) { return p ? p->ws_bytes : 0; }

static void *align256(void *p) { return (void *)(((uintptr_t)p + 255) & ~(uintptr_t)255); }

// One whole transform, directly on `s` or -- unless the per-class timers are on or S2W_NO_GRAPH is set -- as a CUDA
// graph: captured on the plan's private stream at the first call with a given (direction, in, out, work) and replayed
// on the caller's stream afterwards (the legacy default stream cannot be captured, a private one can).
static int run_transform(const s2w_plan *p, int dir, const void *in, void *out, void *work, cudaStream_t s)
{
    auto direct = [&](cudaStream_t st) {
        if (dir == 2) return p->kind == 1 ? ball_forward_adjoint(p, in, out, work, st) : sphere_forward_adjoint(p, in, out, work, st);
        if (dir == 3) return p->kind == 1 ? ball_inverse_adjoint(p, in, out, work, st) : sphere_inverse_adjoint(p, in, out, work, st);
        if (p->kind == 1) return dir == 0 ? ball_forward(p, in, out, work, st) : ball_inverse(p, in, out, work, st);
        return dir == 0 ? sphere_forward(p, in, out, work, st) : sphere_inverse(p, in, out, work, st);
    };
    static const bool no_graph = getenv("S2W_NO_GRAPH") != 0;
    static const bool lanes_direct = getenv("S2W_LANES_DIRECT") != 0;  // debugging: the lanes without a graph
    if (no_graph && lanes_direct && !g_timing) {
        std::lock_guard<std::mutex> lock(p->graph_mu);
        p->lanes_on = true;
        const int rc = direct(s);
        p->lanes_on = false;
        return rc;
    }
    if (no_graph || g_timing) return direct(s);
    std::lock_guard<std::mutex> lock(p->graph_mu);
    for (auto &g : p->graphs)
        if (g.dir == dir && g.in == in && g.out == out && g.work == work) {
            S2W_CUDA_CHECK(cudaGraphLaunch(g.exec, s));
            g_launches += g.launches;
            return S2W_OK;
        }
    if (!p->capture_stream) S2W_CUDA_CHECK(cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking));
    const unsigned long long n0 = g_launches;
    S2W_CUDA_CHECK(cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal));
    p->lanes_on = true;
    const int rc = direct(p->capture_stream);
    p->lanes_on = false;
    cudaGraph_t graph = 0;
    const cudaError_t ce = cudaStreamEndCapture(p->capture_stream, &graph);
    const unsigned long long nl = g_launches - n0;
    g_launches = n0;
    if (rc || ce != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        if (rc) return rc;
        return direct(s);  // capture not possible here: run the launches directly
    }
    s2w_plan::GraphEntry e;
    e.dir = dir;
    e.in = in;
    e.out = out;
    e.work = work;
    e.launches = nl;
    const cudaError_t ci = cudaGraphInstantiate(&e.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ci != cudaSuccess) {
        cudaGetLastError();
        return direct(s);
    }
    if (p->graphs.size() >= 16) {  // bounded cache: drop the oldest
        cudaGraphExecDestroy(p->graphs.front().exec);
        p->graphs.erase(p->graphs.begin());
    }
    p->graphs.push_back(e);
    S2W_CUDA_CHECK(cudaGraphLaunch(e.exec, s));
    g_launches += nl;
    return S2W_OK;
}

// A plan's tables, streams and events live on the device it was created for; its kernels must be launched with that
// device current (nothing checked this, so a call from another device's context launched on the wrong GPU).
static int check_device(const s2w_plan *p)
{
    int dev = -1;
    S2W_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev != p->device) {
        set_error("the current CUDA device (" + std::to_string(dev) + ") is not the plan's device (" +
                  std::to_string(p->device) + "): call cudaSetDevice / torch.cuda.set_device first");
        return S2W_EINVAL;
    }
    return S2W_OK;
}

int s2w_plan_forward(const s2w_plan *p, const void *in, void *out, void *work, void *stream)
{
    if (!p || !in || !out || !work) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    int rc = check_device(p);
    if (rc) return rc;
    return run_transform(p, 0, in, out, align256(work), (cudaStream_t)stream);
}

int s2w_plan_inverse(const s2w_plan *p, const void *in, void *out, void *work, void *stream)
{
    if (!p || !in || !out || !work) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    int rc = check_device(p);
    if (rc) return rc;
    return run_transform(p, 1, in, out, align256(work), (cudaStream_t)stream);
}

static int adjoint_supported(const s2w_plan *p, const void *in, const void *out, const void *work)
{
    if (!p || !in || !out || !work) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    {
        int rcd = check_device(p);
        if (rcd) return rcd;
    }
    if (p->dh) {
        set_error("the adjoint transforms are not available on Driscoll-Healy plans");
        return S2W_EUNSUPPORTED;
    }
    return S2W_OK;
}

int s2w_plan_forward_adjoint(const s2w_plan *p, const void *in, void *out, void *work, void *stream)
{
    int rc = adjoint_supported(p, in, out, work);
    if (rc) return rc;
    return run_transform(p, 2, in, out, align256(work), (cudaStream_t)stream);
}

int s2w_plan_inverse_adjoint(const s2w_plan *p, const void *in, void *out, void *work, void *stream)
{
    int rc = adjoint_supported(p, in, out, work);
    if (rc) return rc;
    return run_transform(p, 3, in, out, align256(work), (cudaStream_t)stream);
}

int s2w_plan_harmonic_forward(const s2w_plan *p, const void *f, void *flm, void *work, void *stream)
{
    if (!p || !f || !flm || !work) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    {
        int rcd = check_device(p);
        if (rcd) return rcd;
    }
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    if (p->kind == 1) {
        const BallWork bw = carve_ball(p, align256(work));
        Work w;
        w.flmT = bw.flm_sh;
        w.F = bw.F;
        w.Ft = bw.Ft;
        const size_t cols = (size_t)(p->real ? p->L : 2 * p->L - 1) * p->L;
        if ((rc = sht_forward_dev(p, p->sht, f, (size_t)p->L * (2 * p->L - 1), p->P, w, true, s))) return rc;
        if ((rc = launch_radial(p->Kfull_fwd, p->P, p->P, bw.flm_sh, bw.flmp, cols, p->L, 0, 0, false, s))) return rc;
        if ((rc = launch_flm_unpack(bw.flmp, (cplx *)flm, p->P, p->L, p->real, s))) return rc;
    } else {
        const Work w = carve(p, align256(work));
        if ((rc = sht_forward_dev(p, p->sht, f, p->signal_elems, p->batch, w, true, s))) return rc;
        if ((rc = launch_flm_unpack(w.flmT, (cplx *)flm, p->batch, p->L, p->real, s))) return rc;
    }
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

int s2w_plan_harmonic_inverse(const s2w_plan *p, const void *flm, void *f, void *work, void *stream)
{
    if (!p || !f || !flm || !work) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    {
        int rcd = check_device(p);
        if (rcd) return rcd;
    }
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    if (p->kind == 1) {
        const BallWork bw = carve_ball(p, align256(work));
        Work w;
        w.flmT = bw.flm_sh;
        w.F = bw.F;
        w.Ft = bw.Ft;
        const size_t cols = (size_t)(p->real ? p->L : 2 * p->L - 1) * p->L;
        if ((rc = launch_flm_pack((const cplx *)flm, bw.flmp, p->P, p->L, p->real, s))) return rc;
        if ((rc = launch_radial(p->Kfull_inv, p->P, p->P, bw.flmp, bw.flm_sh, cols, p->L, 0, 0, false, s))) return rc;
        if ((rc = sht_inverse_dev(p, p->sht, f, (size_t)p->L * (2 * p->L - 1), p->P, w, s))) return rc;
    } else {
        const Work w = carve(p, align256(work));
        if ((rc = launch_flm_pack((const cplx *)flm, w.flmT, p->batch, p->L, p->real, s))) return rc;
        if ((rc = sht_inverse_dev(p, p->sht, f, p->signal_elems, p->batch, w, s))) return rc;
    }
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- the forward harmonic transform with its scratch in a static device array (s2w.h: s2w_plan_harmonic_forward_static)
// For callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).  The scratch of
// steps a1-a3 (flmT, F, Ft) is carved from g_static_scratch instead of a caller buffer.  In host code the name
// g_static_scratch is only a host-side stand-in for the array: its DEVICE address is fetched with cudaGetSymbolAddress,
// once per device and with that device current, and only that pointer goes to the kernels.
static __device__ __align__(256) unsigned char g_static_scratch[S2W_STATIC_SCRATCH_BYTES];

static int static_scratch_ptr(int device, void **out)
{
    enum { MAXDEV = 64 };
    static std::mutex mu;
    static void *ptr[MAXDEV] = {0};
    if (device < 0 || device >= MAXDEV) {
        set_error("s2w_plan_harmonic_forward_static: device ordinal out of range");
        return S2W_EINVAL;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[device]) {  // check_device() has made sure that `device` is the current one
        void *q = 0;
        const cudaError_t e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess || !q) {
            set_error(std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
            cudaGetLastError();
            return S2W_ECUDA;
        }
        ptr[device] = q;
    }
    *out = ptr[device];
    return S2W_OK;
}

int s2w_plan_harmonic_forward_static(const s2w_plan *p, const void *f, void *flm, void *stream)
{
    if (!p || !f || !flm) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    if (p->kind != 0) {
        set_error("s2w_plan_harmonic_forward_static: sphere plans only");
        return S2W_EUNSUPPORTED;
    }
    if (g_timing) {
        set_error("s2w_plan_harmonic_forward_static: the per-class timers create events (s2w_timing_enable(0) first)");
        return S2W_EUNSUPPORTED;
    }
    int rc = check_device(p);
    if (rc) return rc;
    // carve(): flmT, then F and Ft, each rounded up to 16 elements
    const size_t need = (((p->ws_flm_elems + 15) / 16) * 16 + 2 * (((p->ws_F_elems + 15) / 16) * 16)) * sizeof(cplx);
    if (need > (size_t)S2W_STATIC_SCRATCH_BYTES) {
        set_error("s2w_plan_harmonic_forward_static: this plan needs " + std::to_string(need) +
                  " bytes of scratch, the static array holds " + std::to_string((size_t)S2W_STATIC_SCRATCH_BYTES) +
                  " (S2W_STATIC_SCRATCH_BYTES): use s2w_plan_harmonic_forward with a caller workspace");
        return S2W_EINVAL;
    }
    void *scratch = 0;
    if ((rc = static_scratch_ptr(p->device, &scratch))) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const Work w = carve(p, scratch);
    // flmT is accumulated into and is cleared by sht_forward_dev (zero_first); F and Ft are fully overwritten
    if ((rc = sht_forward_dev(p, p->sht, f, p->signal_elems, p->batch, w, true, s))) return rc;
    if ((rc = launch_flm_unpack(w.flmT, (cplx *)flm, p->batch, p->L, p->real, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- Wigner-Laguerre (Q) and spherical-Laguerre (Z) transforms as stand-alone calls (Eqs. 10-11, 24-25) ----------
static int qplan_create(s2w_plan **out, int L, int P, int N, double tau, int device)
{
    *out = 0;
    if (L < 1 || P < 1 || N < 1 || N > L || N > S2W_MAX_N || L > 2048 || !(tau > 0)) {
        set_error("invalid argument: need 1 <= N <= L <= 2048, N <= 32, P >= 1, tau > 0");
        return S2W_EINVAL;
    }
    S2W_CUDA_CHECK(cudaSetDevice(device));
    s2w_plan *p = new s2w_plan();
    int rc;
    p->kind = 2;
    p->spin = 0;
    p->capture_stream = 0;
    for (int i = 0; i < S2W_LANES - 1; ++i) {
        p->lane_stream[i] = 0;
        p->lane_join[i] = 0;
    }
    p->lane_fork = 0;
    p->lanes_on = false;
    p->L = L;
    p->N = N;
    p->P = P;
    p->lambda = p->nu = 2.0;
    p->tau = tau;
    p->J0 = p->J = p->J0p = p->Jp = 0;
    p->multires = 0;
    p->flags = 0;
    p->batch = 1;
    p->device = device;
    p->real = false;
    p->Kfull_fwd = p->Kfull_inv = p->Kfull_fwdT = p->Kfull_invT = 0;
    p->phi_ball = 0;
    p->PS = 0;
    S2W_PLAN_TRY(plan_common(p));
    S2W_PLAN_TRY(build_grid(p, L));
    const double pi = pi_d();
    const int nn = 2 * N - 1;
    std::vector<cplx> fa(L), fs(L);
    for (int l = 0; l < L; ++l) {
        fa[l] = cmake((2.0 * l + 1.0) / (8.0 * pi * pi), 0.0);        // Eq. 5 / Eq. 25
        fs[l] = cmake(4.0 * pi * pi / (2.0 * L - 1.0), 0.0);          // Eq. 4 on the MW x gamma grid
    }
    std::vector<int> all_n, all_rows;
    for (int n = -(N - 1); n <= N - 1; ++n) {
        Stage st;
        memset(&st, 0, sizeof(st));
        st.grid = grid_index(p, L);
        st.Lg = L;
        st.lmin = 0;
        st.nn = 1;
        st.nrows = nn;
        st.n_val[0] = n;
        st.n_tab[0] = find_tab(p, n);
        st.n_row[0] = n + N - 1;
        st.n_rowm[0] = -n + N - 1;   // the mirror columns (-m, -n) belong to the row of -n
        st.n_filtm[0] = 0;
        S2W_PLAN_TRY(make_stage_filters(p, st, fa, fs, (2.0 * L - 1.0) * nn));
        p->qst.push_back(st);
        all_n.push_back(n);
        all_rows.push_back(n + N - 1);
    }
    memset(&p->qall, 0, sizeof(p->qall));
    p->qall.grid = grid_index(p, L);
    p->qall.Lg = L;
    S2W_PLAN_TRY(fill_stage_rows(p, p->qall, all_n, all_rows, nn));
    {
        std::vector<double> x, qw, K;
        gauss_laguerre2(P, x, qw);
        if ((int)x.size() != P) {
            set_error("Gauss-Laguerre root search failed");
            s2w_plan_destroy(p);
            return S2W_EUNSUPPORTED;
        }
        laguerre_basis(P, x, tau, K);
        const double t3 = tau * tau * tau;
        std::vector<double> fwd((size_t)P * P), inv((size_t)P * P);
        for (int pp = 0; pp < P; ++pp)
            for (int i = 0; i < P; ++i) {
                fwd[(size_t)pp * P + i] = t3 * qw[i] * K[(size_t)pp * P + i];
                inv[(size_t)i * P + pp] = K[(size_t)pp * P + i];
            }
        S2W_PLAN_TRY(p->pool.upload(&p->Kfull_fwd, fwd));
        S2W_PLAN_TRY(p->pool.upload(&p->Kfull_inv, inv));
    }
    p->signal_elems = p->coeff_elems = (size_t)P * nn * L * (2 * L - 1);
    p->ws_shell_elems = (((size_t)P * (2 * L - 1) * L + 15) / 16) * 16;      // one internal [P][Mfull][L] array
    p->ws_F_elems = (((size_t)P * nn * L * (2 * L - 1) + 15) / 16) * 16;     // F and Ft
    p->ws_flm_elems = 2 * (size_t)nn * p->ws_shell_elems;                   // H_n and G_n for every signed n
    p->ws_bytes = (p->ws_flm_elems + 2 * p->ws_F_elems) * sizeof(cplx) + 256;
    S2W_PLAN_TRY(cudaDeviceSynchronize() == cudaSuccess ? S2W_OK : S2W_ECUDA);
    *out = p;
    return S2W_OK;
}

// f [P][2N-1][L][2L-1] -> fhat [2N-1][P][L][2L-1]
static int q_forward_dev(const s2w_plan *p, const void *f, void *fhat, void *work, cudaStream_t s)
{
    const int L = p->L, P = p->P, nn = 2 * p->N - 1;
    cplx *H = (cplx *)align256(work), *Gb = H + (size_t)nn * p->ws_shell_elems;
    cplx *F = Gb + (size_t)nn * p->ws_shell_elems, *Ft = F + p->ws_F_elems;
    const GridTab &g = p->grids[p->qall.grid];
    const size_t cols = (size_t)(2 * L - 1) * L, blk = (size_t)P * L * (2 * L - 1);
    int rc;
    So3Args S;
    fill_so3_args(p, p->qall, S);
    if ((rc = launch_so3_fwd(false, f, (size_t)nn * L * (2 * L - 1), F, S, P, g.fft, s))) return rc;
    RwArgs R;
    fill_rw_args(p, p->qall, R);
    if ((rc = g.rw.L ? launch_reweight_th(F, Ft, R, P, g.rw, s) : launch_reweight(F, Ft, R, P, g.fft, s))) return rc;
    S2W_CUDA_CHECK(cudaMemsetAsync(H, 0, (size_t)nn * p->ws_shell_elems * sizeof(cplx), s));
    for (int q = 0; q < nn; ++q) {
        WigArgs A;
        fill_wig_args(p, p->qst[q], true, P, H + (size_t)q * p->ws_shell_elems, Ft, A);
        if ((rc = launch_wigner_forward(A, s))) return rc;
        if ((rc = launch_radial(p->Kfull_fwd, P, P, H + (size_t)q * p->ws_shell_elems, Gb + (size_t)q * p->ws_shell_elems, cols,
                                L, 0, 0, false, s)))
            return rc;
    }
    for (int q = 0; q < nn; ++q)
        if ((rc = launch_flm_unpack_pm(Gb + (size_t)q * p->ws_shell_elems, (cplx *)fhat + (size_t)q * blk,
                                       (cplx *)fhat + (size_t)(nn - 1 - q) * blk, P, L, s)))
            return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

static int q_inverse_dev(const s2w_plan *p, const void *fhat, void *f, void *work, cudaStream_t s)
{
    const int L = p->L, P = p->P, nn = 2 * p->N - 1;
    cplx *H = (cplx *)align256(work), *Gb = H + (size_t)nn * p->ws_shell_elems;
    cplx *F = Gb + (size_t)nn * p->ws_shell_elems;
    const GridTab &g = p->grids[p->qall.grid];
    const size_t cols = (size_t)(2 * L - 1) * L, blk = (size_t)P * L * (2 * L - 1);
    int rc;
    for (int q = 0; q < nn; ++q) {
        cplx *Gq = Gb + (size_t)q * p->ws_shell_elems, *Hq = H + (size_t)q * p->ws_shell_elems;
        if ((rc = launch_flm_pack_pm((const cplx *)fhat + (size_t)q * blk, (const cplx *)fhat + (size_t)(nn - 1 - q) * blk, Gq, P,
                                     L, s)))
            return rc;
        if ((rc = launch_radial(p->Kfull_inv, P, P, Gq, Hq, cols, L, 0, 0, false, s))) return rc;
        WigArgs A;
        fill_wig_args(p, p->qst[q], false, P, Hq, F, A);
        if ((rc = launch_wigner_inverse(A, s))) return rc;
    }
    So3Args S;
    fill_so3_args(p, p->qall, S);
    if ((rc = launch_so3_inv(false, F, f, (size_t)nn * L * (2 * L - 1), S, P, g.fft, s))) return rc;
    S2W_CUDA_CHECK(cudaPeekAtLastError());
    return S2W_OK;
}

// ---- plan cache behind the argument-style entry points ----
namespace {
struct CacheKey {
    int kind, L, P, N, J0, multires, flags, batch, device;
    double lam, nu, tau;
    bool operator<(const CacheKey &o) const
    {
        return std::memcmp(this, &o, sizeof(CacheKey)) < 0;
    }
};
// Users of one cache entry share ONE workspace and one pair of staging buffers: they are serialised.  Host
// threads take `mu` for the duration of their launches; on the device every use waits for the event the previous use
// recorded on its own stream, so two calls with the same parameters on different streams run one after the other.
struct EntrySync {
    std::mutex mu;
    cudaEvent_t done;
    bool used;
    cudaStream_t copy_stream;  // second stream of the host-buffer pipeline, created on the entry's device
};
struct CacheEntry {
    s2w_plan *plan;
    void *work;
    void *d_sig, *d_cof;  // device staging buffers of the host-buffer entry points (allocated on first use)
    EntrySync *sync;
};

// run `fn(stream)` as the next user of entry `e` on `stream`
int entry_serialised(const CacheEntry &e, cudaStream_t stream, const std::function<int(cudaStream_t)> &fn)
{
    std::lock_guard<std::mutex> lock(e.sync->mu);
    if (e.sync->used) S2W_CUDA_CHECK(cudaStreamWaitEvent(stream, e.sync->done, 0));
    const int rc = fn(stream);
    S2W_CUDA_CHECK(cudaEventRecord(e.sync->done, stream));
    e.sync->used = true;
    return rc;
}
std::map<CacheKey, CacheEntry> g_cache;
std::mutex g_cache_mu;

int cached_plan(int kind, int L, int P, int N, double lambda, double nu, double tau, int J0, int multires, int flags,
                int batch, CacheEntry *e)
{
    int device = 0;
    S2W_CUDA_CHECK(cudaGetDevice(&device));
    CacheKey k;
    std::memset(&k, 0, sizeof(k));
    k.kind = kind;
    k.L = L;
    k.P = P;
    k.N = N;
    k.J0 = J0;
    k.multires = multires ? 1 : 0;
    k.flags = flags;
    k.batch = batch;
    k.device = device;
    k.lam = lambda;
    k.nu = nu;
    k.tau = tau;
    std::lock_guard<std::mutex> lock(g_cache_mu);
    auto it = g_cache.find(k);
    if (it == g_cache.end()) {
        CacheEntry ne;
        ne.plan = 0;
        ne.work = 0;
        ne.d_sig = ne.d_cof = 0;
        ne.sync = 0;
        int rc = kind == 0   ? s2wav_plan_create(&ne.plan, L, N, lambda, J0, multires, flags, batch, device)
                 : kind == 1 ? s2ball_plan_create(&ne.plan, L, P, N, lambda, nu, J0, tau, flags, device)
                             : qplan_create(&ne.plan, L, P, N, tau, device);
        if (rc) return rc;
        cudaError_t ce = cudaMalloc(&ne.work, s2w_plan_workspace_bytes(ne.plan));
        if (ce != cudaSuccess) {
            s2w_plan_destroy(ne.plan);
            set_error(std::string("cudaMalloc(workspace): ") + cudaGetErrorString(ce));
            cudaGetLastError();
            return S2W_ENOMEM;
        }
        ne.sync = new EntrySync();
        ne.sync->used = false;
        ne.sync->copy_stream = 0;
        if (cudaEventCreateWithFlags(&ne.sync->done, cudaEventDisableTiming) != cudaSuccess ||
            cudaStreamCreateWithFlags(&ne.sync->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError();
            delete ne.sync;
            cudaFree(ne.work);
            s2w_plan_destroy(ne.plan);
            set_error("cudaEventCreate / cudaStreamCreate for a cache entry failed");
            return S2W_ECUDA;
        }
        it = g_cache.insert(std::make_pair(k, ne)).first;
    }
    *e = it->second;
    return S2W_OK;
}

// as cached_plan, and makes sure the entry owns device staging buffers for one signal batch and one coefficient batch
int cached_plan_staged(int kind, int L, int P, int N, double lambda, double nu, double tau, int J0, int multires,
                       int flags, int batch, CacheEntry *e)
{
    int rc = cached_plan(kind, L, P, N, lambda, nu, tau, J0, multires, flags, batch, e);
    if (rc || e->d_sig) return rc;
    std::lock_guard<std::mutex> lock(g_cache_mu);
    for (auto &kv : g_cache) {
        if (kv.second.plan != e->plan) continue;
        const size_t esz = e->plan->real ? sizeof(double) : sizeof(cplx);
        const size_t sig = e->plan->signal_elems * e->plan->batch * esz, cof = e->plan->coeff_elems * e->plan->batch * esz;
        if (cudaMalloc(&kv.second.d_sig, sig) != cudaSuccess || cudaMalloc(&kv.second.d_cof, cof) != cudaSuccess) {
            cudaFree(kv.second.d_sig);
            kv.second.d_sig = kv.second.d_cof = 0;
            cudaGetLastError();
            set_error("cudaMalloc(staging buffers) failed");
            return S2W_ENOMEM;
        }
        *e = kv.second;
        return S2W_OK;
    }
    return S2W_EINVAL;
}

// host-buffer variant of a cached transform: copy in, transform, copy out, synchronise.  Copies are asynchronous when
// the host buffers are pinned (cudaHostAlloc / cudaHostRegister / torch pin_memory) and staged by the driver otherwise.
int host_transform(bool fwd, const CacheEntry &e, const void *in_h, void *out_h)
{
    if (!in_h || !out_h) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    const s2w_plan *p = e.plan;
    const size_t esz = p->real ? sizeof(double) : sizeof(cplx);
    const size_t sig = p->signal_elems * p->batch * esz, cof = p->coeff_elems * p->batch * esz;
    void *d_in = fwd ? e.d_sig : e.d_cof, *d_out = fwd ? e.d_cof : e.d_sig;
    int rc = S2W_OK;
    // one user of the entry's workspace and staging buffers at a time; the call synchronises before it returns
    std::lock_guard<std::mutex> lock(e.sync->mu);
    if (e.sync->used) S2W_CUDA_CHECK(cudaEventSynchronize(e.sync->done));
    if (p->kind == 0) {
        // sphere: coefficient blocks pipelined over a second stream (see HostPipe)
        cudaStream_t copy_stream = e.sync->copy_stream;
        HostPipe hp;
        hp.copy = copy_stream;
        hp.host = fwd ? (char *)out_h : (char *)const_cast<void *>(in_h);
        hp.dev = (char *)e.d_cof;
        hp.pitch = p->coeff_elems * esz;
        hp.B = p->batch;
        void *work = (void *)(((uintptr_t)e.work + 255) & ~(uintptr_t)255);
        if (fwd) {
            if (cudaMemcpyAsync(d_in, in_h, sig, cudaMemcpyHostToDevice, 0) != cudaSuccess) rc = S2W_ECUDA;
            if (!rc) rc = sphere_forward(p, d_in, d_out, work, 0, &hp);
        } else {
            rc = sphere_inverse(p, d_in, d_out, work, 0, &hp);
            if (!rc && cudaMemcpyAsync(out_h, d_out, sig, cudaMemcpyDeviceToHost, 0) != cudaSuccess) rc = S2W_ECUDA;
        }
        cudaError_t e1 = cudaStreamSynchronize(0), e2 = cudaStreamSynchronize(copy_stream);
        hp.release();
        if ((e1 != cudaSuccess || e2 != cudaSuccess) && !rc) {
            set_error(std::string("stream sync: ") + cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
            rc = S2W_ECUDA;
        }
        return rc;
    }
    if (cudaMemcpyAsync(d_in, in_h, fwd ? sig : cof, cudaMemcpyHostToDevice, 0) != cudaSuccess) rc = S2W_ECUDA;
    if (!rc) rc = fwd ? s2w_plan_forward(e.plan, d_in, d_out, e.work, 0) : s2w_plan_inverse(e.plan, d_in, d_out, e.work, 0);
    if (!rc && cudaMemcpyAsync(out_h, d_out, fwd ? cof : sig, cudaMemcpyDeviceToHost, 0) != cudaSuccess) rc = S2W_ECUDA;
    if (cudaStreamSynchronize(0) != cudaSuccess && !rc) {
        set_error(std::string("stream sync: ") + cudaGetErrorString(cudaGetLastError()));
        rc = S2W_ECUDA;
    }
    return rc;
}
}  // namespace

int s2wav_forward(const void *f, void *w, int L, int N, double lambda, int J0, int multires, int flags, int batch,
                  void *stream)
{
    CacheEntry e;
    int rc = cached_plan(0, L, 1, N, lambda, 0.0, 1.0, J0, multires, flags, batch, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream, [&](cudaStream_t st) { return s2w_plan_forward(e.plan, f, w, e.work, (void *)st); });
}

int s2wav_inverse(const void *w, void *f, int L, int N, double lambda, int J0, int multires, int flags, int batch,
                  void *stream)
{
    CacheEntry e;
    int rc = cached_plan(0, L, 1, N, lambda, 0.0, 1.0, J0, multires, flags, batch, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream, [&](cudaStream_t st) { return s2w_plan_inverse(e.plan, w, f, e.work, (void *)st); });
}

int s2wav_forward_host(const void *f, void *w, int L, int N, double lambda, int J0, int multires, int flags, int batch)
{
    CacheEntry e;
    int rc = cached_plan_staged(0, L, 1, N, lambda, 0.0, 1.0, J0, multires, flags, batch, &e);
    if (rc) return rc;
    return host_transform(true, e, f, w);
}
int s2wav_inverse_host(const void *w, void *f, int L, int N, double lambda, int J0, int multires, int flags, int batch)
{
    CacheEntry e;
    int rc = cached_plan_staged(0, L, 1, N, lambda, 0.0, 1.0, J0, multires, flags, batch, &e);
    if (rc) return rc;
    return host_transform(false, e, w, f);
}

int s2ball_forward(const void *f, void *w, int L, int P, int N, double lambda_l, double lambda_p, int J0, double tau,
                   int flags, void *stream)
{
    CacheEntry e;
    int rc = cached_plan(1, L, P, N, lambda_l, lambda_p, tau, J0, 1, flags, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream, [&](cudaStream_t st) { return s2w_plan_forward(e.plan, f, w, e.work, (void *)st); });
}
int s2ball_inverse(const void *w, void *f, int L, int P, int N, double lambda_l, double lambda_p, int J0, double tau,
                   int flags, void *stream)
{
    CacheEntry e;
    int rc = cached_plan(1, L, P, N, lambda_l, lambda_p, tau, J0, 1, flags, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream, [&](cudaStream_t st) { return s2w_plan_inverse(e.plan, w, f, e.work, (void *)st); });
}

int s2ball_forward_host(const void *f, void *w, int L, int P, int N, double lambda_l, double lambda_p, int J0,
                        double tau, int flags)
{
    CacheEntry e;
    int rc = cached_plan_staged(1, L, P, N, lambda_l, lambda_p, tau, J0, 1, flags, 1, &e);
    if (rc) return rc;
    return host_transform(true, e, f, w);
}
int s2ball_inverse_host(const void *w, void *f, int L, int P, int N, double lambda_l, double lambda_p, int J0,
                        double tau, int flags)
{
    CacheEntry e;
    int rc = cached_plan_staged(1, L, P, N, lambda_l, lambda_p, tau, J0, 1, flags, 1, &e);
    if (rc) return rc;
    return host_transform(false, e, w, f);
}

// Z = K Y, Z^-1 (Eqs. 10-11): the harmonic taps of a cached ball plan
int s2ball_z_forward(const void *f, void *flmp, int L, int P, double tau, int flags, void *stream)
{
    CacheEntry e;
    int rc = cached_plan(1, L, P, 1, 2.0, 2.0, tau, 0, 1, flags, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream,
                            [&](cudaStream_t st) { return s2w_plan_harmonic_forward(e.plan, f, flmp, e.work, (void *)st); });
}
int s2ball_z_inverse(const void *flmp, void *f, int L, int P, double tau, int flags, void *stream)
{
    CacheEntry e;
    int rc = cached_plan(1, L, P, 1, 2.0, 2.0, tau, 0, 1, flags, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream,
                            [&](cudaStream_t st) { return s2w_plan_harmonic_inverse(e.plan, flmp, f, e.work, (void *)st); });
}
// Q = K D, Q^-1 (Eqs. 24-25)
int s2ball_q_forward(const void *f, void *fhat, int L, int P, int N, double tau, void *stream)
{
    if (!f || !fhat) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    CacheEntry e;
    int rc = cached_plan(2, L, P, N, 2.0, 2.0, tau, 0, 0, 0, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream,
                            [&](cudaStream_t st) { return q_forward_dev(e.plan, f, fhat, e.work, st); });
}
int s2ball_q_inverse(const void *fhat, void *f, int L, int P, int N, double tau, void *stream)
{
    if (!f || !fhat) {
        set_error("null pointer");
        return S2W_EINVAL;
    }
    CacheEntry e;
    int rc = cached_plan(2, L, P, N, 2.0, 2.0, tau, 0, 0, 0, 1, &e);
    if (rc) return rc;
    return entry_serialised(e, (cudaStream_t)stream,
                            [&](cudaStream_t st) { return q_inverse_dev(e.plan, fhat, f, e.work, st); });
}

int s2w_cache_clear(void)
{
    std::lock_guard<std::mutex> lock(g_cache_mu);
    for (auto &kv : g_cache) {
        cudaFree(kv.second.work);
        cudaFree(kv.second.d_sig);
        cudaFree(kv.second.d_cof);
        if (kv.second.sync) {
            cudaEventDestroy(kv.second.sync->done);
            cudaStreamDestroy(kv.second.sync->copy_stream);
            delete kv.second.sync;
        }
        s2w_plan_destroy(kv.second.plan);
    }
    g_cache.clear();
    return S2W_OK;
}

int s2w_timing_enable(int on)
{
    std::lock_guard<std::mutex> lock(g_timing_mu);
    g_timing = on != 0;
    return S2W_OK;
}

int s2w_timing_read(double *ms, unsigned long long *launches, int nclass)
{
    if (!ms || !launches || nclass < 1) {
        set_error("invalid argument");
        return S2W_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_timing_mu);
    for (int c = 0; c < nclass; ++c) {
        ms[c] = 0.0;
        launches[c] = 0;
    }
    int rc = S2W_OK;
    for (size_t i = 0; i < g_timed.size(); ++i) {
        float t = 0.f;
        if (cudaEventSynchronize(g_timed[i].b) != cudaSuccess ||
            cudaEventElapsedTime(&t, g_timed[i].a, g_timed[i].b) != cudaSuccess) {
            set_error(std::string("timing events: ") + cudaGetErrorString(cudaGetLastError()));
            rc = S2W_ECUDA;
        } else {
            const int c = g_timed[i].cls < nclass ? g_timed[i].cls : nclass - 1;
            ms[c] += (double)t;
            launches[c] += 1;
        }
        g_ev_free.push_back(g_timed[i]);
    }
    g_timed.clear();
    return rc;
}

int s2w_probe_fp64(int kind, int device, double *tflops)
{
    if (!tflops || kind < 0 || kind > 1) return S2W_EINVAL;
    S2W_CUDA_CHECK(cudaSetDevice(device));
    return probe_fp64(kind, tflops);
}

}  // extern "C"
