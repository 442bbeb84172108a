// fft_core.cuh -- block-cooperative power-of-two complex128 FFT in shared memory.
//
// The MW grids have 2L-1 = 2^k - 1 samples per ring (never a power of two), so every DFT on the path is done as a
// Bluestein chirp convolution of length M = 2^q >= 2n-1.  A convolution needs FFT -> pointwise multiply -> inverse
// FFT, which lets us drop all reordering passes: the forward transform is decimation-in-frequency (natural in,
// digit-reversed out), the kernel spectrum is stored in that same digit-reversed order, and the inverse transform is
// decimation-in-time (digit-reversed in, natural out).  Both run in place on one padded shared-memory buffer with
// radix-8 register butterflies; the innermost pass is fused with the pointwise multiply.
#pragma once
#include "common.cuh"

namespace s2w {

// one 16-byte pad slot after every 8 elements: stride-8 accesses of the small-stride passes become conflict-free
#define S2W_PAD(e) ((e) + ((e) >> 3))
__host__ __device__ inline int fft_padded_len(int M) { return M + (M >> 3) + 1; }

// lengths served by the radix-16 core (fft16_core.cuh)
__host__ __device__ inline bool f16_supported(int M) { return M == 4096 || M == 2048 || M == 1024 || M == 512 || M == 256; }

struct FftTab {
    int n;              // DFT length (2L-1)
    int L;              // band-limit of the grid
    int nt;             // rings of the grid: L (McEwen-Wiaux) or 2L (Driscoll-Healy); the radix-16 and ring-pair kernels
                        // assume nt == L (the launchers route Driscoll-Healy grids to the generic radix-8 kernels)
    int logM, M;        // Bluestein length
    int twmul;          // twiddle table stride: W_M^k = tw[k * twmul]
    int twmask;         // table length - 1
    int twlo;           // low bits of the two-level twiddle split (min(6, log2 table length))
    const cplx *tw;     // exp(-2 pi i k / Mtab)
    const cplx *chirp;  // [n]  exp(-i pi j^2 / n)
    const cplx *bhat_m; // [M]  digit-reversed FFT of the wrapped exp(+i pi d^2/n), times 1/M   (forward DFT, sign -)
    const cplx *bhat_p; // [M]  same for exp(-i pi d^2/n)                                       (inverse DFT, sign +)
    const cplx *what;   // [M]  digit-reversed FFT of the wrapped quadrature kernel w(q), times 1/M   (reweighting)
    const cplx *rw_in1, *rw_out1, *rw_in3, *rw_out3;  // [n] each: reweighting phase tables (ring_fft.cu)
    const cplx *bhat16_m, *bhat16_p;  // [M] the same spectra in the order of fft16_core.cuh (M = 1024, 2048, 4096), else null
};

// Tables of the Toeplitz/Hankel form of the theta reweighting (ring_fft.cu, reweight_th_kernel): length-M2 power-of-two
// transforms, M2 >= 2(L-1) - 1.
struct RwTab {
    int L;                 // band-limit of the grid; 0: not available (tiny grids use the Bluestein kernel)
    FftTab fft;            // M = M2, twiddles only
    int npairs;            // M2/2 + 1 pairs of positions (p, p') holding frequencies (k, -k) in the transform's order
    const int2 *pairs;     // [npairs]
    const cplx *TG;        // [npairs][4]: That(p), Ghat(p), That(p'), Ghat(p') -- spectra of T(d) = 1/sin(pi d/n) and of
                           // H(d + L - 1) times the reversal phase, both times 1/(n M2)
    const double *delta;   // [L] c_t - c_{n-1-t}
    const double *dsum;    // [L] (K_tt + K_{n-1-t,n-1-t}) / n
    const double *vpole;   // [2][L] pole column per parity (sigma = +1, -1), / n
    const double *rpole;   // [2][L] pole row per parity, / n
    const cplx *TG16;      // [2][M2]: That, Ghat in the storage order of fft16_core.cuh's tables (M2 = 1024, 2048), else null
};

template <bool INV>
__device__ __forceinline__ cplx mul_mi(cplx a)  // times -i (forward) or +i (inverse)
{
    return INV ? cmake(-a.y, a.x) : cmake(a.y, -a.x);
}

template <bool INV>
__device__ __forceinline__ void bfly4(cplx &x0, cplx &x1, cplx &x2, cplx &x3)
{
    cplx t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_mi<INV>(csub(x1, x3));
    x0 = cadd(t0, t2);
    x1 = cadd(t1, t3);
    x2 = csub(t0, t2);
    x3 = csub(t1, t3);
}

template <int R, bool INV>
struct Bfly;

template <bool INV>
struct Bfly<2, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[2])
    {
        cplx a = v[0];
        v[0] = cadd(a, v[1]);
        v[1] = csub(a, v[1]);
    }
};
template <bool INV>
struct Bfly<4, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[4]) { bfly4<INV>(v[0], v[1], v[2], v[3]); }
};
template <bool INV>
struct Bfly<8, INV> {
    static __device__ __forceinline__ void run(cplx (&v)[8])
    {
        const double h = 0.70710678118654752440;
        cplx a0 = v[0], a1 = v[2], a2 = v[4], a3 = v[6];
        cplx b0 = v[1], b1 = v[3], b2 = v[5], b3 = v[7];
        bfly4<INV>(a0, a1, a2, a3);
        bfly4<INV>(b0, b1, b2, b3);
        // w^k b_k with w = exp(-+ i pi/4)
        cplx c1, c3;
        if (INV) {
            c1 = cmake((b1.x - b1.y) * h, (b1.x + b1.y) * h);
            c3 = cmake((-b3.x - b3.y) * h, (b3.x - b3.y) * h);
        } else {
            c1 = cmake((b1.x + b1.y) * h, (b1.y - b1.x) * h);
            c3 = cmake((b3.y - b3.x) * h, (-b3.x - b3.y) * h);
        }
        cplx c2 = mul_mi<INV>(b2);
        v[0] = cadd(a0, b0);
        v[4] = csub(a0, b0);
        v[1] = cadd(a1, c1);
        v[5] = csub(a1, c1);
        v[2] = cadd(a2, c2);
        v[6] = csub(a2, c2);
        v[3] = cadd(a3, c3);
        v[7] = csub(a3, c3);
    }
};

// Twiddles W^j, j = 1..R-1, from one table entry W = W_S^i: powers by repeated complex multiplication (at most three
// multiplications deep, error <= ~4 ulp).  One 16-byte table load per butterfly instead of R-1 scattered ones: the
// table does not fit beside three blocks' shared memory in L1, and scattered 16-byte loads cost a wavefront each.
template <int R>
__device__ __forceinline__ void twiddle_powers(cplx w1, cplx (&w)[R])
{
    w[1 % R] = w1;
    if (R >= 4) {
        w[2] = cmul(w1, w1);
        w[3] = cmul(w[2], w1);
    }
    if (R >= 8) {
        w[4] = cmul(w[2], w[2]);
        w[5] = cmul(w[4], w1);
        w[6] = cmul(w[3], w[3]);
        w[7] = cmul(w[4], w[3]);
    }
}

// Two-level twiddle table in shared memory: W^k = W^{(k >> twlo) << twlo} W^{k & (2^twlo - 1)}, at most 128 + 64 entries
// (3 KB) copied from the global table at kernel start, so no pass waits on a global load.
#define S2W_TW_SMEM 192
__device__ __forceinline__ void tw_stage(cplx *stw, const FftTab &T)
{
    const int nh = (T.twmask + 1) >> T.twlo, nl = 1 << T.twlo;
    for (int i = threadIdx.x; i < nh; i += blockDim.x) stw[i] = T.tw[i << T.twlo];
    for (int i = threadIdx.x; i < nl; i += blockDim.x) stw[nh + i] = T.tw[i];
}
__device__ __forceinline__ cplx tw_lookup(const cplx *stw, const FftTab &T, int k)
{
    const int nh = (T.twmask + 1) >> T.twlo;
    return cmul(stw[k >> T.twlo], stw[nh + (k & ((1 << T.twlo) - 1))]);
}

// The same split on the transform's own length M (W_M^k = W^{hi << tl} W^{lo}, tl = ceil(logM / 2)) instead of the
// plan-wide table's: 2 sqrt(M) entries (2 KB at M = 4096), which is what lets a third block of the one-sequence-per-
// block kernels fit on an SM.  T is the caller's local copy and is rewritten to index the staged table.
__host__ __device__ inline int tw_own_entries(int logM)
{
    const int tl = (logM + 1) >> 1;
    return (1 << (logM - tl)) + (1 << tl);
}
__device__ __forceinline__ void tw_stage_own(cplx *stw, FftTab &T)
{
    const int tl = (T.logM + 1) >> 1, nh = T.M >> tl, nl = 1 << tl;
    for (int i = threadIdx.x; i < nh; i += blockDim.x) stw[i] = T.tw[(i << tl) * T.twmul];
    for (int i = threadIdx.x; i < nl; i += blockDim.x) stw[nh + i] = T.tw[i * T.twmul];
    T.twmul = 1;
    T.twmask = T.M - 1;
    T.twlo = tl;
}

// One decimation-in-frequency pass on sub-transforms of size S (radix R): butterflies, then twiddles W_S^{i j}.
// HALF (outermost radix-8 pass only, S = M): the upper half of the buffer is taken as zero without being read.
template <int R, bool HALF = false>
__device__ __forceinline__ void dif_pass(cplx *buf, int M, int logS, const FftTab &T, const cplx *stw)
{
    const int logs = logS - (R == 8 ? 3 : (R == 4 ? 2 : 1));
    const int s = 1 << logs;
    const int twm = T.twmul << (T.logM - logS);  // W_S^k = W_M^{k M/S}
    for (int idx = threadIdx.x; idx < (M / R); idx += blockDim.x) {
        int i = idx & (s - 1);
        int base = ((idx >> logs) << logS) + i;
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = (HALF && 2 * k >= R) ? cmake(0.0, 0.0) : buf[S2W_PAD(base + (k << logs))];
        Bfly<R, false>::run(v);
        cplx w[R];
        twiddle_powers<R>(tw_lookup(stw, T, (i * twm) & T.twmask), w);
#pragma unroll
        for (int j = 1; j < R; ++j) v[j] = cmul(v[j], w[j]);
#pragma unroll
        for (int k = 0; k < R; ++k) buf[S2W_PAD(base + (k << logs))] = v[k];
    }
}

// The matching decimation-in-time inverse pass: conjugate twiddles, then inverse butterflies.
// HALF (outermost radix-8 pass only, S = M): the upper half of the result is neither formed nor stored.
template <int R, bool HALF = false>
__device__ __forceinline__ void dit_pass(cplx *buf, int M, int logS, const FftTab &T, const cplx *stw)
{
    const int logs = logS - (R == 8 ? 3 : (R == 4 ? 2 : 1));
    const int s = 1 << logs;
    const int twm = T.twmul << (T.logM - logS);
    for (int idx = threadIdx.x; idx < (M / R); idx += blockDim.x) {
        int i = idx & (s - 1);
        int base = ((idx >> logs) << logS) + i;
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = buf[S2W_PAD(base + (k << logs))];
        cplx w[R];
        twiddle_powers<R>(tw_lookup(stw, T, (i * twm) & T.twmask), w);
#pragma unroll
        for (int j = 1; j < R; ++j) v[j] = cmulc(v[j], w[j]);
        Bfly<R, true>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k)
            if (!(HALF && 2 * k >= R)) buf[S2W_PAD(base + (k << logs))] = v[k];
    }
}

// Innermost pass of both transforms fused with the pointwise product: groups of R consecutive elements.
template <int R>
__device__ __forceinline__ void mid_pass(cplx *buf, int M, const cplx *__restrict__ khat)
{
    for (int g = threadIdx.x; g < (M / R); g += blockDim.x) {
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = buf[S2W_PAD(g * R + k)];
        Bfly<R, false>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = cmul(v[k], __ldg(&khat[g * R + k]));
        Bfly<R, true>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) buf[S2W_PAD(g * R + k)] = v[k];
    }
}

// Batched variants: nb transforms of length M stored bstride elements apart in one shared-memory buffer; one pass
// works on all of them between two barriers.
template <int R, bool HALF = false>
__device__ __forceinline__ void dif_pass_b(cplx *buf, int M, int logS, const FftTab &T, const cplx *stw, int nb, int bstride)
{
    const int logs = logS - (R == 8 ? 3 : (R == 4 ? 2 : 1));
    const int s = 1 << logs;
    const int twm = T.twmul << (T.logM - logS);
    const int lper = T.logM - (R == 8 ? 3 : (R == 4 ? 2 : 1)), per = 1 << lper;  // M is a power of two
    for (int it = threadIdx.x; it < nb * per; it += blockDim.x) {
        const int bi = it >> lper, idx = it & (per - 1);
        cplx *b = buf + bi * bstride;
        int i = idx & (s - 1);
        int base = ((idx >> logs) << logS) + i;
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = (HALF && 2 * k >= R) ? cmake(0.0, 0.0) : b[S2W_PAD(base + (k << logs))];
        Bfly<R, false>::run(v);
        cplx w[R];
        twiddle_powers<R>(tw_lookup(stw, T, (i * twm) & T.twmask), w);
#pragma unroll
        for (int j = 1; j < R; ++j) v[j] = cmul(v[j], w[j]);
#pragma unroll
        for (int k = 0; k < R; ++k) b[S2W_PAD(base + (k << logs))] = v[k];
    }
}

template <int R, bool HALF = false>
__device__ __forceinline__ void dit_pass_b(cplx *buf, int M, int logS, const FftTab &T, const cplx *stw, int nb, int bstride)
{
    const int logs = logS - (R == 8 ? 3 : (R == 4 ? 2 : 1));
    const int s = 1 << logs;
    const int twm = T.twmul << (T.logM - logS);
    const int lper = T.logM - (R == 8 ? 3 : (R == 4 ? 2 : 1)), per = 1 << lper;  // M is a power of two
    for (int it = threadIdx.x; it < nb * per; it += blockDim.x) {
        const int bi = it >> lper, idx = it & (per - 1);
        cplx *b = buf + bi * bstride;
        int i = idx & (s - 1);
        int base = ((idx >> logs) << logS) + i;
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = b[S2W_PAD(base + (k << logs))];
        cplx w[R];
        twiddle_powers<R>(tw_lookup(stw, T, (i * twm) & T.twmask), w);
#pragma unroll
        for (int j = 1; j < R; ++j) v[j] = cmulc(v[j], w[j]);
        Bfly<R, true>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k)
            if (!(HALF && 2 * k >= R)) b[S2W_PAD(base + (k << logs))] = v[k];
    }
}

// nb forward transforms, natural in, digit-reversed out (radix 8 ... 8, then 4 or 2).  Ends with a barrier.
__device__ inline void fft_dif_full_b(cplx *buf, const FftTab &T, const cplx *stw, int nb, int bstride)
{
    const int M = T.M;
    int logS = T.logM;
    while (logS >= 3) {
        dif_pass_b<8>(buf, M, logS, T, stw, nb, bstride);
        __syncthreads();
        logS -= 3;
    }
    if (logS == 2) {
        dif_pass_b<4>(buf, M, 2, T, stw, nb, bstride);
        __syncthreads();
    } else if (logS == 1) {
        dif_pass_b<2>(buf, M, 1, T, stw, nb, bstride);
        __syncthreads();
    }
}

// the matching inverse: digit-reversed in, natural out, unscaled.  Ends with a barrier.
__device__ inline void fft_dit_full_b(cplx *buf, const FftTab &T, const cplx *stw, int nb, int bstride)
{
    const int M = T.M;
    int logS = T.logM % 3;
    if (logS == 2) {
        dit_pass_b<4>(buf, M, 2, T, stw, nb, bstride);
        __syncthreads();
    } else if (logS == 1) {
        dit_pass_b<2>(buf, M, 1, T, stw, nb, bstride);
        __syncthreads();
    }
    logS += 3;
    while (logS <= T.logM) {
        dit_pass_b<8>(buf, M, logS, T, stw, nb, bstride);
        __syncthreads();
        logS += 3;
    }
}

template <int R>
__device__ __forceinline__ void mid_pass_b(cplx *buf, int M, const cplx *__restrict__ khat, int nb, int bstride)
{
    const int lper = __ffs(M) - 1 - (R == 8 ? 3 : (R == 4 ? 2 : 1)), per = 1 << lper;  // M is a power of two
    for (int it = threadIdx.x; it < nb * per; it += blockDim.x) {
        const int bi = it >> lper, g = it & (per - 1);
        cplx *b = buf + bi * bstride;
        cplx v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = b[S2W_PAD(g * R + k)];
        Bfly<R, false>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = cmul(v[k], __ldg(&khat[g * R + k]));
        Bfly<R, true>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) b[S2W_PAD(g * R + k)] = v[k];
    }
}

// nb circular convolutions (sequences bstride apart) with the same kernel spectrum; see fft_convolve.
template <bool HALF = false>
__device__ inline void fft_convolve_b(cplx *buf, const FftTab &T, const cplx *stw, const cplx *__restrict__ khat,
                                      int nb, int bstride)
{
    const int M = T.M;
    const int r = T.logM % 3;
    const int logMid = (r == 0) ? 3 : r;
    int logS = T.logM;
    if (HALF && logS > logMid) {
        dif_pass_b<8, true>(buf, M, logS, T, stw, nb, bstride);
        __syncthreads();
        logS -= 3;
    }
    while (logS > logMid) {
        dif_pass_b<8>(buf, M, logS, T, stw, nb, bstride);
        __syncthreads();
        logS -= 3;
    }
    if (logMid == 3)
        mid_pass_b<8>(buf, M, khat, nb, bstride);
    else if (logMid == 2)
        mid_pass_b<4>(buf, M, khat, nb, bstride);
    else
        mid_pass_b<2>(buf, M, khat, nb, bstride);
    __syncthreads();
    logS = logMid + 3;
    while (logS <= T.logM) {
        if (HALF && logS == T.logM)
            dit_pass_b<8, true>(buf, M, logS, T, stw, nb, bstride);
        else
            dit_pass_b<8>(buf, M, logS, T, stw, nb, bstride);
        __syncthreads();
        logS += 3;
    }
}

// Forward transform only (used once per table at plan creation): natural in, digit-reversed out.
__device__ inline void fft_dif_full(cplx *buf, const FftTab &T, const cplx *stw)
{
    const int M = T.M;
    int logS = T.logM;
    while (logS >= 3) {
        dif_pass<8>(buf, M, logS, T, stw);
        __syncthreads();
        logS -= 3;
    }
    if (logS == 2) {
        dif_pass<4>(buf, M, 2, T, stw);
        __syncthreads();
    } else if (logS == 1) {
        dif_pass<2>(buf, M, 1, T, stw);
        __syncthreads();
    }
}

// buf <- circular convolution (length M) of buf with the kernel whose digit-reversed, 1/M-scaled spectrum is khat.
// Ends with a __syncthreads().  Requires a __syncthreads() after the caller's writes to buf.
// HALF: the sequence occupies the lower half of the buffer only (Bluestein: n <= M/2 inputs, n outputs wanted): the
// upper half is taken as zero whatever it holds, and holds garbage afterwards -- the outermost pass of each transform
// moves half the data.
template <bool HALF = false>
__device__ inline void fft_convolve(cplx *buf, const FftTab &T, const cplx *stw, const cplx *__restrict__ khat)
{
    const int M = T.M;
    const int r = T.logM % 3;
    const int logMid = (r == 0) ? 3 : r;  // innermost group: 8, 2 or 4 elements
    int logS = T.logM;
    if (HALF && logS > logMid) {
        dif_pass<8, true>(buf, M, logS, T, stw);
        __syncthreads();
        logS -= 3;
    }
    while (logS > logMid) {
        dif_pass<8>(buf, M, logS, T, stw);
        __syncthreads();
        logS -= 3;
    }
    if (logMid == 3)
        mid_pass<8>(buf, M, khat);
    else if (logMid == 2)
        mid_pass<4>(buf, M, khat);
    else
        mid_pass<2>(buf, M, khat);
    __syncthreads();
    logS = logMid + 3;
    while (logS <= T.logM) {
        if (HALF && logS == T.logM)
            dit_pass<8, true>(buf, M, logS, T, stw);
        else
            dit_pass<8>(buf, M, logS, T, stw);
        __syncthreads();
        logS += 3;
    }
}

}  // namespace s2w
