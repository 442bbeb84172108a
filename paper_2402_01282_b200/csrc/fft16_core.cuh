// fft16_core.cuh -- the second-generation block FFT of the path (rows a1, a2, a8): circular convolutions of length
// M = R1 * 256 (R1 = 16, 8, 4, 2, 1: M = 4096 ... 256) on a 4096-element shared-memory buffer holding NB = 16 / R1
// sequences, by 256 threads.
//
// Why a second core (profiles/r01k_notes.md): the radix-8 core of fft_core.cuh moves every sequence through shared
// memory 8 times per convolution (fill, 3 + 1 + 3 passes, read-out) with a block-wide barrier after each, and ncu
// showed the shared-memory pipe (l1tex 80 %) and the barriers, not the FP64 pipe (35 %), as its limit.  Here:
//   * pass 1 (radix R1 over stride 256) takes its inputs from REGISTERS -- the caller loads element tid + 256 k of the
//     sequence straight from global memory, coalesced -- and the last inverse pass hands its outputs back in registers:
//     no fill, no read-out, no zero padding (the upper half of a Bluestein buffer is never formed);
//   * what remains after pass 1 are 16 independent 256-point problems, one per HALF-WARP: radix-16 pass (stride 16),
//     radix-16 pass on 16 contiguous elements fused with the pointwise product and its own inverse, radix-16 inverse
//     pass -- ordered by __syncwarp() only.  A convolution has TWO block-wide barriers instead of nine and 4 instead of
//     8 shared-memory round trips; between the barriers the warps drift apart, so one warp's loads overlap another's
//     FP64 work;
//   * twiddles are powers of one per-thread constant per pass (W_M^tid, W_256^(tid & 15)), kept in registers for the
//     kernel's lifetime: no twiddle table in shared memory at all.
// Element e of the buffer lives at F16_PAD(e) = e + (e >> 4): the three access patterns (consecutive threads ->
// consecutive elements; stride 16; 16 contiguous elements per thread) are all bank-conflict free with it.
//
// Order of the spectrum: position p = j1 * 256 + j2 * 16 + j3 of a sequence holds frequency j1 + R1 (j2 + 16 j3).  Kernel
// spectra are produced in that order by f16_forward_full (plan time), so no reordering pass exists anywhere.
#pragma once
#include "common.cuh"
#include "fft_core.cuh"

namespace s2w {

#define F16_PAD(e) ((e) + ((e) >> 4))
#define F16_ELEMS 4096
#define F16_BUF (F16_ELEMS + (F16_ELEMS >> 4))  // padded elements per block: 69 632 bytes
// where the table entry of position p = j1 256 + j2 16 + j3 is stored: j1 256 + j3 16 + j2
#define F16_TPOS(p) (((p) & ~255) | (((p) & 15) << 4) | (((p) >> 4) & 15))

// a * (c - i s) (forward) or a * (c + i s) (inverse)
template <bool INV>
__device__ __forceinline__ cplx mul_cs(cplx a, double c, double s)
{
    return INV ? cmake(fma(a.x, c, -a.y * s), fma(a.y, c, a.x * s)) : cmake(fma(a.x, c, a.y * s), fma(a.y, c, -a.x * s));
}

// 4-point DFT of (x0, x1, 0, 0)
template <bool INV>
__device__ __forceinline__ void bfly4_half_in(cplx &x0, cplx &x1, cplx &x2, cplx &x3)
{
    const cplx a = x0, b = x1, ib = mul_mi<INV>(b);
    x0 = cadd(a, b);
    x1 = cadd(a, ib);
    x2 = csub(a, b);
    x3 = csub(a, ib);
}

// outputs 0 and 1 only of a 4-point DFT
template <bool INV>
__device__ __forceinline__ void bfly4_half_out(cplx &x0, cplx &x1, cplx x2, cplx x3)
{
    const cplx t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_mi<INV>(csub(x1, x3));
    x0 = cadd(t0, t2);
    x1 = cadd(t1, t3);
}

#define F16_C1 0.92387953251128675613  // cos(pi/8)
#define F16_S1 0.38268343236508977173  // sin(pi/8)
#define F16_H 0.70710678118654752440

// 16-point DFT, natural order in and out: V[j] = sum_k v[k] W16^{jk}, k = k1 + 4 k2, j = 4 j1 + j2.
// HIN: v[8..15] are taken as zero (not read).  HOUT: only V[0..7] are formed.
template <bool INV, bool HIN = false, bool HOUT = false>
__device__ __forceinline__ void bfly16(cplx (&v)[16])
{
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        if (HIN)
            bfly4_half_in<INV>(v[k1], v[k1 + 4], v[k1 + 8], v[k1 + 12]);
        else
            bfly4<INV>(v[k1], v[k1 + 4], v[k1 + 8], v[k1 + 12]);
    }
    // t[k1][j2] sits at v[k1 + 4 j2]; twiddles W16^{k1 j2}
    v[5] = mul_cs<INV>(v[5], F16_C1, F16_S1);
    v[9] = mul_cs<INV>(v[9], F16_H, F16_H);
    v[13] = mul_cs<INV>(v[13], F16_S1, F16_C1);
    v[6] = mul_cs<INV>(v[6], F16_H, F16_H);
    v[10] = mul_mi<INV>(v[10]);
    v[14] = mul_cs<INV>(v[14], -F16_H, F16_H);
    v[7] = mul_cs<INV>(v[7], F16_S1, F16_C1);
    v[11] = mul_cs<INV>(v[11], -F16_H, F16_H);
    v[15] = mul_cs<INV>(v[15], -F16_C1, -F16_S1);
#pragma unroll
    for (int j2 = 0; j2 < 4; ++j2) {
        if (HOUT)
            bfly4_half_out<INV>(v[4 * j2], v[4 * j2 + 1], v[4 * j2 + 2], v[4 * j2 + 3]);
        else
            bfly4<INV>(v[4 * j2], v[4 * j2 + 1], v[4 * j2 + 2], v[4 * j2 + 3]);
    }
    // v[4 j2 + j1] = V[4 j1 + j2]: transpose (register renaming)
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = a + 1; b < 4; ++b) {
            const cplx t = v[4 * a + b];
            v[4 * a + b] = v[4 * b + a];
            v[4 * b + a] = t;
        }
}

// 8-point DFT, natural order; HIN: v[4..7] zero; HOUT: V[0..3] only
template <bool INV, bool HIN = false, bool HOUT = false>
__device__ __forceinline__ void bfly8(cplx (&v)[8])
{
    cplx a0 = v[0], a1 = v[2], a2 = v[4], a3 = v[6];
    cplx b0 = v[1], b1 = v[3], b2 = v[5], b3 = v[7];
    if (HIN) {
        a1 = v[2];
        bfly4_half_in<INV>(a0, a1, a2, a3);
        bfly4_half_in<INV>(b0, b1, b2, b3);
    } else {
        bfly4<INV>(a0, a1, a2, a3);
        bfly4<INV>(b0, b1, b2, b3);
    }
    const cplx c1 = mul_cs<INV>(b1, F16_H, F16_H), c2 = mul_mi<INV>(b2), c3 = mul_cs<INV>(b3, -F16_H, F16_H);
    v[0] = cadd(a0, b0);
    v[1] = cadd(a1, c1);
    v[2] = cadd(a2, c2);
    v[3] = cadd(a3, c3);
    if (!HOUT) {
        v[4] = csub(a0, b0);
        v[5] = csub(a1, c1);
        v[6] = csub(a2, c2);
        v[7] = csub(a3, c3);
    }
}

// 4-point DFT on an array; HIN: v[2..3] zero; HOUT: V[0..1] only
template <bool INV, bool HIN = false, bool HOUT = false>
__device__ __forceinline__ void bfly4a(cplx (&v)[4])
{
    if (HIN)
        bfly4_half_in<INV>(v[0], v[1], v[2], v[3]);
    else if (HOUT)
        bfly4_half_out<INV>(v[0], v[1], v[2], v[3]);
    else
        bfly4<INV>(v[0], v[1], v[2], v[3]);
}

template <int R, bool INV, bool HIN, bool HOUT>
__device__ __forceinline__ void bfly_r(cplx (&v)[R])
{
    if constexpr (R == 16)
        bfly16<INV, HIN, HOUT>(v);
    else if constexpr (R == 8)
        bfly8<INV, HIN, HOUT>(v);
    else if constexpr (R == 4)
        bfly4a<INV, HIN, HOUT>(v);
    else if constexpr (R == 2) {  // HIN: v[1] = 0; HOUT: only v[0] is formed
        const cplx a = v[0], b = HIN ? cmake(0.0, 0.0) : v[1];
        v[0] = HIN ? a : cadd(a, b);
        if (!HOUT) v[1] = HIN ? a : csub(a, b);
    }
    // R == 1: nothing to do
}

__device__ __forceinline__ cplx csqr(cplx a) { return cmake(fma(a.x, a.x, -a.y * a.y), 2.0 * a.x * a.y); }

// v[j] *= w^j (CONJ: conj(w)^j), j = 1..R-1, powers at most four multiplications deep
template <int R, bool CONJ>
__device__ __forceinline__ void twiddle_apply(cplx (&v)[R], cplx w1)
{
    if constexpr (R == 1) return;
    if constexpr (R == 2) {
        v[1] = CONJ ? cmulc(v[1], w1) : cmul(v[1], w1);
        return;
    }
    // opaque to the optimiser: otherwise the powers are hoisted out of the caller's loop over convolutions (loop-invariant)
    // or shared between a forward and an inverse pass, i.e. 15-30 complex values kept live -- in local memory (ptxas
    // spilled 0.85 KB per thread, one LDL.128 per twiddle: as much LSU traffic as half the transform's own)
    asm volatile("" : "+d"(w1.x), "+d"(w1.y));
    if (CONJ) w1 = cconj(w1);
    const cplx w2 = csqr(w1);
    v[1 % R] = cmul(v[1 % R], w1);
    v[2 % R] = cmul(v[2 % R], w2);
    const cplx w3 = cmul(w2, w1);
    v[3 % R] = cmul(v[3 % R], w3);
    if constexpr (R >= 8) {
        const cplx w4 = csqr(w2);
        v[4] = cmul(v[4], w4);
        v[5] = cmul(v[5], cmul(w4, w1));
        v[6] = cmul(v[6], csqr(w3));
        const cplx w7 = cmul(w4, w3);
        v[7] = cmul(v[7], w7);
        if constexpr (R >= 16) {
            const cplx w8 = csqr(w4);
            v[8] = cmul(v[8], w8);
            v[9] = cmul(v[9], cmul(w8, w1));
            v[10] = cmul(v[10], cmul(w8, w2));
            v[11] = cmul(v[11], cmul(w8, w3));
            v[12] = cmul(v[12], cmul(w8, w4));
            v[13] = cmul(v[13], cmul(w8, cmul(w4, w1)));
            v[14] = cmul(v[14], csqr(w7));
            v[15] = cmul(v[15], cmul(w8, w7));
        }
    }
}

// per-thread twiddle bases, computed once per kernel: W_M^tid (pass 1) and W_256^(tid & 15) (pass 2)
struct F16Tw {
    cplx w1, w2;
};
template <int R1>
__device__ __forceinline__ F16Tw f16_twiddles()
{
    F16Tw t;
    double s, c;
    sincospi(-2.0 * (double)threadIdx.x / (double)(R1 * 256), &s, &c);
    t.w1 = cmake(c, s);
    sincospi(-2.0 * (double)(threadIdx.x & 15) / 256.0, &s, &c);
    t.w2 = cmake(c, s);
    return t;
}

// ---- pass 1 (block-wide exchange): radix R1 over stride 256, thread tid <-> column tid of each sequence ---------------

// forward, inputs from registers: x[k] = element tid + 256 k of sequence q (HIN: k < R1/2, the rest zero)
template <int R1, bool HIN>
__device__ __forceinline__ void f16_pass1_fwd(cplx *buf, int q, cplx (&x)[R1], const F16Tw &tw)
{
    bfly_r<R1, false, HIN, false>(x);
    twiddle_apply<R1, false>(x, tw.w1);
    cplx *b = buf + F16_PAD(q * (R1 * 256) + threadIdx.x);
#pragma unroll
    for (int j = 0; j < R1; ++j) b[j * (256 + 16)] = x[j];   // F16_PAD(e + 256 j) = F16_PAD(e) + 272 j
}

// inverse, outputs to registers: y[k] = element tid + 256 k (HOUT: only k < R1/2 are formed)
template <int R1, bool HOUT>
__device__ __forceinline__ void f16_pass1_inv(const cplx *buf, int q, cplx (&y)[R1], const F16Tw &tw)
{
    const cplx *b = buf + F16_PAD(q * (R1 * 256) + threadIdx.x);
#pragma unroll
    for (int j = 0; j < R1; ++j) y[j] = b[j * (256 + 16)];
    twiddle_apply<R1, true>(y, tw.w1);
    bfly_r<R1, true, false, HOUT>(y);
}

// ---- the half-warp's 256-point problem (sub-block hw = tid >> 4 of the buffer) ---------------------------------------

__device__ __forceinline__ void f16_pass2_fwd(cplx *buf, const F16Tw &tw)
{
    cplx *b = buf + F16_PAD((threadIdx.x >> 4) * 256 + (threadIdx.x & 15));   // element sb*256 + l + 16 k -> + 17 k
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = b[17 * k];
    bfly16<false>(v);
    twiddle_apply<16, false>(v, tw.w2);
#pragma unroll
    for (int k = 0; k < 16; ++k) b[17 * k] = v[k];
}

__device__ __forceinline__ void f16_pass2_inv(cplx *buf, const F16Tw &tw)
{
    cplx *b = buf + F16_PAD((threadIdx.x >> 4) * 256 + (threadIdx.x & 15));
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = b[17 * k];
    twiddle_apply<16, true>(v, tw.w2);
    bfly16<true>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) b[17 * k] = v[k];
}

// innermost pass of both transforms around the pointwise product: 16 contiguous elements per thread.
// khat: the kernel's spectrum (1/M folded in) in the transform's own order, indexed by the position inside a sequence
template <int R1>
__device__ __forceinline__ void f16_mid(cplx *buf, const cplx *__restrict__ khat)
{
    const int e0 = (threadIdx.x >> 4) * 256 + (threadIdx.x & 15) * 16;
    cplx *b = buf + F16_PAD(e0);                                            // 16 contiguous slots
    // the table is stored with the two low hex digits of the position swapped (F16_TPOS): the 16 lanes of a half-warp
    // read 256 contiguous bytes per k instead of 16 different cache lines
    const cplx *kh = khat + (((threadIdx.x >> 4) * 256) & (R1 * 256 - 1)) + (threadIdx.x & 15);
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = b[k];
    bfly16<false>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = cmul(v[k], __ldg(&kh[16 * k]));
    bfly16<true>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) b[k] = v[k];
}

// forward only / inverse only innermost passes (reweighting: the spectra of u(k) and u(-k) meet between them)
__device__ __forceinline__ void f16_pass3_fwd(cplx *buf)
{
    cplx *b = buf + F16_PAD((threadIdx.x >> 4) * 256 + (threadIdx.x & 15) * 16);
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = b[k];
    bfly16<false>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) b[k] = v[k];
}

// everything between the two block-wide barriers of a convolution
template <int R1>
__device__ __forceinline__ void f16_middle(cplx *buf, const cplx *__restrict__ khat, const F16Tw &tw)
{
    f16_pass2_fwd(buf, tw);
    __syncwarp();
    f16_mid<R1>(buf, khat);
    __syncwarp();
    f16_pass2_inv(buf, tw);
}

// One round of NB = 16 / R1 Bluestein-style convolutions: x[q][k] = element tid + 256 k (k < R1/2) of sequence q in,
// the same elements of the convolution out (unscaled by anything but khat's 1/M).  Thread-private columns: no barrier is
// needed between consecutive rounds.
template <int R1>
__device__ __forceinline__ void f16_convolve_half(cplx *buf, cplx (&x)[16 / R1][R1], const cplx *__restrict__ khat,
                                                  const F16Tw &tw)
{
#pragma unroll
    for (int q = 0; q < 16 / R1; ++q) f16_pass1_fwd<R1, (R1 > 1)>(buf, q, x[q], tw);
    __syncthreads();
    f16_middle<R1>(buf, khat, tw);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 16 / R1; ++q) f16_pass1_inv<R1, (R1 > 1)>(buf, q, x[q], tw);
}

// plan time: full forward transform of one length-M sequence (natural order in, the core's own order out; TPOSE: in the
// storage order F16_TPOS of the tables)
template <int R1, bool TPOSE>
__device__ __forceinline__ void f16_forward_full(cplx *buf, const cplx *in, cplx *out, const F16Tw &tw)
{
    cplx x[R1];
#pragma unroll
    for (int k = 0; k < R1; ++k) x[k] = in[threadIdx.x + 256 * k];
    f16_pass1_fwd<R1, false>(buf, 0, x, tw);
    __syncthreads();
    if ((int)(threadIdx.x >> 5) < (R1 + 1) / 2) {  // whole warps (a lone half-warp cannot __syncwarp)
        f16_pass2_fwd(buf, tw);
        __syncwarp();
        f16_pass3_fwd(buf);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < R1 * 256; e += blockDim.x) out[TPOSE ? F16_TPOS(e) : e] = buf[F16_PAD(e)];
}

}  // namespace s2w
