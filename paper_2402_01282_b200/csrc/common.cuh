// common.cuh -- shared declarations of the CUDA path (sm_100a, fp64).
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <string>

namespace s2w {

typedef double2 cplx;  // complex128: x = re, y = im

__host__ __device__ __forceinline__ cplx cmake(double r, double i) { return make_double2(r, i); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b)
{
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b)  // a * conj(b)
{
    return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }

void set_error(const std::string &msg);
void count_launch();
void debug_launch(const char *name);  // S2W_DEBUG_LAUNCH=1: report the first launch that leaves a CUDA error behind

#define S2W_CUDA_CHECK(expr)                                                                       \
    do {                                                                                           \
        cudaError_t _e = (expr);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            s2w::set_error(std::string(#expr) + ": " + cudaGetErrorString(_e));                    \
            return S2W_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)

// kernel classes of the per-class device timers (s2w_timing_*; bench.py's roofline and step breakdown)
enum { S2W_K_WIGNER_INV = 0, S2W_K_WIGNER_FWD = 1, S2W_K_RING_FFT = 2, S2W_K_SO3_FFT = 3, S2W_K_REWEIGHT = 4,
       S2W_K_RADIAL = 5, S2W_K_OTHER = 6, S2W_K_NCLASS = 7 };
void timing_begin(int cls, cudaStream_t st);  // no-ops unless s2w_timing_enable(1)
void timing_end(cudaStream_t st);

// launch + count (every kernel of this library goes through these macros)
#define S2W_LAUNCH_C(cls, kernel, grid, block, smem, stream, ...)                                  \
    do {                                                                                           \
        s2w::timing_begin((cls), (stream));                                                        \
        kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);                                \
        s2w::timing_end((stream));                                                                 \
        s2w::count_launch();                                                                       \
        s2w::debug_launch(#kernel);                                                                \
    } while (0)
#define S2W_LAUNCH(kernel, grid, block, smem, stream, ...)                                         \
    S2W_LAUNCH_C(s2w::S2W_K_OTHER, kernel, grid, block, smem, stream, __VA_ARGS__)

}  // namespace s2w
