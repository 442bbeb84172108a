// smem_attr.cuh -- opt-in dynamic shared memory for kernels that need more than 48 KB.
#pragma once
#include <string>

#include "common.cuh"
#include "../../include/s2w.h"

namespace s2w {

// Kernels that may need more than 48 KB of dynamic shared memory are raised to the device's opt-in limit, never to
// the size of one launch: the attribute belongs to the function, not to the launch, so a per-launch value would be
// lowered again by the next (smaller) launch -- under a captured graph, or with two host threads, that is a race with
// the launches that still need the larger size.
template <typename K>
inline int set_smem(K kernel, size_t bytes)
{
    if (bytes == 0) return S2W_OK;
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, kernel) != cudaSuccess) {
        cudaGetLastError();
        fa.sharedSizeBytes = 0;
        fa.maxDynamicSharedSizeBytes = 0;
    }
    // the 48 KB default covers static + dynamic together
    if (fa.sharedSizeBytes + bytes <= 48 * 1024) return S2W_OK;
    int optin = 0, dev = 0;  // per call: the limit and the function attribute below are per device
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) optin = 0;
    const int room = optin - (int)fa.sharedSizeBytes;
    if (room < 0 || (size_t)room < bytes) {
        cudaGetLastError();
        set_error("shared memory per block: the kernel needs more than the device offers");
        return S2W_ECUDA;
    }
    if (fa.maxDynamicSharedSizeBytes == room) return S2W_OK;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, room);
    if (e != cudaSuccess) {
        set_error(std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
        return S2W_ECUDA;
    }
    return S2W_OK;
}

}  // namespace s2w
