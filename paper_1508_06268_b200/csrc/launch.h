// launch.h -- cooperative launch helper (the flow kernel's CTAs wait on one another, so they must
// all be co-resident: cudaLaunchCooperativeKernel guarantees that or fails).
#pragma once
#include <cuda_runtime.h>

namespace rfim {

template <class... KArgs, class... Args>
inline cudaError_t launch_cooperative(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args) {
    void* argv[] = {const_cast<void*>(static_cast<const void*>(&args))...};
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(kernel), grid, block, argv, 0, stream);
}

template <class K>
inline int max_coresident_blocks(K kernel, int threads) {
    int dev = 0, sms = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, 0) != cudaSuccess) return 0;
    return occ * sms;
}

}  // namespace rfim
