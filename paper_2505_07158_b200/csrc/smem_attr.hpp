// smem_attr.hpp -- the opt-in dynamic shared-memory limit of a kernel, only ever raised.
// Internal to libvcrypt.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include <map>
#include <mutex>
#include <utility>

namespace vk {

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the FUNCTION (per device), not to a context of this library: every
// live vcrypt_ctx whose shape takes the same kernel instantiation shares it.  Setting it to "what this shape needs" in every
// vcrypt_init would let a later, smaller context (640 x 480 after 1920 x 1080) lower the limit under the larger one, whose
// next launch would then fail with cudaErrorInvalidValue.  So the limit is remembered per (device, function) and only grows.
// The launch itself still asks for exactly the bytes its plan computed: occupancy is decided there, not by this limit.
// `device` must be the current device.
inline cudaError_t raise_dyn_smem(const void *fn, int device, size_t bytes) {
    static std::mutex mu;
    static std::map<std::pair<int, const void *>, size_t> granted;
    std::lock_guard<std::mutex> lock(mu);
    size_t &have = granted[std::make_pair(device, fn)];
    if (bytes <= have) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

}  // namespace vk
