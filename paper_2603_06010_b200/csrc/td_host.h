// td_host.h - host-side helpers shared by the two translation units of the library (tdlike.cu: fp64 kernels and the
// handle; tdlike_f32.cu: the same FFT-path kernels compiled with real = float).
#pragma once
#include <cuda_runtime.h>

#include "../../include/tdlike.h"

#define CK(call)                                                                               \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess) return e_ == cudaErrorMemoryAllocation ? TD_ENOMEM : TD_ECUDA;      \
  } while (0)


namespace tdhost {

// One-time launch configuration per (kernel instantiation, device): the dynamic shared-memory attribute and the
// occupancy query run on the first use only; td_create makes that first use (a "dry" pass over every kernel its size
// classes can reach), so a batch call contains nothing but launches.  `cache` is the caller's function-local static.
constexpr int TD_MAX_DEV = 64;
template <class K>
td_status kernel_config(K kern, int nt, size_t smem_attr, size_t smem, int device, int* cache, int* blocks_per_sm) {
  if (device < 0 || device >= TD_MAX_DEV) return TD_EUNSUPPORTED;
  if (cache[device] == 0) {
    if (smem_attr > 48 * 1024) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_attr));
    int nb = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, nt, smem));
    cache[device] = nb + 1;
  }
  *blocks_per_sm = cache[device] - 1;
  return TD_OK;
}

}  // namespace tdhost
