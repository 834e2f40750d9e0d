// srhd_common.cuh -- host-side argument checks and small device reductions shared by the kernels.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>

#include "../../include/srhd.h"
#include "srhd_math.cuh"

namespace srhd {

// SMs of the current device (B200: 2 dies x 74 = 148); grid-stride kernels size their grids in multiples of it
inline int num_sms() {
  static int n = 0;
  if (n <= 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
      n = 148;
  }
  return n;
}

inline int check_params(const srhd_params* p) {
  if (!p) return SRHD_ERR_NULL_POINTER;
  if (p->recon != SRHD_RECON_PLM && p->recon != SRHD_RECON_PPM) return SRHD_ERR_BAD_PARAMS;
  if (p->riemann != SRHD_RIEMANN_HLLE && p->riemann != SRHD_RIEMANN_HLLC) return SRHD_ERR_BAD_PARAMS;
  if (p->integrator != SRHD_INTEGRATOR_MHM && p->integrator != SRHD_INTEGRATOR_VL) return SRHD_ERR_BAD_PARAMS;
  if (p->ghost != (p->recon == SRHD_RECON_PLM ? 2 : 3) + p->integrator) return SRHD_ERR_BAD_PARAMS;
  if (!(p->minmod_coeff >= 0.0) || !(p->minmod_coeff <= 2.0)) return SRHD_ERR_BAD_PARAMS;
  if (p->max_retry < 0 || p->max_retry > 64) return SRHD_ERR_BAD_PARAMS;
  if (!(p->newton_rtol >= 0.0) || p->newton_max_iter < 1) return SRHD_ERR_BAD_PARAMS;
  return SRHD_OK;
}

// A positive double and its bit pattern order the same way, so max over doubles >= 0 is an integer
// atomicMax (exact, order independent).
SRHD_DEV void atomic_max_nonneg(double* addr, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(addr),
            static_cast<unsigned long long>(__double_as_longlong(v)));
}
SRHD_DEV void atomic_max_nonneg(float* addr, float v) {
  atomicMax(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}
SRHD_DEV real warp_max(real v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
SRHD_DEV unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace srhd
