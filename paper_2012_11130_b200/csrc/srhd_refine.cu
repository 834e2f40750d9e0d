// srhd_refine.cu -- srhd_refine_flags: the SRHD refinement criteria of the paper evaluated per 8^3
// patch on the same ghosted patch-group tiles the fluid step consumes (section 3.1: gradient of
// the Lorentz factor and the magnitude of |M|/D; Eq. 33: normalised gradient of Q).
//
// One CTA per patch group: Q of the (16+2)^3 cells that the centred differences touch goes to shared
// memory (cons2prim per cell when Q is a primitive quantity -- "computationally expensive" on the
// CPU, which is why it is worth a kernel), then one thread per interior cell evaluates
//   (|Q(i+1)-Q(i-1)| + |Q(j+1)-Q(j-1)| + |Q(k+1)-Q(k-1)|) / (2 |Q|) > C_Q          (Eq. 33, reading S17)
//   |M| / D > threshold
// and the patch flags are OR-reduced with one shared atomic per warp.
#include "srhd_common.cuh"

namespace srhd {

constexpr int kRefineThreads = 256;

template <int G>
__global__ void __launch_bounds__(kRefineThreads) refine_flags_kernel(const real* __restrict__ cons_in,
                                                                      int quantity, real c_q, real mom_thr,
                                                                      real rtol, int max_iter,
                                                                      unsigned char* __restrict__ flags) {
  constexpr int NXT = 16 + 2 * G, T3 = NXT * NXT * NXT, NQ = 18 * 18 * 18;
  __shared__ real Q[NQ];
  __shared__ unsigned int pflag[8];
  const int tid = threadIdx.x, lane = tid & 31;
  const real* __restrict__ tile = cons_in + (size_t)blockIdx.x * 5 * T3;
  if (tid < 8) pflag[tid] = 0u;
  // ---- Q on the 18^3 cells around and including the interior
  if (quantity != SRHD_REFINE_NONE) {
    for (int base = tid - lane; base < NQ; base += kRefineThreads) {     // warp-uniform trip count
      const int item = base + lane;
      const int c = item < NQ ? item : NQ - 1;
      const int i = c % 18, j = (c / 18) % 18, k = c / 324;
      const size_t src = ((size_t)(k + G - 1) * NXT + (j + G - 1)) * NXT + (i + G - 1);
      real q;
      if (quantity == SRHD_REFINE_D) {
        q = tile[src];
      } else if (quantity == SRHD_REFINE_ETILDE) {
        q = tile[4 * (size_t)T3 + src];
      } else {
        real U[1][5], W[1][5];
#pragma unroll
        for (int m = 0; m < 5; ++m) U[0][m] = tile[m * (size_t)T3 + src];
        bool phys[1];
        int it[1];
        Aux aux[1];
        cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
        q = (quantity == SRHD_REFINE_RHO) ? W[0][0]
                                          : sqrt(real(1.0) + (W[0][1] * W[0][1] + W[0][2] * W[0][2] + W[0][3] * W[0][3]));
      }
      if (item < NQ) Q[c] = q;
    }
  }
  __syncthreads();
  // ---- criteria on the 16^3 interior cells
  for (int c = tid; c < 4096; c += kRefineThreads) {
    const int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    bool hit = false;
    if (quantity != SRHD_REFINE_NONE) {
      const int q0 = ((k + 1) * 18 + (j + 1)) * 18 + (i + 1);
      const real gx = fabs(Q[q0 + 1] - Q[q0 - 1]), gy = fabs(Q[q0 + 18] - Q[q0 - 18]),
                   gz = fabs(Q[q0 + 324] - Q[q0 - 324]);
      hit = ((gx + gy) + gz) / (real(2.0) * fabs(Q[q0])) > c_q;
    }
    if (mom_thr > real(0.0)) {
      const size_t src = ((size_t)(k + G) * NXT + (j + G)) * NXT + (i + G);
      const real D = tile[src], mx = tile[(size_t)T3 + src], my = tile[2 * (size_t)T3 + src],
                   mz = tile[3 * (size_t)T3 + src];
      hit = hit || (sqrt((mx * mx + my * my) + mz * mz) / D > mom_thr);
    }
    // the 32 cells of a warp lie in one patch row pair: i spans 0..15 (two patches in x), fixed j pair, k
    const unsigned left = __ballot_sync(0xffffffffu, hit && (i < 8));
    const unsigned right = __ballot_sync(0xffffffffu, hit && (i >= 8));
    if (lane == 0) {
      const int pyz = 2 * (j >> 3) + 4 * (k >> 3);
      if (left) atomicOr(&pflag[pyz], 1u);
      if (right) atomicOr(&pflag[pyz + 1], 1u);
    }
  }
  __syncthreads();
  if (tid < 8) flags[(size_t)blockIdx.x * 8 + tid] = (unsigned char)pflag[tid];
}

}  // namespace srhd

using namespace srhd;

extern "C" int srhd_refine_flags(const real* cons_in, int npg, int quantity, double c_q, double mom_over_d,
                                 const srhd_params* params, unsigned char* flags, void* stream) {
  if (npg > 0 && (!cons_in || !flags)) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  if (npg < 0) return SRHD_ERR_BAD_SIZE;
  if (quantity < SRHD_REFINE_NONE || quantity > SRHD_REFINE_GAMMA) return SRHD_ERR_BAD_PARAMS;
  if (!(c_q >= real(0.0)) || !(mom_over_d >= real(0.0))) return SRHD_ERR_BAD_PARAMS;
  if (npg == 0) return SRHD_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const real rtol = newton_stop_rtol(params->newton_rtol);
  if (params->ghost == 2)
    refine_flags_kernel<2><<<npg, kRefineThreads, 0, st>>>(cons_in, quantity, c_q, mom_over_d, rtol,
                                                           params->newton_max_iter, flags);
  else if (params->ghost == 4)
    refine_flags_kernel<4><<<npg, kRefineThreads, 0, st>>>(cons_in, quantity, c_q, mom_over_d, rtol,
                                                           params->newton_max_iter, flags);
  else
    refine_flags_kernel<3><<<npg, kRefineThreads, 0, st>>>(cons_in, quantity, c_q, mom_over_d, rtol,
                                                           params->newton_max_iter, flags);
  return (int)cudaGetLastError();
}
