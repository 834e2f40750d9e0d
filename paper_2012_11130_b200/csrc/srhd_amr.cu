// srhd_amr.cu -- the coarse-fine hooks an AMR driver needs around srhd_fluid_step:
//   srhd_flux_correction  P:285 section 3.3(4): swap the coarse flux through a coarse-fine interface for the fine
//                         fluxes in the coarse cells next to it; "if unphysical results are found after this flux
//                         correction, we simply ignore the correction on the failed cells";
//   srhd_ghost_interp     P:281 section 3.3(3): 2x interpolation of conserved variables into fine ghost zones,
//                         falling back to the interpolation of PRIMITIVE variables where a child fails Eq. 30.
// Both are memory-bound gathers with a little arithmetic; one thread per face cell / per coarse cell.
#include "srhd_common.cuh"

namespace srhd {

__global__ void __launch_bounds__(64) flux_correction_kernel(real* __restrict__ patches,
                                                             const real* __restrict__ flux_coarse,
                                                             const real* __restrict__ flux_fine,
                                                             const int* __restrict__ face_patch,
                                                             const int* __restrict__ face_id, int cls, real dtdh,
                                                             unsigned long long* __restrict__ n_skipped) {
  const int f = blockIdx.x;
  if (face_id[f] != cls) return;                             // faces are processed class by class (see the ABI)
  const int d = cls >> 1, hi = cls & 1;
  const int a = threadIdx.x >> 3, bb = threadIdx.x & 7;
  int i, j, k;
  if (d == 0) { i = hi ? 7 : 0; j = bb; k = a; }
  else if (d == 1) { i = bb; j = hi ? 7 : 0; k = a; }
  else { i = bb; j = a; k = hi ? 7 : 0; }
  real* P = patches + (size_t)face_patch[f] * 5 * 512 + k * 64 + j * 8 + i;
  real Un[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const size_t o = ((size_t)f * 5 + q) * 64 + threadIdx.x;
    const real dF = flux_fine[o] - flux_coarse[o];
    Un[q] = hi ? P[q * 512] - dtdh * dF : P[q * 512] + dtdh * dF;
  }
  const bool ok = is_physical(Un);                           // Eq. 30 on the corrected cell
  if (ok) {
#pragma unroll
    for (int q = 0; q < 5; ++q) P[q * 512] = Un[q];
  }
  const unsigned long long bad = warp_sum(ok ? 0ull : 1ull);
  if ((threadIdx.x & 31) == 0 && bad) atomicAdd(n_skipped, bad);
}

// limited slopes of the five components of V[0] from its six neighbours, times 1/4 (children sit a quarter cell off)
SRHD_DEV void quarter_slopes(const real V[7][5], real beta, real sl[3][5]) {
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int q = 0; q < 5; ++q)
      sl[d][q] = real(0.25) * limited_slope(V[0][q] - V[1 + 2 * d][q], V[2 + 2 * d][q] - V[0][q], beta);
}
SRHD_DEV void child_of(const real V0[5], const real sl[3][5], int ch, real v[5]) {
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const real ax = (ch & 1) ? sl[0][q] : -sl[0][q], ay = (ch & 2) ? sl[1][q] : -sl[1][q],
                 az = (ch & 4) ? sl[2][q] : -sl[2][q];
    v[q] = ((V0[q] + ax) + ay) + az;
  }
}

__global__ void __launch_bounds__(128) ghost_interp_kernel(const real* __restrict__ coarse, int nx, int ny, int nz,
                                                           real* __restrict__ fine, real beta, real rtol,
                                                           int max_iter, unsigned char* __restrict__ fallback,
                                                           unsigned long long* __restrict__ n_fallback) {
  const int mx = nx - 2, my = ny - 2, mz = nz - 2;
  const long long ncell = (long long)mx * my * mz;
  const size_t n = (size_t)nx * ny * nz;
  const int fx = 2 * mx, fy = 2 * my;
  const size_t nf = (size_t)fx * fy * (2 * mz);
  const unsigned lane = threadIdx.x & 31u;
  unsigned long long nfb = 0;
  for (long long e0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; e0 - lane < ncell;
       e0 += (long long)gridDim.x * blockDim.x) {
    const bool valid = e0 < ncell;
    const long long e = valid ? e0 : ncell - 1;
    const int i = (int)(e % mx) + 1, j = (int)((e / mx) % my) + 1, k = (int)(e / ((long long)mx * my)) + 1;
    const size_t c = ((size_t)k * ny + j) * nx + i;
    const ptrdiff_t stp[3] = {1, nx, (ptrdiff_t)nx * ny};
    real Q[7][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      Q[0][q] = __ldg(coarse + q * n + c);
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        Q[1 + 2 * d][q] = __ldg(coarse + q * n + c - stp[d]);
        Q[2 + 2 * d][q] = __ldg(coarse + q * n + c + stp[d]);
      }
    }
    real sl[3][5], child[8][5];
    quarter_slopes(Q, beta, sl);
    bool ok = true, prim_bad = false;
#pragma unroll
    for (int ch = 0; ch < 8; ++ch) {
      child_of(Q[0], sl, ch, child[ch]);
      ok = ok && is_physical(child[ch]);
    }
    // the fallback converts seven states per cell: a warp-wide loop (cons2prim's Newton iteration votes), entered
    // by every lane as soon as one lane needs it; lanes that do not need it discard the result
    if (__any_sync(0xffffffffu, !ok)) {
      real W[7][5];
#pragma unroll
      for (int m = 0; m < 7; ++m) {
        real U1[1][5], W1[1][5];
#pragma unroll
        for (int q = 0; q < 5; ++q) U1[0][q] = Q[m][q];
        bool phys[1];
        int it[1];
        Aux aux[1];
        cons2prim_multi<1>(U1, W1, aux, rtol, max_iter, phys, it);
#pragma unroll
        for (int q = 0; q < 5; ++q) W[m][q] = W1[0][q];
      }
      if (!ok) {
        quarter_slopes(W, beta, sl);
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
          real v[5];
          child_of(W[0], sl, ch, v);
          // S22: interpolated primitives pass Eq. 30 only while rho and p stay positive (a steep 3-D corner can
          // take three quarter-slopes off the cell value)
          prim_bad = prim_bad || !(v[0] > real(0.0)) || !(v[4] > real(0.0));
          prim2cons(v, child[ch]);
        }
        if (prim_bad) {                         // copy the parent: the vanished-coefficient end of the ladder
#pragma unroll
          for (int ch = 0; ch < 8; ++ch)
#pragma unroll
            for (int q = 0; q < 5; ++q) child[ch][q] = Q[0][q];
        }
        if (valid) ++nfb;
      }
    }
    if (valid) {
      if (fallback) fallback[e] = ok ? 0 : (prim_bad ? 2 : 1);
#pragma unroll
      for (int ch = 0; ch < 8; ++ch) {
        const int I = 2 * (i - 1) + (ch & 1), J = 2 * (j - 1) + ((ch >> 1) & 1), K = 2 * (k - 1) + (ch >> 2);
#pragma unroll
        for (int q = 0; q < 5; ++q) fine[q * nf + ((size_t)K * fy + J) * fx + I] = child[ch][q];
      }
    }
  }
  nfb = warp_sum(nfb);
  if (lane == 0 && nfb) atomicAdd(n_fallback, nfb);
}

}  // namespace srhd

using namespace srhd;

extern "C" int srhd_flux_correction(real* patches, const real* flux_coarse, const real* flux_fine,
                                    const int* face_patch, const int* face_id, int nf, double dt, double dh,
                                    unsigned long long* d_n_skipped, void* stream) {
  if (nf < 0) return SRHD_ERR_BAD_SIZE;
  if (!d_n_skipped || (nf > 0 && (!patches || !flux_coarse || !flux_fine || !face_patch || !face_id)))
    return SRHD_ERR_NULL_POINTER;
  if (!(dt > real(0.0)) || !(dh > real(0.0)) || !std::isfinite(dt) || !std::isfinite(dh)) return SRHD_ERR_BAD_STEP;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaError_t e = cudaMemsetAsync(d_n_skipped, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return (int)e;
  if (nf == 0) return SRHD_OK;
  for (int cls = 0; cls < 6; ++cls)      // a cell on a patch edge belongs to two faces: one class after the other
    flux_correction_kernel<<<nf, 64, 0, st>>>(patches, flux_coarse, flux_fine, face_patch, face_id, cls, dt / dh,
                                              d_n_skipped);
  return (int)cudaGetLastError();
}

extern "C" int srhd_ghost_interp(const real* coarse, int nx, int ny, int nz, real* fine, double minmod_coeff,
                                 const srhd_params* params, unsigned char* fallback,
                                 unsigned long long* d_n_fallback, void* stream) {
  if (!coarse || !fine || !d_n_fallback) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  if (nx < 3 || ny < 3 || nz < 3) return SRHD_ERR_BAD_SIZE;
  if (!(minmod_coeff >= real(0.0)) || !(minmod_coeff <= real(2.0))) return SRHD_ERR_BAD_PARAMS;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaError_t e = cudaMemsetAsync(d_n_fallback, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return (int)e;
  const long long ncell = (long long)(nx - 2) * (ny - 2) * (nz - 2);
  const long long want = (ncell + 127) / 128, cap = (long long)num_sms() * 16;
  ghost_interp_kernel<<<(int)(want < cap ? want : cap), 128, 0, st>>>(coarse, nx, ny, nz, fine, minmod_coeff,
                                                                     newton_stop_rtol(params->newton_rtol),
                                                                     params->newton_max_iter, fallback, d_n_fallback);
  return (int)cudaGetLastError();
}
