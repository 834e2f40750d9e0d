// srhd_vl.cu -- the VL integrator ("VL (Falle 1991; van Leer 2006)"; reading S18 of DESIGN.md) behind
// srhd_fluid_step when params->integrator == SRHD_INTEGRATOR_VL: van Leer's predictor-corrector.
//   V1  W = cons2prim(U) of every tile cell (ghost width: PLM 3, PPM 4)             vl_centre_kernel
//   V2  first-order fluxes F1 from the CELL-CENTRE states of the two cells of a face
//   V3  Uh = U - dt/(2 dh) div F1,  Wh = cons2prim(Uh)                               vl_predictor_kernel
//   V4  PLM / PPM edge values of Wh (retry coefficient beta_k), prim2cons of the edges
//   V5  HLLE / HLLC on the edge states of every face of an interior cell
//   V6  Unew = U - dt/dh div F2, Eq. 30 check; retry ladder over V4-V6 per patch group  vl_corrector_kernel
// Unlike the MUSCL-Hancock path this one is NOT fused: the stages communicate through two primitive tiles
// (W and Wh) in a stream-ordered scratch allocation, one thread per cell, every face solved by both cells
// that share it (the solver is a function of its inputs, so both get the same bits).  It is the second
// integrator of the paper at the same parity bar, not the tuned hot path.
#include "srhd_common.cuh"
#include "srhd_uniform.cuh"

namespace srhd {

constexpr int kVlThreads = 256;

// by-products of a conversion that the production-build solver wants, recomputed from primitives
SRHD_DEV Aux aux_of_prim(const real W[5]) {
  Aux a;
#if SRHD_GENERIC
  a.ht = a.T = a.rg = real(0.0);
#else
  a.T = W[4] * rcp_f(W[0]);
  const real a2 = real(2.25) * a.T * a.T, a1 = a2 + real(1.0);
  a.ht = fma(a2, rcp_f(real(1.0) + a1 * rsqrt_f(a1)), real(2.5) * a.T);     // Eq. 22
  a.rg = rsqrt_f(real(1.0) + (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]));
#endif
  return a;
}

struct VlScratch {
  real* Wc;                 // [npg][5][T3] primitives of the tile
  real* Wh;                 // [npg][5][T3] primitives of the half-step state (predictor cells only)
  unsigned long long* umax;   // bit pattern of max U_max over the interior input cells
};

template <int G>
__global__ void __launch_bounds__(kVlThreads) vl_centre_kernel(const real* __restrict__ cons_in, VlScratch s,
                                                               long long ncell, real rtol, int max_iter,
                                                               srhd_stats* __restrict__ stats,
                                                               const unsigned char* __restrict__ handled) {
  constexpr int NXT = 16 + 2 * G, PL = NXT * NXT, T3 = PL * NXT;
  const unsigned lane = threadIdx.x & 31u;
  const long long step = (long long)gridDim.x * blockDim.x;
  unsigned long long iters = 0, fail = 0, done = 0;
  real umax = real(0.0);
  for (long long i0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; i0 - lane < ncell; i0 += step) {
    const long long i = (i0 < ncell) ? i0 : ncell - 1;
    const long long pg = i / T3;
    const bool valid = (i0 < ncell) && !handled[pg];          // groups the uniform pre-pass has finished are skipped
    if (!__any_sync(0xffffffffu, valid)) continue;             // (whole warps: the conversion votes)
    const int c = (int)(i - pg * T3);
    const real* t = cons_in + pg * 5 * T3 + c;
    real U[1][5], W[1][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[0][q] = __ldg(t + (size_t)q * T3);
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
    if (valid) {
      real* w = s.Wc + pg * 5 * T3 + c;
#pragma unroll
      for (int q = 0; q < 5; ++q) w[(size_t)q * T3] = W[0][q];
      iters += (unsigned)it[0];
      ++done;
      const int ti = c % NXT, tj = (c / NXT) % NXT, tk = c / PL;
      if (ti >= G && ti < G + 16 && tj >= G && tj < G + 16 && tk >= G && tk < G + 16) {
        fail += phys[0] ? 0u : 1u;
        umax = fmax(umax, umax_of_prim(W[0], aux[0]));
      }
    }
  }
  iters = warp_sum(iters);
  fail = warp_sum(fail);
  done = warp_sum(done);
  umax = warp_max(umax);
  if (lane == 0) {
    atomicMax(s.umax, real_bits(umax));
    if (stats) {
      atomicAdd(&stats->newton_iters, iters);
      atomicAdd(&stats->exec_newton, iters);
      atomicAdd(&stats->exec_c2p, done);
      if (fail) atomicAdd(&stats->n_c2p_fail, fail);
    }
  }
}

// first-order flux through the face between tile cells cl and cl + stride_d (centre states)
template <int G, int RS>
SRHD_DEV void flux1(const real* __restrict__ t, const real* __restrict__ w, int d, int cl, real F[5]) {
  constexpr int NXT = 16 + 2 * G, T3 = NXT * NXT * NXT;
  const int cr = cl + ((d == 0) ? 1 : ((d == 1) ? NXT : NXT * NXT));
  real UL[5], UR[5], WL[5], WR[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    UL[q] = __ldg(t + (size_t)q * T3 + cl);
    UR[q] = __ldg(t + (size_t)q * T3 + cr);
    WL[q] = w[(size_t)q * T3 + cl];
    WR[q] = w[(size_t)q * T3 + cr];
  }
  riemann_flux<RS>(d, WL, UL, aux_of_prim(WL), WR, UR, aux_of_prim(WR), F);
}

template <int G, int RS>
__global__ void __launch_bounds__(kVlThreads) vl_predictor_kernel(const real* __restrict__ cons_in, VlScratch s,
                                                                  long long ncell, real dt, real dh, real rtol,
                                                                  int max_iter, srhd_stats* __restrict__ stats,
                                                                  const real* __restrict__ d_smax, real cfl,
                                                                  real min_speed,
                                                                  const unsigned char* __restrict__ handled) {
  constexpr int NXT = 16 + 2 * G, PL = NXT * NXT, T3 = PL * NXT, E = NXT - 2, E3 = E * E * E;
  if (d_smax) dt = cfl * dh / fmax(*d_smax, min_speed);        // Eq. 28 on the device
  const real hdt = dt / (real(2.0) * dh);
  const unsigned lane = threadIdx.x & 31u;
  const long long step = (long long)gridDim.x * blockDim.x;
  unsigned long long iters = 0, fail = 0, done = 0;
  for (long long i0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; i0 - lane < ncell; i0 += step) {
    const long long i = (i0 < ncell) ? i0 : ncell - 1;
    const long long pg = i / E3;
    const bool valid = (i0 < ncell) && !handled[pg];
    if (!__any_sync(0xffffffffu, valid)) continue;
    const int e = (int)(i - pg * E3);
    const int c = ((e / (E * E)) + 1) * PL + (((e / E) % E) + 1) * NXT + (e % E) + 1;   // one layer in from the rim
    const real* t = cons_in + pg * 5 * T3;
    const real* w = s.Wc + pg * 5 * T3;
    real Uh[1][5], W[1][5], df[3][5];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int st = (d == 0) ? 1 : ((d == 1) ? NXT : PL);
      real Fm[5], Fp[5];
      flux1<G, RS>(t, w, d, c - st, Fm);
      flux1<G, RS>(t, w, d, c, Fp);
#pragma unroll
      for (int q = 0; q < 5; ++q) df[d][q] = Fp[q] - Fm[q];
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) Uh[0][q] = __ldg(t + (size_t)q * T3 + c) - hdt * ((df[0][q] + df[1][q]) + df[2][q]);
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(Uh, W, aux, rtol, max_iter, phys, it);
    if (valid) {
      real* wh = s.Wh + pg * 5 * T3 + c;
#pragma unroll
      for (int q = 0; q < 5; ++q) wh[(size_t)q * T3] = W[0][q];
      iters += (unsigned)it[0];
      ++done;
      fail += phys[0] ? 0u : 1u;                               // S15 / S18: counted, no rung can cure it
    }
  }
  iters = warp_sum(iters);
  fail = warp_sum(fail);
  done = warp_sum(done);
  if (lane == 0 && stats) {
    atomicAdd(&stats->newton_iters, iters);
    atomicAdd(&stats->exec_newton, iters);
    atomicAdd(&stats->exec_c2p, done);
    atomicAdd(&stats->exec_riemann, 6ull * done);
    if (fail) atomicAdd(&stats->n_c2p_fail, fail);
  }
}

// edge primitives of tile cell c along d from the half-step primitives, and their conserved form
template <int G>
SRHD_DEV void edges_of(const real* __restrict__ wh, int c, int st, real beta, real beta0, real Wm[5],
                       real Wp[5]) {
  constexpr int NXT = 16 + 2 * G, T3 = NXT * NXT * NXT;
  constexpr bool PPM = (G == 4);
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const real* p = wh + (size_t)q * T3 + c;
    if (PPM) {
      const real a[5] = {p[-2 * st], p[-st], p[0], p[st], p[2 * st]};
      recon_ppm(a, beta, beta0, Wm[q], Wp[q]);
    } else {
      const real a[3] = {p[-st], p[0], p[st]};
      recon_plm(a, beta, Wm[q], Wp[q]);
    }
  }
}

template <int G, int RS>
__global__ void __launch_bounds__(kVlThreads) vl_corrector_kernel(const real* __restrict__ cons_in,
                                                                  real* __restrict__ cons_out,
                                                                  real* __restrict__ flux_out, VlScratch s, real dt,
                                                                  real dh, real beta0, int max_retry,
                                                                  srhd_stats* __restrict__ stats,
                                                                  const real* __restrict__ d_smax, real cfl,
                                                                  real min_speed,
                                                                  const unsigned char* __restrict__ handled) {
  constexpr int NXT = 16 + 2 * G, PL = NXT * NXT, T3 = PL * NXT;
  if (handled[blockIdx.x]) return;                               // a uniform tile: vl_uniform_tiles_kernel wrote its result
  if (d_smax) dt = cfl * dh / fmax(*d_smax, min_speed);
  const real dtdh = dt / dh;
  const long long pg = blockIdx.x;
  const real* t = cons_in + pg * 5 * T3;
  const real* wh = s.Wh + pg * 5 * T3;
  real* out = cons_out + pg * 8 * 5 * 512;
  real* fout = flux_out ? flux_out + pg * 8 * 6 * 5 * 64 : nullptr;
  real beta = beta0;
  int pass = 0, nfail = 0;
  unsigned ex_riemann = 0, ex_edges = 0;
  for (;; ++pass) {
    if (pass > 0) beta = (pass <= max_retry) ? beta * real(0.75) : real(0.0);
    int my_fail = 0;
    for (int cell = threadIdx.x; cell < 4096; cell += kVlThreads) {
      const int i = cell & 15, j = (cell >> 4) & 15, k = cell >> 8;
      const int c = (k + G) * PL + (j + G) * NXT + (i + G);
      real dfs[3][5];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const int st = (d == 0) ? 1 : ((d == 1) ? NXT : PL);
        real Wm0[5], Wp0[5], Wmm[5], Wpm[5], Wmp[5], Wpp[5];
        edges_of<G>(wh, c, st, beta, beta0, Wm0, Wp0);           // this cell
        edges_of<G>(wh, c - st, st, beta, beta0, Wmm, Wpm);      // lower neighbour: its plus edge is used
        edges_of<G>(wh, c + st, st, beta, beta0, Wmp, Wpp);      // upper neighbour: its minus edge is used
        real UL[5], UR[5], Flo[5], Fhi[5];
        Aux aL, aR;
        prim2cons_aux(Wpm, UL, aL);
        prim2cons_aux(Wm0, UR, aR);
        riemann_flux<RS>(d, Wpm, UL, aL, Wm0, UR, aR, Flo);
        prim2cons_aux(Wp0, UL, aL);
        prim2cons_aux(Wmp, UR, aR);
        riemann_flux<RS>(d, Wp0, UL, aL, Wmp, UR, aR, Fhi);
        ex_riemann += 2;
        ex_edges += 3;
#pragma unroll
        for (int q = 0; q < 5; ++q) dfs[d][q] = Fhi[q] - Flo[q];
        if (fout) {                                              // faces on the boundary of an 8^3 patch
          const int x = (d == 0) ? i : ((d == 1) ? j : k);       // coordinate along d
          const int a = (d == 0) ? k : ((d == 1) ? k : j), b = (d == 0) ? j : i;   // in-face coordinates, slower first
          const int p = (i >> 3) + 2 * (j >> 3) + 4 * (k >> 3);
          if ((x & 7) == 0) {
#pragma unroll
            for (int q = 0; q < 5; ++q) fout[(((size_t)p * 6 + 2 * d) * 5 + q) * 64 + (a & 7) * 8 + (b & 7)] = Flo[q];
          }
          if ((x & 7) == 7) {
#pragma unroll
            for (int q = 0; q < 5; ++q) fout[(((size_t)p * 6 + 2 * d + 1) * 5 + q) * 64 + (a & 7) * 8 + (b & 7)] = Fhi[q];
          }
        }
      }
      const int p = (i >> 3) + 2 * (j >> 3) + 4 * (k >> 3);       // S13
      real* o = out + (size_t)p * 5 * 512 + (k & 7) * 64 + (j & 7) * 8 + (i & 7);
      real Un[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        Un[q] = __ldg(t + (size_t)q * T3 + c) - dtdh * ((dfs[0][q] + dfs[1][q]) + dfs[2][q]);   // S12
        o[q * 512] = Un[q];
      }
      if (!is_physical(Un)) ++my_fail;                            // Eq. 30
    }
    nfail = __syncthreads_count(my_fail != 0) ? 1 : 0;
    // the count of failing CELLS of the accepted pass is needed only when the ladder ends here
    if (nfail == 0 || beta == real(0.0)) {
      const unsigned long long tot = warp_sum((unsigned long long)my_fail);
      if ((threadIdx.x & 31) == 0 && tot && stats) atomicAdd(&stats->n_unphys_final, tot);
      break;
    }
  }
  const unsigned long long r = warp_sum((unsigned long long)ex_riemann), e2 = warp_sum((unsigned long long)ex_edges);
  if ((threadIdx.x & 31) == 0 && stats) {
    atomicAdd(&stats->exec_riemann, r);
    atomicAdd(&stats->exec_hancock, e2);
  }
  if (threadIdx.x == 0 && stats) {
    if (pass > 0) atomicAdd(&stats->n_retry_pg, 1ull);
    atomicAdd(&stats->n_passes, (unsigned long long)(pass + 1));
  }
}

// Uniform tiles under the VL integrator (srhd_uniform.cuh; reading S18): W0 = C2P(U0) for every tile cell; the
// first-order fluxes of equal neighbours cancel, so the predictor state is U0 again and its primitives are W0 (the
// same conversion, the same bits); every edge state is (W0, U1 = P2C(W0)); every face solves F_d(W0, U1; W0, U1);
// every update is U0 - dt/dh 0 = U0.  One CTA per group, ahead of the three VL kernels, which skip the groups it
// has finished.
template <int RS>
SRHD_DEV bool uniform_eval_vl(const real U0in[5], real rtol, int max_iter, UniformResult& r) {
  real U0[1][5], W0[1][5], U1[5], F1[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) U0[0][q] = U0in[q];
  bool ph0[1];
  int it0[1];
  Aux a0[1], a1;
  cons2prim_multi<1>(U0, W0, a0, rtol, max_iter, ph0, it0);
  bool ok = ph0[0] && is_physical(U0[0]);
  prim2cons_aux(W0[0], U1, a1);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    riemann_flux<RS>(d, W0[0], U0[0], aux_of_prim(W0[0]), W0[0], U0[0], aux_of_prim(W0[0]), F1);   // predictor fluxes: must be finite
    riemann_flux<RS>(d, W0[0], U1, a1, W0[0], U1, a1, r.F[d]);
#pragma unroll
    for (int q = 0; q < 5; ++q) ok = ok && (fabs(F1[q]) <= kRealMax) && (fabs(r.F[d][q]) <= kRealMax);
  }
  r.it0 = it0[0];
  r.it1 = 0;
  r.umax = umax_of_prim(W0[0], a0[0]);
  return ok;
}

template <int G, int RS>
__global__ void __launch_bounds__(kVlThreads) vl_uniform_tiles_kernel(
    const real* __restrict__ cons_in, real* __restrict__ cons_out, real* __restrict__ flux_out, VlScratch s, real dt,
    real dh, real rtol, int max_iter, srhd_stats* __restrict__ stats, const real* __restrict__ d_smax, real cfl,
    real min_speed, unsigned char* __restrict__ handled) {
  constexpr int NXT = 16 + 2 * G, T3 = NXT * NXT * NXT, E = NXT - 2;
  const int tid = threadIdx.x;
  if (tid == 0) handled[blockIdx.x] = 0;
  real U0[5];
  if (!tile_scan_uniform<T3, kVlThreads>(cons_in + (size_t)blockIdx.x * 5 * T3, U0)) return;
  if (d_smax) dt = cfl * dh / fmax(*d_smax, min_speed);
  if (!(fabs(dt / dh) <= kRealMax)) return;
  uniform_write_state(cons_out + (size_t)blockIdx.x * 8 * 5 * 512, U0, tid, kVlThreads);
  __shared__ UniformResult s_r;
  __shared__ int s_ok;
  if (tid < 32) {
    UniformResult t;
    const bool ok = uniform_eval_vl<RS>(U0, rtol, max_iter, t);
    if (tid == 0) {
      s_r = t;
      s_ok = ok ? 1 : 0;
    }
  }
  __syncthreads();
  if (!s_ok) return;                                             // block uniform: left to the three VL kernels
  if (flux_out) uniform_write_flux(flux_out + (size_t)blockIdx.x * 8 * 6 * 5 * 64, s_r, tid, kVlThreads);
  if (tid == 0) {
    handled[blockIdx.x] = 1;
    atomicMax(s.umax, real_bits(s_r.umax));
    if (stats) {
      const unsigned long long it = (unsigned long long)(T3 + E * E * E) * (unsigned)s_r.it0;   // V1 + V3 conversions
      atomicAdd(&stats->newton_iters, it);
      atomicAdd(&stats->n_passes, 1ull);
      atomicAdd(&stats->n_uniform_pg, 1ull);
      atomicAdd(&stats->exec_newton, (unsigned long long)s_r.it0);
      atomicAdd(&stats->exec_c2p, 1ull);
      atomicAdd(&stats->exec_riemann, 6ull);
    }
  }
}

__global__ void vl_finish_kernel(VlScratch s, srhd_stats* stats) {
  if (!stats) return;
  const real umax = bits_real((rbits)*s.umax);
  atomic_max_nonneg(&stats->max_speed, smax_of_umax(umax));      // Eq. 27 (monotone: max first, convert once)
}

template <int G, int RS>
int launch_vl(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
              const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
              real min_speed) {
  constexpr int NXT = 16 + 2 * G, T3 = NXT * NXT * NXT, E = NXT - 2;
  const int chunk = npg < 4096 ? npg : 4096;                      // bounds the scratch: 2 x 4096 x 5 x T3 doubles
  const size_t tile = (size_t)5 * T3;
  real* buf = nullptr;
  // two primitive tiles per group of a chunk, the U_max word, one flag byte per group of a chunk
  cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&buf),
                                  (2 * (size_t)chunk * tile + 2) * sizeof(real) + 16 + (size_t)chunk, st);
  if (e != cudaSuccess) return (int)e;
  VlScratch s{buf, buf + (size_t)chunk * tile, reinterpret_cast<unsigned long long*>(buf + 2 * (size_t)chunk * tile)};
  unsigned char* handled = reinterpret_cast<unsigned char*>(buf + 2 * (size_t)chunk * tile + 2) + 16;
  e = cudaMemsetAsync(s.umax, 0, sizeof(unsigned long long), st);
  const real rtol = newton_stop_rtol(p->newton_rtol);
  for (int g0 = 0; g0 < npg && e == cudaSuccess; g0 += chunk) {
    const int n = (npg - g0 < chunk) ? npg - g0 : chunk;
    const real* in = cons_in + (size_t)g0 * tile;
    const long long nc = (long long)n * T3, ne = (long long)n * E * E * E;
    const int gc = (int)((nc + kVlThreads - 1) / kVlThreads), ge = (int)((ne + kVlThreads - 1) / kVlThreads);
    const int cap = num_sms() * 8 * 4;
    real* const out = cons_out + (size_t)g0 * 8 * 5 * 512;
    real* const fout = flux_out ? flux_out + (size_t)g0 * 8 * 6 * 5 * 64 : nullptr;
    vl_uniform_tiles_kernel<G, RS><<<n, kVlThreads, 0, st>>>(in, out, fout, s, dt, dh, rtol, p->newton_max_iter, stats,
                                                             d_smax, cfl, min_speed, handled);
    vl_centre_kernel<G><<<gc < cap ? gc : cap, kVlThreads, 0, st>>>(in, s, nc, rtol, p->newton_max_iter, stats, handled);
    vl_predictor_kernel<G, RS><<<ge < cap ? ge : cap, kVlThreads, 0, st>>>(in, s, ne, dt, dh, rtol, p->newton_max_iter,
                                                                            stats, d_smax, cfl, min_speed, handled);
    vl_corrector_kernel<G, RS><<<n, kVlThreads, 0, st>>>(in, out, fout, s, dt, dh, p->minmod_coeff, p->max_retry, stats,
                                                         d_smax, cfl, min_speed, handled);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) {
    vl_finish_kernel<<<1, 1, 0, st>>>(s, stats);
    e = cudaGetLastError();
  }
  const cudaError_t f = cudaFreeAsync(buf, st);
  return (int)(e != cudaSuccess ? e : f);
}

// called by srhd_fluid.cu's dispatcher (arguments already validated, stats already zeroed)
int vl_step(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
            const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
            real min_speed) {
  if (p->recon == SRHD_RECON_PLM) {
    return p->riemann == SRHD_RIEMANN_HLLE
               ? launch_vl<3, 0>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed)
               : launch_vl<3, 1>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed);
  }
  return p->riemann == SRHD_RIEMANN_HLLE
             ? launch_vl<4, 0>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed)
             : launch_vl<4, 1>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed);
}

size_t vl_workspace_bytes(int npg, const srhd_params* p) {
  const int nxt = 16 + 2 * p->ghost;
  const size_t chunk = npg < 4096 ? (size_t)(npg > 0 ? npg : 0) : 4096;
  return (2 * chunk * 5 * nxt * nxt * nxt + 2) * sizeof(real) + 16 + chunk;
}

}  // namespace srhd
