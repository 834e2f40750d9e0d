// srhd_uniform.cuh -- what one step does to a patch group whose whole tile (ghost zones included) holds ONE
// state U0 bit for bit, shared by the two pre-passes that look for such tiles (uniform_tiles_kernel in
// srhd_fluid.cu: tiles already gathered; patch_prepass_kernel in srhd_grid.cu: straight from the patches).
//
// The algorithm of srhd_fluid_step collapses (readings S3-S7, S12): W0 = C2P(U0) for every tile cell; all
// slopes vanish, so every edge state is U1 = P2C(W0) and every flux difference of the half step is +0
// (U1 + (-0) = U1); every face solves the same Riemann problem F_d(U1, U1); every update is
// U0 - dt/dh ((F-F) + (F-F) + (F-F)) = U0 for any finite dt.  Anything unusual (a state that fails Eq. 30, a
// non-finite flux) makes uniform_eval return false and the group takes the general march.
#pragma once
#include "srhd_common.cuh"

namespace srhd {

struct UniformResult {
  int it0, it1;       // Newton-Raphson iterations of C2P(U0) and C2P(U1)
  real umax;        // Eq. 26 of W0
  real F[3][5];     // the Riemann flux of (U1, U1) along x, y, z
};

// every thread of the CTA calls this with the same U0 (the warp votes inside cons2prim_multi need whole warps)
template <int RS>
SRHD_DEV bool uniform_eval(const real U0in[5], real rtol, int max_iter, UniformResult& r) {
  real U0[1][5], W0[1][5], U1[1][5], W1[1][5];
#pragma unroll
  for (int q = 0; q < 5; ++q) U0[0][q] = U0in[q];
  bool ph0[1], ph1[1];
  int it0[1], it1[1];
  Aux a0[1], a1[1], ae;
  cons2prim_multi<1>(U0, W0, a0, rtol, max_iter, ph0, it0);
  prim2cons_aux(W0[0], U1[0], ae);
  cons2prim_multi<1>(U1, W1, a1, rtol, max_iter, ph1, it1);
  bool ok = ph0[0] && ph1[0] && is_physical(U0[0]);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    riemann_flux<RS>(d, W1[0], U1[0], a1[0], W1[0], U1[0], a1[0], r.F[d], true);
#pragma unroll
    for (int q = 0; q < 5; ++q) ok = ok && (fabs(r.F[d][q]) <= kRealMax);
  }
  r.it0 = it0[0];
  r.it1 = it1[0];
  r.umax = umax_of_prim(W0[0], a0[0]);
  return ok;
}

// Does the tile (5 components x T3 values, 16-byte aligned) hold ONE state?  It is streamed once with 16-byte
// loads compared as bit patterns with the first cell (U0 receives it); a tile that is not uniform is dropped at
// its first 4 KB.  NT threads per CTA, all of them call it; the return value is block uniform.
template <int T3, int NT>
SRHD_DEV bool tile_scan_uniform(const real* __restrict__ tile, real U0[5]) {
  constexpr int H = T3 / 2;                                  // 16-byte words per component
  static_assert(T3 % 2 == 0, "tile components must be whole 16-byte words");
  const int tid = threadIdx.x;
  const real2* __restrict__ t2 = reinterpret_cast<const real2*>(tile);
  rbits ref[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) ref[q] = real_bits(__ldg(tile + (size_t)q * T3));
  auto differs = [&](int w, real2 v) {
    const int q = w / H;
    const rbits r = (q == 0) ? ref[0] : (q == 1) ? ref[1] : (q == 2) ? ref[2] : (q == 3) ? ref[3] : ref[4];
    return (real_bits(v.x) != r) || (real_bits(v.y) != r);
  };
  if (__syncthreads_or(differs(tid, __ldg(t2 + tid)) ? 1 : 0)) return false;   // the first 4 KB settle most tiles
  for (int base = NT; base < 5 * H; base += 8 * NT) {
    real2 v[8];
    int w[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      w[u] = min(base + u * NT + tid, 5 * H - 1);
      v[u] = __ldg(t2 + w[u]);
    }
    bool diff = false;
#pragma unroll
    for (int u = 0; u < 8; ++u) diff = diff || differs(w[u], v[u]);
    if (__syncthreads_or(diff ? 1 : 0)) return false;
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) U0[q] = bits_real(ref[q]);
  return true;
}

// the 8 patches of the group, out[patch][component][512] = U0[component]; NT threads, thread tid.  It may be
// issued BEFORE the verdict of uniform_eval is known: a group that is marched after all has every cell rewritten.
SRHD_DEV void uniform_write_state(real* __restrict__ out, const real U0[5], int tid, int NT) {
  real2* __restrict__ o2 = reinterpret_cast<real2*>(out);
  for (int w = tid; w < 8 * 5 * 256; w += NT) {
    const int q = (w >> 8) % 5;
    const real u = (q == 0) ? U0[0] : (q == 1) ? U0[1] : (q == 2) ? U0[2] : (q == 3) ? U0[3] : U0[4];
    o2[w] = make_real2(u, u);
  }
}
// the patch-boundary fluxes, fout[patch][face][component][64] = F[face >> 1][component]
SRHD_DEV void uniform_write_flux(real* __restrict__ fout, const UniformResult& r, int tid, int NT) {
  for (int w = tid; w < 8 * 6 * 5 * 64; w += NT) {
    const int q = (w >> 6) % 5, d = ((w / 320) % 6) >> 1;
    real f = real(0.0);
#pragma unroll
    for (int dd = 0; dd < 3; ++dd)
#pragma unroll
      for (int qq = 0; qq < 5; ++qq) f = (dd == d && qq == q) ? r.F[dd][qq] : f;
    fout[w] = f;
  }
}
// One warp evaluates the uniform state while the others' stores are in flight; the verdict and the result go through
// shared memory.  Block-uniform return value; every thread of the CTA must call it.
template <int RS>
SRHD_DEV bool uniform_eval_by_warp0(const real U0[5], real rtol, int max_iter, UniformResult& r) {
  __shared__ UniformResult s_r;
  __shared__ int s_ok;
  if (threadIdx.x < 32) {
    UniformResult t;
    const bool ok = uniform_eval<RS>(U0, rtol, max_iter, t);
    if (threadIdx.x == 0) {
      s_r = t;
      s_ok = ok ? 1 : 0;
    }
  }
  __syncthreads();
  r = s_r;
  return s_ok != 0;
}

// what the march would have counted for this group (one thread); tile_cells = (16 + 2 ghost)^3
SRHD_DEV void uniform_count(srhd_stats* __restrict__ stats, int tile_cells, const UniformResult& r) {
  if (!stats) return;
  atomicAdd(&stats->newton_iters, (unsigned long long)tile_cells * (unsigned)r.it0 +
                                      (unsigned long long)(2 * 3 * 17 * 256) * (unsigned)r.it1);
  atomicAdd(&stats->n_passes, 1ull);
  atomicAdd(&stats->exec_newton, (unsigned long long)(r.it0 + r.it1));
  atomicAdd(&stats->exec_c2p, 2ull);
  atomicAdd(&stats->exec_riemann, SRHD_EXACT ? 3ull : 0ull);
  atomicAdd(&stats->n_uniform_pg, 1ull);
  atomic_max_nonneg(&stats->max_speed, smax_of_umax(r.umax));
}

// srhd_fluid.cu: the march alone, for patch groups whose handled[] byte is 0 (the caller ran a pre-pass)
int fluid_march(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
                const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
                real min_speed, const unsigned char* handled);

}  // namespace srhd
