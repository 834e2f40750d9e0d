// srhd_grid.cu -- uniform-grid harness helpers (S11, S13): ghost-zone fill into patch-group tiles and
// the scatter of updated patches back to the grid.  They stand in for the AMR driver's ghost-zone
// preparation, are pure data movement (no arithmetic) and are timed as part of a step.
#include "srhd_common.cuh"
#include "srhd_uniform.cuh"

namespace srhd {

struct GridBC {
  int bc[6];
  real inflow[5];
  int has_inflow;
};

// source index of ghost index i along an axis of n cells (S11): periodic wraps, outflow clamps.
// |ghost offset| <= 4 < 16 <= n, so one conditional add replaces the modulo.
SRHD_DEV int map_index(int i, int n, int bc_lo, int bc_hi) {
  if (i < 0) return (bc_lo == SRHD_BC_PERIODIC) ? i + n : 0;
  if (i >= n) return (bc_hi == SRHD_BC_PERIODIC) ? i - n : n - 1;
  return i;
}

// one CTA per (patch group, component): the tile is written as one contiguous run (fully coalesced
// stores, all lanes busy).  The boundary mapping of the 3 x nxt tile coordinates is done once per CTA
// into shared-memory tables, so an element costs one index split (compile-time extents), three table
// reads, one load and one store; four elements in flight per thread.
template <int G>
__global__ void __launch_bounds__(256) grid_gather_kernel(const real* __restrict__ grid,
                                                          real* __restrict__ cons_in, int nx, int ny,
                                                          int nz, GridBC b,
                                                          const unsigned char* __restrict__ mask) {
  constexpr int nxt = 16 + 2 * G, nrow = nxt * nxt, t3 = nrow * nxt;
  __shared__ int xs[nxt], ys[nxt];            // source x index; source y index * nx
  __shared__ long long zs[nxt];               // source z index * ny * nx; -1 - that for a plane below z = 0
  const int px = nx / 16, py = ny / 16;
  const int pg = blockIdx.x, q = blockIdx.y;
  const int gx = pg % px, gy = (pg / px) % py, gz = pg / (px * py);
  const size_t n = (size_t)nx * ny * nz;
  if (threadIdx.x < nxt) {
    const int t = threadIdx.x;
    xs[t] = map_index(gx * 16 + t - G, nx, b.bc[0], b.bc[1]);
    ys[t] = map_index(gy * 16 + t - G, ny, b.bc[2], b.bc[3]) * nx;
    const int kk = gz * 16 + t - G;
    const long long off = (long long)map_index(kk, nz, b.bc[4], b.bc[5]) * ny * nx;
    zs[t] = (b.has_inflow && kk < 0) ? -1 - off : off;
  }
  __syncthreads();
  const real* __restrict__ src = grid + (size_t)q * n;
  real* __restrict__ dst = cons_in + ((size_t)pg * 5 + q) * t3;
  const real inflow_q = b.inflow[q];
  for (int c0 = threadIdx.x; c0 < t3; c0 += 4 * 256) {
    real v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int c = c0 + u * 256;
      if (c < t3) {
        const int k = c / nrow, r = c - k * nrow, j = r / nxt, i = r - j * nxt;
        const int xy = ys[j] + xs[i];
        long long z = zs[k];
        bool inflow = false;
        if (z < 0) {                              // ghost plane below z = 0 of a fixed-inflow boundary
          z = -1 - z;
          inflow = mask[xy] != 0;
        }
        v[u] = inflow ? inflow_q : __ldg(src + z + xy);
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int c = c0 + u * 256;
      if (c < t3) dst[c] = v[u];
    }
  }
}

// one CTA per (patch group, component): 4096 cells, writes coalesced along x in 16-cell rows
__global__ void __launch_bounds__(256) grid_scatter_kernel(const real* __restrict__ cons_out,
                                                           real* __restrict__ grid, int nx, int ny,
                                                           int nz) {
  const int px = nx / 16, py = ny / 16;
  const int pg = blockIdx.x, q = blockIdx.y;
  const int gx = pg % px, gy = (pg / px) % py, gz = pg / (px * py);
  const size_t n = (size_t)nx * ny * nz;
  const real* __restrict__ src = cons_out + (size_t)pg * 8 * 5 * 512;
  real* __restrict__ dst = grid + (size_t)q * n;
  for (int c = threadIdx.x; c < 4096; c += blockDim.x) {
    const int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    const int p = (i >> 3) + 2 * (j >> 3) + 4 * (k >> 3);
    const real v = __ldg(src + ((size_t)p * 5 + q) * 512 + (k & 7) * 64 + (j & 7) * 8 + (i & 7));
    dst[((size_t)(gz * 16 + k) * ny + (gy * 16 + j)) * nx + (gx * 16 + i)] = v;
  }
}

// The scatter fused with the CFL reduction of the state it writes (Eq. 26): one CTA per patch group,
// each thread moves all five components of its cells, converts them (cons2prim) and keeps the
// running max of U_max; the copy is memory bound and the conversion ALU bound, so they overlap.
__global__ void __launch_bounds__(256) grid_scatter_speed_kernel(const real* __restrict__ cons_out,
                                                                 real* __restrict__ grid, int nx, int ny, int nz,
                                                                 real rtol, int max_iter,
                                                                 real* __restrict__ umax_out) {
  const int px = nx / 16, py = ny / 16;
  const int pg = blockIdx.x;
  const int gx = pg % px, gy = (pg / px) % py, gz = pg / (px * py);
  const size_t n = (size_t)nx * ny * nz;
  const real* __restrict__ src = cons_out + (size_t)pg * 8 * 5 * 512;
  real umax = real(0.0);
  for (int c = threadIdx.x; c < 4096; c += 256) {          // 4096 = 16 x 256: every lane of every warp works
    const int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    const int p = (i >> 3) + 2 * (j >> 3) + 4 * (k >> 3);
    const size_t so = (size_t)p * 5 * 512 + (k & 7) * 64 + (j & 7) * 8 + (i & 7);
    const size_t go = ((size_t)(gz * 16 + k) * ny + (gy * 16 + j)) * nx + (gx * 16 + i);
    real U[1][5], W[1][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      U[0][q] = __ldg(src + so + (size_t)q * 512);
      grid[(size_t)q * n + go] = U[0][q];
    }
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
    umax = fmax(umax, umax_of_prim(W[0], aux[0]));
  }
  umax = warp_max(umax);
  if ((threadIdx.x & 31) == 0) atomic_max_nonneg(umax_out, umax);
}
// Ghost-zone fill straight from the patch layout the fluid step wrote (no uniform grid in between) fused
// with the CFL reduction of that state: one CTA per destination patch group.  Loop A copies the
// (16+2g)^3 tile cells of all five components from the source patches (boundary mapping of the three
// tile axes in shared-memory tables, as in grid_gather_kernel); loop B converts the group's own 16^3
// cells (cons2prim) and keeps the running max of U_max (Eq. 26).
template <int G>
__global__ void __launch_bounds__(256) patch_gather_speed_kernel(const real* __restrict__ patches,
                                                                 real* __restrict__ cons_in, int nx, int ny,
                                                                 int nz, GridBC b,
                                                                 const unsigned char* __restrict__ mask,
                                                                 real rtol, int max_iter,
                                                                 real* __restrict__ umax_out) {
  constexpr int nxt = 16 + 2 * G, nrow = nxt * nxt, t3 = nrow * nxt;
  __shared__ int ax[nxt], ay[nxt], mx[nxt], my[nxt];
  __shared__ long long az[nxt];               // -1 - offset for a plane below z = 0 of an inflow boundary
  const int px = nx / 16, py = ny / 16;
  const int pg = blockIdx.x;
  const int gx = pg % px, gy = (pg / px) % py, gz = pg / (px * py);
  if (threadIdx.x < nxt) {
    const int t = threadIdx.x;
    const int X = map_index(gx * 16 + t - G, nx, b.bc[0], b.bc[1]);
    const int Y = map_index(gy * 16 + t - G, ny, b.bc[2], b.bc[3]);
    const int kk = gz * 16 + t - G;
    const int Z = map_index(kk, nz, b.bc[4], b.bc[5]);
    ax[t] = (X >> 4) * 20480 + ((X >> 3) & 1) * 2560 + (X & 7);
    ay[t] = (Y >> 4) * px * 20480 + ((Y >> 3) & 1) * 2 * 2560 + (Y & 7) * 8;
    mx[t] = X;
    my[t] = Y * nx;
    const long long off = (long long)(Z >> 4) * px * py * 20480 + ((Z >> 3) & 1) * 4 * 2560 + (Z & 7) * 64;
    az[t] = (b.has_inflow && kk < 0) ? -1 - off : off;
  }
  __syncthreads();
  real* __restrict__ dst = cons_in + (size_t)pg * 5 * t3;
  for (int c0 = threadIdx.x; c0 < t3; c0 += 2 * 256) {     // loop A: two cells (ten loads) in flight
    real v[2][5];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int c = c0 + u * 256;
      if (c < t3) {
        const int k = c / nrow, r = c - k * nrow, j = r / nxt, i = r - j * nxt;
        long long z = az[k];
        bool inflow = false;
        if (z < 0) {
          z = -1 - z;
          inflow = mask[my[j] + mx[i]] != 0;
        }
        const real* __restrict__ sp = patches + z + ay[j] + ax[i];
#pragma unroll
        for (int q = 0; q < 5; ++q) v[u][q] = inflow ? b.inflow[q] : __ldg(sp + q * 512);
      }
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int c = c0 + u * 256;
      if (c < t3) {
#pragma unroll
        for (int q = 0; q < 5; ++q) dst[(size_t)q * t3 + c] = v[u][q];
      }
    }
  }
  // loop B: S_max of the group's own cells (every lane of every warp works: 4096 = 16 x 256)
  const real* __restrict__ own = patches + (size_t)pg * 8 * 5 * 512;
  real umax = real(0.0);
  for (int c = threadIdx.x; c < 4096; c += 256) {
    const size_t so = (size_t)(c >> 9) * 5 * 512 + (c & 511);
    real U[1][5], W[1][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[0][q] = __ldg(own + so + (size_t)q * 512);
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
    umax = fmax(umax, umax_of_prim(W[0], aux[0]));
  }
  umax = warp_max(umax);
  if ((threadIdx.x & 31) == 0) atomic_max_nonneg(umax_out, umax);
}

// srhd_grid_step_cfl, kernel 0: own_uniform[pg] = 1 if the 8 patches of group pg (20480 contiguous values) hold ONE
// state bit for bit -- a single coalesced pass over the state with 16-byte loads, dropped at the first 4 KB that
// show a difference.  The pre-pass below then knows without reading any ghost cell that a tile is uniform
// whenever the group and its 26 neighbours (after the boundary mapping) all carry this flag with the same state.
__global__ void __launch_bounds__(256) patch_own_uniform_kernel(const real* __restrict__ patches,
                                                               unsigned char* __restrict__ own_uniform) {
  const int pg = blockIdx.x, tid = threadIdx.x;
  const real* __restrict__ own = patches + (size_t)pg * 20480;
  const real2* __restrict__ o2 = reinterpret_cast<const real2*>(own);
  rbits ref[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) ref[q] = real_bits(__ldg(own + q * 512));
  auto differs = [&](int w, real2 v) {                       // w: index of the pair; component = (w / 256) % 5
    const int q = (w >> 8) % 5;
    const rbits r = (q == 0) ? ref[0] : (q == 1) ? ref[1] : (q == 2) ? ref[2] : (q == 3) ? ref[3] : ref[4];
    return (real_bits(v.x) != r) || (real_bits(v.y) != r);
  };
  bool uniform = true;
  // pairs tid + 256 * (0, 1, 2, 3, 4): one of each component of patch 0
  {
    bool diff = false;
#pragma unroll
    for (int u = 0; u < 5; ++u) diff = diff || differs(tid + 256 * u, __ldg(o2 + tid + 256 * u));
    if (__syncthreads_or(diff ? 1 : 0)) uniform = false;
  }
  for (int base = 5 * 256; uniform && base < 10240; base += 8 * 256) {   // 10240 pairs in all; block-uniform trip count
    real2 v[8];
    bool diff = false;
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldg(o2 + min(base + u * 256 + tid, 10239));
#pragma unroll
    for (int u = 0; u < 8; ++u) diff = diff || differs(min(base + u * 256 + tid, 10239), v[u]);
    if (__syncthreads_or(diff ? 1 : 0)) uniform = false;
  }
  if (tid == 0) own_uniform[pg] = uniform ? 1 : 0;
}

// One whole step of a uniform grid kept in the patch layout, first kernel (srhd_grid_step_cfl): patch_gather_speed_kernel
// with the uniform-tile test of srhd_uniform.cuh in front of it.  Phase 1 reads the (16+2g)^3 tile cells of the
// group from the source patches WITHOUT writing them and compares them, as bit patterns, with the group's first
// cell (it stops at the first chunk that shows a difference).  A uniform group is finished here: its 8 patches
// of the NEW state are the old ones (srhd_uniform.cuh), written straight to patches_out, its counters and its
// U_max come from one conversion, handled[pg] = 1 -- the state of such a group crosses HBM once in and once out
// and no tile is ever materialised.  Any other group gets its tile and the U_max of its 4096 cells exactly as
// patch_gather_speed_kernel does it, and handled[pg] = 0 leaves it to fluid_step_kernel.
template <int G, int RS>
__global__ void __launch_bounds__(256, 4) patch_prepass_kernel(const real* __restrict__ patches,
                                                            real* __restrict__ patches_out,
                                                            real* __restrict__ cons_in,
                                                            real* __restrict__ flux_out, int nx, int ny, int nz,
                                                            GridBC b, const unsigned char* __restrict__ mask,
                                                            real rtol, int max_iter, real* __restrict__ umax_out,
                                                            srhd_stats* __restrict__ stats,
                                                            unsigned char* __restrict__ handled,
                                                            const unsigned char* __restrict__ own_uniform) {
  constexpr int nxt = 16 + 2 * G, nrow = nxt * nxt, t3 = nrow * nxt;
  __shared__ int ax[nxt], ay[nxt], mx[nxt], my[nxt];
  __shared__ long long az[nxt];               // -1 - offset for a plane below z = 0 of an inflow boundary
  const int px = nx / 16, py = ny / 16, pz = nz / 16;
  const int pg = blockIdx.x, tid = threadIdx.x;
  const int gx = pg % px, gy = (pg / px) % py, gz = pg / (px * py);
  if (tid < nxt) {
    const int t = tid;
    const int X = map_index(gx * 16 + t - G, nx, b.bc[0], b.bc[1]);
    const int Y = map_index(gy * 16 + t - G, ny, b.bc[2], b.bc[3]);
    const int kk = gz * 16 + t - G;
    const int Z = map_index(kk, nz, b.bc[4], b.bc[5]);
    ax[t] = (X >> 4) * 20480 + ((X >> 3) & 1) * 2560 + (X & 7);
    ay[t] = (Y >> 4) * px * 20480 + ((Y >> 3) & 1) * 2 * 2560 + (Y & 7) * 8;
    mx[t] = X;
    my[t] = Y * nx;
    const long long off = (long long)(Z >> 4) * px * py * 20480 + ((Z >> 3) & 1) * 4 * 2560 + (Z & 7) * 64;
    az[t] = (b.has_inflow && kk < 0) ? -1 - off : off;
  }
  if (tid == 0) handled[pg] = 0;
  __syncthreads();
  const real* __restrict__ own = patches + (size_t)pg * 8 * 5 * 512;
  // the five doubles of tile cell c as the gather would write them
  auto tile_cell = [&](int c, real v[5]) {
    const int k = c / nrow, r = c - k * nrow, j = r / nxt, i = r - j * nxt;
    long long z = az[k];
    bool inflow = false;
    if (z < 0) {
      z = -1 - z;
      inflow = mask[my[j] + mx[i]] != 0;
    }
    const real* __restrict__ sp = patches + z + ay[j] + ax[i];
#pragma unroll
    for (int q = 0; q < 5; ++q) v[q] = inflow ? b.inflow[q] : __ldg(sp + q * 512);
  };
  // ---- phase 1: is the tile one state?
  real U0[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) U0[q] = __ldg(own + q * 512);
  // Shortcut that needs no ghost cell: the group and its 26 neighbours (periodic: wrapped; outflow: the group
  // itself stands in for the missing neighbour, whose ghost cells copy this group's edge cells) each hold one state
  // (patch_own_uniform_kernel) and it is the same state everywhere.  Fixed-inflow ghost cells below z = 0 hold
  // another state, so the bottom layer of groups always takes the full test.
  bool by_flags = false;
  {
    bool bad = false;
    if (tid < 27) {
      const int dx = tid % 3 - 1, dy = (tid / 3) % 3 - 1, dz = tid / 9 - 1;
      int X = gx + dx, Y = gy + dy, Z = gz + dz;
      X = (X < 0) ? (b.bc[0] == SRHD_BC_PERIODIC ? px - 1 : gx) : (X >= px) ? (b.bc[1] == SRHD_BC_PERIODIC ? 0 : gx) : X;
      Y = (Y < 0) ? (b.bc[2] == SRHD_BC_PERIODIC ? py - 1 : gy) : (Y >= py) ? (b.bc[3] == SRHD_BC_PERIODIC ? 0 : gy) : Y;
      Z = (Z < 0) ? (b.bc[4] == SRHD_BC_PERIODIC ? pz - 1 : gz) : (Z >= pz) ? (b.bc[5] == SRHD_BC_PERIODIC ? 0 : gz) : Z;
      const int ng = X + px * (Y + py * Z);
      bad = own_uniform[ng] == 0;
      const real* __restrict__ nb = patches + (size_t)ng * 20480;
#pragma unroll
      for (int q = 0; q < 5; ++q) bad = bad || (real_bits(__ldg(nb + q * 512)) != real_bits(U0[q]));
    }
    by_flags = !__syncthreads_or(bad ? 1 : 0) && !(b.has_inflow && gz == 0);
  }
  // the first 256 cells settle almost every group that is not uniform; then four cells (twenty loads) per thread
  // in flight between two block-wide votes
  bool uniform = true;
  if (!by_flags) {
    real v[5];
    tile_cell(tid, v);
    bool diff = false;
#pragma unroll
    for (int q = 0; q < 5; ++q) diff = diff || (real_bits(v[q]) != real_bits(U0[q]));
    if (__syncthreads_or(diff ? 1 : 0)) uniform = false;
  }
  for (int base = 256; !by_flags && uniform && base < t3; base += 4 * 256) {   // block-uniform trip count: every thread votes
    real v[4][5];
    bool diff = false;
#pragma unroll
    for (int u = 0; u < 4; ++u) tile_cell(min(base + u * 256 + tid, t3 - 1), v[u]);
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int q = 0; q < 5; ++q) diff = diff || (real_bits(v[u][q]) != real_bits(U0[q]));
    if (__syncthreads_or(diff ? 1 : 0)) uniform = false;
  }
  if (uniform) {
    // the stores go out first (harmless if the group is marched after all), one warp evaluates the state meanwhile
    uniform_write_state(patches_out + (size_t)pg * 8 * 5 * 512, U0, tid, 256);
    UniformResult r;
    if (uniform_eval_by_warp0<RS>(U0, rtol, max_iter, r)) {   // block-uniform verdict
      if (flux_out) uniform_write_flux(flux_out + (size_t)pg * 8 * 6 * 5 * 64, r, tid, 256);
      if (tid == 0) {
        handled[pg] = 1;
        uniform_count(stats, t3, r);
        atomic_max_nonneg(umax_out, r.umax);
      }
      return;
    }
  }
  // ---- phase 2 (any other group): the tile and U_max of the group's own cells, as patch_gather_speed_kernel
  real* __restrict__ dst = cons_in + (size_t)pg * 5 * t3;
  for (int c0 = tid; c0 < t3; c0 += 2 * 256) {
    real v[2][5];
#pragma unroll
    for (int u = 0; u < 2; ++u)
      if (c0 + u * 256 < t3) tile_cell(c0 + u * 256, v[u]);
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int c = c0 + u * 256;
      if (c < t3) {
#pragma unroll
        for (int q = 0; q < 5; ++q) dst[(size_t)q * t3 + c] = v[u][q];
      }
    }
  }
  real umax = real(0.0);
  for (int c = tid; c < 4096; c += 256) {
    const size_t so = (size_t)(c >> 9) * 5 * 512 + (c & 511);
    real U[1][5], W[1][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[0][q] = __ldg(own + so + (size_t)q * 512);
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
    umax = fmax(umax, umax_of_prim(W[0], aux[0]));
  }
  umax = warp_max(umax);
  if ((tid & 31) == 0) atomic_max_nonneg(umax_out, umax);
}

__global__ void smax_finish_kernel2(real* v) { *v = smax_of_umax(*v); }   // Eq. 27 once, after the max

}  // namespace srhd

using namespace srhd;

static int check_extents(int nx, int ny, int nz) {
  if (nx <= 0 || ny <= 0 || nz <= 0 || nx % 16 || ny % 16 || nz % 16) return SRHD_ERR_BAD_SIZE;
  // the gather kernels keep the in-plane patch offsets (up to (ny/16)(nx/16) * 20480 values) in 32-bit integers:
  // a very flat grid (e.g. 8192 x 4096 x 16) would overflow them, so it is refused rather than read out of bounds
  if ((long long)(nx / 16) * (ny / 16) * 20480 > 2147483647LL) return SRHD_ERR_BAD_SIZE;
  if ((long long)(nx / 16) * (ny / 16) * (nz / 16) > 2147483647LL / 8) return SRHD_ERR_BAD_SIZE;   // npg * 8 patches in an int
  return SRHD_OK;
}

extern "C" int srhd_grid_gather(const real* grid, real* cons_in, int nx, int ny, int nz, int ghost,
                                const int* bc, const unsigned char* inflow_mask, const double* inflow_cons,
                                void* stream) {
  if (!grid || !cons_in || !bc) return SRHD_ERR_NULL_POINTER;
  if (ghost < 2 || ghost > 4) return SRHD_ERR_BAD_PARAMS;
  const int ce = check_extents(nx, ny, nz);
  if (ce) return ce;
  GridBC b;
  for (int i = 0; i < 6; ++i) {
    if (bc[i] != SRHD_BC_PERIODIC && bc[i] != SRHD_BC_OUTFLOW) return SRHD_ERR_BAD_PARAMS;
    b.bc[i] = bc[i];
  }
  b.has_inflow = (inflow_mask != nullptr);
  if (b.has_inflow && !inflow_cons) return SRHD_ERR_NULL_POINTER;
  for (int q = 0; q < 5; ++q) b.inflow[q] = b.has_inflow ? inflow_cons[q] : real(0.0);
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  if (ghost == 2)
    grid_gather_kernel<2><<<dim3(npg, 5), 256, 0, static_cast<cudaStream_t>(stream)>>>(grid, cons_in, nx, ny, nz,
                                                                                            b, inflow_mask);
  else if (ghost == 4)
    grid_gather_kernel<4><<<dim3(npg, 5), 256, 0, static_cast<cudaStream_t>(stream)>>>(grid, cons_in, nx, ny, nz,
                                                                                            b, inflow_mask);
  else
    grid_gather_kernel<3><<<dim3(npg, 5), 256, 0, static_cast<cudaStream_t>(stream)>>>(grid, cons_in, nx, ny, nz,
                                                                                            b, inflow_mask);
  return (int)cudaGetLastError();
}

extern "C" int srhd_grid_scatter(const real* cons_out, real* grid, int nx, int ny, int nz, void* stream) {
  if (!cons_out || !grid) return SRHD_ERR_NULL_POINTER;
  const int ce = check_extents(nx, ny, nz);
  if (ce) return ce;
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  grid_scatter_kernel<<<dim3(npg, 5), 256, 0, static_cast<cudaStream_t>(stream)>>>(cons_out, grid, nx, ny, nz);
  return (int)cudaGetLastError();
}

extern "C" int srhd_grid_scatter_speed(const real* cons_out, real* grid, int nx, int ny, int nz,
                                       const srhd_params* params, real* d_max_speed, void* stream) {
  if (!cons_out || !grid || !d_max_speed) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  const int ce = check_extents(nx, ny, nz);
  if (ce) return ce;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const cudaError_t e = cudaMemsetAsync(d_max_speed, 0, sizeof(real), st);
  if (e != cudaSuccess) return (int)e;
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  grid_scatter_speed_kernel<<<npg, 256, 0, st>>>(cons_out, grid, nx, ny, nz, newton_stop_rtol(params->newton_rtol),
                                                 params->newton_max_iter, d_max_speed);
  smax_finish_kernel2<<<1, 1, 0, st>>>(d_max_speed);
  return (int)cudaGetLastError();
}

extern "C" int srhd_patch_gather_speed(const real* patches, real* cons_in, int nx, int ny, int nz,
                                       const int* bc, const unsigned char* inflow_mask, const double* inflow_cons,
                                       const srhd_params* params, real* d_max_speed, void* stream) {
  if (!patches || !cons_in || !bc || !d_max_speed) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  const int ce = check_extents(nx, ny, nz);
  if (ce) return ce;
  GridBC b;
  for (int i = 0; i < 6; ++i) {
    if (bc[i] != SRHD_BC_PERIODIC && bc[i] != SRHD_BC_OUTFLOW) return SRHD_ERR_BAD_PARAMS;
    b.bc[i] = bc[i];
  }
  b.has_inflow = (inflow_mask != nullptr);
  if (b.has_inflow && !inflow_cons) return SRHD_ERR_NULL_POINTER;
  for (int q = 0; q < 5; ++q) b.inflow[q] = b.has_inflow ? inflow_cons[q] : real(0.0);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const cudaError_t e = cudaMemsetAsync(d_max_speed, 0, sizeof(real), st);
  if (e != cudaSuccess) return (int)e;
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  const real rtol = newton_stop_rtol(params->newton_rtol);
  if (params->ghost == 2)
    patch_gather_speed_kernel<2><<<npg, 256, 0, st>>>(patches, cons_in, nx, ny, nz, b, inflow_mask, rtol,
                                                      params->newton_max_iter, d_max_speed);
  else if (params->ghost == 4)
    patch_gather_speed_kernel<4><<<npg, 256, 0, st>>>(patches, cons_in, nx, ny, nz, b, inflow_mask, rtol,
                                                      params->newton_max_iter, d_max_speed);
  else
    patch_gather_speed_kernel<3><<<npg, 256, 0, st>>>(patches, cons_in, nx, ny, nz, b, inflow_mask, rtol,
                                                      params->newton_max_iter, d_max_speed);
  smax_finish_kernel2<<<1, 1, 0, st>>>(d_max_speed);
  return (int)cudaGetLastError();
}

template <int G, int RS>
static void launch_prepass(const real* patches, real* patches_out, real* cons_in, real* flux_out, int nx,
                           int ny, int nz, const GridBC& b, const unsigned char* mask, real rtol, int max_iter,
                           real* umax_out, srhd_stats* stats, unsigned char* handled, cudaStream_t st) {
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  unsigned char* own_uniform = handled + npg;                 // second half of the scratch allocation
  patch_own_uniform_kernel<<<npg, 256, 0, st>>>(patches, own_uniform);
  patch_prepass_kernel<G, RS><<<npg, 256, 0, st>>>(patches, patches_out, cons_in, flux_out, nx, ny, nz, b, mask, rtol,
                                                   max_iter, umax_out, stats, handled, own_uniform);
}

extern "C" int srhd_grid_step_cfl(const real* patches_in, real* patches_out, real* cons_in, real* flux_out,
                                  int nx, int ny, int nz, const int* bc, const unsigned char* inflow_mask,
                                  const double* inflow_cons, double cfl, double dh, double min_speed,
                                  const srhd_params* params, srhd_stats* stats, real* d_max_speed, void* stream) {
  if (!patches_in || !patches_out || !cons_in || !bc || !d_max_speed) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  const int ce = check_extents(nx, ny, nz);
  if (ce) return ce;
  if (!(cfl > real(0.0)) || !std::isfinite(cfl) || !(min_speed >= real(0.0)) || !(dh > real(0.0)) || !std::isfinite(dh))
    return SRHD_ERR_BAD_STEP;
  // patches_in / patches_out are read and written as pairs of srhd_real (own-uniform scan, uniform-tile stores);
  // cons_in is the target of the ghost-zone fill and the source of the march's 16-byte TMA bulk copies
  if ((reinterpret_cast<uintptr_t>(patches_in) & (sizeof(real2) - 1)) ||
      (reinterpret_cast<uintptr_t>(patches_out) & (sizeof(real2) - 1)) || (reinterpret_cast<uintptr_t>(cons_in) & 15u))
    return SRHD_ERR_BAD_ALIGN;
  const int npg = (nx / 16) * (ny / 16) * (nz / 16);
  {
    // the three state buffers must be pairwise disjoint (the pre-pass reads patches_in while it writes the other two)
    const int nxt = 16 + 2 * params->ghost;
    const size_t patch_bytes = (size_t)npg * 8 * 5 * 512 * sizeof(real);
    const size_t tile_bytes = (size_t)npg * 5 * nxt * nxt * nxt * sizeof(real);
    const uintptr_t a = reinterpret_cast<uintptr_t>(patches_in), b = reinterpret_cast<uintptr_t>(patches_out),
                    c = reinterpret_cast<uintptr_t>(cons_in);
    if ((a < b + patch_bytes && b < a + patch_bytes) || (a < c + tile_bytes && c < a + patch_bytes) ||
        (b < c + tile_bytes && c < b + patch_bytes))
      return SRHD_ERR_ALIAS;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (params->integrator != SRHD_INTEGRATOR_MHM) {           // no pre-pass for the VL kernels: the two plain calls
    const int e = srhd_patch_gather_speed(patches_in, cons_in, nx, ny, nz, bc, inflow_mask, inflow_cons, params,
                                          d_max_speed, stream);
    if (e) return e;
    return srhd_fluid_step_cfl(cons_in, patches_out, flux_out, npg, cfl, dh, d_max_speed, min_speed, params, stats,
                               stream);
  }
  GridBC b;
  for (int i = 0; i < 6; ++i) {
    if (bc[i] != SRHD_BC_PERIODIC && bc[i] != SRHD_BC_OUTFLOW) return SRHD_ERR_BAD_PARAMS;
    b.bc[i] = bc[i];
  }
  b.has_inflow = (inflow_mask != nullptr);
  if (b.has_inflow && !inflow_cons) return SRHD_ERR_NULL_POINTER;
  for (int q = 0; q < 5; ++q) b.inflow[q] = b.has_inflow ? inflow_cons[q] : real(0.0);
  cudaError_t e = cudaMemsetAsync(d_max_speed, 0, sizeof(real), st);
  if (e != cudaSuccess) return (int)e;
  if (stats) {
    e = cudaMemsetAsync(stats, 0, sizeof(srhd_stats), st);
    if (e != cudaSuccess) return (int)e;
  }
  unsigned char* handled = nullptr;
  e = cudaMallocAsync(reinterpret_cast<void**>(&handled), 2 * (size_t)npg, st);   // handled[npg] + own_uniform[npg]
  if (e != cudaSuccess) return (int)e;
  const real rtol = newton_stop_rtol(params->newton_rtol);
  const int mi = params->newton_max_iter;
  if (params->recon == SRHD_RECON_PLM) {
    if (params->riemann == SRHD_RIEMANN_HLLE)
      launch_prepass<2, 0>(patches_in, patches_out, cons_in, flux_out, nx, ny, nz, b, inflow_mask, rtol, mi, d_max_speed, stats, handled, st);
    else
      launch_prepass<2, 1>(patches_in, patches_out, cons_in, flux_out, nx, ny, nz, b, inflow_mask, rtol, mi, d_max_speed, stats, handled, st);
  } else {
    if (params->riemann == SRHD_RIEMANN_HLLE)
      launch_prepass<3, 0>(patches_in, patches_out, cons_in, flux_out, nx, ny, nz, b, inflow_mask, rtol, mi, d_max_speed, stats, handled, st);
    else
      launch_prepass<3, 1>(patches_in, patches_out, cons_in, flux_out, nx, ny, nz, b, inflow_mask, rtol, mi, d_max_speed, stats, handled, st);
  }
  smax_finish_kernel2<<<1, 1, 0, st>>>(d_max_speed);
  e = cudaGetLastError();
  int rc = (int)e;
  if (e == cudaSuccess)
    rc = fluid_march(cons_in, patches_out, flux_out, npg, real(1.0), dh, params, stats, st, d_max_speed, cfl, min_speed, handled);
  const cudaError_t e2 = cudaFreeAsync(handled, st);
  return rc ? rc : (int)e2;
}

extern "C" void srhd_default_params(srhd_params* p, int recon, int riemann) {
  if (!p) return;
  p->recon = recon;
  p->riemann = riemann;
  p->minmod_coeff = real(1.5);
  p->max_retry = 8;
  p->newton_rtol = SRHD_IS_F32 ? 1e-6 : 1e-15;   // a few eps_machine of the build's precision
  p->newton_max_iter = 20;
  p->ghost = (recon == SRHD_RECON_PLM) ? 2 : 3;
  p->integrator = SRHD_INTEGRATOR_MHM;
}

extern "C" const char* srhd_error_string(int code) {
  switch (code) {
    case SRHD_OK: return "ok";
    case SRHD_ERR_NULL_POINTER: return "null pointer argument";
    case SRHD_ERR_BAD_PARAMS: return "bad srhd_params (recon / riemann / ghost / coefficients)";
    case SRHD_ERR_BAD_SIZE: return "bad size (stride < n, negative count, extent not a multiple of 16)";
    case SRHD_ERR_BAD_STEP: return "dt and dh must be positive and finite";
    case SRHD_ERR_ALIAS: return "state buffers overlap (cons_in / cons_out; patches_in / patches_out / cons_in)";
    case SRHD_ERR_BAD_ALIGN: return "cons_in must be 16-byte aligned; cons_out, patches_in and patches_out aligned to two srhd_real";
    case SRHD_ERR_TOO_LARGE: return "srhd_fluid_step_noalloc: npg exceeds SRHD_NOALLOC_MAX_NPG (65536); split the batch";
    default: break;
  }
  if (code > 0) return cudaGetErrorString(static_cast<cudaError_t>(code));
  return "unknown srhd error code";
}

extern "C" int srhd_build_is_exact(void) { return SRHD_EXACT; }

#define SRHD_STR2(x) #x
#define SRHD_STR(x) SRHD_STR2(x)
extern "C" const char* srhd_build_variant(void) {
  return "eos="
#if SRHD_EOS == 0
         "taub-mathews"
#else
         "gamma-" SRHD_STR(SRHD_GAMMA_NUM) "/" SRHD_STR(SRHD_GAMMA_DEN)
#endif
         " energy="
#if SRHD_SCHEME == 0
         "reduced"
#else
         "total"
#endif
         " precision="
#if SRHD_IS_F32
         "f32"
#else
         "f64"
#endif
         " arithmetic="
#if SRHD_EXACT
         "exact"
#elif SRHD_GENERIC
         "generic"
#else
         "production"
#endif
      ;
}

// SRHD_F64_ONLY_BEGIN (measurement helpers: double precision in every build)
// ---- fp64 ALU roof: register-only DFMA loop, 8 independent chains per thread, 8 CTAs x 256 threads
// per SM (full occupancy).  Used by bench.py for the MEASURED denominator of the "alu" roofline.
namespace srhd {
__global__ void __launch_bounds__(256) fp64_peak_kernel(double* __restrict__ sink, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = 1.0 + 1e-3 * (threadIdx.x + k);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
    }
  }
  double acc = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) acc += x[k];
  if (acc == 12345.678) sink[0] = acc;    // never true: keeps the chains alive without a store
}
}  // namespace srhd

// ---- issue-port probe: the same DFMA loop with NI independent FFMA interleaved per 8 DFMA.  If an fp64
// warp instruction held only the fp64 pipe, up to 8 FFMA per 8 DFMA would issue in its shadow for free; the
// measured DFMA rate instead falls as 16/(16 + NI): every fp64 warp instruction occupies its scheduler's issue
// port for two cycles and any other instruction for one, with no overlap.
namespace srhd {
template <int NI>
__global__ void __launch_bounds__(256) issue_probe_kernel(double* __restrict__ sink, int iters, double a, double b,
                                                          float fa, float fb) {
  double x[8];
  float y[16];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = 1.0 + 1e-3 * (threadIdx.x + k);
#pragma unroll
  for (int k = 0; k < 16; ++k) y[k] = 1.0f + 1e-3f * (threadIdx.x + k);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
#pragma unroll
      for (int k = 0; k < NI; ++k) y[k] = fmaf(y[k], fa, fb);
    }
  }
  double acc = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) acc += x[k];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc += y[k];
  if (acc == 12345.678) sink[0] = acc;    // never true
}
}  // namespace srhd

extern "C" int srhd_issue_probe(double* d_sink, int iters, int ffma_per_8_dfma, unsigned long long* dfma_flops,
                                void* stream) {
  if (!d_sink) return SRHD_ERR_NULL_POINTER;
  if (iters < 1) return SRHD_ERR_BAD_SIZE;
  const int grid = srhd::num_sms() * 8, block = 256;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (ffma_per_8_dfma) {
    case 0: srhd::issue_probe_kernel<0><<<grid, block, 0, st>>>(d_sink, iters, 0.999999, 1e-6, 0.99999f, 1e-6f); break;
    case 4: srhd::issue_probe_kernel<4><<<grid, block, 0, st>>>(d_sink, iters, 0.999999, 1e-6, 0.99999f, 1e-6f); break;
    case 8: srhd::issue_probe_kernel<8><<<grid, block, 0, st>>>(d_sink, iters, 0.999999, 1e-6, 0.99999f, 1e-6f); break;
    case 12: srhd::issue_probe_kernel<12><<<grid, block, 0, st>>>(d_sink, iters, 0.999999, 1e-6, 0.99999f, 1e-6f); break;
    case 16: srhd::issue_probe_kernel<16><<<grid, block, 0, st>>>(d_sink, iters, 0.999999, 1e-6, 0.99999f, 1e-6f); break;
    default: return SRHD_ERR_BAD_PARAMS;
  }
  if (dfma_flops) *dfma_flops = 2ull * 32ull * (unsigned long long)iters * (unsigned long long)grid * block;
  return (int)cudaGetLastError();
}

extern "C" int srhd_fp64_peak_probe(double* d_sink, int iters, unsigned long long* flops, void* stream) {
  if (!d_sink) return SRHD_ERR_NULL_POINTER;
  if (iters < 1) return SRHD_ERR_BAD_SIZE;
  const int grid = srhd::num_sms() * 8, block = 256;
  srhd::fp64_peak_kernel<<<grid, block, 0, static_cast<cudaStream_t>(stream)>>>(d_sink, iters, 0.999999, 1e-6);
  if (flops) *flops = 2ull * 32ull * (unsigned long long)iters * (unsigned long long)grid * block;
  return (int)cudaGetLastError();
}

// SRHD_F64_ONLY_END
