// srhd_fluid.cu -- srhd_fluid_step: one fused kernel per batch of patch groups.
//
// One CTA advances one patch group (16^3 interior cells + ghost zones) and marches through
// its z planes, keeping all three directional sweeps on chip.  Two barrier intervals per plane s:
//   interval Y  (plane kh = s - 2g + 1)  Hancock stage: one LANE per (cell, direction) -- 10 cells x
//               3 directions per warp -- does the PLM/PPM edge values of the five primitives along its
//               direction, prim2cons + physical flux of both edge states; the three flux differences
//               of a cell are combined with warp shuffles in the fixed order (x + y) + z, and every
//               lane stores its two evolved edge states to shared memory (S3-S5);
//   interval X  a CTA-wide work queue of 32-item chunks: (i) one Riemann problem per face of plane kh
//               (z faces below it: 16x16, bound to the thread that owns the column and therefore
//               updates cell (i,j,kh-1), checks Eq. 30 and stores it; x: 17x16, y: 16x17): cons2prim
//               of both sides as two interleaved Newton chains per lane, HLLE/HLLC; (ii) cons2prim of
//               the NEXT tile plane s+1 (staged by TMA bulk copies, cp.async.bulk + mbarrier, one plane
//               ahead) into the ring of 2g-1 primitive planes; interior cells feed the CFL reduction
//               (Eq. 26) and the Eq. 30 counter.  Mixing the two kinds of chunk fills the ragged tail of
//               the face list.
// If any face state or updated cell of the group fails Eq. 30 the CTA repeats the march with
// beta <- 0.75 beta, finally with beta = 0.  Each cell's state crosses HBM once on the way
// in (plus ghost layers) and once on the way out; the update re-reads its own cell through L2.
#include <mutex>

#include "srhd_common.cuh"
#include "srhd_uniform.cuh"

namespace srhd {

constexpr int kFluidThreads = 512;   // 16 warps, <= 128 registers per thread, one CTA per SM (384 ... 768
                                     // threads were measured in round 1: 512 is best)

// ---- TMA bulk copy + mbarrier (PTX; SASS: UBLKCP / SYNCS) -------------------------------------
SRHD_DEV uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
SRHD_DEV void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
SRHD_DEV void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
SRHD_DEV bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
SRHD_DEV void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
SRHD_DEV void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
SRHD_DEV void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }


// ---- shared-memory plan -----------------------------------------------------------------------
template <int G>
struct Plan {
  static constexpr int NXT = 16 + 2 * G;      // tile extent
  static constexpr int PL = NXT * NXT;        // cells per tile plane
  static constexpr int T3 = PL * NXT;         // cells per tile component
  static constexpr int R = 2 * G - 1;         // primitive planes kept (z stencil of the reconstruction)
  static constexpr int XS = 16 * 18;          // x edge states: row j in 0..15, cell i in -1..16
  static constexpr int YS = 18 * 16;          // y edge states: cell j in -1..16, column i in 0..15
  static constexpr int ZS = 256;              // z edge states: interior columns
  static constexpr int NFXY = 272;            // faces per plane along x (17x16) and along y (16x17)
  // offsets in doubles
  static constexpr int oW = 0;
  static constexpr int oStg = oW + R * 5 * PL;        // conserved plane staged by TMA, one plane ahead
  static constexpr int oXSm = oStg + 5 * PL;
  static constexpr int oXSp = oXSm + 5 * XS;
  static constexpr int oYSm = oXSp + 5 * XS;
  static constexpr int oYSp = oYSm + 5 * YS;
  static constexpr int oZSm = oYSp + 5 * YS;
  static constexpr int oZSp = oZSm + 5 * ZS;          // two buffers (plane parity)
  static constexpr int oFX = oZSp + 2 * 5 * ZS;
  static constexpr int oFY = oFX + 5 * NFXY;
  static constexpr int oFZ = oFY + 5 * NFXY;          // z flux through the lower face of each column's cell
  static constexpr int oCtl = oFZ + 5 * ZS;           // control block (struct Ctl)
  static_assert(oCtl % 2 == 0, "the control block needs 8-byte alignment in every precision");
  static constexpr size_t bytes = (size_t)oCtl * sizeof(real) + 96;   // + struct Ctl
};

struct Ctl {                       // lives in shared memory
  uint64_t mbar;
  unsigned long long newton;
  rbits umax_bits;
  unsigned int face_fail, cell_fail, in_fail;
  int queue;                       // next chunk of interval X
  unsigned int abort;              // a failure was seen in this (non-final) pass: abandon it at the plane's end
  unsigned int exec_c2p, exec_riemann, exec_hancock;
  unsigned long long exec_newton;
};
static_assert(sizeof(Ctl) <= 96, "Plan<G>::bytes reserves 96 bytes for the control block");

// Hancock stage of one (cell, direction) lane: PLM/PPM edge values of the five primitives along d
// (stencil offsets o[] into the primitive ring, component stride PL), prim2cons and physical flux
// of both edge states; returns the un-evolved conserved edge states and dF = F(W+) - F(W-).
template <int G>
SRHD_DEV bool hancock_lane(const real* __restrict__ Wr, int d, const int o[2 * G - 1], real beta,
                           real beta0, real um[5], real up[5], real dF[5]) {
  using P = Plan<G>;
  real wm[5], wp[5];
  bool allflat = true;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    real a[2 * G - 1];
#pragma unroll
    for (int m = 0; m < 2 * G - 1; ++m) a[m] = Wr[o[m] + q * P::PL];
    // A constant stencil (ambient gas ahead of a blast wave or a jet) has zero slopes and edge values
    // equal to the cell value BIT FOR BIT in both schemes, so it skips the limiter arithmetic.
    bool flat = true;
#pragma unroll
    for (int m = 0; m < 2 * G - 1; ++m) flat = flat && (a[m] == a[G - 1]);
    allflat = allflat && flat;
    if (flat) {
      wm[q] = a[G - 1];
      wp[q] = a[G - 1];
    } else if (G == 2) {
      recon_plm(a, beta, wm[q], wp[q]);
    } else {
      recon_ppm(a, beta, beta0, wm[q], wp[q]);
    }
  }
  real Fm[5], Fp[5];
  Aux am, ap;
  if (__all_sync(0xffffffffu, allflat)) {
    // every lane's two edge states are the same state: one conversion, and F(W+) - F(W-) = +0 exactly
    prim2cons_aux(wm, um, am);
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      up[q] = um[q];
      dF[q] = real(0.0);
    }
    return true;
  }
  prim2cons_aux(wm, um, am);      // two independent chains: the compiler interleaves them
  prim2cons_aux(wp, up, ap);
  phys_flux_rt(d, wm, um, am, Fm);
  phys_flux_rt(d, wp, up, ap, Fp);
#pragma unroll
  for (int q = 0; q < 5; ++q) dF[q] = Fp[q] - Fm[q];
  return false;
}

// Uniform tiles (undisturbed ambient gas ahead of a blast wave or a jet; srhd_uniform.cuh): this pre-pass (one
// CTA per patch group, launched ahead of fluid_step_kernel on the same stream) streams a tile once from HBM
// (16-byte loads, compared as bit patterns); if every cell holds the same state it writes the 8 patches, adds
// what the march would have counted to the counters and sets handled[pg] = 1, which makes the main kernel's CTA
// return at once.  A tile that is not uniform is dropped at its first 4 KB.  It is a kernel of its own, not a
// branch of the main one: a data-dependent early exit there makes nvcc guard every warp collective of the march
// with a divergence test (BRA.DIV; measured +25 % kernel time on data without a single uniform tile).
constexpr int kScanThreads = 256;
template <int G, int RS>
__global__ void __launch_bounds__(kScanThreads) uniform_tiles_kernel(
    const real* __restrict__ cons_in, real* __restrict__ cons_out, real* __restrict__ flux_out, real dt,
    real dh, real rtol, int max_iter, srhd_stats* __restrict__ stats, const real* __restrict__ d_smax,
    real cfl, real min_speed, unsigned char* __restrict__ handled) {
  using P = Plan<G>;
  constexpr int NT = kScanThreads, T3 = P::T3;
  const int tid = threadIdx.x;
  const real* __restrict__ tile = cons_in + (size_t)blockIdx.x * 5 * T3;
  if (tid == 0) handled[blockIdx.x] = 0;
  real U0[5];
  if (!tile_scan_uniform<T3, NT>(tile, U0)) return;
  if (d_smax) dt = cfl * dh / fmax(*d_smax, min_speed);      // as the main kernel (srhd_fluid_step_cfl)
  if (!(fabs(dt / dh) <= kRealMax)) return;                   // U0 - (dt/dh) 0 = U0 needs a finite dt/dh
  uniform_write_state(cons_out + (size_t)blockIdx.x * 8 * 5 * 512, U0, tid, NT);   // (rewritten by the march if the verdict is no)
  UniformResult r;
  if (!uniform_eval_by_warp0<RS>(U0, rtol, max_iter, r)) return;      // block-uniform verdict
  if (flux_out) uniform_write_flux(flux_out + (size_t)blockIdx.x * 8 * 6 * 5 * 64, r, tid, NT);
  if (tid == 0) {
    handled[blockIdx.x] = 1;
    uniform_count(stats, T3, r);
  }
}

template <int G, int RS>
__global__ void __launch_bounds__(kFluidThreads, 1)
fluid_step_kernel(const real* __restrict__ cons_in, real* __restrict__ cons_out,
                  real* __restrict__ flux_out, real dt, real dh, real beta0, int max_retry, real rtol,
                  int max_iter, srhd_stats* __restrict__ stats, const real* __restrict__ d_smax, real cfl,
                  real min_speed, const unsigned char* __restrict__ handled) {
  using P = Plan<G>;
  constexpr int NT = kFluidThreads, NW = NT / 32;
  if (handled[blockIdx.x]) return;              // a uniform tile: uniform_tiles_kernel wrote its result
  constexpr int NXT = P::NXT, PL = P::PL, T3 = P::T3, R = P::R;
  constexpr int NP1 = (PL + 31) / 32;           // cons2prim chunks per tile plane
  constexpr int NXY = 2 * P::NFXY / 32;         // x and y face chunks per plane (544 faces = 17 x 32)
  static_assert(2 * P::NFXY % 32 == 0 && NW >= 8, "face list must be whole warps; z faces need 8 warps");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* sm = reinterpret_cast<real*>(smem_raw);
  real* Wr = sm + P::oW;
  real* Stg = sm + P::oStg;
  real* XSm = sm + P::oXSm;
  real* XSp = sm + P::oXSp;
  real* YSm = sm + P::oYSm;
  real* YSp = sm + P::oYSp;
  real* ZSm = sm + P::oZSm;
  real* ZSp = sm + P::oZSp;
  real* FX = sm + P::oFX;
  real* FY = sm + P::oFY;
  real* FZ = sm + P::oFZ;     // written and read by the thread that owns the column: no barrier needed
  Ctl* ctl = reinterpret_cast<Ctl*>(sm + P::oCtl);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const real* __restrict__ tile = cons_in + (size_t)blockIdx.x * 5 * T3;
  real* __restrict__ out = cons_out + (size_t)blockIdx.x * 8 * 5 * 512;
  real* __restrict__ fout = flux_out ? flux_out + (size_t)blockIdx.x * 8 * 6 * 5 * 64 : nullptr;
  // flux through a patch-boundary face -> flux_out[patch][face][comp][a][b] (include/srhd.h)
  auto put_flux = [&](int p, int f, int a, int b, const real F[5]) {
#pragma unroll
    for (int q = 0; q < 5; ++q) fout[(((size_t)p * 6 + f) * 5 + q) * 64 + a * 8 + b] = F[q];
  };

  if (tid == 0) {
    mbar_init(&ctl->mbar, 1);
    ctl->newton = 0ull;
    ctl->umax_bits = 0;
    ctl->face_fail = ctl->cell_fail = ctl->in_fail = 0u;
    ctl->queue = 0;
    ctl->abort = 0u;
    ctl->exec_c2p = ctl->exec_riemann = ctl->exec_hancock = 0u;
    ctl->exec_newton = 0ull;
    fence_proxy_async();
  }
  __syncthreads();

  // Hancock stage: lane -> (cell of the warp's ten, direction); lanes 30, 31 shadow lane 29
  const int hd = (lane < 30) ? lane % 3 : 2;
  const int hc = (lane < 30) ? lane / 3 : 9;
  const int hbase = 3 * hc;
  // Each thread meets the same two (cell, direction) items in every plane (chunks warp and warp + NW
  // of the 32): decode them once.  info = in-plane tile index | store offset << 9 | has-edge-array
  // << 18 | interior-column << 19
  static_assert(NW == 16, "the Hancock stage maps 32 chunks of 10 cells onto exactly two rounds of 16 warps");
  real* const hpm = (hd == 0) ? XSm : ((hd == 1) ? YSm : ZSm);
  real* const hpp = (hd == 0) ? XSp : ((hd == 1) ? YSp : ZSp);
  const int hqs = (hd == 0) ? P::XS : ((hd == 1) ? P::YS : P::ZS);
  int hinfo[2];
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    int cell = (warp + NW * r) * 10 + hc;
    if (cell > 319) cell = 319;
    int i, j;
    if (cell < 256) {
      i = cell & 15;
      j = cell >> 4;
    } else {
      const int e = cell - 256, side = e >> 4, t = e & 15;
      i = (side == 0) ? -1 : ((side == 1) ? 16 : t);
      j = (side == 2) ? -1 : ((side == 3) ? 16 : t);
    }
    const int cidx = (j + G) * NXT + (i + G);
    const int soff = (hd == 0) ? j * 18 + (i + 1) : ((hd == 1) ? (j + 1) * 16 + i : cell);
    const bool hs = (hd == 0) ? (j >= 0 && j <= 15) : ((hd == 1) ? (i >= 0 && i <= 15) : (cell < 256));
    hinfo[r] = cidx | ((hs ? soff : 0) << 9) | ((hs ? 1 : 0) << 18) | ((cell < 256 ? 1 : 0) << 19);
  }

  if (d_smax) dt = cfl * dh / fmax(*d_smax, min_speed);   // Eq. 28 formed on the device (srhd_fluid_step_cfl)
  const real hdt = dt / (real(2.0) * dh);
  const real dtdh = dt / dh;

  unsigned long long my_iters = 0;     // iterations of the algorithm's conversions (centre cells + accepted pass)
  unsigned long long ex_newton = 0;    // executed work (every pass, shortcuts taken into account)
  unsigned ex_c2p = 0, ex_riemann = 0, ex_hancock = 0;
  int phase_base = 0;                  // TMA phases completed before the current pass (mbarrier parity)
  int planes_counted = 0;              // tile planes whose cells already fed newton_iters / S_max / Eq. 30 counters
  unsigned my_in_fail = 0;
  real my_umax = real(0.0);
  real beta = beta0;
  int pass = 0;
  unsigned n_face_fail = 0, n_cell_fail = 0;

  // TMA: conserved tile plane pl -> staging buffer (thread 0 only)
  auto issue_plane = [&](int pl) {
    fence_proxy_async();
    mbar_expect_tx(&ctl->mbar, 5u * PL * (uint32_t)sizeof(real));
#pragma unroll
    for (int q = 0; q < 5; ++q)
      bulk_g2s(Stg + q * PL, tile + (size_t)q * T3 + (size_t)pl * PL, PL * (uint32_t)sizeof(real), &ctl->mbar);
  };
  // cons2prim of 32 cells of the staged plane pl into its ring slot (Eq. 15-18); pass 0 also feeds
  // the CFL reduction (Eq. 26) and the Eq. 30 counter from the input-interior cells
  auto convert_chunk = [&](int pl, int chunk) {
    mbar_wait(&ctl->mbar, (uint32_t)((phase_base + pl) & 1));   // one phase per staged plane, in order
    real* Ws = Wr + (pl % R) * 5 * PL;
    const int item = chunk * 32 + lane;
    const bool valid = item < PL;
    const int c = valid ? item : PL - 1;
    real U[1][5], W[1][5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[0][q] = Stg[q * PL + c];
    bool phys[1];
    int it[1];
    Aux aux[1];
    cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
    if (valid) {
#pragma unroll
      for (int q = 0; q < 5; ++q) Ws[q * PL + c] = W[0][q];
      ++ex_c2p;
      ex_newton += (unsigned)it[0];
      if (pl >= planes_counted) {          // each tile plane feeds the input-state counters exactly once
        my_iters += (unsigned)it[0];
        const int ti = c % NXT, tj = c / NXT;
        const bool interior = (ti >= G) && (ti < G + 16) && (tj >= G) && (tj < G + 16) && (pl >= G) &&
                              (pl < G + 16);
        if (interior) {
          if (!phys[0]) ++my_in_fail;
          my_umax = fmax(my_umax, umax_of_prim(W[0], aux[0]));
        }
      }
    }
  };

  for (;; ++pass) {
    if (pass > 0) beta = (pass <= max_retry) ? beta * real(0.75) : real(0.0);
    if (tid == 0) {
      ctl->face_fail = 0u;
      ctl->cell_fail = 0u;
      ctl->abort = 0u;
      issue_plane(0);
    }
    unsigned my_face_fail = 0, my_cell_fail = 0;
    unsigned long long pass_iters = 0;            // Newton iterations of this pass's face conversions
    bool flagged = false, aborted = false;
    int planes_staged = NXT;
    real part[5] = {real(0.0), real(0.0), real(0.0), real(0.0), real(0.0)};   // (Fx+ - Fx-) + (Fy+ - Fy-) of this thread's column cell

    // ---- prologue: tile plane 0 -> primitives; stage plane 1
    for (int chunk = warp; chunk < NP1; chunk += NW) convert_chunk(0, chunk);
    __syncthreads();
    if (tid == 0) issue_plane(1);

    for (int s = 0; s < NXT; ++s) {
      const int kh = s - 2 * G + 1;               // physical plane of the Hancock stage and the faces

      // ---- in-plane flux differences of plane kh-1 (fluxes written in the previous interval X)
      if (tid < 256 && kh - 1 >= 0 && kh - 1 <= 15) {
        const int i = tid & 15, j = tid >> 4;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const real dfx = FX[q * P::NFXY + j * 17 + i + 1] - FX[q * P::NFXY + j * 17 + i];
          const real dfy = FY[q * P::NFXY + (j + 1) * 16 + i] - FY[q * P::NFXY + j * 16 + i];
          part[q] = dfx + dfy;
        }
      }

      // ---- interval Y: edge states + Hancock half step of plane kh (S3-S5)
      if (kh >= -1 && kh <= 16) {
        const bool inplane = (kh >= 0) && (kh <= 15);
        const int nchunk = inplane ? 32 : 26;     // 320 cells (interior columns + the ring around them) or 256
        const int tk = kh + G;
        const int zb = (kh + 2) & 1;
        for (int r = 0; r < 2; ++r) {
          if (warp + NW * r >= nchunk) break;       // warp uniform
          const int info = hinfo[r];
          const int cidx = info & 511, soff = (info >> 9) & 511;
          const bool valid = (lane < 30) && (inplane || ((info >> 19) & 1));
          int o[2 * G - 1];
#pragma unroll
          for (int m = -(G - 1); m <= G - 1; ++m)
            o[m + G - 1] = (hd == 2) ? (((tk + m) % R) * 5 * PL + cidx)
                                     : ((tk % R) * 5 * PL + cidx + m * ((hd == 0) ? 1 : NXT));
          real um[5], up[5], dF[5];
          const bool warp_flat = hancock_lane<G>(Wr, hd, o, beta, beta0, um, up, dF);
          ex_hancock += (valid && !warp_flat) ? 1u : 0u;
          real* pm = hpm + soff;
          real* pp = hpp + soff + ((hd == 2) ? zb * 5 * P::ZS : 0);
          const int qs = hqs;
          bool has = ((info >> 18) & 1) && (hd == 2 || inplane);
          has = has && valid;
          if (warp_flat) {
            // every flux difference of the warp is +0: the common increment is -hdt*0 = -0 and
            // x + (-0) = x bit for bit, so the evolved edge states are the un-evolved ones
            if (has) {
#pragma unroll
              for (int q = 0; q < 5; ++q) {
                pm[q * qs] = um[q];
                pp[q * qs] = up[q];
              }
            }
            continue;
          }
          // `has` differs from lane to lane and nvcc likes to test it BEFORE the warp-uniform warp_flat (jump
          // threading), which sends the two groups of lanes to the shuffles below along different paths: a
          // diverged warp executes every shuffle through the slow collective path (measured: +25 % kernel time).
          // The explicit convergence point keeps the lanes together whatever the compiler does above it.
          __syncwarp();
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            const real fx = __shfl_sync(0xffffffffu, dF[q], hbase);
            const real fy = __shfl_sync(0xffffffffu, dF[q], hbase + 1);
            const real fz = __shfl_sync(0xffffffffu, dF[q], hbase + 2);
            const real dU = -hdt * ((fx + fy) + fz);
            if (has) {
              pm[q * qs] = um[q] + dU;
              pp[q * qs] = up[q] + dU;
            }
          }
        }
      }
      if (tid == 0) ctl->queue = 0;
      __syncthreads();

      // ---- interval X: Riemann problems of plane kh + update of plane kh-1; cons2prim of plane s+1
      {
        const int nxy = (kh >= 0 && kh <= 15) ? NXY : 0;
        const int np1 = (s + 1 < NXT) ? NP1 : 0;
        const int zbl = (kh + 1) & 1;             // buffer of plane kh-1
        bool zfirst = (kh >= 0) && (kh <= 16) && (warp < 8);
        int cq = -1;                              // queue ticket that turned out to be a cons2prim chunk
        for (;;) {                                // ---- face chunks
          int idx;
          if (zfirst) {
            zfirst = false;
            idx = tid;
          } else {
            int c = 0;
            if (lane == 0) c = atomicAdd(&ctl->queue, 1);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= nxy) {
              cq = c;
              break;
            }
            idx = 256 + c * 32 + lane;
          }
          int d, qs;
          const real *pL, *pR;
          if (idx < 256) {
            d = 2;
            qs = P::ZS;
            pL = ZSp + zbl * 5 * P::ZS + idx;
            pR = ZSm + idx;
          } else if (idx < 256 + P::NFXY) {
            const int f = idx - 256, jj = f / 17, fi = f - jj * 17;
            d = 0;
            qs = P::XS;
            pL = XSp + jj * 18 + fi;
            pR = XSm + jj * 18 + fi + 1;
          } else {
            const int f = idx - 256 - P::NFXY;
            d = 1;
            qs = P::YS;
            pL = YSp + f;
            pR = YSm + f + 16;
          }
          real U[2][5], W[2][5], F[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            U[0][q] = pL[q * qs];
            U[1][q] = pR[q * qs];
          }
          bool phys[2];
          int it[2];
          Aux aux[2];
          // Faces inside a uniform region carry the same state on both sides: when that holds for
          // the whole warp one conversion serves both (cons2prim is a function of its input, so the
          // bits are those of converting twice; the iteration counter still counts both).
          bool same = true;
#pragma unroll
          for (int q = 0; q < 5; ++q) same = same && (U[0][q] == U[1][q]);
          same = __all_sync(0xffffffffu, same);
          if (same) {
            cons2prim_multi<1>(U, W, aux, rtol, max_iter, phys, it);
#pragma unroll
            for (int q = 0; q < 5; ++q) W[1][q] = W[0][q];
            aux[1] = aux[0];
            phys[1] = phys[0];
            it[1] = it[0];
          } else {
            cons2prim_multi<2>(U, W, aux, rtol, max_iter, phys, it);
          }
          riemann_flux<RS>(d, W[0], U[0], aux[0], W[1], U[1], aux[1], F, same);
          pass_iters += (unsigned)(it[0] + it[1]);
          ex_c2p += same ? 1u : 2u;
          ex_newton += (unsigned)(same ? it[0] : it[0] + it[1]);
          ex_riemann += (SRHD_EXACT || !same) ? 1u : 0u;
          my_face_fail += (phys[0] ? 0u : 1u) + (phys[1] ? 0u : 1u);      // S15
          if (fout) {                               // faces on the boundary of an 8^3 patch
            if (idx < 256) {
              if ((kh & 7) == 0) {
                const int i = idx & 15, j = idx >> 4, pxy = (i >> 3) + 2 * (j >> 3);
                if (kh < 16) put_flux(pxy + 4 * (kh >> 3), 4, j & 7, i & 7, F);
                if (kh > 0) put_flux(pxy + 4 * ((kh - 1) >> 3), 5, j & 7, i & 7, F);
              }
            } else if (idx < 256 + P::NFXY) {
              const int f = idx - 256, jj = f / 17, fi = f - jj * 17;
              if ((fi & 7) == 0) {
                const int pyz = 2 * (jj >> 3) + 4 * (kh >> 3);
                if (fi < 16) put_flux((fi >> 3) + pyz, 0, kh & 7, jj & 7, F);
                if (fi > 0) put_flux(((fi - 1) >> 3) + pyz, 1, kh & 7, jj & 7, F);
              }
            } else {
              const int f = idx - 256 - P::NFXY, jf = f >> 4, i = f & 15;
              if ((jf & 7) == 0) {
                const int pxz = (i >> 3) + 4 * (kh >> 3);
                if (jf < 16) put_flux(pxz + 2 * (jf >> 3), 2, kh & 7, i & 7, F);
                if (jf > 0) put_flux(pxz + 2 * ((jf - 1) >> 3), 3, kh & 7, i & 7, F);
              }
            }
          }
          if (idx < 256) {
            if (kh >= 1) {                          // update cell (i, j, kh-1): Eq. 4a, 4b, 7; S12
              const int ku = kh - 1, i = idx & 15, j = idx >> 4;
              const real* uin = tile + ((size_t)(ku + G) * NXT + (j + G)) * NXT + (i + G);
              const int p = (i >> 3) + 2 * (j >> 3) + 4 * (ku >> 3);   // S13
              real* o = out + (size_t)p * 5 * 512 + (ku & 7) * 64 + (j & 7) * 8 + (i & 7);
              real Un[5];
#pragma unroll
              for (int q = 0; q < 5; ++q) {
                const real dfz = F[q] - FZ[q * P::ZS + idx];
                Un[q] = __ldg(uin + (size_t)q * T3) - dtdh * (part[q] + dfz);
                o[q * 512] = Un[q];
              }
              if (!is_physical(Un)) ++my_cell_fail;                      // Eq. 30
            }
#pragma unroll
            for (int q = 0; q < 5; ++q) FZ[q * P::ZS + idx] = F[q];
          } else if (idx < 256 + P::NFXY) {
#pragma unroll
            for (int q = 0; q < 5; ++q) FX[q * P::NFXY + (idx - 256)] = F[q];
          } else {
#pragma unroll
            for (int q = 0; q < 5; ++q) FY[q * P::NFXY + (idx - 256 - P::NFXY)] = F[q];
          }
        }
        while (cq < nxy + np1) {                  // ---- cons2prim chunks of the next tile plane
          convert_chunk(s + 1, cq - nxy);
          int c = 0;
          if (lane == 0) c = atomicAdd(&ctl->queue, 1);
          cq = __shfl_sync(0xffffffffu, c, 0);
        }
        // A failure anywhere fails the whole pass (S9, S15), so a pass that is not the last rung of the
        // ladder can be abandoned as soon as one is seen: same verdict, same accepted pass, less work.
        if (!flagged && beta != real(0.0) && (my_face_fail | my_cell_fail) != 0u) {
          *reinterpret_cast<volatile unsigned int*>(&ctl->abort) = 1u;
          flagged = true;
        }
      }
      __syncthreads();
      if (beta != real(0.0) && s + 1 < NXT && *reinterpret_cast<volatile unsigned int*>(&ctl->abort) != 0u) {
        aborted = true;                           // block uniform; planes 0 .. s+1 were staged and consumed
        planes_staged = s + 2;
        break;
      }
      // the staging buffer is free again: stage conserved plane s+2
      if (tid == 0 && s + 2 < NXT) issue_plane(s + 2);
    }

    phase_base += planes_staged;
    planes_counted = max(planes_counted, planes_staged);
    if (aborted) {
      __syncthreads();                            // everyone has read ctl->abort before thread 0 clears it
      continue;                                   // (the loop header moves on to the next rung)
    }

    // ---- verdict of this pass for the whole patch group (S9, S10, S15)
    my_face_fail = (unsigned)warp_sum(my_face_fail);
    my_cell_fail = (unsigned)warp_sum(my_cell_fail);
    if (lane == 0) {
      if (my_face_fail) atomicAdd(&ctl->face_fail, my_face_fail);
      if (my_cell_fail) atomicAdd(&ctl->cell_fail, my_cell_fail);
    }
    __syncthreads();
    n_face_fail = ctl->face_fail;
    n_cell_fail = ctl->cell_fail;
    __syncthreads();
    if ((n_face_fail == 0 && n_cell_fail == 0) || beta == real(0.0)) {
      my_iters += pass_iters;                     // the accepted pass's face conversions count, no other pass's
      break;
    }
  }

  // ---- per-call counters
  my_iters = warp_sum(my_iters);
  my_in_fail = (unsigned)warp_sum(my_in_fail);
  my_umax = warp_max(my_umax);
  ex_newton = warp_sum(ex_newton);
  ex_c2p = (unsigned)warp_sum(ex_c2p);
  ex_riemann = (unsigned)warp_sum(ex_riemann);
  ex_hancock = (unsigned)warp_sum(ex_hancock);
  if (lane == 0) {
    atomicAdd(&ctl->exec_newton, ex_newton);
    atomicAdd(&ctl->exec_c2p, ex_c2p);
    atomicAdd(&ctl->exec_riemann, ex_riemann);
    atomicAdd(&ctl->exec_hancock, ex_hancock);
    atomicAdd(&ctl->newton, my_iters);
    if (my_in_fail) atomicAdd(&ctl->in_fail, my_in_fail);
    atomicMax(&ctl->umax_bits, real_bits(my_umax));
  }
  __syncthreads();
  if (tid == 0 && stats) {
    atomicAdd(&stats->newton_iters, ctl->newton);
    const unsigned long long nf = (unsigned long long)ctl->in_fail + n_face_fail;
    if (nf) atomicAdd(&stats->n_c2p_fail, nf);
    if (n_cell_fail) atomicAdd(&stats->n_unphys_final, (unsigned long long)n_cell_fail);
    if (pass > 0) atomicAdd(&stats->n_retry_pg, 1ull);
    atomicAdd(&stats->n_passes, (unsigned long long)(pass + 1));
    atomicAdd(&stats->exec_newton, ctl->exec_newton);
    atomicAdd(&stats->exec_c2p, (unsigned long long)ctl->exec_c2p);
    atomicAdd(&stats->exec_riemann, (unsigned long long)ctl->exec_riemann);
    atomicAdd(&stats->exec_hancock, (unsigned long long)ctl->exec_hancock);
    const real umax = bits_real((rbits)ctl->umax_bits);
    atomic_max_nonneg(&stats->max_speed, smax_of_umax(umax));      // Eq. 27 per group, then max
  }
}

// handled == nullptr: run the uniform-tile pre-pass first (flags in a stream-ordered scratch allocation);
// else the caller has run a pre-pass of its own and only the march is launched
template <int G, int RS>
int launch_fluid(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
                 const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
                 real min_speed, const unsigned char* handled) {
  auto kern = fluid_step_kernel<G, RS>;
  const size_t smem = Plan<G>::bytes;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  const real rtol = newton_stop_rtol(p->newton_rtol);
  unsigned char* scratch = nullptr;
  if (!handled) {
    e = cudaMallocAsync(reinterpret_cast<void**>(&scratch), (size_t)npg, st);
    if (e != cudaSuccess) return (int)e;
    uniform_tiles_kernel<G, RS><<<npg, kScanThreads, 0, st>>>(cons_in, cons_out, flux_out, dt, dh, rtol,
                                                              p->newton_max_iter, stats, d_smax, cfl, min_speed, scratch);
    handled = scratch;
  }
  kern<<<npg, kFluidThreads, smem, st>>>(cons_in, cons_out, flux_out, dt, dh, p->minmod_coeff, p->max_retry, rtol,
                                         p->newton_max_iter, stats, d_smax, cfl, min_speed, handled);
  e = cudaGetLastError();
  const cudaError_t e2 = scratch ? cudaFreeAsync(scratch, st) : cudaSuccess;
  return (int)(e != cudaSuccess ? e : e2);
}

int fluid_march(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
                const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
                real min_speed, const unsigned char* handled) {
  if (p->recon == SRHD_RECON_PLM) {
    return p->riemann == SRHD_RIEMANN_HLLE
               ? launch_fluid<2, 0>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed, handled)
               : launch_fluid<2, 1>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed, handled);
  }
  return p->riemann == SRHD_RIEMANN_HLLE
             ? launch_fluid<3, 0>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed, handled)
             : launch_fluid<3, 1>(cons_in, cons_out, flux_out, npg, dt, dh, p, stats, st, d_smax, cfl, min_speed, handled);
}

}  // namespace srhd

namespace srhd {   // srhd_vl.cu
int vl_step(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt, real dh,
            const srhd_params* p, srhd_stats* stats, cudaStream_t st, const real* d_smax, real cfl,
            real min_speed);
size_t vl_workspace_bytes(int npg, const srhd_params* p);
}  // namespace srhd

using namespace srhd;

extern "C" size_t srhd_workspace_bytes(int npg, const srhd_params* params) {
  if (check_params(params) != SRHD_OK || npg <= 0) return 0;
  if (params->integrator == SRHD_INTEGRATOR_MHM) return (size_t)npg;   // the uniform-tile flags, one byte per group
  return vl_workspace_bytes(npg, params);
}

static int fluid_step_impl(const real* cons_in, real* cons_out, real* flux_out, int npg, real dt,
                           real dh, const srhd_params* params, srhd_stats* stats, void* stream,
                           const real* d_smax, real cfl, real min_speed) {
  if (npg > 0 && (!cons_in || !cons_out)) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  if (npg < 0) return SRHD_ERR_BAD_SIZE;
  if (!(dt > real(0.0)) || !(dh > real(0.0)) || !std::isfinite(dt) || !std::isfinite(dh)) return SRHD_ERR_BAD_STEP;
  // cons_in: TMA bulk copies (16 bytes) and the pair loads of the uniform-tile scan; cons_out: the uniform-tile
  // path stores pairs of srhd_real (flux_out is written one value at a time)
  if ((reinterpret_cast<uintptr_t>(cons_in) & 15u) || (reinterpret_cast<uintptr_t>(cons_out) & (sizeof(real2) - 1)))
    return SRHD_ERR_BAD_ALIGN;
  const int nxt = 16 + 2 * params->ghost;
  const size_t in_bytes = (size_t)npg * 5 * nxt * nxt * nxt * sizeof(real);
  const size_t out_bytes = (size_t)npg * 8 * 5 * 512 * sizeof(real);
  const uintptr_t a = reinterpret_cast<uintptr_t>(cons_in), b = reinterpret_cast<uintptr_t>(cons_out);
  if (a < b + out_bytes && b < a + in_bytes) return SRHD_ERR_ALIAS;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (stats) {
    const cudaError_t e = cudaMemsetAsync(stats, 0, sizeof(srhd_stats), st);
    if (e != cudaSuccess) return (int)e;
  }
  if (npg == 0) return SRHD_OK;
  if (params->integrator == SRHD_INTEGRATOR_VL)
    return vl_step(cons_in, cons_out, flux_out, npg, dt, dh, params, stats, st, d_smax, cfl, min_speed);
  return fluid_march(cons_in, cons_out, flux_out, npg, dt, dh, params, stats, st, d_smax, cfl, min_speed, nullptr);
}

extern "C" int srhd_fluid_step_fluxes(const real* cons_in, real* cons_out, real* flux_out, int npg,
                                      double dt, double dh, const srhd_params* params, srhd_stats* stats,
                                      void* stream) {
  return fluid_step_impl(cons_in, cons_out, flux_out, npg, dt, dh, params, stats, stream, nullptr, real(0.0), real(0.0));
}

extern "C" int srhd_fluid_step(const real* cons_in, real* cons_out, int npg, double dt, double dh,
                               const srhd_params* params, srhd_stats* stats, void* stream) {
  return fluid_step_impl(cons_in, cons_out, nullptr, npg, dt, dh, params, stats, stream, nullptr, real(0.0), real(0.0));
}

extern "C" int srhd_fluid_step_cfl(const real* cons_in, real* cons_out, real* flux_out, int npg, double cfl,
                                   double dh, const real* d_max_speed, double min_speed,
                                   const srhd_params* params, srhd_stats* stats, void* stream) {
  if (!d_max_speed) return SRHD_ERR_NULL_POINTER;
  if (!(cfl > real(0.0)) || !std::isfinite(cfl) || !(min_speed >= real(0.0))) return SRHD_ERR_BAD_STEP;
  // dt is formed on the device; the host-side check of dt is replaced by the one of cfl (dt = 1 passes it)
  return fluid_step_impl(cons_in, cons_out, flux_out, npg, real(1.0), dh, params, stats, stream, d_max_speed, cfl,
                         min_speed);
}

// ---------------------------------------------------------------------------------------------------------------
// srhd_fluid_step_noalloc (include/srhd.h): the MUSCL-Hancock step for hosts that cannot let this library
// allocate -- codes whose own pool owns the whole GPU, step loops with a fixed memory budget, processes whose
// footprint is policed from outside.  Same two kernels as srhd_fluid_step; the only difference is where the
// pre-pass's one-byte-per-group flags live: in the fixed array below instead of a cudaMallocAsync block.
// ---------------------------------------------------------------------------------------------------------------
namespace srhd {

// 64 KiB per GPU that runs this library's code, from module load to process exit.  Shared by every call on the
// device and never cleared behind the caller's back: each call zeroes the bytes it will use (below).
static __device__ __align__(256) unsigned char g_noalloc_handled[SRHD_NOALLOC_MAX_NPG];

// In host code `g_noalloc_handled` is only a handle for the runtime, not an address a kernel may dereference.
// The real device address is asked for once per device, with that device current, and cached here.
constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static unsigned char* g_noalloc_addr[kNoAllocMaxDevices] = {};

// Returns 0 and the device address of the flag array on the CURRENT device; a cudaError_t if the look-up fails.
// First use on a device does the look-up (set-up; keep it out of stream capture), later uses read the cache.
static int noalloc_flags_on_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= kNoAllocMaxDevices) return (int)cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_handled);
    if (e != cudaSuccess) return (int)e;
    if (!p) return (int)cudaErrorInvalidSymbol;
    g_noalloc_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_addr[dev];
  return 0;
}

template <int G, int RS>
static int launch_fluid_noalloc(const real* cons_in, real* cons_out, int npg, real dt, real dh,
                                const srhd_params* p, srhd_stats* stats, cudaStream_t st, unsigned char* flags) {
  // the flags of this call's groups start at zero whatever the previous call left there (stream-ordered, so it
  // cannot overtake a kernel of an earlier call on the same stream)
  cudaError_t e = cudaMemsetAsync(flags, 0, (size_t)npg, st);
  if (e != cudaSuccess) return (int)e;
  const real rtol = newton_stop_rtol(p->newton_rtol);
  uniform_tiles_kernel<G, RS><<<npg, kScanThreads, 0, st>>>(cons_in, cons_out, nullptr, dt, dh, rtol,
                                                            p->newton_max_iter, stats, nullptr, real(0.0), real(0.0),
                                                            flags);
  e = cudaGetLastError();
  if (e != cudaSuccess) return (int)e;
  // with the flags handed in, launch_fluid launches the march only: no allocation on that branch
  return launch_fluid<G, RS>(cons_in, cons_out, nullptr, npg, dt, dh, p, stats, st, nullptr, real(0.0), real(0.0), flags);
}

}  // namespace srhd

extern "C" int srhd_fluid_step_noalloc(const real* cons_in, real* cons_out, int npg, double dt_, double dh_,
                                       const srhd_params* params, srhd_stats* stats, void* stream) {
  const real dt = (real)dt_, dh = (real)dh_;
  // the argument checks of srhd_fluid_step, then the two limits of this variant
  if (npg > 0 && (!cons_in || !cons_out)) return SRHD_ERR_NULL_POINTER;
  const int pc = check_params(params);
  if (pc) return pc;
  if (params->integrator != SRHD_INTEGRATOR_MHM) return SRHD_ERR_BAD_PARAMS;   // VL scratch does not fit a fixed array
  if (npg < 0) return SRHD_ERR_BAD_SIZE;
  if (npg > SRHD_NOALLOC_MAX_NPG) return SRHD_ERR_TOO_LARGE;
  if (!(dt > real(0.0)) || !(dh > real(0.0)) || !std::isfinite(dt) || !std::isfinite(dh)) return SRHD_ERR_BAD_STEP;
  if ((reinterpret_cast<uintptr_t>(cons_in) & 15u) || (reinterpret_cast<uintptr_t>(cons_out) & (sizeof(real2) - 1)))
    return SRHD_ERR_BAD_ALIGN;
  const int nxt = 16 + 2 * params->ghost;
  const size_t in_bytes = (size_t)npg * 5 * nxt * nxt * nxt * sizeof(real);
  const size_t out_bytes = (size_t)npg * 8 * 5 * 512 * sizeof(real);
  const uintptr_t a = reinterpret_cast<uintptr_t>(cons_in), b = reinterpret_cast<uintptr_t>(cons_out);
  if (a < b + out_bytes && b < a + in_bytes) return SRHD_ERR_ALIAS;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (stats) {
    const cudaError_t e = cudaMemsetAsync(stats, 0, sizeof(srhd_stats), st);
    if (e != cudaSuccess) return (int)e;
  }
  if (npg == 0) return SRHD_OK;
  unsigned char* flags = nullptr;
  const int rc = noalloc_flags_on_current_device(&flags);
  if (rc) return rc;
  if (params->recon == SRHD_RECON_PLM) {
    return params->riemann == SRHD_RIEMANN_HLLE
               ? launch_fluid_noalloc<2, 0>(cons_in, cons_out, npg, dt, dh, params, stats, st, flags)
               : launch_fluid_noalloc<2, 1>(cons_in, cons_out, npg, dt, dh, params, stats, st, flags);
  }
  return params->riemann == SRHD_RIEMANN_HLLE
             ? launch_fluid_noalloc<3, 0>(cons_in, cons_out, npg, dt, dh, params, stats, st, flags)
             : launch_fluid_noalloc<3, 1>(cons_in, cons_out, npg, dt, dh, params, stats, st, flags);
}
