/* include/srhd.h -- C ABI of the B200-native GAMER-SR hot path (arXiv 2012.11130).
 *
 * One data-parallel path of the paper: the per-patch-group special-relativistic hydrodynamics
 * update with the Taub-Mathews equation of state, in fp64, as hand-written CUDA for sm_100a.
 *
 * Citations: "P:n" = line n of the paper text; "S#"/"G#" = readings listed in
 * DESIGN.md section 4.  Units c = k_B = m = 1.
 *
 * State vectors (Eq. 5-8, "equations actually solved"):
 *   primitive  W = (rho, U^x, U^y, U^z, p)       -- U^i is the FOUR-velocity (Eq. 8)
 *   conserved  U = (D, M^x, M^y, M^z, Etilde)    -- Etilde = E - D, the REDUCED energy (Eq. 6)
 *
 * Conventions common to every call
 *   - every data pointer is a DEVICE pointer owned by the caller (allocate / free is the caller's
 *     job; the library keeps no state between calls).  `const srhd_params*` is a HOST pointer and is
 *     read before the call returns.  `srhd_stats*` / `double* d_max_speed` are DEVICE pointers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream); every call is
 *     asynchronous on that stream and returns after the launch.
 *   - SoA state lists: component c of state i lives at ptr[c*stride + i], stride >= n (in doubles).
 *   - return value: 0 = OK; negative = bad argument (SRHD_ERR_*); positive = a cudaError_t raised by
 *     the launch.  UNPHYSICAL STATES ARE NOT ERRORS: they are counted in srhd_stats and evaluated
 *     by the deterministic rules S9/S10/S15 so that results are reproducible.
 *   - n == 0 / npg == 0 is a no-op that returns 0 (stats are still zeroed).
 *   - there is no CPU fallback: without a CUDA device every compute call returns a cudaError_t.
 */
#ifndef SRHD_H_
#define SRHD_H_

#include <stddef.h>

/* Every state array (and the max-speed scalar) is an array of srhd_real: double, or float in the library built
 * with -DSRHD_F32 (libsrhd_b200_f32*.so: the precision of every performance number in the paper; Eq. 30
 * then uses eps_machine = FLT_EPSILON).  Scalar arguments (dt, dh, cfl, thresholds), srhd_params and
 * srhd_stats have the same types in every build. */
#ifdef SRHD_F32
typedef float srhd_real;
#else
typedef double srhd_real;
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define SRHD_OK                 0
#define SRHD_ERR_NULL_POINTER  (-1)
#define SRHD_ERR_BAD_PARAMS    (-2)   /* recon/riemann out of range, ghost != 2 (PLM) / 3 (PPM), ... */
#define SRHD_ERR_BAD_SIZE      (-3)   /* stride < n, negative npg, grid extent not a multiple of 16, */
                                      /* or (nx/16)*(ny/16) > 104857 (32-bit in-plane offsets)      */
#define SRHD_ERR_BAD_STEP      (-4)   /* dt <= 0 or dh <= 0 (or not finite)                         */
#define SRHD_ERR_ALIAS         (-5)   /* cons_in and cons_out (srhd_grid_step_cfl: any two of       */
                                      /* patches_in, patches_out, cons_in) overlap                  */
#define SRHD_ERR_BAD_ALIGN     (-6)   /* cons_in not 16-byte aligned (TMA bulk copies), or cons_out */
                                      /* / patches_in / patches_out not aligned to 2*sizeof(srhd_real) */
                                      /* (16 bytes in the fp64 builds: pair loads and stores)       */
#define SRHD_ERR_TOO_LARGE     (-7)   /* srhd_fluid_step_noalloc: npg > SRHD_NOALLOC_MAX_NPG         */

#define SRHD_RECON_PLM   0
#define SRHD_RECON_PPM   1
#define SRHD_RIEMANN_HLLE 0
#define SRHD_RIEMANN_HLLC 1
#define SRHD_INTEGRATOR_MHM 0   /* MUSCL-Hancock (Toro 2011), the fused hot path                 */
#define SRHD_INTEGRATOR_VL  1   /* VL: van Leer predictor-corrector (Falle 1991; van Leer 2006; S18) */

#define SRHD_REFINE_NONE   0   /* no gradient criterion */
#define SRHD_REFINE_D      1   /* Q = D        (conserved: no root finding)            */
#define SRHD_REFINE_ETILDE 2   /* Q = Etilde   (conserved)                                    */
#define SRHD_REFINE_RHO    3   /* Q = rho      (primitive: cons2prim per cell; P:346 uses it) */
#define SRHD_REFINE_GAMMA  4   /* Q = Lorentz factor ("gradient of the Lorentz factor") */

#define SRHD_BC_PERIODIC 0
#define SRHD_BC_OUTFLOW  1

/* Run-time parameters of the solver (values the paper leaves open are the
 * readings S2, S3, S9 of DESIGN.md). */
typedef struct {
  int    recon;            /* SRHD_RECON_PLM or SRHD_RECON_PPM (BASELINE.json configs 3, 5)   */
  int    riemann;          /* SRHD_RIEMANN_HLLE or SRHD_RIEMANN_HLLC                          */
  double minmod_coeff;     /* beta0 in [1,2], "original minmod coefficient"; default 1.5 (S3) */
  int    max_retry;        /* K reductions of beta by 0.75, then beta = 0; default 8 (S9)     */
  double newton_rtol;      /* Newton-Raphson stop: |delta| <= rtol*|htilde|; default 1e-15, 1e-6 in the f32 build (S2) */
  int    newton_max_iter;  /* iteration cap; default 20 (S2)                                          */
  int    ghost;            /* ghost width of cons_in: MUSCL-Hancock 2 (PLM) / 3 (PPM); VL one more    */
  int    integrator;       /* SRHD_INTEGRATOR_MHM (default) or SRHD_INTEGRATOR_VL             */
} srhd_params;

/* Per-call counters, DEVICE resident, zeroed by the callee at call start (on the stream). */
typedef struct {
  unsigned long long n_c2p_fail;      /* states violating Eq. 30 on input to a conversion:
                                         srhd_cons2prim: every failing state; srhd_fluid_step: failing
                                         input interior cells + failing half-step face states of the
                                         accepted beta = 0 pass (S15)                                 */
  unsigned long long n_retry_pg;      /* patch groups that needed >= 1 retry pass         */
  unsigned long long n_unphys_final;  /* updated cells still violating Eq. 30 after beta = 0 (S10)    */
  unsigned long long newton_iters;    /* Newton-Raphson iterations of the ALGORITHM's conversions: every
                                         tile cell once + both states of every face in the accepted pass
                                         (for the flop model; retries that were thrown away not counted) */
  double             max_speed;       /* max S_max (Eq. 27) over the INPUT interior cells       */
  unsigned long long n_passes;        /* passes over patch groups, retry passes included (>= npg)     */
  /* work the kernel actually EXECUTED (srhd_fluid_step only; for the executed-flop roofline figure):
   * retry passes are abandoned at the first plane that shows a failure, uniform regions take shortcuts */
  unsigned long long exec_c2p;        /* conversions executed (cons2prim calls)                       */
  unsigned long long exec_newton;     /* Newton-Raphson iterations executed                           */
  unsigned long long exec_riemann;    /* HLLE / HLLC solves executed                                  */
  unsigned long long exec_hancock;    /* (cell, direction) edge-state pairs reconstructed + converted */
  unsigned long long n_uniform_pg;    /* patch groups whose whole tile held one state bit for bit and took
                                         the uniform-tile path (the result is the input; see srhd_fluid.cu) */
} srhd_stats;

/* Fill *p with the defaults above for the given recon / riemann choice (host pointer). */
void srhd_default_params(srhd_params* p, int recon, int riemann);

/* prim -> cons for n independent states (Fig. 15 right; Eq. 5a-b; Eq. 22-23).
 * prim, cons: device, SoA with `stride`; the two arrays must not overlap. */
int srhd_prim2cons(const srhd_real* prim, srhd_real* cons, size_t n, size_t stride, void* stream);

/* cons -> prim for n independent states (Fig. 15 left; Eq. 15-18; App. A):
 * Newton-Raphson on htilde = h - 1 from the two-branch guess A4/A6, canonical left-hand side
 * L = fma(x, x+2, -mu^2).  A state that fails Eq. 30 is counted in
 * stats->n_c2p_fail and evaluated with L <- eps_machine (S10).  stats may be NULL. */
int srhd_cons2prim(const srhd_real* cons, srhd_real* prim, size_t n, size_t stride,
                   const srhd_params* params, srhd_stats* stats, void* stream);

/* CFL signal speed (Eq. 24-28; G1): *d_max_speed = S_max(max_i U_max,i) with
 * U_max = gamma_s (|U^x|+|U^y|+|U^z|) + 3 gamma U_s from cons2prim of each state.  The time step is
 * dt = C_CFL * dh / *d_max_speed (Eq. 28), formed by the caller.  n == 0 gives 0. */
int srhd_max_signal_speed(const srhd_real* cons, size_t n, size_t stride,
                          const srhd_params* params, srhd_real* d_max_speed, void* stream);

/* One MUSCL-Hancock step (readings S3-S7, S9-S15) of npg patch groups.
 *   cons_in : [npg][5][nxt][nxt][nxt] doubles, nxt = 16 + 2*ghost, x fastest: the 16^3 interior
 *             cells of the patch group (2^3 patches of 8^3 cells) plus `ghost` layers of
 *             ghost zones on every side, already filled by the caller (srhd_grid_gather below, or
 *             an AMR driver -- P:219).
 *   cons_out: [npg][8][5][8][8][8] doubles: patch p = ix + 2*iy + 4*iz (S13), component, z, y, x.
 *   dt, dh  : time step and cell size.
 * Per patch group: cons2prim of every tile cell -> PLM/PPM edge values on primitives -> Hancock
 * half step -> cons2prim of both states at every face -> HLLE/HLLC flux -> flux-difference update
 * -> Eq. 30 check; if any interior cell or face state of the group fails, the whole group is redone
 * with beta <- 0.75 beta, after max_retry reductions with beta = 0, whose result is accepted.
 * cons_in and cons_out must not overlap.  stats may be NULL. */
int srhd_fluid_step(const srhd_real* cons_in, srhd_real* cons_out, int npg, double dt, double dh,
                    const srhd_params* params, srhd_stats* stats, void* stream);

/* The same step, additionally returning the fluxes through the six boundary faces of every 8^3 patch
 * -- what the AMR driver's flux-correction step at coarse-fine interfaces consumes (P:285 section
 * 3.3(4); the solver runs on the GPU, the correction on the host side).
 *   flux_out: device, [npg][8][6][5][8][8] doubles: patch p (S13), face (0 x-lo, 1 x-hi, 2 y-lo, 3 y-hi,
 *             4 z-lo, 5 z-hi), component (D, M^x, M^y, M^z, Etilde), then the two in-face cell
 *             coordinates, slower one first: (z,y) on x faces, (z,x) on y faces, (y,x) on z faces.
 *             Values are the HLLE/HLLC fluxes of the ACCEPTED pass, positive along +axis; the face shared
 *             by two patches of the group is written to both.  NULL = srhd_fluid_step.
 * Must not overlap cons_in / cons_out.  Same errors and asynchrony as srhd_fluid_step. */
int srhd_fluid_step_fluxes(const srhd_real* cons_in, srhd_real* cons_out, srhd_real* flux_out, int npg,
                           double dt, double dh, const srhd_params* params, srhd_stats* stats,
                           void* stream);

/* The same step with the time step formed ON THE DEVICE from a signal speed that is already there
 * (srhd_max_signal_speed / srhd_grid_scatter_speed wrote it): dt = cfl * dh / max(*d_max_speed, min_speed)
 * (Eq. 28).  No host round trip for dt, so a sequence of steps can be enqueued without a
 * synchronisation.  d_max_speed: device, one srhd_real, read by every CTA at kernel start; min_speed >= 0
 * bounds the speed from below (e.g. the signal speed of a fixed-inflow state that is not in the
 * grid yet); the caller guarantees max(*d_max_speed, min_speed) > 0.  flux_out may be NULL. */
int srhd_fluid_step_cfl(const srhd_real* cons_in, srhd_real* cons_out, srhd_real* flux_out, int npg, double cfl,
                        double dh, const srhd_real* d_max_speed, double min_speed,
                        const srhd_params* params, srhd_stats* stats, void* stream);

/* Refinement criteria of the SRHD module (section 3.1; Eq. 33), one flag per 8^3 patch,
 * on the same ghosted tiles as srhd_fluid_step (cons_in: [npg][5][nxt]^3, nxt = 16 + 2*params->ghost).
 *   flags[pg*8 + p] = 1 if ANY cell of patch p (S13) satisfies
 *     (|Q(i+1)-Q(i-1)| + |Q(j+1)-Q(j-1)| + |Q(k+1)-Q(k-1)|) / (2 |Q|) > c_q        (Eq. 33 with centred
 *         differences, reading S17; the cell size cancels)       -- skipped if quantity == SRHD_REFINE_NONE
 *     or  |M| / D > mom_over_d
 *                                                                 -- skipped if mom_over_d == 0
 *   else 0.  flags: device, npg*8 bytes.  Thresholds per level are the caller's business. */
int srhd_refine_flags(const srhd_real* cons_in, int npg, int quantity, double c_q, double mom_over_d,
                      const srhd_params* params, unsigned char* flags, void* stream);

/* Flux correction at coarse-fine interfaces with the paper's guard (section 3.3(4)): the coarse cells
 * next to the interface were updated with the coarse flux through it (flux_out of srhd_fluid_step_fluxes); this
 * call swaps that flux for the fine one (already averaged over the fine faces and sub-steps by the driver):
 *     lo face: U' = U + dt/dh (F_fine - F_coarse),    hi face: U' = U - dt/dh (F_fine - F_coarse),
 * and "if unphysical results are found after this flux correction, we simply ignore the correction on the
 * failed cells": U' that fails Eq. 30 is dropped and counted.
 *   patches     : device, [np][5][8][8][8] (cons_out layout, updated in place)
 *   flux_coarse, flux_fine : device, [nf][5][8][8], in-face layout of flux_out
 *   face_patch, face_id    : device, [nf] ints: patch index, face 0 x-lo .. 5 z-hi
 *   d_n_skipped : device, one unsigned long long (zeroed by the call): cells whose correction was ignored
 * Faces are processed class by class (x-lo, x-hi, y-lo, ...), so a cell on a patch edge is corrected through
 * one face after the other, in that order; within a class a (patch, face) pair may appear once.
 * The two index arrays are TRUSTED (the call does not know how many patches `patches` holds): a face_id outside
 * 0..5 is silently never applied and a face_patch beyond the array is an out-of-bounds access -- validate them
 * where they are built (binding.py checks both before the call). */
int srhd_flux_correction(srhd_real* patches, const srhd_real* flux_coarse, const srhd_real* flux_fine,
                         const int* face_patch, const int* face_id, int nf, double dt, double dh,
                         unsigned long long* d_n_skipped, void* stream);

/* Ghost-zone interpolation with the primitive-variable fallback (section 3.3(3)): every coarse cell with six
 * neighbours gives its 2^3 children Q -+ d_x/4 -+ d_y/4 -+ d_z/4 with the limited slopes of reading S3
 * (coefficient minmod_coeff) on the CONSERVED variables (conservative); where a child fails Eq. 30 the
 * same interpolation is done on the PRIMITIVE variables of the seven cells and converted back ("Eq. 30 is
 * always satisfied ... ghost zones do not affect conservation").  That holds while every child's rho and p stay
 * positive; where the primitive interpolation would give a child rho <= 0 or p <= 0 (a steep 3-D corner) the eight
 * children are copies of the parent state (vanished minmod coefficient = copy from the parent; reading S22).
 *   coarse: device, [5][nz][ny][nx];  fine: device, [5][2(nz-2)][2(ny-2)][2(nx-2)]
 *   fallback: device, (nz-2)(ny-2)(nx-2) bytes: 0 conserved interpolation, 1 primitive interpolation, 2 parent
 *             copied (may be NULL)
 *   d_n_fallback: device, one unsigned long long (zeroed by the call): cells with fallback != 0 */
int srhd_ghost_interp(const srhd_real* coarse, int nx, int ny, int nz, srhd_real* fine, double minmod_coeff,
                      const srhd_params* params, unsigned char* fallback, unsigned long long* d_n_fallback,
                      void* stream);

/* Bytes of scratch a srhd_fluid_step call uses: for MUSCL-Hancock one byte per patch group (the flags by
 * which the uniform-tile pre-pass tells the main kernel which groups it has already written); for the VL
 * integrator the two primitive tiles its stages communicate through.  The call allocates and frees them itself
 * in stream order (cudaMallocAsync / cudaFreeAsync on `stream`): informational, nothing for the caller to provide. */
size_t srhd_workspace_bytes(int npg, const srhd_params* params);

/* srhd_fluid_step for callers that must not allocate.
 *
 * Who this is for: srhd_fluid_step obtains its one-byte-per-group flag array (srhd_workspace_bytes) with
 * cudaMallocAsync / cudaFreeAsync.  Some hosts of this library cannot afford that: a simulation code whose own
 * allocator already owns every byte of the GPU (a later cudaMalloc* fails or fragments its pool), a step loop
 * that has promised its scheduler a fixed memory footprint, a process sharing the GPU whose memory budget is
 * enforced from outside, or a context in which the stream-ordered pool is disabled.  This variant computes
 * exactly what srhd_fluid_step computes (same kernels, same arguments, same results bit for bit, same stats),
 * but calls no cudaMalloc / cudaMallocAsync / cudaFree* and no library routine that allocates.
 *
 * Where the scratch lives: in a fixed array of SRHD_NOALLOC_MAX_NPG bytes (64 KiB) that is part of the library
 * image, so every GPU on which this library is used carries those 64 KiB from the moment the library's code is
 * loaded there until the process exits, whether or not this call is ever made.
 *
 * Limits and rules
 *   - npg <= SRHD_NOALLOC_MAX_NPG (65 536 patch groups = 2.7e8 cells, the size of the largest BASELINE config);
 *     a larger npg returns SRHD_ERR_TOO_LARGE and launches nothing: split the batch and call again.
 *   - MUSCL-Hancock only (params->integrator == SRHD_INTEGRATOR_MHM): the VL integrator's scratch is two
 *     primitive tiles per group, far beyond a fixed array; it returns SRHD_ERR_BAD_PARAMS here.
 *   - First call per device: the first call made with a given device current looks up the array's device
 *     address (once per device, then cached; a cudaGetSymbolAddress call, which may make the runtime load the
 *     library's code onto that device).  Make that first call during set-up, outside any stream capture and
 *     before the phase in which allocation is forbidden; later calls on that device do no set-up.
 *   - The array is shared by every call on the device and keeps whatever the last call left in it.  Each call
 *     re-zeroes the npg bytes it is going to use, in stream order, before its kernels run, so stale flags are
 *     never read.  Two calls whose kernels can overlap on one GPU (different streams without an ordering
 *     between them, or two host threads) RACE on the array and give wrong results: keep calls to this entry
 *     point on one device ordered one after the other.  Calls on different devices do not interact.
 *   - Every other argument, error code and the asynchrony are those of srhd_fluid_step. */
#define SRHD_NOALLOC_MAX_NPG 65536
int srhd_fluid_step_noalloc(const srhd_real* cons_in, srhd_real* cons_out, int npg, double dt, double dh,
                            const srhd_params* params, srhd_stats* stats, void* stream);

/* Harness helpers for a uniform grid (reading S11, S13; NOT part of the paper's solver: they stand in
 * for the AMR driver's ghost-zone fill).  grid: [5][nz][ny][nx] conserved, extents multiples
 * of 16.  bc[6] (HOST pointer) = {x-lo, x-hi, y-lo, y-hi, z-lo, z-hi}, each SRHD_BC_PERIODIC (wrap)
 * or SRHD_BC_OUTFLOW (copy the nearest interior cell).  inflow_mask (device, [ny][nx] bytes, may be
 * NULL): ghost cells below z = 0 whose column is marked hold inflow_cons[5] (HOST pointer) instead.
 * Patch group pg = gx + (nx/16)*(gy + (ny/16)*gz). */
int srhd_grid_gather(const srhd_real* grid, srhd_real* cons_in, int nx, int ny, int nz, int ghost,
                     const int* bc, const unsigned char* inflow_mask, const double* inflow_cons,
                     void* stream);
int srhd_grid_scatter(const srhd_real* cons_out, srhd_real* grid, int nx, int ny, int nz, void* stream);

/* srhd_grid_scatter fused with srhd_max_signal_speed of the state it writes: *d_max_speed (device)
 * receives S_max (Eq. 26-27) of the scattered grid, ready for the next step's dt (Eq. 28).  The copy is
 * memory bound and the conversion ALU bound, so the fused kernel costs about as much as the slower one. */
int srhd_grid_scatter_speed(const srhd_real* cons_out, srhd_real* grid, int nx, int ny, int nz,
                            const srhd_params* params, srhd_real* d_max_speed, void* stream);

/* Ghost-zone fill straight from the PATCH layout srhd_fluid_step wrote (cons_out of the previous
 * step of the same uniform grid: patch group pg = gx + (nx/16)*(gy + (ny/16)*gz)), fused with
 * srhd_max_signal_speed of that state: patches -> cons_in tiles (as srhd_grid_gather would build them
 * from the scattered grid, bit for bit) and *d_max_speed = S_max.  With it a uniform-grid step is two
 * kernels (this one and srhd_fluid_step_cfl) and the grid is only materialised on demand.  The ghost
 * width is params->ghost.  Boundary arguments as srhd_grid_gather. */
int srhd_patch_gather_speed(const srhd_real* patches, srhd_real* cons_in, int nx, int ny, int nz, const int* bc,
                            const unsigned char* inflow_mask, const double* inflow_cons,
                            const srhd_params* params, srhd_real* d_max_speed, void* stream);

/* One whole step of a uniform grid kept in the patch layout: srhd_patch_gather_speed + srhd_fluid_step_cfl behind
 * one call, with the uniform-tile test done on the way (same results, bit for bit, as the two calls).
 *   patches_in : device, [npg][8][5][8][8][8], the current state (cons_out of the previous step)
 *   patches_out: device, same shape, the new state; must not be patches_in (neighbouring groups still read it)
 *   cons_in    : device scratch for the ghosted tiles, [npg][5][nxt]^3, nxt = 16 + 2*params->ghost; only the
 *                tiles of groups that are not uniform are written
 *   flux_out   : as srhd_fluid_step_fluxes, may be NULL
 *   d_max_speed: device, one srhd_real: receives S_max of the CURRENT state (Eq. 26-27); the step then uses
 *                dt = cfl * dh / max(S_max, min_speed) (Eq. 28) without a host round trip
 * A patch group whose whole tile (ghost zones after the boundary mapping included) holds one state bit for bit is
 * finished by the first kernel: its new patches are its old ones (srhd_stats.n_uniform_pg counts them), so its
 * state crosses HBM once in and once out and no tile is materialised for it; every other group goes through
 * fluid_step_kernel as in srhd_fluid_step_cfl.  Boundary arguments as srhd_grid_gather; errors as the two calls. */
int srhd_grid_step_cfl(const srhd_real* patches_in, srhd_real* patches_out, srhd_real* cons_in, srhd_real* flux_out,
                       int nx, int ny, int nz, const int* bc, const unsigned char* inflow_mask,
                       const double* inflow_cons, double cfl, double dh, double min_speed,
                       const srhd_params* params, srhd_stats* stats, srhd_real* d_max_speed, void* stream);

/* Measurement helper (not part of the solver): launches a register-only DFMA loop that fills every
 * fp64 lane of the GPU (148 x 8 CTAs x 256 threads, 32*iters dependent-chain DFMA per thread in 8
 * independent chains) on `stream`; *flops (HOST pointer, may be NULL) receives the flop count of the
 * launch (2 per DFMA).  The caller times it with events.  d_sink: device, >= 1 double, never written
 * in practice.  bench.py uses it for the measured fp64 ALU roof. */
int srhd_fp64_peak_probe(double* d_sink, int iters, unsigned long long* flops, void* stream);

/* Measurement helper: srhd_fp64_peak_probe's DFMA loop with `ffma_per_8_dfma` (0, 4, 8, 12 or 16) independent
 * single-precision FMAs interleaved per 8 DFMA.  *dfma_flops (HOST pointer) = flops of the DFMA part only.
 * Timed by the caller; shows how issue slots are shared between the fp64 pipe and everything else
 * (output kept under profiles/). */
int srhd_issue_probe(double* d_sink, int iters, int ffma_per_8_dfma, unsigned long long* dfma_flops, void* stream);

/* Verification helper (not part of the solver): evaluates the library's canonical quotient a/b (the one
 * that feeds the Eq. 30 verdict: one shared reciprocal + a Markstein correction in the production build, IEEE
 * division in the exact build) and IEEE division side by side on n seeded pairs generated on the device;
 * d_out (device, 2 x unsigned long long) receives {number of bit mismatches, index of the first one or
 * ~0}.  dist: 0 = the value ranges of BASELINE.json configs 2-5, 1 = operands within 2^15 ulp of powers of two
 * and of each other, 2 = exponents over [1e-150, 1e150]
 * (quotients that underflow to subnormal numbers are outside the claim: such a state fails Eq. 30 either way).  Used by tests/test_gpu_quotient.py. */
int srhd_quotient_check(unsigned long long n, unsigned long long seed, int dist,
                        unsigned long long* d_out, void* stream);

/* Human-readable text for a return code of this library (negative) or of CUDA (positive). */
const char* srhd_error_string(int code);

/* 1 if this build reproduces the reference operation order without fused multiply-add contraction
 * (libsrhd_b200_exact.so, used by the bit-parity tests), 0 for the production build. */
int srhd_build_is_exact(void);

/* Which compile-time variant this library is (one library per variant, like the EoS
 * choice of the paper's code): "eos=taub-mathews|gamma-5/3|gamma-4/3 energy=reduced|total precision=f64|f32
 * arithmetic=production|generic|exact".  eos: Eq. 10 or the polytropic P:107 Eq. 11; energy=total is the paper's "original scheme"
 * (the fifth conserved variable is E, evolved by the flux M) kept for its A/B runs; arithmetic=generic means
 * the paper's formulas as written with IEEE division and square root, exact the same without FMA contraction. */
const char* srhd_build_variant(void);

#ifdef __cplusplus
}
#endif
#endif /* SRHD_H_ */
