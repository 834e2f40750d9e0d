// oracle/srhd_ref.hpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle for the GAMER-SR hot path
// (arXiv 2012.11130).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, link, import or call anything in oracle/.  It shares no code,
// header, table or helper with the CUDA path in paper_2012_11130_b200/csrc.
//
// Citations: "P:n" = /root/reference/PAPER.md line n; "S#/G#" = reading listed in DESIGN.md.
// Units c = k_B = m = 1.  T == Theta == p/rho (Eq. 18).
//
// State vectors:
//   primitive W = (rho, U^x, U^y, U^z, p)   -- FOUR-velocity (Eq. 8)
//   conserved U = (D, M^x, M^y, M^z, Etilde) -- REDUCED energy Etilde = E - D (Eq. 6)
// SoA convention of the C entry points: component c of state i at ptr[c*stride + i].
//
// Pin status (tests/test_oracle_*.py): EoS, prim2cons, cons2prim, max speed (incl. the
// relativistic factors of Eq. 26), wave speeds and their differences, HLLE/HLLC values, PLM/PPM properties, the
// fluid step (3-D diagonal wave of section 4.1, 40-digit one-step evaluation), the retry ladder (Python re-assembly of
// a pass; beta = 0 == first-order Godunov), the VL integrator, the coarse-fine hooks, the refinement flags and the
// variants (polytropic EoS, original scheme, single precision): pinned; tests/mutants.py checks that one-line
// mistakes in any of them fail a pin.  The values K, beta0 and the per-patch-group granularity of the ladder are
// readings (S3, S9); the PPM / limiter DETAILS (PPM is named by BASELINE.json only; S3, S4) are "parity unpinned"
// against the paper -- pinned by textbook properties only.
#pragma once
#include <cstddef>

// every state array and every scalar of the arithmetic is a `real`: double, or float in the SRHD_REF_F32 variant
// (the run-time parameters and the counters keep their types)
// SRHD_REF_EXT: x87 extended precision (64-bit significand, eps = 1.1e-19): the SAME algorithm with the SAME
// thresholds (Eq. 30 and the S10 floor stay at double's eps_machine / DBL_MIN) evaluated 2048 times more finely --
// the stand-in for "the true update" against which the fp64 oracle and the fp64 CUDA build are both measured
// (tests/test_gpu_truth.py); never the parity reference
#if defined(SRHD_REF_F32)
typedef float real;
#elif defined(SRHD_REF_EXT)
typedef long double real;
#else
typedef double real;
#endif

extern "C" {

struct srhd_ref_params {
  int    recon;            // 0 PLM, 1 PPM                           (PPM per BASELINE.json)
  int    riemann;          // 0 HLLE, 1 HLLC
  double minmod_coeff;     // beta0 in [1,2]                         (value: reading S3)
  int    max_retry;        // K reductions by 0.75, then beta = 0    (K: reading S9)
  double newton_rtol;      // stop when |delta| <= rtol*|htilde|     (reading S2)
  int    newton_max_iter;  // iteration cap                          (reading S2)
  int    ghost;            // MUSCL-Hancock: 2 (PLM) or 3 (PPM); VL: one more
  int    integrator;       // 0 MUSCL-Hancock (Toro 2011), 1 VL (Falle 1991; van Leer 2006)   (reading S18)
};

struct srhd_ref_stats {
  unsigned long long n_c2p_fail;      // Eq. 30 violations on input to a conversion
  unsigned long long n_retry_pg;      // patch groups that needed >= 1 retry
  unsigned long long n_unphys_final;  // output cells still violating Eq. 30 in the accepted pass
  unsigned long long newton_iters;    // Newton iterations of the algorithm's conversions (informational): every
                                      // tile cell once + both states of every face in the ACCEPTED pass
  double             max_speed;       // max S_max (Eq. 27) over the input interior cells
  unsigned long long n_passes;        // passes over patch groups, retries included (>= number of groups)
};

// --- O1 EoS (Eq. 10, Eq. 22, Eq. 16, Eq. 14) --------------------------
real srhd_ref_htilde_of_T(real T);
real srhd_ref_T_of_htilde(real ht);
real srhd_ref_dT_dhtilde(real ht);                       // P:591 Eq. A2
real srhd_ref_cs2_of_T(real T);                          // P:129 Eq. 14 (squared)
real srhd_ref_f_eq15(real ht, real musq);              // P:140-144 Eq. 15 right-hand side
real srhd_ref_df_eqA1(real ht, real musq);             // P:587 Eq. A1
real srhd_ref_htilde_guess(real L, real musq);         // P:602-618 Eq. A4 (reading G2), A6, A7

// --- O2/O3 conversions on n SoA states; all pointers are HOST pointers --------------------------
void srhd_ref_prim2cons(const real* prim, real* cons, size_t n, size_t stride);
void srhd_ref_cons2prim(const real* cons, real* prim, size_t n, size_t stride,
                        const srhd_ref_params* par, srhd_ref_stats* stats);
// optional diagnostics: per-state root htilde, iteration count and Eq.-30 flag (may be null)
void srhd_ref_cons2prim_diag(const real* cons, real* prim, size_t n, size_t stride,
                             const srhd_ref_params* par, real* htilde, int* iters,
                             unsigned char* unphys);

// --- O4 time step (Eq. 26-28) -------------------------------------------------------
// per-state U_max (Eq. 26, reading G1) from PRIMITIVES, and S_max = U_max/sqrt(1+U_max^2) (Eq. 27)
real srhd_ref_umax_of_prim(const real W[5]);
real srhd_ref_smax_of_umax(real umax);
void   srhd_ref_max_signal_speed(const real* cons, size_t n, size_t stride,
                                 const srhd_ref_params* par, real* max_speed);
// Eq. 30 as applied to an UPDATED cell (O9): ok[i] = 1 iff D > 0, Etilde > 0 and L > eps_machine
void   srhd_ref_is_physical(const real* cons, unsigned char* ok, size_t n, size_t stride);

// --- O5-O9 one fluid step ---------------------------------------------------------------------
// Box form: cons_in [5][nz+2g][ny+2g][nx+2g] (x fastest) -> cons_out [5][nz][ny][nx].
// Retry granularity = the whole box.  Returns the number of passes used (1 = no retry).
int srhd_ref_step_box(const real* cons_in, real* cons_out, int nx, int ny, int nz,
                      real dt, real dh, const srhd_ref_params* par, srhd_ref_stats* stats);
// Patch-group form (the C-ABI shape of SURVEY.md 8b):
//   cons_in  [npg][5][nxt][nxt][nxt], nxt = 16 + 2*ghost
//   cons_out [npg][8][5][8][8][8],    patch p = ix + 2*iy + 4*iz   (reading S13)
void srhd_ref_fluid_step(const real* cons_in, real* cons_out, int npg, real dt, real dh,
                         const srhd_ref_params* par, srhd_ref_stats* stats, int nthreads);

// The same step that also returns the fluxes through the six boundary faces of every 8^3 patch, as
// the AMR flux-correction step needs them (section 3.3(4)): flux_out [npg][8][6][5][8][8]
// (patch, face x-lo x-hi y-lo y-hi z-lo z-hi, component, in-face coordinates slower one first:
// (z,y) / (z,x) / (y,x)); fluxes of the accepted pass, positive along +axis.  May be null.
void srhd_ref_fluid_step_fluxes(const real* cons_in, real* cons_out, real* flux_out, int npg,
                                real dt, real dh, const srhd_ref_params* par,
                                srhd_ref_stats* stats, int nthreads);

// single Riemann flux along direction dir (0,1,2), for tests: WL/UL/WR/UR are 5-vectors
void srhd_ref_riemann_flux(int riemann, int dir, const real* WL, const real* UL,
                           const real* WR, const real* UR, real* F);
// acoustic wave speeds (reading S6) of one primitive state along dir, for tests:
// out[6] = {lambda_-, lambda_+, lambda_+ - v_n, v_n - lambda_-, 1 - lambda_+, 1 + lambda_-}
void srhd_ref_wave_speeds(int dir, const real* W, real* out);
// physical flux along dir (Eq. 4a, 4b; Eq. 7)
void srhd_ref_phys_flux(int dir, const real* W, const real* U, real* F);
// limited slope (reading S3) and 1-D face reconstruction of one component for tests:
real srhd_ref_limited_slope(real sL, real sR, real beta);
void   srhd_ref_recon_1d(int recon, const real* a /*5 values: i-2..i+2*/, real beta,
                         real beta0, real* am, real* ap);

// --- O10 uniform-grid helpers -------------------------------------------------------------------
// grid [5][nz][ny][nx].  bc[6] = {x_lo,x_hi,y_lo,y_hi,z_lo,z_hi}: 0 periodic, 1 outflow (copy).
// inflow_mask (may be null): [ny][nx] bytes; ghost cells with k<0 whose (wrapped/clamped) (i,j)
// has mask!=0 hold inflow_cons[5] (fixed inflow at the z_lo face), outflow elsewhere.
void srhd_ref_grid_pad(const real* grid, real* padded, int nx, int ny, int nz, int g,
                       const int* bc, const unsigned char* inflow_mask, const real* inflow_cons);
void srhd_ref_grid_gather(const real* grid, real* cons_in, int nx, int ny, int nz, int g,
                          const int* bc, const unsigned char* inflow_mask,
                          const real* inflow_cons);
void srhd_ref_grid_scatter(const real* cons_out, real* grid, int nx, int ny, int nz);

// --- coarse-fine hooks (section 3.3(3), section 3.3(4)); see srhd_ref.cpp for layouts ------------
// flux correction of the coarse cells next to a coarse-fine interface, skipped where the corrected cell fails
// Eq. 30; returns the number of skipped cells
unsigned long long srhd_ref_flux_correction(real* patches, const real* flux_coarse, const real* flux_fine,
                                            const int* face_patch, const int* face_id, int nf, real dt, real dh);
// 2x ghost-zone interpolation of conserved variables with the primitive-variable fallback; returns the number
// of coarse cells that fell back
unsigned long long srhd_ref_ghost_interp(const real* coarse, int nx, int ny, int nz, real* fine, real beta,
                                         const srhd_ref_params* par, unsigned char* fallback);

// --- refinement criteria of the SRHD module (section 3.1; Eq. 33) -----------------
// per 8^3 patch of ghosted patch-group tiles: flag = any cell with
//   (|dQ_x| + |dQ_y| + |dQ_z|) / (2|Q|) > c_q  (centred differences over two cells: reading S17)
//   or |M|/D > mom_over_d (skipped when 0).  quantity: 0 none, 1 D, 2 Etilde, 3 rho, 4 Lorentz factor.
void srhd_ref_refine_flags(const real* cons_in, int npg, int quantity, real c_q, real mom_over_d,
                           const srhd_ref_params* par, unsigned char* flags);
}
