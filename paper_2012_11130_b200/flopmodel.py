"""Algorithmic operation counts of the hot path, used by bench.py's roofline.

Hand count of the paper's formulas exactly as written in DESIGN.md section 4 (no common-subexpression
sharing beyond what the formula shows): every +, -, *, /, sqrt and each half of an explicit fma is
ONE flop; comparisons, abs, min/max, selects and sign flips are free.  Counts are per call of the
named formula; `k` is the number of Newton-Raphson iterations (measured: srhd_stats.newton_iters).

These are ALGORITHMIC figures: halo cells a tiled kernel recomputes, and the instruction expansion
of fp64 division / sqrt on the SM (about 10 / 13 fp64-pipe instructions), are not counted.
"""

HTILDE_OF_T = 8            # Eq. 22
T_OF_HTILDE = 14           # Eq. 16
T_DT_OF_HTILDE = 26        # Eq. 16 + Eq. A2 sharing the square root
F_EQ15 = 13                # Eq. 15 right-hand side
DF_EQA1 = 25               # Eq. A1
NEWTON_ITER = T_DT_OF_HTILDE + F_EQ15 + DF_EQA1 + 3 + 1   # (f-L)/f', update, stop test  = 68
C2P_SETUP = 12             # canonical L: 4 divisions, two fma + one product, x+2, one fma
C2P_GUESS = 15             # A7 threshold + A4 or A6 (mean of the two branches)
C2P_FINISH = 29            # Eq. 17, 8, 5a, 16, 18
C2P_FIXED = C2P_SETUP + C2P_GUESS + C2P_FINISH            # 56, plus NEWTON_ITER per iteration
P2C = 45                   # Eq. 18, 22, 8, 5a, 5b, 15, 23
PHYS_FLUX = 15             # Eq. 4a, 4b, 7 along one direction (incl. gamma and v)
UMAX = 36                  # Eq. 14, 26 from primitives
LIMITED_SLOPE = 5          # reading S3
PLM_COMPONENT = 10         # two differences, slope, two edge values
PPM_COMPONENT = 42         # four differences, three slopes, two faces, CW84 monotonisation
SIDE_SETUP = 46            # one side of a Riemann problem: Eq. 14, S6 eigenvalues, physical flux
HLLE = 37
HLLC = 113                 # reading S7
UPDATE = 35                # reading S12: seven operations per component
EQ30_CHECK = 12


def c2p(k):
    return C2P_FIXED + NEWTON_ITER * k


def fluid_step_flops_per_cell(recon, riemann, k_mean):
    """One interior cell advanced one step with no halo redundancy: centre cons2prim + U_max,
    reconstruction in 3 directions, Hancock half step (6 prim2cons, 6 fluxes), 3 faces per cell
    (2 cons2prim + Riemann solver each), update + Eq. 30 check."""
    rec = 15 * (PLM_COMPONENT if recon in (0, "plm") else PPM_COMPONENT)
    hancock = 6 * (P2C + PHYS_FLUX) + 15 + 15 + 30
    face = 2 * c2p(k_mean) + 2 * SIDE_SETUP + (HLLE if riemann in (0, "hlle") else HLLC)
    return c2p(k_mean) + UMAX + rec + hancock + 3 * face + UPDATE + EQ30_CHECK


def conversions_per_cell_in_kernel(ghost):
    """cons2prim calls the fused kernel performs per interior cell: every tile cell once (pass 0)
    plus two per face of the 3 x 17 x 16^2 faces of a patch group."""
    nxt = 16 + 2 * ghost
    return (nxt ** 3 + 2 * 3 * 17 * 256) / 4096.0


# Algorithmic HBM bytes per cell update of srhd_fluid_step: 5 doubles in + 5 doubles out.
FLUID_STEP_BYTES_PER_CELL = 80.0
# B200 fp64 ALU peak from the unit counts: 148 SMs x 64 fp64 lanes x 2 flops (DFMA) x clock
FP64_LANES_PER_SM = 64
NUM_SMS = 148


def fp64_peak_tflops(sm_mhz=1965.0):
    return NUM_SMS * FP64_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def fluid_step_flops_executed(recon, riemann, ncell, exec_c2p, exec_newton, exec_riemann, exec_hancock):
    """Flops of the work the kernel actually executed (srhd_stats.exec_*): conversions and their Newton
    iterations (retry passes, ghost-zone cells and shortcuts as they happened), Riemann solves, edge-state
    pairs of the Hancock stage, plus the per-cell update / Eq. 30 check / U_max of the interior cells."""
    solver = HLLE if riemann in (0, "hlle") else HLLC
    rec = 5 * (PLM_COMPONENT if recon in (0, "plm") else PPM_COMPONENT)
    hancock = rec + 2 * (P2C + PHYS_FLUX) + 5 + 10 + 10       # per (cell, direction): dF, share of the sum, two adds
    return (exec_c2p * C2P_FIXED + exec_newton * NEWTON_ITER + exec_riemann * (2 * SIDE_SETUP + solver) +
            exec_hancock * hancock + ncell * (UPDATE + EQ30_CHECK + UMAX))


def fluid_step_flops_per_cell_survey(recon, riemann, k_mean):
    """The same quantity with SURVEY.md section 8(a)'s own per-step counts (simple / div / sqrt operations, each
    counted as ONE flop): A1 cons->prim (40+38k)/(5+4k)/(2.5+k); A2 16/1/2; A3 PLM 210/15/0 or PPM 420/15/0;
    A4 282/30/18; A5 = 6 x A1; A6 per face HLLC 123/9/5 or HLLE 85/7/4, three faces per cell; A7 30; A8 10/1/0.
    It charges 43 flops per Newton iteration where the count above charges 68 (it shares T and dT/dhtilde between f
    and f'), so it comes out about 15-20 % lower; bench.py prints both and says which one `frac` uses."""
    a1 = 47.5 + 43.0 * k_mean
    a3 = 225.0 if recon in (0, "plm") else 435.0
    a6 = 3 * (96.0 if riemann in (0, "hlle") else 137.0)
    return a1 + 19.0 + a3 + 330.0 + 6 * a1 + a6 + 30.0 + 11.0
