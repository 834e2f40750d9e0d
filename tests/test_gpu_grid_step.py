"""-m gpu: srhd_grid_step_cfl (one whole step of a uniform grid behind one call, uniform patch groups finished by
its pre-pass) against the two separate calls and against the oracle's tiled grid step."""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200.driver import GridStepper

pytestmark = pytest.mark.gpu


def _field(shape, seed):
    """Ambient gas at rest with a hot, moving, rough blob in one corner region: most patch groups are uniform."""
    nz, ny, nx = shape
    rng = np.random.default_rng(seed)
    prim = np.empty((5,) + shape)
    prim[0], prim[1:4], prim[4] = 1.0, 0.0, 1e-6
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    blob = (x - 20) ** 2 + (y - 12) ** 2 + (z - 24) ** 2 < 9 ** 2
    prim[0][blob] = 0.5 + rng.random(blob.sum())
    prim[4][blob] = 10.0 ** rng.uniform(-2, 2, blob.sum())
    for c in (1, 2, 3):
        prim[c][blob] = rng.normal(0, 2.0, blob.sum())
    return prim


@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("ppm", "hllc")])
@pytest.mark.parametrize("bc", [["periodic"] * 6, ["outflow"] * 6])
def test_fused_step_equals_two_calls_and_oracle(ref, recon, riemann, bc):
    shape, dh = (64, 32, 48), 1.0 / 64
    prim = _field(shape, seed=3)
    for exact in (True, False):
        a = GridStepper(shape, dh, bc, recon, riemann, cfl=0.4, exact=exact, fused=True).set_prim(prim)
        b = GridStepper(shape, dh, bc, recon, riemann, cfl=0.4, exact=exact, fused=False).set_prim(prim)
        n_uniform = []
        for step in range(4):                       # the first step starts from the grid (both take the same calls)
            a.step_async()
            b.step_async()
            torch.cuda.synchronize()
            sa, sb = a.last_stats(), b.last_stats()
            assert torch.equal(a.patches, b.patches), (exact, step)
            assert float(a.smax.cpu()) == float(b.smax.cpu())
            assert sa.algorithm_dict() == sb.algorithm_dict()
            assert sa.n_uniform_pg == sb.n_uniform_pg
            n_uniform.append(sa.n_uniform_pg)
        assert 0 < n_uniform[-1] < a.npg, n_uniform  # both kinds of patch group were present
        if exact:                                    # and the oracle, free running from the same start, bit for bit
            po = ref.params(recon, riemann)
            cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
            for step in range(4):
                cons, _ = ref.grid_step_tiled(cons, ref.cfl_dt(cons, 0.4, dh, po), dh, po, bc)
            assert np.array_equal(a.grid.cpu().numpy(), cons)


def test_fused_step_inflow_and_flux_output(ref):
    """Fixed-inflow ghost cells make the groups under the nozzle non-uniform; flux_out of a uniform group holds the
    flux of its one state on every patch face."""
    shape, dh, bc = (32, 32, 32), 1.0 / 32, ["outflow"] * 6
    prim = np.empty((5,) + shape)
    prim[0], prim[1:4], prim[4] = 1.0, 0.0, 1e-6
    mask = np.zeros(shape[1:], dtype=np.uint8)
    mask[3:7, 4:9] = 1
    pj = np.array([1e-2, 0.0, 0.0, 30.0, 1e-1])
    cj = B.prim2cons(torch.from_numpy(pj.reshape(5, 1).copy()).cuda()).cpu().numpy().ravel()
    for exact in (True, False):
        a = GridStepper(shape, dh, bc, "ppm", "hllc", exact=exact, inflow=(mask, cj), fused=True).set_prim(prim)
        b = GridStepper(shape, dh, bc, "ppm", "hllc", exact=exact, inflow=(mask, cj), fused=False).set_prim(prim)
        for step in range(3):
            a.step_async()
            b.step_async()
            torch.cuda.synchronize()
            assert torch.equal(a.patches, b.patches)
            assert a.last_stats().algorithm_dict() == b.last_stats().algorithm_dict()
        assert 0 < a.last_stats().n_uniform_pg < a.npg
    # flux output through the fused call == through srhd_patch_gather_speed + srhd_fluid_step_cfl
    par = B.params("ppm", "hllc")
    st = GridStepper(shape, dh, bc, "ppm", "hllc", inflow=(mask, cj)).set_prim(prim)
    st.step_async()
    inflow = st.inflow
    p_in = st.patches.clone()
    tiles, smax = B.patch_gather_speed(p_in, shape, par, bc, inflow)
    flux_b = torch.zeros((st.npg, 8, 6, 5, 8, 8), dtype=torch.float64, device="cuda")
    out_b, sb = B.fluid_step_cfl(tiles, 0.4, dh, smax, par, min_speed=st.smax_inflow, flux_out=flux_b)
    flux_a = torch.zeros_like(flux_b)
    out_a, smax_a, sa = B.grid_step_cfl(p_in, torch.empty_like(p_in), torch.empty_like(tiles), shape, 0.4, dh, par, bc,
                                        inflow, min_speed=st.smax_inflow, flux_out=flux_a)
    torch.cuda.synchronize()
    assert torch.equal(out_a, out_b) and torch.equal(flux_a, flux_b) and float(smax_a.cpu()) == float(smax.cpu())


@pytest.mark.parametrize("name", ["blast256", "jet_half"])
def test_fused_step_equals_two_calls_at_config_size(name):
    """The launch configuration bench.py times (GridStepper.step_async -> srhd_grid_step_cfl, production library) against
    the two separate calls on the blast wave at full size and on the jet at half size (nozzle, outflow): identical
    patches, S_max and counters after every one of 24 steps, with both kinds of patch group present."""
    from paper_2012_11130_b200 import workloads as wl
    inflow = None
    if name == "blast256":
        prim, dh, bc = wl.blast_wave(n=256)
    else:
        prim, dh, bc, (mask, pj) = wl.jet(nx=256, ny=256, nz=512, radius=0.04)
        cj = B.prim2cons(torch.from_numpy(pj.reshape(5, 1).copy()).cuda()).cpu().numpy().ravel()
        inflow = (mask, cj)
    shape = prim.shape[1:]
    a = GridStepper(shape, dh, bc, "ppm", "hllc", cfl=0.4, inflow=inflow, fused=True).set_prim(prim)
    b = GridStepper(shape, dh, bc, "ppm", "hllc", cfl=0.4, inflow=inflow, fused=False).set_prim(prim)
    del prim
    for step in range(24):
        a.step_async()
        b.step_async()
        if step % 6 == 5 or step < 2:
            torch.cuda.synchronize()
            sa, sb = a.last_stats(), b.last_stats()
            assert torch.equal(a.patches, b.patches), (name, step)
            assert float(a.smax.cpu()) == float(b.smax.cpu())
            assert sa.algorithm_dict() == sb.algorithm_dict() and sa.n_uniform_pg == sb.n_uniform_pg
    assert 0 < sa.n_uniform_pg < a.npg and sa.n_uniform_pg > 0.8 * a.npg
