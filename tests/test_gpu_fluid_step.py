"""-m gpu parity: srhd_fluid_step (and the grid helpers) vs the CPU oracle on seeded patch groups.

exact build: bit-identical output and identical counters (same IEEE operations, same decisions);
production build: per-cell error (norm S14) <= 1e-11 after one step (north_star).
"""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200 import workloads as wl
from tests.gpu_util import step_err

pytestmark = pytest.mark.gpu
TOL_STEP = 1e-11   # BASELINE.json north_star: relative error per cell after one step

COMBOS = [("plm", "hlle"), ("plm", "hllc"), ("ppm", "hlle"), ("ppm", "hllc")]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_tiles(ref, npg, ghost, seed, **kw):
    prim = wl.random_patch_groups(npg, ghost, seed=seed, **kw)
    nxt = 16 + 2 * ghost
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    return np.ascontiguousarray(cons.reshape(5, npg, nxt, nxt, nxt).transpose(1, 0, 2, 3, 4))


def cfl_dt(ref, tiles, dh, cfl=0.4):
    return cfl * dh / ref.max_signal_speed(tiles.transpose(1, 0, 2, 3, 4).reshape(5, -1))


@pytest.mark.parametrize("recon,riemann", COMBOS)
def test_one_step_parity(ref, recon, riemann):
    po = ref.params(recon, riemann)
    npg, dh = 5, 1.0 / 64
    tiles = make_tiles(ref, npg, po.ghost, seed=11 + po.ghost)
    dt = cfl_dt(ref, tiles, dh)
    want, st = ref.fluid_step(tiles, dt, dh, po)
    # exact build: bit for bit, counters included
    pe = B.params(recon, riemann, exact=True)
    got, sbuf = B.fluid_step(dev(tiles), dt, dh, pe, exact=True)
    s = B.stats_to_host(sbuf)
    got = got.cpu().numpy()
    assert np.array_equal(got, want), float(np.nanmax(step_err(got, want, 2)))
    assert s.algorithm_dict() == st.as_dict()
    # production build: tolerance
    got, sbuf = B.fluid_step(dev(tiles), dt, dh, B.params(recon, riemann))
    s = B.stats_to_host(sbuf)
    got = got.cpu().numpy()
    assert np.all(np.isfinite(got))
    err = step_err(got, want, 2)
    assert err.max() <= TOL_STEP, err.max()
    assert (s.n_retry_pg, s.n_unphys_final, s.n_c2p_fail) == (st.n_retry_pg, st.n_unphys_final, st.n_c2p_fail)
    assert abs(s.max_speed - st.max_speed) <= 1e-13 * st.max_speed


@pytest.mark.parametrize("recon,riemann", [("plm", "hllc"), ("ppm", "hllc")])
def test_retry_ladder_parity(ref, recon, riemann):
    """A time step far above the CFL limit on rough, fast data forces Eq. 30 failures: the retry
    decisions (per patch group, beta *= 0.75 ... then 0) must match the oracle's exactly."""
    po = ref.params(recon, riemann, max_retry=3)
    npg, dh = 4, 1.0 / 64
    tiles = make_tiles(ref, npg, po.ghost, seed=5, umax=30.0, rough=3.0, log_theta=(-8.0, 2.0))
    dt = 4.0 * cfl_dt(ref, tiles, dh)
    want, st = ref.fluid_step(tiles, dt, dh, po)
    assert st.n_retry_pg > 0, "test input must trigger the retry ladder"
    pe = B.params(recon, riemann, max_retry=3, exact=True)
    got, sbuf = B.fluid_step(dev(tiles), dt, dh, pe, exact=True)
    s = B.stats_to_host(sbuf)
    assert np.array_equal(got.cpu().numpy(), want, equal_nan=True)
    assert s.algorithm_dict() == st.as_dict()


def test_uniform_state_is_a_fixed_point(ref):
    """All flux differences are x - x: bit-exact fixed point for any gamma, T (SURVEY 8c pin)."""
    for recon in ("plm", "ppm"):
        p = B.params(recon, "hllc")
        nxt = 16 + 2 * p.ghost
        W = np.array([0.7, 3.0e2, -1.0e2, 5.0e1, 1e-4])
        prim = np.broadcast_to(W[:, None], (5, 2 * nxt ** 3)).copy()
        cons = B.prim2cons(dev(prim))
        tiles = cons.reshape(5, 2, nxt, nxt, nxt).permute(1, 0, 2, 3, 4).contiguous()
        out, sbuf = B.fluid_step(tiles, 1e-3, 1e-2, p)
        out = out.cpu().numpy()
        c0 = cons[:, 0].cpu().numpy()
        assert np.array_equal(out, np.broadcast_to(c0[None, None, :, None, None, None], out.shape))
        assert B.stats_to_host(sbuf).n_retry_pg == 0


def test_npg_zero_and_many(ref):
    p = B.params("plm", "hlle")
    e = torch.empty((0, 5, 20, 20, 20), dtype=torch.float64, device="cuda")
    out, sbuf = B.fluid_step(e, 0.1, 1.0, p)
    assert out.shape[0] == 0 and B.stats_to_host(sbuf).newton_iters == 0
    # more patch groups than SMs (several waves, ragged last wave): sampled parity
    po = ref.params("plm", "hlle")
    base = make_tiles(ref, 3, 2, seed=3)
    npg = 2 * 148 + 5
    tiles = np.ascontiguousarray(base[np.arange(npg) % 3])
    dt = cfl_dt(ref, base, 1.0 / 64)
    want, _ = ref.fluid_step(base, dt, 1.0 / 64, po)
    got, _ = B.fluid_step(dev(tiles), dt, 1.0 / 64, B.params("plm", "hlle", exact=True), exact=True)
    got = got.cpu().numpy()
    for pg in (0, 1, 2, 147, 148, 149, npg - 2, npg - 1):
        assert np.array_equal(got[pg], want[pg % 3])


@pytest.mark.parametrize("ghost", [2, 3])
def test_grid_gather_scatter_bit_exact(ref, ghost):
    rng = np.random.default_rng(ghost)
    grid = rng.standard_normal((5, 32, 16, 48))
    mask = (rng.random((16, 48)) < 0.2).astype(np.uint8)
    vals = np.arange(5) + 0.5
    for bc in (["periodic"] * 6, ["outflow"] * 6, ["outflow", "periodic", "periodic", "outflow", "outflow", "outflow"]):
        for inflow in (None, (mask, vals)):
            want = ref.grid_gather(grid, ghost, bc, inflow)
            di = None if inflow is None else (dev(mask), vals)
            got = B.grid_gather(dev(grid), ghost, bc, di).cpu().numpy()
            assert np.array_equal(got, want)
    out = rng.standard_normal((6, 8, 5, 8, 8, 8))
    want = ref.grid_scatter(out, (32, 16, 48))
    got = B.grid_scatter(dev(out), (32, 16, 48)).cpu().numpy()
    assert np.array_equal(got, want)


@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("ppm", "hllc")])
def test_patch_boundary_fluxes_parity(ref, recon, riemann):
    """srhd_fluid_step_fluxes: the fluxes through the faces of every 8^3 patch; a retry pass
    must leave the ACCEPTED pass's fluxes behind.  Exact build bit for bit, production to 1e-11 of the
    largest flux of the face."""
    po = ref.params(recon, riemann, max_retry=3)
    npg, dh = 4, 1.0 / 64
    for rough_dt in (False, True):
        kw = dict(umax=30.0, rough=3.0, log_theta=(-8.0, 2.0)) if rough_dt else {}
        tiles = make_tiles(ref, npg, po.ghost, seed=5 if rough_dt else 11 + po.ghost, **kw)
        dt = (4.0 if rough_dt else 1.0) * cfl_dt(ref, tiles, dh)
        want, wflux, st = ref.fluid_step_fluxes(tiles, dt, dh, po)
        assert st.n_retry_pg > 0 or not rough_dt          # the rough case must go through the ladder
        got, gflux, sbuf = B.fluid_step_fluxes(dev(tiles), dt, dh, B.params(recon, riemann, max_retry=3, exact=True),
                                               exact=True)
        assert np.array_equal(got.cpu().numpy(), want, equal_nan=True)
        assert np.array_equal(gflux.cpu().numpy(), wflux, equal_nan=True)
        assert B.stats_to_host(sbuf).algorithm_dict() == st.as_dict()
        if not rough_dt:
            got, gflux, sbuf = B.fluid_step_fluxes(dev(tiles), dt, dh, B.params(recon, riemann, max_retry=3))
            assert B.stats_to_host(sbuf).n_retry_pg == st.n_retry_pg      # same rungs of the ladder
            gf = gflux.cpu().numpy()
            scale = np.abs(wflux).max(axis=(4, 5), keepdims=True)
            assert (np.abs(gf - wflux) / scale).max() <= 1e-11
            plain, _ = B.fluid_step(dev(tiles), dt, dh, B.params(recon, riemann, max_retry=3))
            assert np.array_equal(plain.cpu().numpy(), got.cpu().numpy())


def test_speed_of_light_time_step_option(ref):
    """the second CFL condition replaces S_max by c: dt = C dh exactly, no reduction kernel."""
    from paper_2012_11130_b200 import workloads as wl
    from paper_2012_11130_b200.driver import GridStepper
    prim, dh, bc = wl.shock_tube(n_long=32, n_trans=16)
    a = GridStepper(prim.shape[1:], dh, bc, "plm", "hllc", cfl=0.5, dt_speed="light").set_prim(prim)
    b = GridStepper(prim.shape[1:], dh, bc, "plm", "hllc", cfl=0.5).set_prim(prim)
    assert a.step() == 0.5 * dh
    assert b.step() > 0.5 * dh                        # S_max < c: the signal-speed condition allows more
    po = ref.params("plm", "hllc")
    o = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    want, _ = ref.grid_step_tiled(o, 0.5 * dh, dh, po, bc)
    from tests.gpu_util import l1_rel
    assert l1_rel(a.grid.cpu().numpy(), want).max() <= 1e-11


def test_fused_scatter_speed_equals_scatter_then_max_signal_speed(ref):
    rng = np.random.default_rng(4)
    prim = wl.random_patch_groups(6, 0, seed=8, rough=0.1)             # (6,5,16,16,16) primitives
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1)).reshape(5, 6, 16, 16, 16)
    # patch layout (npg,8,5,8,8,8) of a 32x16x48 grid
    blocks = cons.transpose(1, 0, 2, 3, 4)
    patches = np.ascontiguousarray(
        blocks.reshape(6, 5, 2, 8, 2, 8, 2, 8).transpose(0, 2, 4, 6, 1, 3, 5, 7).reshape(6, 8, 5, 8, 8, 8))
    for exact in (True, False):
        par = B.params("plm", "hllc", exact=exact)
        grid, smax = B.grid_scatter_speed(dev(patches), (32, 16, 48), par, exact=exact)
        plain = B.grid_scatter(dev(patches), (32, 16, 48), exact=exact)
        assert torch.equal(grid, plain)
        assert np.array_equal(grid.cpu().numpy(), ref.grid_scatter(patches, (32, 16, 48)))
        sep = B.max_signal_speed(plain.reshape(5, -1).contiguous(), par, exact=exact)
        assert float(smax.cpu()) == float(sep.cpu())
        want = ref.max_signal_speed(ref.grid_scatter(patches, (32, 16, 48)).reshape(5, -1))
        assert abs(float(smax.cpu()) - want) <= (0.0 if exact else 1e-13) * want
    assert rng is not None


def test_device_side_time_step_equals_host_side(ref):
    """srhd_fluid_step_cfl forms dt = C dh / max(S_max, floor) on the device (Eq. 28): a run enqueued
    without any host synchronisation must equal, bit for bit, the run whose dt went through the host."""
    from paper_2012_11130_b200.driver import GridStepper
    prim, dh, bc, inflow = wl.jet(nx=32, ny=32, nz=64, radius=0.16)
    mask, prim_jet = inflow
    cj = B.prim2cons(dev(prim_jet.reshape(5, 1))).cpu().numpy().ravel()
    a = GridStepper(prim.shape[1:], dh, bc, "ppm", "hllc", cfl=0.4, inflow=(mask, cj)).set_prim(prim)
    b = GridStepper(prim.shape[1:], dh, bc, "ppm", "hllc", cfl=0.4, inflow=(mask, cj)).set_prim(prim)
    for _ in range(4):
        a.step()
        b.step_async()
    torch.cuda.synchronize()
    assert torch.equal(a.grid, b.grid)
    assert float(a.smax.cpu()) == float(b.smax.cpu())
    assert a.last_stats().as_dict() == b.last_stats().as_dict()


@pytest.mark.parametrize("ghost", [2, 3])
def test_patch_gather_speed_equals_scatter_then_gather(ref, ghost):
    """srhd_patch_gather_speed: ghost-zone fill straight from the patch layout (+ S_max) must equal
    srhd_grid_scatter -> srhd_grid_gather (+ srhd_max_signal_speed) bit for bit, for every boundary type."""
    rng = np.random.default_rng(ghost)
    shape = (32, 16, 48)
    prim = np.empty((5,) + shape)
    prim[0] = 10.0 ** rng.uniform(-1, 1, shape)
    prim[1:4] = rng.standard_normal((3,) + shape)
    prim[4] = prim[0] * 10.0 ** rng.uniform(-3, 1, shape)
    grid = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    npg = 6
    # grid -> patch layout (the inverse of the oracle's scatter)
    patches = np.empty((npg, 8, 5, 8, 8, 8))
    for pg in range(npg):
        gx, gy, gz = pg % 3, (pg // 3) % 1, pg // 3
        blk = grid[:, gz * 16:gz * 16 + 16, gy * 16:gy * 16 + 16, gx * 16:gx * 16 + 16]
        patches[pg] = blk.reshape(5, 2, 8, 2, 8, 2, 8).transpose(1, 3, 5, 0, 2, 4, 6).reshape(8, 5, 8, 8, 8)
    assert np.array_equal(ref.grid_scatter(patches, shape), grid)
    mask = (rng.random((16, 48)) < 0.2).astype(np.uint8)
    vals = ref.prim2cons(np.array([[1e-2], [0.0], [0.0], [5.0], [1e-1]]))[:, 0]
    recon = "plm" if ghost == 2 else "ppm"
    for bc in (["periodic"] * 6, ["outflow"] * 6, ["outflow", "periodic", "periodic", "outflow", "outflow", "outflow"]):
        for inflow in (None, (mask, vals)):
            want = ref.grid_gather(grid, ghost, bc, inflow)
            for exact in (True, False):
                par = B.params(recon, "hllc", exact=exact)
                di = None if inflow is None else (dev(mask), vals)
                tiles, smax = B.patch_gather_speed(dev(patches), shape, par, bc, di, exact=exact)
                assert np.array_equal(tiles.cpu().numpy(), want)
                sep = B.max_signal_speed(dev(grid).reshape(5, -1).contiguous(), par, exact=exact)
                assert float(smax.cpu()) == float(sep.cpu())


@pytest.mark.parametrize("recon,riemann", [("plm", "hllc"), ("ppm", "hllc"), ("plm", "hlle")])
def test_retry_ladder_parity_production_build(ref, recon, riemann):
    """the PRODUCTION library on data that walks the retry ladder: every patch group ends on
    the same rung as the oracle's (same number of passes in total, same retried groups, same count of cells
    left unphysical after the last rung), and the cells of groups that end physically agree to 1e-11."""
    po = ref.params(recon, riemann, max_retry=3)
    dh = 1.0 / 64
    for seed, mult, kw in ((5, 4.0, dict(umax=30.0, rough=3.0, log_theta=(-8.0, 2.0))),
                           (9, 1.0, dict(umax=10.0, rough=1.0, log_theta=(-6.0, 2.0))),
                           (11 + po.ghost, 1.0, {})):
        tiles = make_tiles(ref, 6, po.ghost, seed=seed, **kw)
        dt = mult * cfl_dt(ref, tiles, dh)
        per_group = [ref.fluid_step(tiles[g:g + 1], dt, dh, po) for g in range(tiles.shape[0])]
        want = np.concatenate([w for w, _ in per_group])
        par = B.params(recon, riemann, max_retry=3)
        for g, (w, st) in enumerate(per_group):       # group by group: the rung of EACH group
            got, sbuf = B.fluid_step(dev(tiles[g:g + 1]), dt, dh, par)
            s = B.stats_to_host(sbuf)
            assert (s.n_passes, s.n_retry_pg, s.n_unphys_final, s.n_c2p_fail) == \
                   (st.n_passes, st.n_retry_pg, st.n_unphys_final, st.n_c2p_fail), (seed, g)
            if st.n_unphys_final == 0:
                assert step_err(got.cpu().numpy(), w, 2).max() <= TOL_STEP, (seed, g, st.n_passes)
        got, sbuf = B.fluid_step(dev(tiles), dt, dh, par)       # and the batch as one launch
        s = B.stats_to_host(sbuf)
        assert s.n_passes == sum(st.n_passes for _, st in per_group)
        assert s.exec_c2p >= tiles.shape[0] * ((16 + 2 * po.ghost) ** 3)      # the executed-work counters are live
        assert np.array_equal(np.isfinite(got.cpu().numpy()), np.isfinite(want))


@pytest.mark.parametrize("recon,riemann", COMBOS)
def test_uniform_tile_path_parity(ref, recon, riemann):
    """Tiles that hold ONE state bit for bit take the uniform-tile path of the kernel (srhd_stats.n_uniform_pg):
    output, patch-boundary fluxes and every algorithm counter must be what the oracle's full march gives.  Tiles
    that differ from uniform in one cell (first / last tile cell, one interior cell), and a uniform state that fails
    Eq. 30, must take the general path and match too."""
    po = ref.params(recon, riemann)
    nxt, dh = 16 + 2 * po.ghost, 1.0 / 64
    states = np.array([[0.7, 3.0e2, -1.0e2, 5.0e1, 1e-4],        # fast and cold
                       [1.0, 0.0, 0.0, 0.0, 1e-6],               # ambient gas at rest (blast / jet configs)
                       [2.5e-3, -0.4, 0.3, 2.0, 40.0]])          # hot
    cons = ref.prim2cons(states.T.copy())                         # (5, 3)
    npg = 7
    tiles = np.empty((npg, 5, nxt, nxt, nxt))
    for pg in range(npg):
        tiles[pg] = cons[:, pg % 3][:, None, None, None]
    tiles[3, 0, 0, 0, 0] *= 1.0 + 2.0 ** -52                      # one ulp in the first tile cell
    tiles[4, 4, -1, -1, -1] *= 1.0 + 2.0 ** -52                   # ... in the last one
    tiles[5, 2, nxt // 2, nxt // 2, nxt // 2] += 1e-3             # one interior cell
    tiles[6, 4] = -1e-9                                           # uniform but unphysical (Etilde < 0): general path
    dt = 0.4 * dh
    want, wflux, st = ref.fluid_step_fluxes(tiles, dt, dh, po)
    pe = B.params(recon, riemann, exact=True)
    got, gflux, sbuf = B.fluid_step_fluxes(dev(tiles), dt, dh, pe, exact=True)
    s = B.stats_to_host(sbuf)
    assert s.n_uniform_pg == 3
    assert np.array_equal(got.cpu().numpy(), want, equal_nan=True)
    assert np.array_equal(gflux.cpu().numpy(), wflux, equal_nan=True)
    assert s.algorithm_dict() == st.as_dict()
    got, sbuf = B.fluid_step(dev(tiles), dt, dh, pe, exact=True)  # without flux output
    assert np.array_equal(got.cpu().numpy(), want, equal_nan=True)
    assert B.stats_to_host(sbuf).algorithm_dict() == st.as_dict()
    # production build: the uniform tiles reproduce their input bit for bit, the rest to the step tolerance
    got, gflux, sbuf = B.fluid_step_fluxes(dev(tiles), dt, dh, B.params(recon, riemann))
    s = B.stats_to_host(sbuf)
    got = got.cpu().numpy()
    assert s.n_uniform_pg == 3
    assert np.array_equal(got[:3], want[:3])
    assert step_err(got[:6], want[:6], 2).max() <= TOL_STEP
    fscale = np.abs(wflux[:3]).max(axis=(1, 2, 3, 4, 5), keepdims=True)
    assert (np.abs(gflux.cpu().numpy()[:3] - wflux[:3]) / fscale).max() <= 1e-13
    assert (s.n_retry_pg, s.n_passes) == (st.n_retry_pg, st.n_passes)
