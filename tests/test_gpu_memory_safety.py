"""-m gpu: bounds, initialisation and determinism checks of our own (compute-sanitizer is closed on this GPU
pool -- gpurun answers "closed on this pool and stays closed" -- so SURVEY.md section 5's memcheck / initcheck /
racecheck runs are replaced by what can be checked from outside the kernels):

  * out-of-bounds WRITES: every output buffer sits between guard regions filled with a bit pattern that must
    survive the launch; inputs are followed by poisoned (NaN) memory so that an out-of-bounds READ that
    matters turns the bit-exact comparison with the oracle red;
  * uninitialised output: outputs are pre-filled with NaN and must be overwritten completely;
  * races: a data race in the shared-memory pipeline shows up as run-to-run differences; the same launch is
    repeated 12 times (and interleaved with another kernel on a second stream) and must give the same bits.

All four fluid_step_kernel instantiations, with and without the flux output, with a forced retry.
"""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200 import workloads as wl

pytestmark = pytest.mark.gpu
GUARD = 4096          # doubles on each side
PATTERN = -1.2345678901234567e+123


def guarded(shape, fill=float("nan")):
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * GUARD,), PATTERN, dtype=torch.float64, device="cuda")
    view = buf[GUARD:GUARD + n].view(*shape)
    view.fill_(fill)
    return buf, view


def guards_intact(buf):
    return bool((buf[:GUARD] == PATTERN).all()) and bool((buf[-GUARD:] == PATTERN).all())


def _tiles(ref, npg, ghost, seed, **kw):
    prim = wl.random_patch_groups(npg, ghost, seed=seed, **kw)
    nxt = 16 + 2 * ghost
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    return np.ascontiguousarray(cons.reshape(5, npg, nxt, nxt, nxt).transpose(1, 0, 2, 3, 4))


@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("plm", "hllc"), ("ppm", "hlle"), ("ppm", "hllc")])
@pytest.mark.parametrize("forced_retry", [False, True])
def test_guards_poison_and_determinism(ref, recon, riemann, forced_retry):
    po = ref.params(recon, riemann, max_retry=2)
    npg, dh = 3, 1.0 / 64
    kw = dict(umax=30.0, rough=3.0, log_theta=(-8.0, 2.0)) if forced_retry else {}
    tiles = _tiles(ref, npg, po.ghost, seed=5 if forced_retry else 11 + po.ghost, **kw)
    dt = (4.0 if forced_retry else 0.4) * dh / ref.max_signal_speed(tiles.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    want, wflux, st = ref.fluid_step_fluxes(tiles, dt, dh, po)
    ibuf, d_in = guarded(tiles.shape)                 # input followed (and preceded) by poison
    ibuf[:GUARD] = float("nan")
    ibuf[-GUARD:] = float("nan")
    d_in.copy_(torch.from_numpy(tiles))
    side = torch.cuda.Stream()
    for exact in (True, False):
        par = B.params(recon, riemann, max_retry=2, exact=exact)
        first = None
        for rep in range(12):
            obuf, out = guarded((npg, 8, 5, 8, 8, 8))
            fbuf, flux = guarded((npg, 8, 6, 5, 8, 8))
            sbuf_g, stats = guarded((B.new_stats().numel() // 8,), fill=0.0)
            if rep % 3 == 2:                          # another kernel of ours in flight on a second stream
                with torch.cuda.stream(side):
                    B.cons2prim(d_in[0].reshape(5, -1).contiguous(), exact=exact)
            B.fluid_step_fluxes(d_in, dt, dh, par, cons_out=out, flux_out=flux, stats=stats.view(torch.uint8), exact=exact)
            plain, _ = B.fluid_step(d_in, dt, dh, par, exact=exact)
            torch.cuda.synchronize()
            assert guards_intact(obuf) and guards_intact(fbuf) and guards_intact(sbuf_g), (recon, riemann, rep)
            assert not bool(torch.isnan(out).any()) or forced_retry      # every output cell was written
            assert not bool((flux != flux).all())
            assert torch.equal(out, plain) or forced_retry and bool(torch.isnan(out).any())
            res = (out.clone(), flux.clone(), stats.clone())
            if first is None:
                first = res
                if exact:
                    assert np.array_equal(out.cpu().numpy(), want, equal_nan=True)
                    assert np.array_equal(flux.cpu().numpy(), wflux, equal_nan=True)
            else:
                for a, b in zip(first, res):          # bit-identical from run to run
                    assert torch.equal(a.view(torch.int64), b.view(torch.int64)), (recon, riemann, exact, rep)


def test_state_list_kernels_respect_their_bounds(ref):
    for n in (1, 31, 32, 33, 1000, 4097):            # ragged tails of the vectorised loads
        prim = wl.conversion_states(n, seed=n, log_gamma=(0, 2))
        for exact in (True, False):
            pbuf, d_prim = guarded((5, n))
            d_prim.copy_(torch.from_numpy(prim))
            cbuf, d_cons = guarded((5, n))
            bbuf, d_back = guarded((5, n))
            B.prim2cons(d_prim, cons=d_cons, exact=exact)
            B.cons2prim(d_cons, prim=d_back, exact=exact)
            s = B.max_signal_speed(d_cons, exact=exact)
            torch.cuda.synchronize()
            assert guards_intact(cbuf) and guards_intact(bbuf) and guards_intact(pbuf)
            assert bool(torch.isfinite(d_cons).all()) and bool(torch.isfinite(d_back).all()) and float(s.cpu()) > 0


@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("ppm", "hllc")])
def test_grid_step_guards_and_determinism(recon, riemann):
    """srhd_grid_step_cfl (own-uniform flags, pre-pass, march) on a grid with both kinds of patch group: the two
    patch buffers and the tile scratch sit between guard regions, the output is pre-filled with NaN, the tile scratch
    of a uniform group must stay untouched, and 8 repetitions (every third with another kernel in flight on a second
    stream) give the same bits.  The tile-based calls with the uniform-tile pre-pass (MUSCL-Hancock and VL) likewise."""
    shape, dh, bc = (32, 32, 48), 1.0 / 32, ["periodic", "periodic", "outflow", "outflow", "periodic", "periodic"]
    rng = np.random.default_rng(7)
    prim = np.empty((5,) + shape)
    prim[0], prim[1:4], prim[4] = 1.0, 0.0, 1e-6
    prim[:, 4:12, 6:14, 20:30] = np.stack([0.5 + rng.random((8, 8, 10)), *rng.normal(0, 1.0, (3, 8, 8, 10)),
                                           10.0 ** rng.uniform(-2, 1, (8, 8, 10))])
    par = B.params(recon, riemann)
    npg = (shape[0] // 16) * (shape[1] // 16) * (shape[2] // 16)
    nxt = 16 + 2 * par.ghost
    cons = B.prim2cons(torch.from_numpy(prim.reshape(5, -1)).cuda()).reshape(5, *shape).contiguous()
    tiles0 = B.grid_gather(cons, par.ghost, bc)
    smax = B.max_signal_speed(cons.view(5, -1), par)
    p0, _ = B.fluid_step_cfl(tiles0, 0.4, dh, smax, par)              # a state in the patch layout to start from
    ibuf, p_in = guarded((npg, 8, 5, 8, 8, 8))
    ibuf[:GUARD] = float("nan")
    ibuf[-GUARD:] = float("nan")
    p_in.copy_(p0)
    side = torch.cuda.Stream()
    first = None
    for rep in range(8):
        obuf, p_out = guarded((npg, 8, 5, 8, 8, 8))
        tbuf, tiles = guarded((npg, 5, nxt, nxt, nxt))
        fbuf, flux = guarded((npg, 8, 6, 5, 8, 8))
        if rep % 3 == 2:
            with torch.cuda.stream(side):
                B.cons2prim(cons.view(5, -1))
        _, sm, stats = B.grid_step_cfl(p_in, p_out, tiles, shape, 0.4, dh, par, bc, flux_out=flux)
        torch.cuda.synchronize()
        s = B.stats_to_host(stats)
        assert guards_intact(obuf) and guards_intact(tbuf) and guards_intact(fbuf)
        assert torch.equal(p_in, p0)                                    # the input state is read only
        assert not bool(torch.isnan(p_out).any()) and not bool(torch.isnan(flux).any())
        assert 0 < s.n_uniform_pg < npg
        written = ~torch.isnan(tiles).reshape(npg, -1).all(1)          # groups whose tile was materialised
        assert int(written.sum()) == npg - s.n_uniform_pg
        res = (p_out.clone(), flux.clone(), sm.clone())
        if first is None:
            first = res
        else:
            for a, b in zip(first, res):
                assert torch.equal(a.view(torch.int64), b.view(torch.int64)), (recon, riemann, rep)
    # tile-based calls on tiles that are partly uniform: MUSCL-Hancock and VL pre-passes
    for integ in ("mhm", "vl"):
        pv = B.params(recon, riemann, integrator=integ)
        tl = B.grid_gather(cons, pv.ghost, bc)
        obuf, out = guarded((npg, 8, 5, 8, 8, 8))
        fbuf, flux = guarded((npg, 8, 6, 5, 8, 8))
        _, _, stats = B.fluid_step_fluxes(tl, 0.1 * dh, dh, pv, cons_out=out, flux_out=flux)
        torch.cuda.synchronize()
        assert guards_intact(obuf) and guards_intact(fbuf)
        assert not bool(torch.isnan(out).any()) and not bool(torch.isnan(flux).any())
        assert 0 < B.stats_to_host(stats).n_uniform_pg < npg
