"""-m gpu: the small case the compute-sanitizer runs use (summaries in profiles/).

Two patch groups through every <ghost, riemann> instantiation of fluid_step_kernel, with and without the
patch-face flux output, once at a CFL-sized step and once at a step that forces the retry ladder, in
both builds; plus the ghost-zone fill, the refinement flags and the three state-list calls.  Run as

    compute-sanitizer --tool {memcheck|racecheck|initcheck|synccheck} python -m pytest -q -m gpu tests/test_gpu_sanitizer_case.py

It is also an ordinary parity test: every output is compared with the oracle.
"""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200 import workloads as wl
from tests.gpu_util import step_err

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _tiles(ref, npg, ghost, seed, **kw):
    prim = wl.random_patch_groups(npg, ghost, seed=seed, **kw)
    nxt = 16 + 2 * ghost
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    return np.ascontiguousarray(cons.reshape(5, npg, nxt, nxt, nxt).transpose(1, 0, 2, 3, 4))


@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("plm", "hllc"), ("ppm", "hlle"), ("ppm", "hllc")])
@pytest.mark.parametrize("forced_retry", [False, True])
def test_two_patch_groups_all_instantiations(ref, recon, riemann, forced_retry):
    po = ref.params(recon, riemann, max_retry=2)
    dh = 1.0 / 64
    kw = dict(umax=30.0, rough=3.0, log_theta=(-8.0, 2.0)) if forced_retry else {}
    tiles = _tiles(ref, 2, po.ghost, seed=5 if forced_retry else 11 + po.ghost, **kw)
    smax = ref.max_signal_speed(tiles.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    dt = (4.0 if forced_retry else 0.4) * dh / smax
    want, wflux, st = ref.fluid_step_fluxes(tiles, dt, dh, po)
    assert st.n_retry_pg > 0 or not forced_retry, "the over-long step must go through the retry ladder"
    for exact in (True, False):
        par = B.params(recon, riemann, max_retry=2, exact=exact)
        got, sb = B.fluid_step(dev(tiles), dt, dh, par, exact=exact)
        got2, gflux, sb2 = B.fluid_step_fluxes(dev(tiles), dt, dh, par, exact=exact)
        torch.cuda.synchronize()
        assert torch.equal(got, got2)
        s = B.stats_to_host(sb)
        assert s.n_retry_pg == st.n_retry_pg
        if exact:
            assert np.array_equal(got.cpu().numpy(), want, equal_nan=True)
            assert np.array_equal(gflux.cpu().numpy(), wflux, equal_nan=True)
            assert s.algorithm_dict() == st.as_dict()
        elif st.n_retry_pg == 0:
            assert step_err(got.cpu().numpy(), want, 2).max() <= 1e-11


def test_helpers_and_state_lists(ref):
    rng = np.random.default_rng(0)
    shape = (16, 16, 32)
    prim = np.empty((5,) + shape)
    prim[0] = 10.0 ** rng.uniform(-1, 1, shape)
    prim[1:4] = rng.standard_normal((3,) + shape)
    prim[4] = prim[0] * 10.0 ** rng.uniform(-3, 1, shape)
    n = prim[0].size
    for exact in (True, False):
        d_cons = B.prim2cons(dev(prim.reshape(5, -1)), exact=exact)
        back, _ = B.cons2prim(d_cons, exact=exact)
        smax = B.max_signal_speed(d_cons, exact=exact)
        for ghost, recon in ((2, "plm"), (3, "ppm")):
            par = B.params(recon, "hllc", exact=exact)
            t = B.grid_gather(d_cons.reshape(5, *shape), ghost, ["outflow"] * 6, exact=exact)
            out, _ = B.fluid_step(t, 1e-4, 1.0 / 32, par, exact=exact)
            t2, s2 = B.patch_gather_speed(out, shape, par, ["periodic"] * 6, exact=exact)
            g = B.grid_scatter(out, shape, exact=exact)
            B.refine_flags(t2, par, "rho", 0.3, 2.0, exact=exact)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(back).all()) and float(smax.cpu()) > 0 and g.shape[0] == 5
    o = ref.prim2cons(prim.reshape(5, -1))
    assert np.abs(d_cons.cpu().numpy() - o).max() <= 1e-12 * np.abs(o).max() and n > 0
