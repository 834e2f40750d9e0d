"""-m gpu: srhd_fluid_step_noalloc against srhd_fluid_step.

srhd_fluid_step_noalloc exists for programs that embed this library but cannot let it allocate GPU memory: a
simulation code whose own pool has claimed the whole device (so a cudaMallocAsync inside the step would fail or
eat into memory the code thinks it owns), or a step loop that runs under a fixed, externally enforced memory
budget.  It runs the same two kernels as srhd_fluid_step; only the home of the pre-pass's per-group flags differs
(a 64 KiB array inside the library, shared by all calls on the GPU, instead of a fresh stream-ordered block).

What can go wrong with that, and what this file therefore checks: the array keeps the flags of the previous
call, so the second of two back-to-back calls must not see the first one's verdicts.  The two calls below use
batches in which uniform ("already finished by the pre-pass", flag 1) and general (flag 0) groups swap places,
and a different group count, so a stale flag would skip a group that needs the solver and leave garbage in its
output.  Both calls must reproduce srhd_fluid_step on the same input: bit for bit (same kernels, same order of
operations) and hence inside the 1e-11 per-cell one-step tolerance the other parity tests use.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide
the parity tests proper.  It passes alone in a fresh process (first call on the device = the set-up call) and
after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200 import workloads as wl
from tests.gpu_util import step_err

TOL_STEP = 1e-11   # the per-cell one-step tolerance of tests/test_gpu_fluid_step.py (BASELINE.json north_star)


def _tiles(npg, ghost, seed, uniform_groups):
    """Seeded conserved tiles (npg,5,nxt,nxt,nxt) on the GPU; the groups listed in `uniform_groups` hold one state
    in every cell (the pre-pass finishes those and raises their flag)."""
    prim = wl.random_patch_groups(npg, ghost, seed=seed)              # (npg,5,nxt,nxt,nxt) primitives
    for g in uniform_groups:
        prim[g] = prim[g][:, 3:4, 5:6, 7:8]
    nxt = 16 + 2 * ghost
    flat = torch.from_numpy(np.ascontiguousarray(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1))).cuda()
    cons = B.prim2cons(flat)
    return cons.reshape(5, npg, nxt, nxt, nxt).permute(1, 0, 2, 3, 4).contiguous()


@pytest.mark.gpu
@pytest.mark.parametrize("recon,riemann", [("plm", "hlle"), ("ppm", "hllc")])
def test_noalloc_matches_fluid_step_on_two_calls_in_a_row(recon, riemann):
    par = B.params(recon, riemann)
    dh = 1.0 / 64
    # call 1: groups 0, 2, 3, 5 uniform; call 2: fewer groups, and exactly the other ones uniform
    batches = [_tiles(7, par.ghost, 101, (0, 2, 3, 5)), _tiles(6, par.ghost, 202, (1, 4))]
    dts = [0.4 * dh / float(B.max_signal_speed(t.permute(1, 0, 2, 3, 4).reshape(5, -1).contiguous(), par).item())
           for t in batches]
    # everything the no-allocation path writes to is created up front, as its callers would
    outs = [torch.full((t.shape[0], 8, 5, 8, 8, 8), float("nan"), dtype=t.dtype, device="cuda") for t in batches]
    stats = [B.new_stats(), B.new_stats()]
    torch.cuda.synchronize()
    for t, dt, o, s in zip(batches, dts, outs, stats):              # back to back on one stream, no sync between
        B.fluid_step_noalloc(t, dt, dh, par, o, s)
    torch.cuda.synchronize()
    for i, (t, dt, o, s) in enumerate(zip(batches, dts, outs, stats)):
        want, ws = B.fluid_step(t, dt, dh, par)
        got, want = o.cpu().numpy(), want.cpu().numpy()
        assert np.all(np.isfinite(got)), f"call {i + 1}: a group was skipped (stale flag?)"
        err = step_err(got, want, 2)
        assert err.max() <= TOL_STEP, (i, float(err.max()))
        assert np.array_equal(got, want), f"call {i + 1} differs from srhd_fluid_step"
        assert B.stats_to_host(s).as_dict() == B.stats_to_host(ws).as_dict()
    # the uniform groups were in fact taken by the pre-pass (otherwise the flags were never exercised)
    assert [B.stats_to_host(s).n_uniform_pg for s in stats] == [4, 2]


@pytest.mark.gpu
def test_noalloc_limits_are_reported_not_launched():
    """Beyond SRHD_NOALLOC_MAX_NPG groups, or with the VL integrator, the call refuses with a clear error before it
    touches the GPU (the pointers below are never dereferenced)."""
    L = B.load_library()
    par = B.params("plm", "hllc")
    assert L.srhd_fluid_step_noalloc(1 << 20, 1 << 44, B.NOALLOC_MAX_NPG + 1, 0.1, 1.0, C.byref(par), None, None) == -7
    assert b"SRHD_NOALLOC_MAX_NPG" in L.srhd_error_string(-7)
    vl = B.params("plm", "hllc", integrator="vl")
    assert L.srhd_fluid_step_noalloc(1 << 20, 1 << 44, 4, 0.1, 1.0, C.byref(vl), None, None) == -2
