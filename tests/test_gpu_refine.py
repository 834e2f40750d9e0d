"""-m gpu parity: srhd_refine_flags vs the oracle (byte work: bit-exact flags) on seeded tiles."""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from tests.test_gpu_fluid_step import dev, make_tiles

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("recon", ["plm", "ppm"])
def test_refine_flags_parity(ref, recon):
    po = ref.params(recon, "hllc")
    npg = 2 * 148 + 3                                  # several waves and a ragged last one
    base = make_tiles(ref, 7, po.ghost, seed=31, umax=5.0)
    tiles = np.ascontiguousarray(base[np.arange(npg) % 7])
    d = dev(tiles)
    hits = 0
    for quantity, c_q, thr in (("rho", 4.0, 0.0), ("gamma", 0.4, 0.0), ("D", 4.0, 0.0), ("Etilde", 8.0, 0.0),
                               ("none", 0.0, 16.0), ("rho", 8.0, 16.0)):
        want = ref.refine_flags(tiles, po, quantity, c_q, thr)
        for exact in (True, False):
            got = B.refine_flags(d, B.params(recon, "hllc", exact=exact), quantity, c_q, thr, exact=exact)
            assert np.array_equal(got.cpu().numpy(), want), (quantity, exact)
        hits += int(want.sum())
        assert 0 < want[:7].sum() < 56, (quantity, want[:7].sum())      # thresholds that discriminate
    empty = torch.empty((0, 5, 16 + 2 * po.ghost) + (16 + 2 * po.ghost,) * 2, dtype=torch.float64, device="cuda")
    assert B.refine_flags(empty, B.params(recon, "hllc")).shape == (0, 8)
