"""band x octant sharding of one box.  One GPU stands in for the ranks one after the other: every
rank's context sweeps its own units; the sum of the partial results (what the NCCL all-reduce forms) must equal
the unsharded solve and the oracle."""
import numpy as np
import pytest
import torch

from paper_2107_08145_b200 import inputs, multi, rts
import oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nranks", [2, 3, 8])
def test_shards_sum_to_the_whole_solve(nranks):
    inp = inputs.make_config(3, grid=(40, 36, 33), nbands=4)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    full = rts.from_inputs(inp)
    Q0, I0 = full.solve(rho, T, P)
    full.sync_check()
    Qs = torch.zeros_like(Q0, dtype=torch.float64)
    Is = torch.zeros_like(I0, dtype=torch.float64)
    owned = []
    n_all = None
    for r in range(nranks):
        s = rts.from_inputs(inp, shard=(r, nranks))
        mine, n_all = s.shard_info()
        owned.append(mine)
        assert mine == len(multi.shard_units(n_all, r, nranks))
        Q, I = s.solve(rho, T, P)
        s.sync_check()
        Qs += Q.double(); Is += I.double()
        # a (band, ray) slice of I_top belongs to exactly one rank: everybody else leaves zeros there
        s.close()
    assert sum(owned) == n_all
    Q0d, I0d = Q0.double(), I0.double()
    assert float((Qs - Q0d).abs().max() / Q0d.abs().max()) <= 2e-6       # only the order of the fp32 sums differs
    assert float(((Is - I0d).abs() / I0d.abs()).max()) <= 1e-6
    Qo, Io = oracle.solve(inp)
    assert np.abs(Qs.cpu().numpy() - Qo).max() / np.abs(Qo).max() <= 1e-4
    assert (np.abs(Is.cpu().numpy() - Io) / np.abs(Io)).max() <= 1e-5
    full.close()


def test_shard_argument_checks():
    inp = inputs.make_config(1, grid=(8, 8, 6))
    s = rts.from_inputs(inp)
    with pytest.raises(rts.RTSError):
        s.set_shard(2, 2)
    with pytest.raises(rts.RTSError):
        s.set_shard(0, 0)
    s.close()
