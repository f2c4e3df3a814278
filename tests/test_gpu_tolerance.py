"""error-controlled iteration and warm start on the GPU against oracle O-12 (global mode:
one pass count for the whole solve)."""
import math

import numpy as np
import pytest
import torch

from paper_2107_08145_b200 import inputs, rts
import oracle

pytestmark = pytest.mark.gpu
TOL_Q, TOL_I = 1e-4, 1e-5


def _dev(inp):
    return tuple(torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))


def _cmp(Q, I, Qo, Io, what):
    Q = Q.cpu().numpy().astype(np.float64); I = I.cpu().numpy().astype(np.float64)
    eq = np.abs(Q - Qo).max() / np.abs(Qo).max()
    ei = (np.abs(I - Io) / np.abs(Io)).max()
    print(f"{what}: dQ/maxQ = {eq:.3e}  rel dItop = {ei:.3e}")
    assert eq <= TOL_Q and ei <= TOL_I, (what, eq, ei)


@pytest.mark.parametrize("cfg,grid,nb,tiling", [(1, None, None, None), (3, (40, 36, 33), 4, {0: (16, 12), 1: (16, 12), 2: (16, 12)}),
                                               (5, (48, 40, 36), 4, None)])
def test_one_pass_per_launch_reproduces_the_fixed_pass_solve_bit_for_bit(cfg, grid, nb, tiling):
    """A negative tolerance never stops: max_passes = 3 launches of one pass each carry the same seam histories and
    last planes through HBM that the 3-pass launch carries in shared memory."""
    kw = dict(grid=grid, nbands=nb) if grid else {}
    inp = inputs.make_config(cfg, **kw)
    rho, T, P = _dev(inp)
    a = rts.from_inputs(inp, tiling=tiling)
    a.set_thick_skip(False)
    Qa, Ia = a.solve(rho, T, P); a.sync_check()
    b = rts.from_inputs(inp, tiling=tiling, tolerance=(-1.0, 3))
    Qb, Ib = b.solve(rho, T, P); b.sync_check()
    assert b.passes_used()[0] == 3
    assert torch.equal(Qa, Qb) and torch.equal(Ia, Ib)
    a.close(); b.close()


@pytest.mark.parametrize("cfg,grid,nb", [(1, None, None), (2, None, None), (3, (40, 36, 33), 4), (5, (48, 40, 36), 4)])
def test_pass_count_and_result_match_the_oracle(cfg, grid, nb):
    kw = dict(grid=grid, nbands=nb) if grid else {}
    inp = inputs.make_config(cfg, **kw)
    # the oracle's error history with no early stop; tolerances in the gaps between consecutive passes, so that
    # the fp32 error measure cannot tip the count
    _, _, _, _, rel = oracle.solve_tol(inp, -1.0, 8, mode=1)
    rho, T, P = _dev(inp)
    for k in (1, 2, 3):
        if not (rel[k] > 0 and rel[k - 1] > 4 * rel[k]):
            continue
        tol = math.sqrt(rel[k - 1] * rel[k])
        Qo, Io, _, used, relo = oracle.solve_tol(inp, tol, 8, mode=1)
        assert (used == k + 1).all()
        s = rts.from_inputs(inp, tolerance=(tol, 8))
        Q, I = s.solve(rho, T, P); s.sync_check()
        n, e = s.passes_used()
        assert n == k + 1, (n, k + 1, e, relo)
        assert abs(e - relo[-1]) <= 0.02 * relo[-1] + 1e-7       # the same error measure (fp32 vs fp64)
        _cmp(Q, I, Qo, Io, f"{inp.name} tol={tol:.2e} passes={n}")
        s.close()


def test_warm_start_needs_one_pass_and_matches_the_oracle():
    inp = inputs.make_config(3, grid=(40, 36, 33), nbands=4)
    _, _, _, _, rel = oracle.solve_tol(inp, -1.0, 8, mode=1)
    print('oracle relative seam change per pass:', rel)
    tol = math.sqrt(rel[1] * rel[2])                           # well above the fp32 resolution of the GPU's error measure
    Qo, Io, faces, used, _ = oracle.solve_tol(inp, tol, 12, mode=1)
    Qw, Iw, _, usedw, relw = oracle.solve_tol(inp, tol, 12, mode=1, faces=faces)
    assert (usedw == 1).all()
    rho, T, P = _dev(inp)
    s = rts.from_inputs(inp, tolerance=(tol, 12))
    s.set_warm_start(True)
    Q, I = s.solve(rho, T, P); s.sync_check()
    assert s.passes_used()[0] == int(used.max())
    _cmp(Q, I, Qo, Io, "cold")
    Q2, I2 = s.solve(rho, T, P); s.sync_check()               # same atmosphere again: starts from the converged seams
    n2, e2 = s.passes_used()
    assert n2 == 1 and e2 <= tol
    _cmp(Q2, I2, Qw, Iw, "warm")
    s.set_warm_start(False)
    Q3, I3 = s.solve(rho, T, P); s.sync_check()               # cold again
    assert s.passes_used()[0] == int(used.max()) and torch.equal(Q3, Q)
    s.close()


def test_tolerance_api_state():
    inp = inputs.make_config(1, grid=(8, 8, 6))
    s = rts.from_inputs(inp)
    with pytest.raises(rts.RTSError):
        s.passes_used()                                        # mode off
    with pytest.raises(rts.RTSError):
        s.set_tolerance(1e-3, -1)
    s.close()
