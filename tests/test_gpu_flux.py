"""Radiative flux, flux-divergence heating and deterministic accumulation on the CUDA path (NEXT #2) -- needs a B200.

F is compared element by element with the oracle's O-10 at 1e-5 of max|F|, Qdiv / Qblend
(O-11) at 1e-4 of their maxima (differences of fp32 fluxes over two cells amplify the rounding of F).
"""
import numpy as np
import pytest

from paper_2107_08145_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_F = 1e-5
TOL_Q = 1e-4


def _run(inp, tau0=0.1, **kw):
    import torch
    from paper_2107_08145_b200 import rts
    s = rts.from_inputs(inp, flux=True, **kw)
    s.set_flux_blend(tau0)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    out = s.solve_flux(rho, T, P)
    s.sync_check()
    s.close()
    return [o.cpu().numpy().astype(np.float64) for o in out]


@pytest.mark.parametrize("cfg,grid,nb", [(1, None, None), (2, None, None), (3, (40, 36, 33), None),
                                         (5, (48, 40, 36), None), (4, (24, 28, 20), 3)])
def test_flux_and_flux_heating_parity(cfg, grid, nb):
    import oracle
    inp = inputs.make_config(cfg, grid=grid, nbands=nb)
    Qo, Io, Fo = oracle.solve(inp, want_F=True)
    kap, _ = oracle.coefficients(inp)
    Qdo, Qbo = oracle.flux_heating(inp, Fo, Qo, kap[0], tau0=0.1)
    Q, I, F, Qd, Qb = _run(inp)
    eF = np.abs(F - Fo).max() / np.abs(Fo).max()
    eQ = np.abs(Q - Qo).max() / np.abs(Qo).max()
    eD = np.abs(Qd - Qdo).max() / np.abs(Qdo).max()
    eB = np.abs(Qb - Qbo).max() / np.abs(Qbo).max()
    eI = (np.abs(I - Io) / np.abs(Io)).max()
    print(f"{inp.name}: dF/maxF = {eF:.2e}  dQ/maxQ = {eQ:.2e}  dQdiv/max = {eD:.2e}  dQblend/max = {eB:.2e}  dItop = {eI:.2e}")
    assert eF <= TOL_F and eQ <= TOL_Q and eI <= 1e-5
    assert eD <= TOL_Q and eB <= TOL_Q


def test_flux_with_unnormalised_and_unequal_rays():
    import oracle
    inp = inputs.make_config(2, grid=(24, 24, 20))
    inp.mu = np.array([[0.6, -1.0, 1.62], [-0.9, 0.2, -0.38], [0.1, 0.95, 0.3], [0.2, 0.1, -0.97]])
    inp.wq = np.array([0.1, 0.4, 0.3, 0.2])
    _, _, Fo = oracle.solve(inp, want_F=True)
    _, _, F, _, _ = _run(inp)
    assert np.abs(F - Fo).max() <= TOL_F * np.abs(Fo).max()


def test_heating_and_flux_are_bitwise_reproducible():
    """No atomics on the heating path: every sweep unit writes its own partial field, the units are summed in a
    fixed order -> identical bits from run to run and from context to context."""
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(3, grid=(52, 44, 40))
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    outs = []
    for rep in range(2):
        s = rts.from_inputs(inp, flux=True)
        for _ in range(2):
            o = s.solve_flux(rho, T, P)
            s.sync_check()
            outs.append([t.clone() for t in o])
        s.close()
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert torch.equal(a, b)
    s = rts.from_inputs(inp)
    Q, I = s.solve(rho, T, P)
    s.sync_check()
    assert torch.equal(Q, outs[0][0]) and torch.equal(I, outs[0][1])      # the flux fields do not change Q or I_top
    s.close()


def test_flux_needs_enable_before_workspace():
    import ctypes
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(1, grid=(8, 8, 6))
    s = rts.from_inputs(inp)                       # flux not enabled
    lib = rts.load_library()
    buf = torch.zeros(3 * 8 * 8 * 6, dtype=torch.float32, device="cuda")
    p = ctypes.c_void_p(buf.data_ptr())
    assert lib.rts_solve_flux(s._ctx, p, p, p, p, None, p, None, None, None) == -2
    assert lib.rts_set_flux_blend(s._ctx, -1.0) == -1
    s.close()
