"""rts_scatter_solve_static: the scattering solve for callers that cannot allocate device memory (scratch in a static
device array inside the library) against the existing rts_scatter_solve (caller-owned workspace), through the C-ABI.

Collected last on purpose (the suite runs with pytest -x).  Two calls in a row with different inputs: the static
array keeps the previous call's contents, and nothing of them may reach the next call.
"""
import numpy as np
import pytest

from paper_2107_08145_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-10          # the tolerance of tests/test_gpu_scatter.py (the two paths run the same kernel: they agree bitwise)


def _setup(grid=(40, 36, 33)):
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(3, grid=grid)
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    k, B = s.coefficients(rho, T, P)
    s.sync_check()
    return torch, rts, inp, s, k, B


def test_static_scratch_entry_matches_the_workspace_path_on_two_calls_in_a_row():
    torch, rts, inp, s, k, B = _setup()
    rng = np.random.default_rng(23)
    eps_a = torch.from_numpy((0.05 + 0.95 * rng.random(inp.shape)).astype(np.float32)).cuda()
    eps_b = torch.from_numpy((0.3 + 0.7 * rng.random(inp.shape)).astype(np.float32)).cuda()
    calls = [(k[2].contiguous(), B[2].contiguous(), eps_a, 4, True),      # a thick band, Gauss-Seidel
             (k[0].contiguous(), B[0].contiguous(), eps_b, 3, False)]     # another band, fewer iterations, Jacobi
    # outputs allocated by the test: the entry point itself allocates nothing
    S = torch.empty(inp.shape, dtype=torch.float64, device="cuda")
    J = torch.empty(inp.shape, dtype=torch.float64, device="cuda")
    for kk, BB, ee, niter, gs in calls:
        S.fill_(float("nan")); J.fill_(float("nan"))
        _, _, ch = s.scatter_solve_static(kk, BB, ee, niter, gauss_seidel=gs, S=S, J=J)
        S_ref, J_ref, ch_ref = s.scatter_solve(kk, BB, ee, niter, gauss_seidel=gs)
        s.sync_check()
        assert torch.isfinite(S).all() and torch.isfinite(J).all()
        assert float((S - S_ref).abs().max()) <= TOL * float(S_ref.abs().max())
        assert float((J - J_ref).abs().max()) <= TOL * float(J_ref.abs().max())
        assert np.allclose(ch, ch_ref, rtol=1e-12, atol=0.0)
    s.close()


def test_static_scratch_entry_rejects_what_does_not_fit():
    torch, rts, inp, s, k, B = _setup()
    eps = torch.full_like(k[:2], 0.5)
    need = int(s._lib.rts_scatter_workspace_bytes(s._ctx, 2, 2))
    assert need > (16 << 20)                                   # two bands of this grid exceed the static array
    with pytest.raises(rts.RTSError, match="bytes of scratch"):
        s.scatter_solve_static(k[:2].contiguous(), B[:2].contiguous(), eps, 2)
    with pytest.raises(rts.RTSError, match="2048"):
        s.scatter_solve_static(k[0].contiguous(), B[0].contiguous(), eps[0].contiguous(), 5000)
    # the context stays usable after a rejected call
    S, J, ch = s.scatter_solve_static(k[0].contiguous(), B[0].contiguous(), eps[0].contiguous(), 1)
    assert torch.isfinite(S).all() and len(ch) == 1
    s.close()
