"""NEXT #4 on the GPU: scattering source function with the source update along the ray against
the fp64 oracle O-13, element by element, through the C-ABI.  Both sides get the same fp32 kaprho, B and eps (the
CUDA path's stage-A output); the kernel computes in fp64, so the tolerance is that of a different summation order."""
import numpy as np
import pytest

from paper_2107_08145_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _case(cfg, grid, band, eps_lo):
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(cfg, grid=grid)
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    k, B = s.coefficients(rho, T, P)
    s.sync_check()
    rng = np.random.default_rng(17)
    eps = (eps_lo + (1.0 - eps_lo) * rng.random(inp.shape)).astype(np.float32)
    return inp, s, k[band].contiguous(), B[band].contiguous(), torch.from_numpy(eps).cuda()


@pytest.mark.parametrize("cfg,grid,band,niter,gs", [
    (1, (24, 20, 18), 0, 6, True),
    (1, (24, 20, 18), 0, 6, False),
    (3, (37, 41, 30), 2, 4, True),      # ragged widths, a thick band
    (5, (30, 34, 61), 1, 3, True),
    (2, (5, 3, 2), 0, 5, True),         # two levels: every node is a Dirichlet node for half of the rays
    (3, (288, 280, 5), 1, 3, True),     # planes beyond 2 x 256 threads per SM: the kernel build with y-fastest copies for
    (3, (288, 280, 5), 3, 2, False),    # the x-march rays (rts_scatter.cuh), Gauss-Seidel and Jacobi
])
def test_scatter_against_oracle(cfg, grid, band, niter, gs):
    import oracle
    inp, s, k, B, eps = _case(cfg, grid, band, 0.05)
    S, J, change = s.scatter_solve(k, B, eps, niter, gauss_seidel=gs)
    s.sync_check()
    So, Jo, cho = oracle.scatter_solve(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu, inp.wq,
                                       k.cpu().numpy().astype(np.float64), B.cpu().numpy().astype(np.float64),
                                       eps.cpu().numpy().astype(np.float64), niter, gs=gs)
    s.close()
    S = S.cpu().numpy(); J = J.cpu().numpy()
    assert np.isfinite(S).all() and np.isfinite(J).all()
    assert np.abs(S - So).max() <= TOL * np.abs(So).max()
    assert np.abs(J - Jo).max() <= TOL * np.abs(Jo).max()
    assert np.allclose(change, cho, rtol=1e-6, atol=1e-14)


def test_several_bands_in_one_call_are_independent_problems():
    """All bands of a call share the plane steps; every band must equal the oracle's one-band solve (and so the
    one-band call) element by element."""
    import oracle
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(4, grid=(20, 24, 17))                # 12 bands, opacity scales up to 1e5
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    k, B = s.coefficients(rho, T, P)
    rng = np.random.default_rng(3)
    eps = torch.from_numpy((0.02 + 0.98 * rng.random((inp.nbands,) + inp.shape)).astype(np.float32)).cuda()
    S, J, change = s.scatter_solve(k, B, eps, 4)
    S1, J1, ch1 = s.scatter_solve(k[5].contiguous(), B[5].contiguous(), eps[5].contiguous(), 4)
    s.sync_check(); s.close()
    assert torch.equal(S[5], S1) and torch.equal(J[5], J1) and [c[5] for c in change] == ch1
    for b in (0, 7, 11):
        So, Jo, cho = oracle.scatter_solve(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu, inp.wq,
                                           k[b].cpu().numpy().astype(np.float64), B[b].cpu().numpy().astype(np.float64),
                                           eps[b].cpu().numpy().astype(np.float64), 4, gs=True)
        assert np.abs(S[b].cpu().numpy() - So).max() <= TOL * np.abs(So).max()
        assert np.abs(J[b].cpu().numpy() - Jo).max() <= TOL * np.abs(Jo).max()
        assert np.allclose([c[b] for c in change], cho, rtol=1e-6, atol=1e-14)


@pytest.mark.parametrize("rays", ["axis_parallel_and_aligned", "single", "z_face_only"])
def test_scatter_with_other_ray_sets(rays):
    """Rays with a zero component (f = 0), lattice-aligned rays (f = 1), one ray alone, and a set whose rays all
    march along z: the per-ray geometry of the kernel against the oracle's."""
    import oracle
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(1, grid=(16, 12, 14))
    if rays == "axis_parallel_and_aligned":
        inp.dz = inp.dx * 0.9082483 / 0.2958759
        inp.mu = np.array([[0.0, 0.6, 0.8], [0.6, 0.0, -0.8], [0.0, 0.0, 1.0], [0.0, 0.0, -1.0],
                           [0.2958759, 0.2958759, 0.9082483], [-0.2958759, 0.2958759, -0.9082483]])
        inp.wq = np.full(6, 1.0 / 6.0)
    elif rays == "single":
        inp.mu = np.array([[0.3, -0.5, 0.81]]); inp.wq = np.array([1.0])
    else:
        mu, w = inputs.carlson24()
        sel = [r for r in range(24) if r % 3 == 2]
        inp.mu = np.ascontiguousarray(mu[sel]); inp.wq = np.full(len(sel), 1.0 / len(sel))
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    k, B = s.coefficients(rho, T, P)
    rng = np.random.default_rng(5)
    eps = torch.from_numpy((0.1 + 0.9 * rng.random(inp.shape)).astype(np.float32)).cuda()
    S, J, change = s.scatter_solve(k[0].contiguous(), B[0].contiguous(), eps, 5)
    s.sync_check(); s.close()
    So, Jo, cho = oracle.scatter_solve(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu, inp.wq,
                                       k[0].cpu().numpy().astype(np.float64), B[0].cpu().numpy().astype(np.float64),
                                       eps.cpu().numpy().astype(np.float64), 5, gs=True)
    assert np.abs(S.cpu().numpy() - So).max() <= TOL * np.abs(So).max()
    assert np.abs(J.cpu().numpy() - Jo).max() <= TOL * np.abs(Jo).max()
    assert np.allclose(change, cho, rtol=1e-6, atol=1e-14)


def test_many_bands_on_the_large_plane_build():
    """12 bands x 80 x 80 nodes per plane step select the kernel build for large planes; every band against the oracle."""
    import oracle
    import torch
    from paper_2107_08145_b200 import rts
    inp = inputs.make_config(4, grid=(80, 80, 6))
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    k, B = s.coefficients(rho, T, P)
    rng = np.random.default_rng(11)
    eps = torch.from_numpy((0.05 + 0.95 * rng.random((inp.nbands,) + inp.shape)).astype(np.float32)).cuda()
    S, J, change = s.scatter_solve(k, B, eps, 3)
    s.sync_check(); s.close()
    for b in range(0, inp.nbands, 5):
        So, Jo, cho = oracle.scatter_solve(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu, inp.wq,
                                           k[b].cpu().numpy().astype(np.float64), B[b].cpu().numpy().astype(np.float64),
                                           eps[b].cpu().numpy().astype(np.float64), 3, gs=True)
        assert np.abs(S[b].cpu().numpy() - So).max() <= TOL * np.abs(So).max()
        assert np.abs(J[b].cpu().numpy() - Jo).max() <= TOL * np.abs(Jo).max()
        assert np.allclose([c[b] for c in change], cho, rtol=1e-6, atol=1e-14)


def test_eps_one_is_the_lte_source_and_zero_iterations_return_the_start():
    import torch
    inp, s, k, B, eps = _case(1, (16, 12, 10), 0, 0.05)
    one = torch.ones_like(eps)
    S, J, change = s.scatter_solve(k, B, one, 3)
    assert torch.equal(S, B.double()) and change == [0.0, 0.0, 0.0]
    S0, J0, ch0 = s.scatter_solve(k, B, eps, 0)
    assert torch.equal(S0, B.double()) and ch0 == []
    # J of the start: sum_r w_r I(0), I(0) = S except 0 on the top plane of the downward rays
    wdown = float(sum(w for m, w in zip(inp.mu, inp.wq) if m[2] < 0))
    Jref = B.double().clone(); Jref[-1] *= (1.0 - wdown)
    assert torch.allclose(J0, Jref, rtol=1e-13, atol=0.0)
    s.close()


def test_gauss_seidel_needs_fewer_iterations_than_jacobi_on_the_gpu():
    """The point of the scheme: after the same number of iterations the Gauss-Seidel form is closer
    to the converged source function."""
    inp, s, k, B, eps = _case(3, (20, 16, 24), 1, 0.02)
    Sref, _, ch = s.scatter_solve(k, B, eps, 400)
    assert ch[-1] < 1e-9
    Sg, _, _ = s.scatter_solve(k, B, eps, 8, gauss_seidel=True)
    Sj, _, _ = s.scatter_solve(k, B, eps, 8, gauss_seidel=False)
    s.close()
    eg = float((Sg - Sref).abs().max()); ej = float((Sj - Sref).abs().max())
    assert eg < ej
