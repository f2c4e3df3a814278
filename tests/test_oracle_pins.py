"""Pins of the fp64 oracle against what the paper and the mathematics fix.

Each test names the SURVEY.md 8(c) pin it implements and what part of the oracle a
plausible mistake in it would break.  None of these re-types the oracle's formulas:
closed forms of the transfer equation, an independent quadrature / geometric /
recursive evaluator (tests/independent.py), symmetries and golden check values.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2107_08145_b200 import inputs
from tests import independent as ind

GOLD = os.path.join(os.path.dirname(__file__), "golden")
A, B = inputs.CARLSON_A, inputs.CARLSON_B
KM = 1e5


def _read_table(name):
    rows = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    return rows


# --------------------------------------------------------------------------- O-6
def test_psi_golden_values():
    for dtau, E, pu, pp in _read_table("psi_check_values.txt"):
        e, u, p = oracle.psi(dtau)
        assert e == pytest.approx(E, rel=2e-9)
        assert u == pytest.approx(pu, rel=2e-9)
        assert p == pytest.approx(pp, rel=2e-9)
        assert e + u + p == pytest.approx(1.0, abs=1e-15)


def test_psi_matches_quadrature_of_formal_integral():
    # psi_u, psi_p are the responses to (S_u,S_p) = (1,0) and (0,1); E to I_u = 1.
    for dtau in [1e-7, 3e-4, 9.99e-4, 1.0e-3, 1.01e-3, 0.02, 0.5, 3.0, 7.5, 40.0, 500.0]:
        e, u, p = oracle.psi(dtau)
        assert e == pytest.approx(ind.formal_integral(1.0, 0.0, 0.0, dtau), rel=1e-12, abs=1e-300)
        assert u == pytest.approx(ind.formal_integral(0.0, 1.0, 0.0, dtau), rel=1e-11)
        assert p == pytest.approx(ind.formal_integral(0.0, 0.0, 1.0, dtau), rel=1e-11)
    assert oracle.psi(0.0) == (1.0, 0.0, 0.0)


# --------------------------------------------------------------------------- O-3
def test_ray_geometry_numbers_of_survey():
    # cfg 1/2 big-x ray -> x-face, ds = 52.848984 km, f_y = 0.325765, f_z = 0.488648
    ax, sg, ds, f = oracle.ray_geometry(48 * KM, 48 * KM, 32 * KM, [B, A, A])
    assert ax == 0 and sg == (1, 1, 1)
    assert ds / KM == pytest.approx(52.848984, abs=1e-6)
    assert f[1] == pytest.approx(0.325765, abs=1e-6) and f[2] == pytest.approx(0.488648, abs=1e-6)
    # big-z ray -> z-face, ds = 35.232656 km, f_x = f_y = 0.217177
    ax, sg, ds, f = oracle.ray_geometry(48 * KM, 48 * KM, 32 * KM, [-A, A, -B])
    assert ax == 2 and sg == (-1, 1, -1)
    assert ds / KM == pytest.approx(35.232656, abs=1e-6)
    assert f[0] == pytest.approx(0.217177, abs=1e-6) and f[1] == pytest.approx(0.217177, abs=1e-6)
    # cfg 3/4: big-x ds = 35.232656 km, f_y = 0.325765, f_z = 0.651531; big-z ds = 17.616328, f = 0.162883
    ax, sg, ds, f = oracle.ray_geometry(32 * KM, 32 * KM, 16 * KM, [B, A, A])
    assert ax == 0 and ds / KM == pytest.approx(35.232656, abs=1e-6)
    assert f[1] == pytest.approx(0.325765, abs=1e-6) and f[2] == pytest.approx(0.651531, abs=1e-6)
    ax, sg, ds, f = oracle.ray_geometry(32 * KM, 32 * KM, 16 * KM, [A, A, B])
    assert ax == 2 and ds / KM == pytest.approx(17.616328, abs=1e-6)
    assert f[0] == pytest.approx(0.162883, abs=1e-6)


def test_ray_geometry_matches_geometric_walkback():
    rng = np.random.default_rng(5)
    for _ in range(50):
        mu = rng.uniform(0.05, 1.0, 3) * rng.choice([-1, 1], 3)
        mu /= np.linalg.norm(mu)
        h = rng.uniform(1.0, 4.0, 3)
        ax, sg, ds, f = oracle.ray_geometry(h[0], h[1], h[2], mu)
        pt, ds2 = ind.upwind_point((5, 5, 5), mu, h)
        assert ds == pytest.approx(ds2, rel=1e-14)
        for a in range(3):
            assert 5 - sg[a] * f[a] == pytest.approx(pt[a], abs=1e-12)
        assert f[ax] == 1.0


def test_quadrature_set_moments():
    mu, w = inputs.carlson24()
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    assert np.abs((w[:, None] * mu).sum(0)).max() < 1e-15          # first moment
    m2 = (w[:, None, None] * mu[:, :, None] * mu[:, None, :]).sum(0)
    assert np.allclose(m2, np.eye(3) * 0.3333333570, atol=2e-10)
    assert np.all(mu[:12, 2] > 0) and np.all(mu[12:, 2] < 0)
    # r = 3*o + m, m = axis of the large cosine
    for r in range(24):
        assert np.argmax(np.abs(mu[r])) == r % 3
        o = r // 3
        for a in range(3):
            assert (mu[r, a] < 0) == bool((o >> a) & 1)


# --------------------------------------------------------------------------- P1
def test_P1_exponential_attenuation_zface():
    nx = ny = 6
    nz = 12
    dx = dy = 48 * KM
    dz = 32 * KM
    kap = np.full((nz, ny, nx), 2.5e-7)
    S = np.zeros((nz, ny, nx))
    I0 = 3.7
    for mu in ([A, A, B], [-A, A, B], [A, -A, B], [-A, -A, B]):
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mu, nz + 1, kap, S, inflow=np.full((ny, nx), I0))
        k = np.arange(nz)
        expect = I0 * np.exp(-2.5e-7 * k * dz / B)
        assert np.allclose(I, expect[:, None, None], rtol=1e-13, atol=0)
    # downward: inflow on the top plane
    I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, [A, -A, -B], nz + 1, kap, S, inflow=np.full((ny, nx), I0))
    expect = I0 * np.exp(-2.5e-7 * (nz - 1 - np.arange(nz)) * dz / B)
    assert np.allclose(I, expect[:, None, None], rtol=1e-13)


def test_P1b_lattice_aligned_pattern_shift():
    # dz chosen so that dx/|mu_x| = dy/|mu_y| = dz/|mu_z|: the upwind point is the corner node.
    nx, ny, nz = 7, 5, 5
    dx = dy = 10 * KM
    dz = dx * B / A
    kap = np.full((nz, ny, nx), 1.3e-6)
    S = np.zeros((nz, ny, nx))
    rng = np.random.default_rng(11)
    I0 = rng.uniform(1.0, 2.0, (ny, nx))
    for sx, sy in ((1, 1), (-1, 1), (1, -1), (-1, -1)):
        mu = [sx * A, sy * A, B]
        ax, sg, ds, f = oracle.ray_geometry(dx, dy, dz, mu)
        assert f[0] == pytest.approx(1.0, abs=1e-12) and f[1] == pytest.approx(1.0, abs=1e-12)
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mu, 3, kap, S, inflow=I0)
        for k in range(nz):
            shifted = np.roll(np.roll(I0, k * sx, axis=1), k * sy, axis=0)
            expect = shifted * math.exp(-1.3e-6 * ds * k)
            assert np.allclose(I[k], expect, rtol=1e-12), (sx, sy, k)


# --------------------------------------------------------------------------- P2
def test_P2_linear_source_in_tau_golden_and_closed_form():
    rows = _read_table("linear_source_values.txt")
    nx = ny = 3
    nz = 8
    dz = 20 * KM
    dtau = 0.5
    ds = dz / B
    kap = np.full((nz, ny, nx), dtau / ds)
    g, S0 = 0.3, 1.0
    t = dtau * np.arange(nz)
    S = np.broadcast_to((S0 + g * t)[:, None, None], (nz, ny, nx)).copy()
    I = oracle.sweep_ray(nx, ny, nz, 50 * KM, 50 * KM, dz, [A, A, B], nz + 1, kap, S)
    for (tt, val), k in zip(rows, (1, 2, 3)):
        assert tt == pytest.approx(t[k])
        assert I[k, 1, 1] == pytest.approx(val, abs=6e-11)          # 10 printed digits
    expect = S0 + g * t - g * (1.0 - np.exp(-t))
    assert np.allclose(I, expect[:, None, None], rtol=1e-14)
    # downward ray, source linear in the downward optical depth, I(top) = 0
    Sdn = np.broadcast_to((S0 + g * t[::-1])[:, None, None], (nz, ny, nx)).copy()
    I = oracle.sweep_ray(nx, ny, nz, 50 * KM, 50 * KM, dz, [A, -A, -B], nz + 1, kap, Sdn)
    td = t[::-1]
    expect = S0 + g * td - g * (1 - np.exp(-td)) - S0 * np.exp(-td)     # minus the missing I(0)=S0 part
    assert np.allclose(I, expect[:, None, None], rtol=1e-13)


# --------------------------------------------------------------------------- P3
def test_P3_thick_limit_all_rays_and_flux():
    nx = ny = 8
    nz = 24
    dx = dy = 48 * KM
    dz = 32 * KM
    kr = 6.0 / dz                                  # ~6-19 optical depths per segment
    kap = np.full((nz, ny, nx), kr)
    dSdz = 2.0e3 / dz
    S = np.broadcast_to((5.0e4 + dSdz * dz * np.arange(nz))[:, None, None], (nz, ny, nx)).copy()
    mus, w = inputs.carlson24()
    Fz = 0.0
    kmid = nz // 2
    for r in range(24):
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mus[r], 12, kap, S)
        D = I[kmid] - S[kmid]
        expect = -mus[r, 2] * dSdz / kr
        assert np.allclose(D, expect, rtol=1e-9), r
        Fz += 4 * math.pi * w[r] * mus[r, 2] * I[kmid, 0, 0]
    assert Fz == pytest.approx(-(4 * math.pi / 3) * dSdz / kr * (1 + 7.1e-8), rel=5e-9)


# --------------------------------------------------------------------------- P4
def test_P4_isothermal():
    nx = ny = 5
    nz = 10
    dx, dy, dz = 30 * KM, 40 * KM, 25 * KM
    rng = np.random.default_rng(2)
    kz = 10.0 ** rng.uniform(-8, -5.5, nz)
    kap = np.broadcast_to(kz[:, None, None], (nz, ny, nx)).copy()
    S = np.full((nz, ny, nx), 4.2e10)
    mus, _ = inputs.carlson24()
    for r in range(12):                           # upward: I == S everywhere, any kappa
        kap3 = 10.0 ** rng.uniform(-8, -5.5, (nz, ny, nx))
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mus[r], 3, kap3, S)
        assert np.allclose(I, S, rtol=1e-14)
    for r in range(12, 24):                       # downward z-face rays: I = S (1 - exp(-tau_r))
        ax, sg, ds, f = oracle.ray_geometry(dx, dy, dz, mus[r])
        if ax != 2:
            continue
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mus[r], nz + 1, kap, S)
        tau = np.zeros(nz)
        for k in range(nz - 2, -1, -1):
            tau[k] = tau[k + 1] + 0.5 * (kz[k] + kz[k + 1]) * ds
        assert np.allclose(I, (4.2e10 * (1 - np.exp(-tau)))[:, None, None], rtol=1e-13)


# --------------------------------------------------------------------------- P7
def test_P7_one_dimensional_reduction():
    nx = ny = 4
    nz = 40
    dx = dy = 48 * KM
    dz = 32 * KM
    z = np.arange(nz) / (nz - 1)
    kz = 3e-7 * np.exp(-9 * z) * 20
    Sz = 1e10 * (1 + 3 * (1 - z) ** 2)
    kap = np.broadcast_to(kz[:, None, None], (nz, ny, nx)).copy()
    S = np.broadcast_to(Sz[:, None, None], (nz, ny, nx)).copy()
    for mu in ([A, A, B], [-A, -A, B], [A, -A, -B], [-A, A, -B]):
        I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mu, nz + 1, kap, S)
        ref = ind.oned_zface(kz, Sz, mu[2], dz)
        assert np.allclose(I, ref[:, None, None], rtol=2e-12)


# --------------------------------------------------------------------------- P10
@pytest.mark.parametrize("shape", [(3, 3, 3), (4, 3, 2), (2, 5, 4)])
def test_P10_recursive_bruteforce(shape):
    nx, ny, nz = shape
    rng = np.random.default_rng(nx * 100 + ny * 10 + nz)
    kap = 10.0 ** rng.uniform(-7.5, -5.0, (nz, ny, nx))
    S = rng.uniform(1.0, 5.0, (nz, ny, nx)) * 1e10
    mus, _ = inputs.carlson24()
    for (dx, dy, dz) in ((48 * KM, 48 * KM, 32 * KM), (10 * KM, 35 * KM, 90 * KM)):
        for r in (0, 1, 2, 4, 8, 11, 13, 17, 21, 23):
            for P in (1, 2, 3):
                I = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mus[r], P, kap, S)
                ref = ind.recursive_solve(kap, S, mus[r], (dx, dy, dz), P)
                assert np.allclose(I, ref, rtol=1e-12), (r, P)


def test_P10_zero_component_ray():
    # a ray with mu_x = 0: the x-shifted stencil nodes carry zero weight
    nx, ny, nz = 3, 4, 3
    rng = np.random.default_rng(3)
    kap = 10.0 ** rng.uniform(-7.5, -5.5, (nz, ny, nx))
    S = rng.uniform(1.0, 5.0, (nz, ny, nx))
    for mu in ([0.0, 0.6, 0.8], [0.0, 0.0, -1.0], [0.6, 0.0, 0.8]):
        I = oracle.sweep_ray(nx, ny, nz, 20 * KM, 20 * KM, 20 * KM, mu, 2, kap, S)
        ref = ind.recursive_solve(kap, S, mu, (20 * KM,) * 3, 2)
        assert np.allclose(I, ref, rtol=1e-12)


# --------------------------------------------------------------------------- P11
def test_P11_I_form_equals_D_form():
    inp = inputs.make_config(1, grid=(12, 10, 14))
    kap, S = oracle.coefficients(inp)
    for r in (0, 1, 2, 14, 19, 21):
        I0 = oracle.sweep_ray(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu[r], 3, kap[0], S[0], form=0)
        I1 = oracle.sweep_ray(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu[r], 3, kap[0], S[0], form=1)
        assert np.max(np.abs(I0 - I1)) <= 1e-12 * np.max(np.abs(I0))


# --------------------------------------------------------------------------- P12
def _table_problem(nb=2, nT=5, nP=4, noise=True):
    rng = np.random.default_rng(9)
    logT = (3.5, 4.3)
    logP = (2.0, 7.0)
    xT = np.linspace(*logT, nT)
    xP = np.linspace(*logP, nP)
    L = (4.5 * xT[None, :, None] + 0.7 * xP[None, None, :] - 18.5
         + np.arange(nb)[:, None, None])
    if noise:
        L = L + 0.3 * rng.standard_normal(L.shape)
    f = rng.uniform(0.1, 0.9, (nb, nT))
    return logT, logP, xT, xP, L.astype(np.float32), f.astype(np.float32)


def test_P12_table_nodes_and_clamping():
    logT, logP, xT, xP, L, f = _table_problem()
    nb, nT, nP = L.shape
    # nodes of the table as a (nT x nP x 1) "grid"; plus out-of-range points
    T = np.repeat((10.0 ** xT)[None, :], nP, 0)            # [nP][nT] -> ny=nP, nx=nT
    P = np.repeat((10.0 ** xP)[:, None], nT, 1)
    T2 = np.stack([T, T * 0 + 10 ** 3.0, T * 0 + 10 ** 4.9])    # nz=3: in-range, below, above
    P2 = np.stack([P, P * 0 + 10 ** 1.0, P * 0 + 10 ** 8.5])
    rho = np.full_like(T2, 2.0e-7)
    inp = inputs.make_custom(nT, nP, 3, 1e6, 1e6, 1e6, rho, T2, P2, L, f, logT, logP)
    kap, S = oracle.coefficients(inp)
    Tf = inp.T.astype(np.float64)
    rh = inp.rho.astype(np.float64)
    for b in range(nb):
        # float32 rounding of T,P moves the lookup point by ~1e-7 of a table cell
        expect = 10.0 ** L[b].astype(np.float64).T * 2.0e-7       # [nP][nT]
        assert np.allclose(kap[b, 0], expect * (rh[0] / 2.0e-7), rtol=3e-5)
        assert np.allclose(kap[b, 1], 10.0 ** float(L[b, 0, 0]) * rh[1], rtol=1e-13)
        assert np.allclose(kap[b, 2], 10.0 ** float(L[b, -1, -1]) * rh[2], rtol=1e-13)
        sig = 5.670374e-5
        assert np.allclose(S[b, 1], float(f[b, 0]) * sig * Tf[1] ** 4 / math.pi, rtol=1e-13)
        assert np.allclose(S[b, 2], float(f[b, -1]) * sig * Tf[2] ** 4 / math.pi, rtol=1e-13)
        fb = np.repeat(f[b].astype(np.float64)[None, :], nP, 0)
        assert np.allclose(S[b, 0], fb * sig * Tf[0] ** 4 / math.pi, rtol=3e-6)


def test_P12_bilinear_exact_on_loglinear_table():
    logT, logP, xT, xP, L, f = _table_problem(nb=1, nT=9, nP=7, noise=False)
    L64 = (4.5 * xT[None, :, None] + 0.7 * xP[None, None, :] - 18.5)
    rng = np.random.default_rng(4)
    n = 64
    T = 10.0 ** rng.uniform(3.5, 4.3, n)
    P = 10.0 ** rng.uniform(2.0, 7.0, n)
    rho = 10.0 ** rng.uniform(-9, -6, n)
    inp = inputs.make_custom(n, 1, 1, 1e6, 1e6, 1e6, rho, T, P, L64.astype(np.float32), np.ones((1, 9)), logT, logP)
    kap, S = oracle.coefficients(inp)
    Tf, Pf, rf = (inp.T.astype(np.float64).ravel(), inp.P.astype(np.float64).ravel(), inp.rho.astype(np.float64).ravel())
    expect = 10.0 ** (4.5 * np.log10(Tf) + 0.7 * np.log10(Pf) - 18.5) * rf
    # the table itself was rounded to fp32 (abs 1e-6 in log10 -> 2.5e-6 relative)
    assert np.allclose(kap.ravel(), expect, rtol=5e-6)
    assert np.allclose(S.ravel(), 5.670374e-5 * Tf ** 4 / math.pi, rtol=1e-14)


# --------------------------------------------------------------------------- full solve
def _small_problem(nx=10, ny=10, nz=9, nb=2, P=3, seed=0):
    inp = inputs.make_config(3, grid=(nx, ny, nz), nbands=nb, npasses=P, seed_offset=seed)
    return inp


def test_solve_equals_sum_of_sweeps():
    """O-7: Q = 4 pi sum_b kaprho_b (J_b - S_b), J_b = sum_r w_r I; I_top order = upward rays."""
    inp = _small_problem()
    Q, Itop, J = oracle.solve(inp, want_J=True)
    kap, S = oracle.coefficients(inp)
    Jm = np.zeros_like(J)
    for b in range(inp.nbands):
        for r in range(24):
            I = ind.recursive_solve(kap[b], S[b], inp.mu[r], (inp.dx, inp.dy, inp.dz), inp.npasses) \
                if (b == 0 and r in (0, 13)) else \
                oracle.sweep_ray(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu[r], inp.npasses, kap[b], S[b])
            Jm[b] += I / 24.0
            if r < 12:
                assert np.allclose(Itop[b, r], I[-1], rtol=1e-12)
    assert np.allclose(J, Jm, rtol=1e-12)
    Qm = (4 * math.pi * kap * (Jm - S)).sum(0)
    assert np.allclose(Q, Qm, rtol=1e-8, atol=1e-10 * np.abs(Qm).max())  # J - S cancels ~6 digits


def _transform(inp, fn):
    return inputs.make_custom(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz,
                              fn(inp.rho), fn(inp.T), fn(inp.P), inp.logkappa, inp.bandfrac,
                              (inp.logT_min, inp.logT_max), (inp.logP_min, inp.logP_max),
                              npasses=inp.npasses)


def _ray_perm(mu, M):
    """index map r -> r' with mu[r'] == M @ mu[r]"""
    out = []
    for r in range(mu.shape[0]):
        v = M @ mu[r]
        d = np.abs(mu - v[None, :]).sum(1)
        out.append(int(np.argmin(d)))
        assert d[out[-1]] < 1e-14
    return out


def test_P5_symmetries():
    inp = _small_problem(nx=9, ny=9, nz=8, nb=2)
    Q, Itop = oracle.solve(inp)
    kap, S = oracle.coefficients(inp)
    # Q = 4 pi kaprho (J - S) carries the rounding of J (sum order differs under a symmetry)
    tol = 1e-11 * np.abs(Q).max() + 64 * np.finfo(np.float64).eps * (4 * math.pi * kap * S).max()
    # mirror x
    Qm, Im = oracle.solve(_transform(inp, lambda a: a[:, :, ::-1].copy()))
    assert np.abs(Qm - Q[:, :, ::-1]).max() < tol
    perm = _ray_perm(inp.mu, np.diag([-1.0, 1.0, 1.0]))
    for r in range(12):
        assert np.allclose(Im[:, perm[r]], Itop[:, r][:, :, ::-1], rtol=1e-11)
    # transpose x <-> y
    Qt, It = oracle.solve(_transform(inp, lambda a: a.transpose(0, 2, 1).copy()))
    assert np.abs(Qt - Q.transpose(0, 2, 1)).max() < tol
    perm = _ray_perm(inp.mu, np.array([[0.0, 1, 0], [1, 0, 0], [0, 0, 1]]))
    for r in range(12):
        assert np.allclose(It[:, perm[r]], Itop[:, r].transpose(0, 2, 1), rtol=1e-11)
    # rotate by 90 degrees about z: (x, y) -> (-y, x)
    Qr, Ir = oracle.solve(_transform(inp, lambda a: np.rot90(a, 1, axes=(2, 1)).copy()))
    assert np.abs(Qr - np.rot90(Q, 1, axes=(2, 1))).max() < tol


def test_P6_translation_invariance_at_seam_convergence():
    inp = _small_problem(nx=8, ny=6, nz=6, nb=1, P=14)
    Q, Itop = oracle.solve(inp)
    sh = lambda a: np.roll(np.roll(a, 3, axis=2), -2, axis=1)
    Qs, Is = oracle.solve(_transform(inp, sh))
    kap, S = oracle.coefficients(inp)
    assert np.abs(Qs - sh(Q)).max() < 1e-9 * np.abs(Q).max() + 64 * np.finfo(np.float64).eps * (4 * math.pi * kap * S).max()
    assert np.allclose(Is, np.roll(np.roll(Itop, 3, axis=3), -2, axis=2), rtol=1e-9)


def test_P6_horizontal_uniformity():
    inp = inputs.make_config(1, grid=(6, 5, 12), npasses=16)
    flat = lambda a: np.broadcast_to(a.reshape(inp.nz, -1).mean(1)[:, None, None], a.shape).copy()
    u = _transform(inp, flat)
    Q, Itop = oracle.solve(u)
    assert np.abs(Q - Q[:, :1, :1]).max() < 1e-10 * np.abs(Q).max()
    assert np.abs(Itop - Itop[:, :, :1, :1]).max() < 1e-10 * np.abs(Itop).max()


def test_P8_pass_fixed_point_geometric_decay():
    base = inputs.make_config(1, grid=(8, 8, 16), npasses=1)
    kap, S = oracle.coefficients(base)
    mu = base.mu[0]                               # big-x ray, crosses the seam
    prev = None
    diffs = []
    for P in range(1, 9):
        I = oracle.sweep_ray(8, 8, 16, base.dx, base.dy, base.dz, mu, P, kap[0], S[0])
        if prev is not None:
            diffs.append(np.abs(I - prev).max())
        prev = I
    assert diffs[0] > 0
    assert all(b <= a * 1.0000001 for a, b in zip(diffs[:-1], diffs[1:]))
    assert diffs[-1] < 1e-3 * diffs[0]
    # pass 1 really starts from I^(0) = S at the seam: column i = 0 of pass 1 equals the
    # formal integral fed with S at the wrapped stencil nodes
    I1 = oracle.sweep_ray(8, 8, 16, base.dx, base.dy, base.dz, mu, 1, kap[0], S[0])
    ref = ind.recursive_solve(kap[0], S[0], mu, (base.dx, base.dy, base.dz), 1)
    assert np.allclose(I1, ref, rtol=1e-12)


def test_P9_energy_balance_trend():
    """sum Q dV ~ -(F_top - F_bottom) A; not exact for this scheme -- it must improve on refinement."""
    def imbalance(n):
        nz = 2 * n
        L = 6.0e7                                   # 600 km box
        z = (np.arange(nz) / (nz - 1))[:, None, None]
        x = (np.arange(n) / n)[None, None, :]
        y = (np.arange(n) / n)[None, :, None]
        T = 9000 - 4000 * z + 300 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) * (1 - z)
        rho = 3e-7 * np.exp(-5 * z) * (1 + 0.1 * np.cos(2 * np.pi * x)) + 0 * y
        P = rho * 1.380649e-16 * T / (1.3 * 1.6735575e-24)
        nT = nP = 32
        xT = np.linspace(3.5, 4.3, nT)
        xP = np.linspace(2, 7, nP)
        # opacity offset chosen so that the box is ~2 optical depths deep: every cell is resolved
        Lk = (4.5 * xT[None, :, None] + 0.7 * xP[None, None, :] - 21.5)
        inp = inputs.make_custom(n, n, nz, L / n, L / n, L / (nz - 1), rho, T, P, Lk, np.ones((1, nT)),
                                 (3.5, 4.3), (2, 7), npasses=10)
        Q, Itop, J = oracle.solve(inp, want_J=True)
        kap, S = oracle.coefficients(inp)
        Fz = np.zeros((nz, n, n))
        for r in range(24):
            I = oracle.sweep_ray(n, n, nz, inp.dx, inp.dy, inp.dz, inp.mu[r], 10, kap[0], S[0])
            Fz += 4 * math.pi * inp.wq[r] * inp.mu[r, 2] * I
        # trapezoid in z (node planes), periodic in x, y
        wz = np.ones(nz); wz[0] = wz[-1] = 0.5
        lhs = (Q * wz[:, None, None]).sum() * inp.dx * inp.dy * inp.dz
        rhs = -(Fz[-1].sum() - Fz[0].sum()) * inp.dx * inp.dy
        return abs(lhs - rhs) / abs(rhs), lhs, rhs
    e1, l1, r1 = imbalance(8)
    e2, l2, r2 = imbalance(16)
    assert l1 * r1 > 0 and l2 * r2 > 0             # same sign: Q is a cooling where flux leaves
    assert e2 < 0.7 * e1                           # measured 1.5% -> 0.8% (-> 0.4% at n = 32)
    assert e2 < 0.02


# ------------------------------------------------------------------ O-9 grid staggering (NEXT #1)
def test_O9_cells_to_nodes_constant_linear_and_edges():
    """Trilinear interpolation at a corner = mean of 8 cells: constants are kept, a field linear
    in z lands on the midpoints, and the bottom / top corner levels repeat the edge cell level
    (reading R20)."""
    ncz, ncy, ncx = 6, 4, 5
    c = np.full((ncz, ncy, ncx), 3.25, dtype=np.float32)
    assert np.array_equal(oracle.cells_to_nodes(c), np.full((ncz + 1, ncy, ncx), 3.25, dtype=np.float32))
    z = (np.arange(ncz, dtype=np.float64) + 0.5)                  # cell-centre heights
    c = np.broadcast_to((2.0 + 0.5 * z)[:, None, None], (ncz, ncy, ncx)).astype(np.float32)
    n = oracle.cells_to_nodes(c).astype(np.float64)
    for k in range(1, ncz):
        assert np.allclose(n[k], 2.0 + 0.5 * k, rtol=0, atol=1e-6)      # corner height k = midpoint
    assert np.allclose(n[0], c[0]) and np.allclose(n[ncz], c[ncz - 1])  # zero-gradient ghost levels


def test_O9_cells_to_nodes_fourier_mode_attenuation():
    """A horizontal Fourier mode sin(2 pi m (i + 1/2) / n) of the cell centres arrives at the corners
    x = i as cos(pi m / n) sin(2 pi m i / n): the closed form of the two-point mean, in x and in y."""
    ncz, ncy, ncx = 3, 12, 16
    for axis, n_, m in ((2, ncx, 3), (1, ncy, 2)):
        idx = np.arange(n_, dtype=np.float64)
        mode = np.sin(2 * np.pi * m * (idx + 0.5) / n_)
        shape = [1, 1, 1]; shape[axis] = n_
        c = np.broadcast_to(mode.reshape(shape), (ncz, ncy, ncx)).astype(np.float32)
        n = oracle.cells_to_nodes(c).astype(np.float64)
        want = np.cos(np.pi * m / n_) * np.sin(2 * np.pi * m * idx / n_)
        got = n[1, 0, :] if axis == 2 else n[1, :, 0]
        assert np.abs(got - want).max() < 2e-7


def test_O9_cells_to_nodes_is_the_rounded_exact_mean():
    """The fp32 node value is the correctly rounded mean of the 8 fp32 cells (brute force in
    exact rational arithmetic on a tiny grid)."""
    from fractions import Fraction
    rng = np.random.default_rng(5)
    c = (rng.standard_normal((2, 3, 3)) * 10 ** rng.uniform(-3, 3, (2, 3, 3))).astype(np.float32)
    n = oracle.cells_to_nodes(c)
    ncz, ncy, ncx = c.shape
    for k in range(ncz + 1):
        for j in range(ncy):
            for i in range(ncx):
                tot = Fraction(0)
                for dk in (0, 1):
                    kk = min(max(k - dk, 0), ncz - 1)
                    for dj in (0, 1):
                        for di in (0, 1):
                            tot += Fraction(float(c[kk, (j - dj) % ncy, (i - di) % ncx]))
                assert n[k, j, i] == np.float32(float(tot / 8))


def test_O9_nodes_to_cells_linear_exact_and_sum_rule():
    """Back-averaging: exact on a field linear in z; sum over cells = sum over nodes with the
    trapezoid weights (1/2 on the two boundary levels) -- every node is a corner of 8 cells, or of
    4 on the bottom / top level."""
    nz, ny, nx = 7, 5, 6
    q = np.broadcast_to((1.0 - 0.25 * np.arange(nz))[:, None, None], (nz, ny, nx)).copy()
    qc = oracle.nodes_to_cells(q)
    assert qc.shape == (nz - 1, ny, nx)
    assert np.allclose(qc, (1.0 - 0.25 * (np.arange(nz - 1) + 0.5))[:, None, None], rtol=0, atol=1e-15)
    rng = np.random.default_rng(9)
    q = rng.standard_normal((nz, ny, nx))
    w = np.ones(nz); w[0] = w[-1] = 0.5
    assert abs(oracle.nodes_to_cells(q).sum() - (w[:, None, None] * q).sum()) < 1e-12


def test_O9_solve_cells_of_horizontally_uniform_atmosphere_is_uniform():
    """A horizontally uniform cell atmosphere stays uniform through staggering, solve and
    back-averaging (with enough passes for the seams, pin P6)."""
    inp = inputs.make_config(1, grid=(6, 6, 9), npasses=14)
    for f in (inp.rho, inp.T, inp.P):
        f[...] = f[:, :1, :1]
    Qc, Itop, node = oracle.solve_cells(inp)
    assert node.nz == inp.nz + 1 and Qc.shape == inp.shape
    assert np.abs(Qc - Qc[:, :1, :1]).max() <= 1e-9 * np.abs(Qc).max()


# --------------------------------------------------------------------------- O-10 / O-11 (NEXT #2): flux
def _flat_table_problem(nx, ny, nz, dx, dy, dz, S3, kaprho, P=8, nb=1):
    """Inputs whose stage A gives kaprho = const and S = S3 exactly up to the fp32 rounding of T:
    flat opacity table (log10 kappa = 0), rho = kaprho, band fraction 1, T = (pi S / sigma)^(1/4)."""
    T = (math.pi * S3 / 5.670374e-5) ** 0.25
    rho = np.full((nz, ny, nx), kaprho)
    Pg = np.full((nz, ny, nx), 1.0e4)
    logk = np.zeros((nb, 4, 4), dtype=np.float32)
    bf = np.ones((nb, 4), dtype=np.float32)
    return inputs.make_custom(nx, ny, nz, dx, dy, dz, rho, T, Pg, logk, bf, (3.0, 5.0), (2.0, 6.0), npasses=P)


def test_O10_flux_of_tilted_linear_source_in_the_thick_limit():
    """P3 for all three components: with S linear in space and uniform kaprho every ray carries
    D_r = -Omega_r . grad S / kaprho (bilinear interpolation is exact on linear fields), so
    F = 4 pi sum_r w_r Omega_r I_r = -(4 pi / 3) (1 + 7.1e-8) grad S / kaprho  (second moment of the ray set)."""
    nx, ny, nz = 16, 16, 20
    dx, dy, dz = 48 * KM, 40 * KM, 32 * KM
    kr = 8.0 / dz
    gx, gy, gz = 1.1e3 / dx, -0.7e3 / dy, 2.0e3 / dz
    z, y, x = np.meshgrid(np.arange(nz) * dz, np.arange(ny) * dy, np.arange(nx) * dx, indexing="ij")
    S3 = 6.0e5 + gx * x + gy * y + gz * z
    inp = _flat_table_problem(nx, ny, nz, dx, dy, dz, S3, kr)
    Q, Itop, F = oracle.solve(inp, want_F=True)
    c = -(4 * math.pi / 3) * (1 + 7.1e-8) / kr
    sl = (slice(6, nz - 6), slice(5, ny - 5), slice(5, nx - 5))      # away from the seams (gradient jump) and the inflow planes
    for a, g in enumerate((gx, gy, gz)):
        assert np.allclose(F[a][sl], c * g, rtol=1e-4), a              # fp32 rounding of T: 2.4e-7 on S against dS per cell ~ 2e-3 S


def test_O10_flux_vanishes_in_an_isothermal_thick_medium_and_flips_under_mirror():
    nx, ny, nz = 10, 8, 14
    dx, dy, dz = 48 * KM, 48 * KM, 32 * KM
    S3 = np.full((nz, ny, nx), 3.0e9)
    inp = _flat_table_problem(nx, ny, nz, dx, dy, dz, S3, 10.0 / dz, P=3)
    _, _, F = oracle.solve(inp, want_F=True)
    assert np.abs(F[:, 2:6]).max() <= 1e-9 * 4 * math.pi * 3.0e9      # I = S for every ray deep inside: sum_r w_r Omega_r = 0
    # mirror x: F_x flips sign, F_y and F_z do not (the ray set is mirror symmetric)
    inp = _small_problem(nx=12, ny=10, nz=9, nb=2, P=4)
    _, _, F = oracle.solve(inp, want_F=True)
    _, _, Fm = oracle.solve(_transform(inp, lambda a: np.ascontiguousarray(a[:, :, ::-1])), want_F=True)
    s = np.abs(F).max()
    assert np.allclose(Fm[0], -F[0][:, :, ::-1], rtol=0, atol=1e-12 * s)
    assert np.allclose(Fm[1], F[1][:, :, ::-1], rtol=0, atol=1e-12 * s)
    assert np.allclose(Fm[2], F[2][:, :, ::-1], rtol=0, atol=1e-12 * s)


def test_O10_flux_is_the_weighted_vector_sum_of_sweeps():
    inp = _small_problem(nx=8, ny=6, nz=7, nb=2, P=2)
    _, _, F = oracle.solve(inp, want_F=True)
    kap, S = oracle.coefficients(inp)
    Fm = np.zeros_like(F)
    for b in range(inp.nbands):
        for r in range(24):
            I = oracle.sweep_ray(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.mu[r], inp.npasses, kap[b], S[b])
            Fm += 4 * math.pi * inp.wq[r] * (inp.mu[r] / np.linalg.norm(inp.mu[r]))[:, None, None, None] * I[None]
    assert np.allclose(F, Fm, rtol=1e-12, atol=1e-12 * np.abs(Fm).max())


def test_O11_flux_divergence_against_numpy_gradient_closed_form_and_telescoping():
    nx, ny, nz = 12, 10, 9
    dx, dy, dz = 3.0, 2.0, 1.5
    rng = np.random.default_rng(11)
    F = rng.normal(size=(3, nz, ny, nx))
    inp = _small_problem(nx=nx, ny=ny, nz=nz, nb=1)
    inp.dx, inp.dy, inp.dz = dx, dy, dz
    Qdiv, _ = oracle.flux_heating(inp, F, want_blend=False)
    # library routine: np.gradient (central inside, first-order one-sided at the ends) on periodically padded x, y
    gx = np.gradient(np.concatenate([F[0][:, :, -1:], F[0], F[0][:, :, :1]], axis=2), dx, axis=2)[:, :, 1:-1]
    gy = np.gradient(np.concatenate([F[1][:, -1:, :], F[1], F[1][:, :1, :]], axis=1), dy, axis=1)[:, 1:-1, :]
    gz = np.gradient(F[2], dz, axis=0, edge_order=1)
    assert np.allclose(Qdiv, -(gx + gy + gz), rtol=1e-13, atol=1e-13)
    # closed form: central difference of sin is cos * sin(h k)/(h k)
    x = np.arange(nx) * dx
    kx = 2 * math.pi / (nx * dx)
    F2 = np.zeros_like(F)
    F2[0] = np.sin(kx * x)[None, None, :]
    Qd2, _ = oracle.flux_heating(inp, F2, want_blend=False)
    assert np.allclose(Qd2, -(kx * np.cos(kx * x) * np.sin(kx * dx) / (kx * dx))[None, None, :], atol=1e-14)
    # telescoping: sum_k Qdiv dz = -(1.5 Fz[top] - 0.5 Fz[top-1] + 0.5 Fz[1] - 1.5 Fz[0]) for a purely vertical flux
    F3 = np.zeros_like(F)
    F3[2] = F[2]
    Qd3, _ = oracle.flux_heating(inp, F3, want_blend=False)
    lhs = Qd3.sum(axis=0) * dz
    rhs = -(1.5 * F[2][-1] - 0.5 * F[2][-2] + 0.5 * F[2][1] - 1.5 * F[2][0])
    assert np.allclose(lhs, rhs, atol=1e-12)


def test_O11_blend_weights():
    nx, ny, nz = 6, 5, 8
    dz = 2.0e6
    inp = _small_problem(nx=nx, ny=ny, nz=nz, nb=1)
    inp.dz = dz
    rng = np.random.default_rng(3)
    F = rng.normal(size=(3, nz, ny, nx))
    QJ = rng.normal(size=(nz, ny, nx))
    kr = 0.05 / dz
    k0 = np.full((nz, ny, nx), kr)
    tau0 = 0.1
    Qdiv, Qb = oracle.flux_heating(inp, F, QJ, k0, tau0=tau0)
    w = np.exp(-kr * dz * (nz - np.arange(nz)) / tau0)               # uniform medium: taubar(k) = kaprho dz (nz - k)
    assert np.allclose(Qb, w[:, None, None] * QJ + (1 - w)[:, None, None] * Qdiv, rtol=1e-13, atol=1e-15)
    # horizontally varying opacity enters through its level mean only
    k1 = k0 * (1 + 0.5 * np.sin(np.arange(nx)))[None, None, :]
    k1 *= k0.mean() / k1.mean(axis=(1, 2), keepdims=True)
    _, Qb1 = oracle.flux_heating(inp, F, QJ, k1, tau0=tau0)
    assert np.allclose(Qb1, Qb, rtol=1e-12, atol=1e-15)
    # limits: tau0 -> infinity gives the J - S form, tau0 -> 0 the flux divergence
    assert np.allclose(oracle.flux_heating(inp, F, QJ, k0, tau0=1e30)[1], QJ, rtol=1e-12)
    assert np.allclose(oracle.flux_heating(inp, F, QJ, k0, tau0=1e-30)[1], Qdiv, rtol=1e-12)


# --------------------------------------------------------------------------- O-12 (NEXT #3): error-controlled iteration
def _faces(I, mu):
    """The two faces O-5 keeps: i = iface (all j, k) and j = jface (all i, k)."""
    nz, ny, nx = I.shape
    iface = nx - 1 if mu[0] > 0 else 0
    jface = ny - 1 if mu[1] > 0 else 0
    return I[:, :, iface].copy(), I[:, jface, :].copy()


def test_O12_error_is_the_face_change_of_the_fixed_pass_sweeps_and_the_stop_rule():
    """The error-controlled sweep is tied to the pinned fixed-pass one: after p passes it holds the same field
    bit for bit, its err_p / scale_p is the change of the two seam faces between the p-pass and the (p-1)-pass
    solution (pass 0: I^(0) = S, Dirichlet value on the Dirichlet plane) over the largest face intensity, and it
    stops at the first pass whose error is within the tolerance."""
    base = inputs.make_config(1, grid=(8, 8, 16), npasses=1)
    kap, S = oracle.coefficients(base)
    g = (8, 8, 16, base.dx, base.dy, base.dz)
    for mu in (base.mu[0], base.mu[7], base.mu[14]):           # an x-, a y- and a z-march ray, different octants
        fixed = [None] + [oracle.sweep_ray(*g, mu, P, kap[0], S[0]) for P in range(1, 9)]
        I0 = S[0].copy()
        kdir = 0 if mu[2] > 0 else 15
        if mu[2] < 0:
            I0[kdir] = 0.0
        fixed[0] = I0
        want = []
        for P in range(1, 9):
            (ax, ay), (bx, by) = _faces(fixed[P], mu), _faces(fixed[P - 1], mu)
            err = max(np.abs(ax - bx).max(), np.abs(ay - by).max())
            want.append(err / max(np.abs(ax).max(), np.abs(ay).max()))
        I, fc, rel, used = oracle.sweep_ray_tol(*g, mu, -1.0, 8, kap[0], S[0])
        assert used == 8 and np.array_equal(I, fixed[8])       # a negative tolerance never stops early
        assert np.allclose(rel, want, rtol=1e-12, atol=0)
        assert np.array_equal(fc[0], _faces(fixed[8], mu)[0]) and np.array_equal(fc[1], _faces(fixed[8], mu)[1])
        # P8: the change decays from pass to pass and reaches exactly 0 once every characteristic has been traced
        # back to the inflow plane (the dependence of an upward ray only ever runs downwards)
        assert all(b <= a for a, b in zip(rel[:-1], rel[1:])) and rel[-1] < 1e-3 * rel[0] and rel[0] > 0
        nz_ = int((rel > 0).sum())
        assert nz_ >= 3
        for k in range(1, nz_):                                # a tolerance between err_k and err_{k+1} stops after k+1 passes
            tol = math.sqrt(want[k - 1] * want[k])
            Ik, _, relk, usedk = oracle.sweep_ray_tol(*g, mu, tol, 8, kap[0], S[0])
            assert usedk == k + 1 and np.array_equal(Ik, fixed[k + 1]) and np.array_equal(relk, rel[:k + 1])
        assert oracle.sweep_ray_tol(*g, mu, 1e-30, 3, kap[0], S[0])[3] == 3      # the cap


def test_O12_warm_start_continues_the_iteration():
    """Warm start = the faces of an earlier solve as the faces of I^(0): one more pass from the P-pass faces is
    pass P+1 bit for bit, and from converged faces the first pass already meets the tolerance."""
    base = inputs.make_config(1, grid=(8, 8, 16), npasses=1)
    kap, S = oracle.coefficients(base)
    g = (8, 8, 16, base.dx, base.dy, base.dz)
    mu = base.mu[3]
    I3, f3, rel3, _ = oracle.sweep_ray_tol(*g, mu, -1.0, 3, kap[0], S[0])
    I4w, f4w, rel4w, used = oracle.sweep_ray_tol(*g, mu, -1.0, 1, kap[0], S[0], warm=f3)
    I4 = oracle.sweep_ray(*g, mu, 4, kap[0], S[0])
    assert used == 1 and np.array_equal(I4w, I4)
    I8, f8, rel8, _ = oracle.sweep_ray_tol(*g, mu, -1.0, 8, kap[0], S[0])
    tol = 2.0 * rel8[-1]
    cold = oracle.sweep_ray_tol(*g, mu, tol, 20, kap[0], S[0])
    warm = oracle.sweep_ray_tol(*g, mu, tol, 20, kap[0], S[0], warm=cold[1])
    assert cold[3] >= 7 and warm[3] == 1 and warm[2][0] <= tol
    assert np.abs(warm[0] - cold[0]).max() <= tol * np.abs(cold[0]).max()


def test_O12_solve_modes_against_the_fixed_pass_solve():
    """All bands and rays: with a negative tolerance and max_passes = P both modes are the fixed P-pass solve (Q to summation
    rounding, I_top bit for bit); mode 0 stops every (band, ray) problem on its own error, mode 1 runs all of
    them as long as the slowest one needs; a warm restart from the returned faces needs one pass."""
    inp = _small_problem(nx=10, ny=8, nz=9, nb=2, P=3)
    Q3, I3 = oracle.solve(inp)
    for mode in (0, 1):
        Q, It, fc, used, rel = oracle.solve_tol(inp, -1.0, 3, mode=mode)
        assert (used == 3).all() and np.array_equal(It, I3)
        assert np.abs(Q - Q3).max() <= 1e-12 * np.abs(Q3).max()
    kap, S = oracle.coefficients(inp)
    g = (inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz)
    tol = 1e-4
    each = np.array([oracle.sweep_ray_tol(*g, inp.mu[r], tol, 30, kap[b], S[b])[3]
                     for b in range(inp.nbands) for r in range(inp.nrays)])
    Q0, I0, f0, used0, _ = oracle.solve_tol(inp, tol, 30, mode=0)
    assert np.array_equal(used0, each) and each.min() < each.max()
    Q1, I1, f1, used1, rel1 = oracle.solve_tol(inp, tol, 30, mode=1)
    assert (used1 == each.max()).all() and len(rel1) == each.max()
    assert rel1[-1] <= tol < rel1[-2]
    inp_fixed = _small_problem(nx=10, ny=8, nz=9, nb=2, P=int(each.max()))
    Qf, If = oracle.solve(inp_fixed)
    assert np.array_equal(I1, If) and np.abs(Q1 - Qf).max() <= 1e-12 * np.abs(Qf).max()
    Qw, Iw, fw, usedw, relw = oracle.solve_tol(inp, tol, 30, mode=1, faces=f1)
    assert (usedw == 1).all() and relw[0] <= tol
    assert np.abs(Qw - Q1).max() <= 10 * tol * np.abs(Q1).max()


# --------------------------------------------------------------------------- O-13 (NEXT #4: scattering, source update along the ray)
def _scatter_case(nx=4, ny=3, nz=6, seed=5):
    rng = np.random.default_rng(seed)
    mu, w = inputs.carlson24()
    dx = dy = dz = 30 * KM
    z = np.arange(nz)[:, None, None]
    kap = 3e-7 * np.exp(-0.5 * z) * (1.0 + 0.3 * rng.random((nz, ny, nx)))       # ~0.9 per cell at the bottom
    Bt = 2.0 * np.exp(-0.3 * z) * (1.0 + 0.2 * rng.random((nz, ny, nx)))
    eps = 0.05 + 0.5 * rng.random((nz, ny, nx))
    return nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps


def test_O13_with_eps_one_is_the_fixed_pass_formal_solution():
    """eps = 1: S stays B, and n iterations are n Jacobi-seam passes of O-5 for every ray (the plane-by-plane
    visiting order of O-13 against the k, j, i order of the pinned O-5) and J their weighted sum."""
    nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, _ = _scatter_case()
    S, J, ch, I = oracle.scatter_solve(nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, 1.0, 3, gs=True, want_I=True)
    assert np.array_equal(S, Bt) and np.all(ch == 0.0)
    Jref = np.zeros_like(J)
    for r in range(24):
        Ir = oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mu[r], 3, kap, Bt)
        assert np.abs(I[r] - Ir).max() <= 1e-13 * np.abs(Ir).max()
        Jref += w[r] * Ir
    assert np.abs(J - Jref).max() <= 1e-12 * np.abs(Jref).max()


def test_O13_fixed_point_is_the_solution_of_the_linear_system():
    """J is linear in S (the bottom inflow I = S included), so the converged source function solves
    (1 - (1 - eps) L) S = eps B with L built column by column from the pinned periodic formal solution (O-5 with
    enough passes for the seams to converge).  Both iterations must end there; the incremental J of the
    Gauss-Seidel form must equal the weighted sum of its intensities."""
    nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps = _scatter_case()
    N = nx * ny * nz
    L = np.zeros((N, N))
    for c in range(N):
        e = np.zeros(N); e[c] = 1.0
        e = e.reshape(nz, ny, nx)
        col = np.zeros((nz, ny, nx))
        for r in range(24):
            col += w[r] * oracle.sweep_ray(nx, ny, nz, dx, dy, dz, mu[r], 60, kap, e)
        L[:, c] = col.ravel()
    Sstar = np.linalg.solve(np.eye(N) - (1.0 - eps.ravel())[:, None] * L, (eps * Bt).ravel()).reshape(nz, ny, nx)
    Sg, Jg, chg, Ig = oracle.scatter_solve(nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps, 300, gs=True, want_I=True)
    Sj, Jj, chj = oracle.scatter_solve(nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps, 300, gs=False)
    assert np.abs(Sg - Sstar).max() <= 1e-10 * Sstar.max()
    assert np.abs(Sj - Sstar).max() <= 1e-10 * Sstar.max()
    assert np.abs(Jg - np.tensordot(w, Ig, axes=1)).max() <= 1e-12 * Jg.max()
    assert np.abs(Sg - ((1.0 - eps) * Jg + eps * Bt)).max() <= 1e-13 * Sg.max()
    # the reason for the scheme: fewer iterations than the Jacobi form
    e_g = [np.abs(oracle.scatter_solve(nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps, n, gs=True)[0] - Sstar).max() for n in (5, 10)]
    e_j = [np.abs(oracle.scatter_solve(nx, ny, nz, dx, dy, dz, mu, w, kap, Bt, eps, n, gs=False)[0] - Sstar).max() for n in (5, 10)]
    assert e_g[0] < e_j[0] and e_g[1] < e_j[1]


def test_O13_sqrt_eps_law_of_the_isothermal_semi_infinite_atmosphere():
    """Isothermal, constant eps, semi-infinite: S(tau = 0) = sqrt(eps) B, exact in every discrete-ordinate
    approximation (Chandrasekhar, Radiative Transfer, ch. XI).  Horizontally uniform column of vertical optical depth
    100 whose cells thin out by 1e5 towards the top; what is left is the linear-source discretisation of tau, which
    halves when the number of levels doubles."""
    mu, w = inputs.carlson24()
    nx = ny = 2
    dz = 10 * KM
    err = {}
    for nz in (90, 180):
        prof = np.exp(-(np.arange(nz) / (nz - 1.0)) * math.log(1e5))
        kap = np.broadcast_to((prof / prof.sum() * 100.0 / dz)[:, None, None], (nz, ny, nx)).copy()
        Bt = np.ones((nz, ny, nx))
        for eps in (0.1, 0.3):
            S, J, ch = oracle.scatter_solve(nx, ny, nz, dz, dz, dz, mu, w, kap, Bt, eps, 1000, gs=True)
            assert ch[-1] < 1e-8
            err[nz, eps] = S[nz - 1, 0, 0] / math.sqrt(eps) - 1.0
            assert abs(err[nz, eps]) <= 0.01
            assert S[0, 0, 0] == pytest.approx(1.0, rel=1e-6)             # thermalised at depth
            assert np.all(np.diff(S[:, 0, 0]) <= 1e-12)                   # monotonic outward
    for eps in (0.1, 0.3):
        assert abs(err[180, eps]) < 0.6 * abs(err[90, eps])
