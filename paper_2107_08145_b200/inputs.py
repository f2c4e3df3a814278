"""Seeded synthetic inputs for the RTS hot path (serves BOTH the oracle and the CUDA path).

This module holds NONE of the method's arithmetic: no opacity lookup, no source
function, no ray geometry, no transfer integration.  It only manufactures the
fields (rho, T, P), the opacity / band-fraction tables and the quadrature data
(the 24 direction cosines quoted by BASELINE.json configs[0]) that both sides
consume as plain fp32 / fp64 arrays.

Recipe: SURVEY.md section 8(d) ("Synthetic inputs"), which fills in the constants
BASELINE.json `configs` leave open.  The paper's own inputs (MURaM snapshots and
opacity tables, sections 4.1 / 5 / 6.2) are not
public, so these stand in for them.  Everything is generated in fp64 and cast to
fp32 once; those fp32 arrays are the inputs of both sides.
"""
from __future__ import annotations

import dataclasses
from typing import Optional, Sequence, Tuple

import numpy as np

# physical constants used only to build a consistent ideal-gas pressure (cgs)
K_B = 1.380649e-16
M_H = 1.6735575e-24
MU_MOL = 1.3

# BASELINE.json configs[0]: direction cosines of the Carlson-type 24-ray set
CARLSON_A = 0.2958759
CARLSON_B = 0.9082483


@dataclasses.dataclass
class RTSInputs:
    """One synthetic RTS problem. Arrays are C-contiguous, x fastest."""
    name: str
    nx: int
    ny: int
    nz: int
    dx: float            # cm
    dy: float            # cm
    dz: float            # cm
    nbands: int
    npasses: int
    rho: np.ndarray      # float32 [nz][ny][nx]  g cm^-3
    T: np.ndarray        # float32 [nz][ny][nx]  K
    P: np.ndarray        # float32 [nz][ny][nx]  dyn cm^-2
    nT: int
    nP: int
    logT_min: float
    logT_max: float
    logP_min: float
    logP_max: float
    logkappa: np.ndarray  # float32 [nbands][nT][nP]   log10 kappa (cm^2 g^-1)
    bandfrac: np.ndarray  # float32 [nbands][nT]
    mu: np.ndarray        # float64 [nrays][3]  direction of photon travel
    wq: np.ndarray        # float64 [nrays]     quadrature weights (sum 1)

    @property
    def shape(self) -> Tuple[int, int, int]:
        return (self.nz, self.ny, self.nx)

    @property
    def ncells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def nrays(self) -> int:
        return int(self.mu.shape[0])

    @property
    def n_up(self) -> int:
        return int(np.count_nonzero(self.mu[:, 2] > 0))

    @property
    def updates(self) -> int:
        """Nominal cell*band*ray updates of one solve, U = N*nb*nrays*P."""
        return self.ncells * self.nbands * self.nrays * self.npasses


def carlson24() -> Tuple[np.ndarray, np.ndarray]:
    """The 24 directions of BASELINE.json configs[0] in the order of SURVEY 8(c) O-8.

    r = 3*o + m; octant o = bx + 2*by + 4*bz with b_a = 0 if mu_a > 0 else 1;
    m = axis carrying the large cosine (0:x, 1:y, 2:z).  Weights 1/24 (J is the
    mean over the sphere).  The 7-digit cosines are used as given (not
    renormalised).  Upward rays (mu_z > 0) are exactly r = 0..11.
    """
    mu = np.empty((24, 3), dtype=np.float64)
    for o in range(8):
        sgn = [1.0 if ((o >> a) & 1) == 0 else -1.0 for a in range(3)]
        for m in range(3):
            for a in range(3):
                mu[3 * o + m, a] = sgn[a] * (CARLSON_B if a == m else CARLSON_A)
    w = np.full(24, 1.0 / 24.0, dtype=np.float64)
    return mu, w


# ----------------------------------------------------------------------------
# smoothing helpers (input synthesis only)
# ----------------------------------------------------------------------------
def _box3(g: np.ndarray) -> np.ndarray:
    """3-point box filter: periodic along x, y; edge-replicate along z."""
    g = (np.roll(g, 1, axis=2) + g + np.roll(g, -1, axis=2)) / 3.0
    g = (np.roll(g, 1, axis=1) + g + np.roll(g, -1, axis=1)) / 3.0
    gp = np.concatenate([g[:1], g, g[-1:]], axis=0)
    g = (gp[:-2] + gp[1:-1] + gp[2:]) / 3.0
    return g


def _gauss_periodic_axis(g: np.ndarray, sigma_cells: float, axis: int) -> np.ndarray:
    """Periodic Gaussian smoothing along one axis (exact circular convolution via FFT)."""
    import scipy.fft as sfft
    n = g.shape[axis]
    k = sfft.rfftfreq(n)  # cycles per cell
    resp = np.exp(-2.0 * (np.pi * k * sigma_cells) ** 2)
    shape = [1, 1, 1]
    shape[axis] = resp.shape[0]
    G = sfft.rfft(g, axis=axis, workers=-1)
    G *= resp.reshape(shape)
    return sfft.irfft(G, n=n, axis=axis, workers=-1)


def _gauss_replicate_z(g: np.ndarray, sigma_cells: float) -> np.ndarray:
    """Gaussian smoothing along z with edge replication (kernel truncated at 4 sigma)."""
    from scipy.ndimage import gaussian_filter1d
    return gaussian_filter1d(g, sigma_cells, axis=0, mode="nearest", truncate=4.0)


def _granulation(g: np.ndarray, sig_h_cells_x: float, sig_h_cells_y: float,
                 sig_v_cells: float) -> np.ndarray:
    g = _gauss_periodic_axis(g, sig_h_cells_x, axis=2)
    g = _gauss_periodic_axis(g, sig_h_cells_y, axis=1)
    g = _gauss_replicate_z(g, sig_v_cells)
    # unit standard deviation on every horizontal level: edge replication in z would
    # otherwise leave ~4x larger fluctuations on the top and bottom planes
    g = g - g.mean(axis=(1, 2), keepdims=True)
    sd = g.std(axis=(1, 2), keepdims=True)
    return g / np.where(sd > 0, sd, 1.0)


def _unit_std(g: np.ndarray) -> np.ndarray:
    g = g - g.mean()
    s = g.std()
    return g / s if s > 0 else g


# ----------------------------------------------------------------------------
# mean profiles
# ----------------------------------------------------------------------------
def _profile_photosphere(zeta: np.ndarray):
    T0 = 8250.0 - 3750.0 * np.tanh((zeta - 0.5) / 0.15)
    rho0 = 3e-7 * np.exp(-6.613 * zeta)
    return T0, rho0


def _profile_tallbox(zeta: np.ndarray):
    T0 = (4000.0 + 8000.0 * 0.5 * (1.0 - np.tanh((zeta - 0.35) / 0.08))
          + 16000.0 * 0.5 * (1.0 + np.tanh((zeta - 0.8) / 0.05)))
    rho0 = 3e-7 * 10.0 ** (-6.0 * zeta)
    return T0, rho0


_CFG = {
    # id: grid, spacing km, nbands, table n, logT range, logP range, scales, profile, perturb
    1: dict(grid=(32, 32, 32), dkm=(48.0, 48.0, 32.0), nb=1, ntab=64,
            logT=(3.5, 4.3), logP=(2.0, 7.0), scales=[1.0], profile="phot", pert="box"),
    2: dict(grid=(96, 96, 96), dkm=(48.0, 48.0, 32.0), nb=1, ntab=64,
            logT=(3.5, 4.3), logP=(2.0, 7.0), scales=[1.0], profile="phot", pert="box"),
    3: dict(grid=(288, 288, 288), dkm=(32.0, 32.0, 16.0), nb=4, ntab=128,
            logT=(3.5, 4.3), logP=(2.0, 7.0), scales=[1.0, 10.0, 100.0, 1000.0],
            profile="phot", pert="gran"),
    4: dict(grid=(288, 288, 288), dkm=(32.0, 32.0, 16.0), nb=12, ntab=128,
            logT=(3.5, 4.3), logP=(2.0, 7.0),
            scales=[10.0 ** (5.0 * m / 11.0) for m in range(12)],
            profile="phot", pert="gran"),
    5: dict(grid=(512, 512, 192), dkm=(24.0, 24.0, 12.0), nb=4, ntab=128,
            logT=(3.5, 4.4), logP=(-1.5, 7.0), scales=[1.0, 10.0, 100.0, 1000.0],
            profile="tall", pert="gran"),
}


def config_ids() -> Sequence[int]:
    return tuple(sorted(_CFG))


def make_config(cfg: int, grid: Optional[Tuple[int, int, int]] = None,
                nbands: Optional[int] = None, npasses: int = 3,
                seed_offset: int = 0) -> RTSInputs:
    """Build BASELINE.json config `cfg` (1..5).

    `grid=(nx,ny,nz)` and `nbands` override the size (the recipe is expressed in
    the normalised height zeta = k/(nz-1) and in physical correlation lengths, so
    a reduced grid keeps the same atmosphere "scaled to the box"); used by the
    parity tests to get small cases of the multi-band / tall-box recipes.
    """
    c = _CFG[cfg]
    nx, ny, nz = grid if grid is not None else c["grid"]
    dx, dy, dz = (d * 1e5 for d in c["dkm"])
    scales = list(c["scales"])
    nb = nbands if nbands is not None else c["nb"]
    if nb != len(scales):
        # log-spaced between the recipe's smallest and largest scale
        lo, hi = np.log10(scales[0]), np.log10(scales[-1])
        scales = [10.0 ** (lo + (hi - lo) * m / max(nb - 1, 1)) for m in range(nb)]
    ntab = c["ntab"]
    rng = np.random.Generator(np.random.PCG64(2107081450 + cfg + seed_offset))

    # draw order fixed: g_T, g_rho, table noise, alpha, beta
    gT = rng.standard_normal((nz, ny, nx))
    gR = rng.standard_normal((nz, ny, nx))
    tnoise = rng.standard_normal((nb, ntab, ntab))
    alpha = rng.standard_normal(nb)
    beta = rng.standard_normal(nb)

    zeta = (np.arange(nz, dtype=np.float64) / max(nz - 1, 1)).reshape(nz, 1, 1)
    if c["profile"] == "phot":
        T0, rho0 = _profile_photosphere(zeta)
    else:
        T0, rho0 = _profile_tallbox(zeta)

    if c["pert"] == "box":
        gT = _unit_std(_box3(gT))
        gR = _unit_std(_box3(gR))
        T = T0 * (1.0 + 0.03 * gT)
        rho = rho0 * (1.0 + 0.05 * gR)
    else:
        sh, sv = 0.5e8, 0.25e8     # 0.5 Mm horizontal, 0.25 Mm vertical (cm)
        gT = _unit_std(_granulation(gT, sh / dx, sh / dy, sv / dz))
        gR = _unit_std(_granulation(gR, sh / dx, sh / dy, sv / dz))
        T = T0 * np.exp(0.10 * gT)
        rho = rho0 * np.exp(0.20 * gR)
    P = rho * K_B * T / (MU_MOL * M_H)

    logT_min, logT_max = c["logT"]
    logP_min, logP_max = c["logP"]
    xT = np.linspace(logT_min, logT_max, ntab).reshape(1, ntab, 1)
    xP = np.linspace(logP_min, logP_max, ntab).reshape(1, 1, ntab)
    lsc = np.log10(np.asarray(scales, dtype=np.float64)).reshape(nb, 1, 1)
    logkappa = 4.5 * xT + 0.7 * xP - 18.5 + lsc + 0.05 * tnoise

    if nb > 1:
        arg = alpha.reshape(nb, 1) + 2.0 * beta.reshape(nb, 1) * (xT.reshape(1, ntab) - 3.9) / 0.4
        arg = arg - arg.max(axis=0, keepdims=True)
        e = np.exp(arg)
        bandfrac = e / e.sum(axis=0, keepdims=True)
    else:
        bandfrac = np.ones((1, ntab), dtype=np.float64)

    mu, wq = carlson24()
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return RTSInputs(
        name=f"cfg{cfg}_{nx}x{ny}x{nz}_b{nb}", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz,
        nbands=nb, npasses=npasses, rho=f32(rho), T=f32(T), P=f32(P),
        nT=ntab, nP=ntab, logT_min=logT_min, logT_max=logT_max,
        logP_min=logP_min, logP_max=logP_max,
        logkappa=f32(logkappa), bandfrac=f32(bandfrac), mu=mu, wq=wq)


def make_custom(nx: int, ny: int, nz: int, dx: float, dy: float, dz: float,
                rho: np.ndarray, T: np.ndarray, P: np.ndarray,
                logkappa: np.ndarray, bandfrac: np.ndarray,
                logT_rng: Tuple[float, float], logP_rng: Tuple[float, float],
                npasses: int = 3, mu: Optional[np.ndarray] = None,
                wq: Optional[np.ndarray] = None, name: str = "custom") -> RTSInputs:
    """Wrap hand-built arrays (closed-form pins, edge cases) in the same container."""
    nb, nT, nP = logkappa.shape
    if mu is None:
        mu, wq = carlson24()
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return RTSInputs(name=name, nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, nbands=nb,
                     npasses=npasses, rho=f32(rho).reshape(nz, ny, nx),
                     T=f32(T).reshape(nz, ny, nx), P=f32(P).reshape(nz, ny, nx),
                     nT=nT, nP=nP, logT_min=logT_rng[0], logT_max=logT_rng[1],
                     logP_min=logP_rng[0], logP_max=logP_rng[1],
                     logkappa=f32(logkappa), bandfrac=f32(bandfrac).reshape(nb, nT),
                     mu=np.ascontiguousarray(mu, dtype=np.float64),
                     wq=np.ascontiguousarray(wq, dtype=np.float64))
