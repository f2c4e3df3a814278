"""fp64 CPU oracle of the RTS hot path -- TEST INFRASTRUCTURE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this package.  It shares no code with the CUDA
path (`paper_2107_08145_b200/csrc`); the product path never routes through it.

The arithmetic lives in `rts_oracle.c` (plain C, fp64, one OpenMP loop over the
independent (band, ray) sweeps); this file only compiles it with gcc and marshals
numpy arrays through ctypes.  Passages followed: see the header of rts_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rts_oracle.c")
_LIB = os.path.join(_HERE, "librts_oracle.so")
_lib = None

_D = ctypes.c_double
_I = ctypes.c_int
_PD = ctypes.POINTER(ctypes.c_double)
_PF = ctypes.POINTER(ctypes.c_float)
_PI = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile rts_oracle.c -> librts_oracle.so (gcc -O3, OpenMP, no fast-math, no -march: the .so built on the
    CPU-only box travels to the GPU box)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O3", "-fopenmp", "-fPIC", "-shared", "-std=c11",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_coefficients.restype = _I
        _lib.oracle_coefficients.argtypes = [_I] * 6 + [_D] * 4 + [_PF] * 5 + [_PD] * 2
        _lib.oracle_cells_to_nodes.restype = _I
        _lib.oracle_cells_to_nodes.argtypes = [_I] * 3 + [_PF] * 2
        _lib.oracle_nodes_to_cells.restype = _I
        _lib.oracle_nodes_to_cells.argtypes = [_I] * 3 + [_PD] * 2
        _lib.oracle_ray_geometry.restype = _I
        _lib.oracle_ray_geometry.argtypes = [_D, _D, _D, _PD, _PI, _PI, _PD, _PD]
        _lib.oracle_psi.restype = None
        _lib.oracle_psi.argtypes = [_D, _PD, _PD, _PD]
        _lib.oracle_sweep_ray.restype = _I
        _lib.oracle_sweep_ray.argtypes = [_I, _I, _I, _D, _D, _D, _PD, _I, _PD, _PD, _PD, _I, _PD]
        _lib.oracle_solve.restype = _I
        _lib.oracle_solve.argtypes = ([_I, _I, _I, _D, _D, _D, _I, _I, _I, _D, _D, _D, _D,
                                       _PF, _PF, _I, _I, _PD, _PD, _PF, _PF, _PF,
                                       _PD, _PD, _PD, _PD, _I])
        _lib.oracle_sweep_ray_tol.restype = _I
        _lib.oracle_sweep_ray_tol.argtypes = [_I, _I, _I, _D, _D, _D, _PD, _D, _I, _PD, _PD, _PD, _PD, _PD, _PD, _PD, _PD, _PI]
        _lib.oracle_solve_tol.restype = _I
        _lib.oracle_solve_tol.argtypes = ([_I, _I, _I, _D, _D, _D, _I, _I, _I, _D, _D, _D, _D, _PF, _PF,
                                           _D, _I, _I, _I, _I, _PD, _PD, _PF, _PF, _PF, _PD, _PD, _PD, _PI, _PD, _I])
        _lib.oracle_scatter_solve.restype = _I
        _lib.oracle_scatter_solve.argtypes = [_I, _I, _I, _D, _D, _D, _I, _PD, _PD, _PD, _PD, _PD, _I, _I, _PD, _PD, _PD, _PD]
        _lib.oracle_flux_heating.restype = _I
        _lib.oracle_flux_heating.argtypes = [_I, _I, _I, _D, _D, _D, _PD, _PD, _PD, _D, _PD, _PD]
        _lib.oracle_num_threads.restype = _I
        _lib.oracle_num_threads.argtypes = []
    return _lib


def _pf(a):
    return a.ctypes.data_as(_PF)


def _pd(a):
    return a.ctypes.data_as(_PD) if a is not None else None


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def coefficients(inp) -> Tuple[np.ndarray, np.ndarray]:
    """O-2: (kaprho, S), each float64 [nb][nz][ny][nx]."""
    lib = _load()
    N = inp.ncells
    kap = np.empty((inp.nbands,) + inp.shape, dtype=np.float64)
    S = np.empty_like(kap)
    rc = lib.oracle_coefficients(inp.nx, inp.ny, inp.nz, inp.nbands, inp.nT, inp.nP,
                                 inp.logT_min, inp.logT_max, inp.logP_min, inp.logP_max,
                                 _pf(inp.logkappa), _pf(inp.bandfrac),
                                 _pf(inp.rho), _pf(inp.T), _pf(inp.P), _pd(kap), _pd(S))
    if rc != 0:
        raise RuntimeError(f"oracle_coefficients failed: {rc}")
    return kap, S


def ray_geometry(dx: float, dy: float, dz: float, mu) -> Tuple[int, Tuple[int, int, int], float, Tuple[float, float, float]]:
    """O-3: (entry-face axis, signs, ds, fractions f_a)."""
    lib = _load()
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    axis = ctypes.c_int()
    sg = (ctypes.c_int * 3)()
    ds = ctypes.c_double()
    f = (ctypes.c_double * 3)()
    rc = lib.oracle_ray_geometry(dx, dy, dz, _pd(mu), ctypes.byref(axis), sg, ctypes.byref(ds), f)
    if rc != 0:
        raise ValueError("ray has mu_z == 0")
    return axis.value, tuple(sg), ds.value, tuple(f)


def psi(dtau: float) -> Tuple[float, float, float]:
    """O-6: (E, psi_u, psi_p)."""
    lib = _load()
    E, pu, pp = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    lib.oracle_psi(float(dtau), ctypes.byref(E), ctypes.byref(pu), ctypes.byref(pp))
    return E.value, pu.value, pp.value


def sweep_ray(nx, ny, nz, dx, dy, dz, mu, npasses, kaprho, S,
              inflow: Optional[np.ndarray] = None, form: int = 0) -> np.ndarray:
    """O-4..O-6 for one band and one ray; returns I^(P) float64 [nz][ny][nx]."""
    lib = _load()
    kaprho = np.ascontiguousarray(kaprho, dtype=np.float64)
    S = np.ascontiguousarray(S, dtype=np.float64)
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    if inflow is not None:
        inflow = np.ascontiguousarray(inflow, dtype=np.float64)
    I = np.empty((nz, ny, nx), dtype=np.float64)
    rc = lib.oracle_sweep_ray(nx, ny, nz, dx, dy, dz, _pd(mu), npasses,
                              _pd(kaprho), _pd(S), _pd(inflow), form, _pd(I))
    if rc != 0:
        raise RuntimeError(f"oracle_sweep_ray failed: {rc}")
    return I


def sweep_ray_tol(nx, ny, nz, dx, dy, dz, mu, tol, max_passes, kaprho, S, warm=None):
    """O-12 for one band and one ray: iterate until the seam faces change by <= tol * max|I| on them.
    warm = (faceX [nz][ny], faceY [nz][nx]) of I^(0), or None.  Returns (I, (faceX, faceY), relerr per pass, passes)."""
    lib = _load()
    kaprho = np.ascontiguousarray(kaprho, dtype=np.float64)
    S = np.ascontiguousarray(S, dtype=np.float64)
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    wx = np.ascontiguousarray(warm[0], dtype=np.float64) if warm is not None else None
    wy = np.ascontiguousarray(warm[1], dtype=np.float64) if warm is not None else None
    I = np.empty((nz, ny, nx), dtype=np.float64)
    fx = np.empty((nz, ny), dtype=np.float64); fy = np.empty((nz, nx), dtype=np.float64)
    rel = np.zeros(max_passes, dtype=np.float64)
    used = ctypes.c_int(0)
    rc = lib.oracle_sweep_ray_tol(nx, ny, nz, dx, dy, dz, _pd(mu), float(tol), int(max_passes), _pd(kaprho), _pd(S),
                                  _pd(wx), _pd(wy), _pd(I), _pd(fx), _pd(fy), _pd(rel), ctypes.byref(used))
    if rc != 0:
        raise RuntimeError(f"oracle_sweep_ray_tol failed: {rc}")
    return I, (fx, fy), rel[:used.value].copy(), used.value


def solve_tol(inp, tol: float, max_passes: int, mode: int = 1, faces: Optional[np.ndarray] = None, nthreads: int = 0):
    """O-12, all bands and rays.  mode 0: every (band, ray) stops on its own error; mode 1: one pass count for all.
    faces: None (cold start) or the array returned by an earlier call (warm start).
    Returns (Q, Itop, faces [nb*nrays][nz*ny + nz*nx], passes_used [nb*nrays], relerr per pass (mode 1))."""
    lib = _load()
    Q = np.empty(inp.shape, dtype=np.float64)
    Itop = np.empty((inp.nbands, inp.n_up, inp.ny, inp.nx), dtype=np.float64)
    mu = np.ascontiguousarray(inp.mu, dtype=np.float64)
    wq = np.ascontiguousarray(inp.wq, dtype=np.float64)
    ntask = inp.nbands * inp.nrays
    nf = inp.nz * inp.ny + inp.nz * inp.nx
    warm = faces is not None
    fc = np.ascontiguousarray(faces, dtype=np.float64).copy() if warm else np.empty((ntask, nf), dtype=np.float64)
    assert fc.shape == (ntask, nf)
    used = np.zeros(ntask, dtype=np.int32)
    rel = np.zeros(max_passes, dtype=np.float64)
    rc = lib.oracle_solve_tol(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, inp.nbands, inp.nT, inp.nP,
                              inp.logT_min, inp.logT_max, inp.logP_min, inp.logP_max,
                              _pf(inp.logkappa), _pf(inp.bandfrac),
                              float(tol), int(max_passes), int(mode), int(warm),
                              inp.nrays, _pd(mu), _pd(wq), _pf(inp.rho), _pf(inp.T), _pf(inp.P),
                              _pd(Q), _pd(Itop), _pd(fc), used.ctypes.data_as(_PI), _pd(rel), nthreads)
    if rc != 0:
        raise RuntimeError(f"oracle_solve_tol failed: {rc}")
    return Q, Itop, fc, used, rel[:int(used.max())].copy()


def scatter_solve(nx, ny, nz, dx, dy, dz, mu, wq, kaprho, B, eps, niter: int, gs: bool = True, want_I: bool = False):
    """O-13, one band: S = (1 - eps) J + eps B iterated niter times with the source update along the ray (gs) or
    as a Jacobi / Lambda iteration.  Returns (S, J [nz][ny][nx], change [niter]) (+ I [nrays][nz][ny][nx])."""
    lib = _load()
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    wq = np.ascontiguousarray(wq, dtype=np.float64)
    kaprho = np.ascontiguousarray(kaprho, dtype=np.float64)
    B = np.ascontiguousarray(B, dtype=np.float64)
    eps = np.ascontiguousarray(np.broadcast_to(eps, (nz, ny, nx)), dtype=np.float64)
    assert kaprho.shape == (nz, ny, nx) and B.shape == (nz, ny, nx)
    S = np.empty((nz, ny, nx), dtype=np.float64)
    J = np.empty((nz, ny, nx), dtype=np.float64)
    Iall = np.empty((len(wq), nz, ny, nx), dtype=np.float64) if want_I else None
    change = np.zeros(max(niter, 1), dtype=np.float64)
    rc = lib.oracle_scatter_solve(nx, ny, nz, dx, dy, dz, len(wq), _pd(mu), _pd(wq), _pd(kaprho), _pd(B), _pd(eps),
                                  int(niter), 1 if gs else 0, _pd(S), _pd(J), _pd(Iall), _pd(change))
    if rc != 0:
        raise RuntimeError(f"oracle_scatter_solve failed: {rc}")
    out = (S, J, change[:niter].copy())
    return out + (Iall,) if want_I else out


def solve(inp, nthreads: int = 0, want_J: bool = False, want_F: bool = False):
    """O-7: returns (Q [nz][ny][nx], Itop [nb][n_up][ny][nx]) (+ J [nb][nz][ny][nx]) (+ O-10 F [3][nz][ny][nx])."""
    lib = _load()
    Q = np.empty(inp.shape, dtype=np.float64)
    Itop = np.empty((inp.nbands, inp.n_up, inp.ny, inp.nx), dtype=np.float64)
    J = np.empty((inp.nbands,) + inp.shape, dtype=np.float64) if want_J else None
    F = np.empty((3,) + inp.shape, dtype=np.float64) if want_F else None
    mu = np.ascontiguousarray(inp.mu, dtype=np.float64)
    wq = np.ascontiguousarray(inp.wq, dtype=np.float64)
    rc = lib.oracle_solve(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz,
                          inp.nbands, inp.nT, inp.nP,
                          inp.logT_min, inp.logT_max, inp.logP_min, inp.logP_max,
                          _pf(inp.logkappa), _pf(inp.bandfrac),
                          inp.npasses, inp.nrays, _pd(mu), _pd(wq),
                          _pf(inp.rho), _pf(inp.T), _pf(inp.P),
                          _pd(Q), _pd(Itop), _pd(J), _pd(F), nthreads)
    if rc != 0:
        raise RuntimeError(f"oracle_solve failed: {rc}")
    out = (Q, Itop)
    if want_J:
        out += (J,)
    if want_F:
        out += (F,)
    return out


def flux_heating(inp, F, QJ=None, kaprho0=None, tau0: float = 0.1, want_blend: bool = True):
    """O-11: (Qdiv, Qblend) from the flux F [3][nz][ny][nx]; Qblend needs QJ and the band-0 kaprho."""
    lib = _load()
    F = np.ascontiguousarray(F, dtype=np.float64)
    Qdiv = np.empty(inp.shape, dtype=np.float64)
    Qb = np.empty(inp.shape, dtype=np.float64) if want_blend else None
    if want_blend:
        QJ = np.ascontiguousarray(QJ, dtype=np.float64)
        kaprho0 = np.ascontiguousarray(kaprho0, dtype=np.float64)
    rc = lib.oracle_flux_heating(inp.nx, inp.ny, inp.nz, inp.dx, inp.dy, inp.dz, _pd(F),
                                 _pd(QJ) if want_blend else None, _pd(kaprho0) if want_blend else None,
                                 float(tau0), _pd(Qdiv), _pd(Qb))
    if rc != 0:
        raise RuntimeError(f"oracle_flux_heating failed: {rc}")
    return Qdiv, Qb


def cells_to_nodes(cell: np.ndarray) -> np.ndarray:
    """O-9: fp32 cell-centred field [ncz][ncy][ncx] -> fp32 corner-node field [ncz+1][ncy][ncx]."""
    lib = _load()
    cell = np.ascontiguousarray(cell, dtype=np.float32)
    ncz, ncy, ncx = cell.shape
    node = np.empty((ncz + 1, ncy, ncx), dtype=np.float32)
    rc = lib.oracle_cells_to_nodes(ncx, ncy, ncz, _pf(cell), _pf(node))
    assert rc == 0, rc
    return node


def nodes_to_cells(qn: np.ndarray) -> np.ndarray:
    """O-9: fp64 node field [nz][ny][nx] -> fp64 cell field [nz-1][ny][nx] (mean of the 8 corners)."""
    lib = _load()
    qn = np.ascontiguousarray(qn, dtype=np.float64)
    nz, ny, nx = qn.shape
    qc = np.empty((nz - 1, ny, nx), dtype=np.float64)
    rc = lib.oracle_nodes_to_cells(nx, ny, nz, _pd(qn), _pd(qc))
    assert rc == 0, rc
    return qc


def solve_cells(inp_cells, nthreads: int = 0):
    """Staggered solve: `inp_cells` holds cell-centred rho, T, P [ncz][ncy][ncx]; the RT grid has
    nz = ncz + 1 levels.  Returns (Q on cells fp64, I_top fp64, node-grid inputs)."""
    import copy
    node = copy.copy(inp_cells)
    node.rho = cells_to_nodes(inp_cells.rho)
    node.T = cells_to_nodes(inp_cells.T)
    node.P = cells_to_nodes(inp_cells.P)
    node.nz = inp_cells.nz + 1
    Qn, Itop = solve(node, nthreads=nthreads)
    return nodes_to_cells(Qn), Itop, node
