"""Thin Python binding of the C-ABI in include/rts.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of librts.so.  PyTorch is used for
device memory and the current stream only.  There is no fallback: if librts.so is
missing (and cannot be built) or no CUDA device is present, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

RTS_OK = 0
_ERR = {-1: "RTS_EINVAL", -2: "RTS_ESTATE", -3: "RTS_ECUDA", -4: "RTS_ENOMEM", -5: "RTS_ETIMEOUT"}

EXPORTS = [
    "rts_create", "rts_destroy", "rts_set_tables", "rts_set_passes", "rts_set_rays", "rts_get_rays",
    "rts_num_up_rays", "rts_set_tiling", "rts_set_exchange_interval", "rts_set_ctas_per_sm", "rts_set_ring_depth", "rts_workspace_bytes",
    "rts_set_workspace", "rts_solve", "rts_solve_host", "rts_coefficients", "rts_sync_check",
    "rts_plan_info", "rts_last_error", "rts_enable_timing", "rts_last_timing",
    "rts_cells_to_nodes", "rts_nodes_to_cells", "rts_solve_cells", "rts_set_thick_skip", "rts_thick_levels",
    "rts_enable_flux", "rts_set_flux_blend", "rts_solve_flux", "rts_set_shard", "rts_shard_info",
    "rts_set_tolerance", "rts_set_warm_start", "rts_passes_used",
    "rts_scatter_workspace_bytes", "rts_scatter_solve", "rts_scatter_solve_static",
]


def load_library(build_if_missing: bool = True) -> ctypes.CDLL:
    """dlopen librts.so (building it first if it is missing or stale) and declare prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_missing and not _build.up_to_date():
        _build.build()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2107_08145_b200.build`")
    lib = ctypes.CDLL(path)
    c_void_p, c_int, c_double, c_size_t = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    PF, PD, PI = ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    lib.rts_create.restype = c_int
    lib.rts_create.argtypes = [ctypes.POINTER(c_void_p), c_int, c_int, c_int, c_double, c_double, c_double, c_int]
    lib.rts_destroy.restype = c_int
    lib.rts_destroy.argtypes = [c_void_p]
    lib.rts_set_tables.restype = c_int
    lib.rts_set_tables.argtypes = [c_void_p, c_int, c_int, c_double, c_double, c_double, c_double, PF, PF]
    lib.rts_set_passes.restype = c_int
    lib.rts_set_passes.argtypes = [c_void_p, c_int]
    lib.rts_set_rays.restype = c_int
    lib.rts_set_rays.argtypes = [c_void_p, c_int, PD, PD]
    lib.rts_get_rays.restype = c_int
    lib.rts_get_rays.argtypes = [c_void_p, PI, PD, PD]
    lib.rts_num_up_rays.restype = c_int
    lib.rts_num_up_rays.argtypes = [c_void_p]
    lib.rts_set_tiling.restype = c_int
    lib.rts_set_tiling.argtypes = [c_void_p, c_int, c_int, c_int]
    lib.rts_set_exchange_interval.restype = c_int
    lib.rts_set_exchange_interval.argtypes = [c_void_p, c_int]
    lib.rts_set_ctas_per_sm.restype = c_int
    lib.rts_set_ctas_per_sm.argtypes = [c_void_p, c_int]
    lib.rts_set_ring_depth.restype = c_int
    lib.rts_set_ring_depth.argtypes = [c_void_p, c_int]
    lib.rts_workspace_bytes.restype = c_size_t
    lib.rts_workspace_bytes.argtypes = [c_void_p]
    lib.rts_set_workspace.restype = c_int
    lib.rts_set_workspace.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.rts_solve.restype = c_int
    lib.rts_solve.argtypes = [c_void_p] + [c_void_p] * 5 + [c_void_p]
    lib.rts_solve_host.restype = c_int
    lib.rts_solve_host.argtypes = [c_void_p] + [c_void_p] * 5 + [c_void_p]
    lib.rts_coefficients.restype = c_int
    lib.rts_coefficients.argtypes = [c_void_p] + [c_void_p] * 5 + [c_void_p]
    lib.rts_sync_check.restype = c_int
    lib.rts_sync_check.argtypes = [c_void_p, c_void_p]
    lib.rts_plan_info.restype = c_int
    lib.rts_plan_info.argtypes = [c_void_p, PI, c_int]
    lib.rts_enable_timing.restype = c_int
    lib.rts_enable_timing.argtypes = [c_void_p, c_int]
    lib.rts_last_timing.restype = c_int
    lib.rts_last_timing.argtypes = [c_void_p, PF]
    lib.rts_cells_to_nodes.restype = c_int
    lib.rts_cells_to_nodes.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.rts_nodes_to_cells.restype = c_int
    lib.rts_nodes_to_cells.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.rts_solve_cells.restype = c_int
    lib.rts_solve_cells.argtypes = [c_void_p] + [c_void_p] * 5 + [c_void_p]
    lib.rts_set_thick_skip.restype = c_int
    lib.rts_set_thick_skip.argtypes = [c_void_p, c_int]
    lib.rts_thick_levels.restype = c_int
    lib.rts_thick_levels.argtypes = [c_void_p, PI, c_void_p]
    lib.rts_enable_flux.restype = c_int
    lib.rts_enable_flux.argtypes = [c_void_p, c_int]
    lib.rts_set_flux_blend.restype = c_int
    lib.rts_set_flux_blend.argtypes = [c_void_p, c_double]
    lib.rts_solve_flux.restype = c_int
    lib.rts_solve_flux.argtypes = [c_void_p] + [c_void_p] * 8 + [c_void_p]
    lib.rts_scatter_workspace_bytes.restype = ctypes.c_size_t
    lib.rts_scatter_workspace_bytes.argtypes = [c_void_p, c_int, c_int]
    lib.rts_scatter_solve.restype = c_int
    lib.rts_scatter_solve.argtypes = [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p, ctypes.c_size_t,
                                      c_void_p, c_void_p, ctypes.POINTER(ctypes.c_double), c_void_p]
    lib.rts_scatter_solve_static.restype = c_int
    lib.rts_scatter_solve_static.argtypes = [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int,
                                             c_void_p, c_void_p, ctypes.POINTER(ctypes.c_double), c_void_p]
    lib.rts_set_tolerance.restype = c_int
    lib.rts_set_tolerance.argtypes = [c_void_p, c_double, c_int]
    lib.rts_set_warm_start.restype = c_int
    lib.rts_set_warm_start.argtypes = [c_void_p, c_int]
    lib.rts_passes_used.restype = c_int
    lib.rts_passes_used.argtypes = [c_void_p, PI, PF]
    lib.rts_set_shard.restype = c_int
    lib.rts_set_shard.argtypes = [c_void_p, c_int, c_int]
    lib.rts_shard_info.restype = c_int
    lib.rts_shard_info.argtypes = [c_void_p, PI, PI]
    lib.rts_last_error.restype = ctypes.c_char_p
    lib.rts_last_error.argtypes = [c_void_p]
    _lib = lib
    return lib


class RTSError(RuntimeError):
    pass


class RTS:
    """Handle around rts_ctx.  Names follow include/rts.h."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, nbands: int):
        import torch
        if not torch.cuda.is_available():
            raise RTSError("no CUDA device: the RTS path has no CPU fallback")
        self._torch = torch
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.nx, self.ny, self.nz, self.nbands = nx, ny, nz, nbands
        torch.cuda.init()
        torch.zeros(1, device="cuda")          # make sure the primary context exists and is current
        rc = self._lib.rts_create(ctypes.byref(self._ctx), nx, ny, nz, dx, dy, dz, nbands)
        if rc != RTS_OK:
            msg = self._lib.rts_last_error(None)
            raise RTSError(f"rts_create failed: {_ERR.get(rc, rc)}: {msg.decode() if msg else ''}")
        self._ws = None

    # -- helpers
    def _check(self, rc: int, what: str):
        if rc != RTS_OK:
            msg = self._lib.rts_last_error(self._ctx)
            raise RTSError(f"{what}: {_ERR.get(rc, rc)}: {msg.decode() if msg else ''}")

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.rts_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- configuration
    def set_tables(self, nT, nP, logT_min, logT_max, logP_min, logP_max, logkappa, bandfrac):
        lk = np.ascontiguousarray(logkappa, dtype=np.float32)
        bf = np.ascontiguousarray(bandfrac, dtype=np.float32)
        assert lk.shape == (self.nbands, nT, nP) and bf.shape == (self.nbands, nT)
        PF = ctypes.POINTER(ctypes.c_float)
        self._check(self._lib.rts_set_tables(self._ctx, nT, nP, logT_min, logT_max, logP_min, logP_max,
                                             lk.ctypes.data_as(PF), bf.ctypes.data_as(PF)), "rts_set_tables")

    def set_passes(self, n: int):
        self._check(self._lib.rts_set_passes(self._ctx, n), "rts_set_passes")

    def set_rays(self, mu, w):
        mu = np.ascontiguousarray(mu, dtype=np.float64)
        w = np.ascontiguousarray(w, dtype=np.float64)
        PD = ctypes.POINTER(ctypes.c_double)
        self._check(self._lib.rts_set_rays(self._ctx, mu.shape[0], mu.ctypes.data_as(PD), w.ctypes.data_as(PD)),
                    "rts_set_rays")

    def get_rays(self) -> Tuple[np.ndarray, np.ndarray]:
        n = ctypes.c_int()
        self._check(self._lib.rts_get_rays(self._ctx, ctypes.byref(n), None, None), "rts_get_rays")
        mu = np.empty((n.value, 3), dtype=np.float64)
        w = np.empty(n.value, dtype=np.float64)
        PD = ctypes.POINTER(ctypes.c_double)
        self._check(self._lib.rts_get_rays(self._ctx, ctypes.byref(n), mu.ctypes.data_as(PD), w.ctypes.data_as(PD)),
                    "rts_get_rays")
        return mu, w

    def num_up_rays(self) -> int:
        return int(self._lib.rts_num_up_rays(self._ctx))

    def set_tiling(self, march: int, tile_u: int, tile_v: int):
        self._check(self._lib.rts_set_tiling(self._ctx, march, tile_u, tile_v), "rts_set_tiling")

    def set_exchange_interval(self, k: int):
        self._check(self._lib.rts_set_exchange_interval(self._ctx, k), "rts_set_exchange_interval")

    def set_ctas_per_sm(self, n: int):
        self._check(self._lib.rts_set_ctas_per_sm(self._ctx, n), "rts_set_ctas_per_sm")

    def set_ring_depth(self, n: int):
        self._check(self._lib.rts_set_ring_depth(self._ctx, n), "rts_set_ring_depth")

    def workspace_bytes(self) -> int:
        n = int(self._lib.rts_workspace_bytes(self._ctx))
        if n == 0:
            msg = self._lib.rts_last_error(self._ctx)
            raise RTSError(f"rts_workspace_bytes: {msg.decode() if msg else 'failed'}")
        return n

    def allocate_workspace(self):
        """torch-allocated device workspace handed to rts_set_workspace (caller-owned memory)."""
        n = self.workspace_bytes()
        self._ws = self._torch.empty(n + 256, dtype=self._torch.uint8, device="cuda")
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        self._check(self._lib.rts_set_workspace(self._ctx, ctypes.c_void_p(ptr), n), "rts_set_workspace")

    def plan_info(self) -> dict:
        arr = (ctypes.c_int * 16)()
        self._check(self._lib.rts_plan_info(self._ctx, arr, 16), "rts_plan_info")
        keys = ["launches", "tasks", "ctas_per_sm", "units", "threads", "smem_bytes",
                "grid", "exchange_interval", "tile_v_x", "tile_v_y", "tile_v_z",
                "tile_u_x", "tile_u_y", "tile_u_z", "z_march_rays", "units_all"]
        return dict(zip(keys, [int(v) for v in arr]))

    # -- the hot path
    def _stream(self):
        return ctypes.c_void_p(self._torch.cuda.current_stream().cuda_stream)

    def solve(self, rho, T, P, Q=None, Itop=None, want_itop: bool = True):
        """rho, T, P: float32 CUDA tensors [nz][ny][nx].  Returns (Q, Itop) CUDA tensors."""
        torch = self._torch
        for t in (rho, T, P):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            assert tuple(t.shape) == (self.nz, self.ny, self.nx)
        if self._ws is None:
            self.allocate_workspace()
        if Q is None:
            Q = torch.empty((self.nz, self.ny, self.nx), dtype=torch.float32, device="cuda")
        if want_itop and Itop is None:
            Itop = torch.empty((self.nbands, self.num_up_rays(), self.ny, self.nx), dtype=torch.float32, device="cuda")
        ip = ctypes.c_void_p(Itop.data_ptr()) if (want_itop and Itop is not None) else None
        self._check(self._lib.rts_solve(self._ctx, ctypes.c_void_p(rho.data_ptr()), ctypes.c_void_p(T.data_ptr()),
                                        ctypes.c_void_p(P.data_ptr()), ctypes.c_void_p(Q.data_ptr()), ip,
                                        self._stream()), "rts_solve")
        return Q, (Itop if want_itop else None)

    def enable_flux(self, on: bool = True):
        """Must precede allocate_workspace (three more partial fields per sweep unit)."""
        self._check(self._lib.rts_enable_flux(self._ctx, 1 if on else 0), "rts_enable_flux")
        self._ws = None

    def set_flux_blend(self, tau0: float):
        self._check(self._lib.rts_set_flux_blend(self._ctx, float(tau0)), "rts_set_flux_blend")

    def solve_flux(self, rho, T, P, want_div: bool = True, want_blend: bool = True):
        """rts_solve_flux: returns (Q, Itop, F[3][nz][ny][nx], Qdiv or None, Qblend or None) as CUDA tensors."""
        torch = self._torch
        if self._ws is None:
            self.allocate_workspace()
        shp = (self.nz, self.ny, self.nx)
        Q = torch.empty(shp, dtype=torch.float32, device="cuda")
        Itop = torch.empty((self.nbands, self.num_up_rays(), self.ny, self.nx), dtype=torch.float32, device="cuda")
        F = torch.empty((3,) + shp, dtype=torch.float32, device="cuda")
        Qd = torch.empty(shp, dtype=torch.float32, device="cuda") if want_div else None
        Qb = torch.empty(shp, dtype=torch.float32, device="cuda") if want_blend else None
        p = lambda t: ctypes.c_void_p(t.data_ptr()) if t is not None else None
        self._check(self._lib.rts_solve_flux(self._ctx, p(rho), p(T), p(P), p(Q), p(Itop), p(F), p(Qd), p(Qb), self._stream()),
                    "rts_solve_flux")
        return Q, Itop, F, Qd, Qb

    def solve_host(self, rho, T, P, Q, Itop=None):
        """Host numpy / pinned torch buffers in and out (copies inside the call, synchronous)."""
        if self._ws is None:
            self.allocate_workspace()

        def ptr(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float32 and a.flags.c_contiguous
                return ctypes.c_void_p(a.ctypes.data)
            assert (not a.is_cuda) and a.dtype == self._torch.float32 and a.is_contiguous()
            return ctypes.c_void_p(a.data_ptr())
        self._check(self._lib.rts_solve_host(self._ctx, ptr(rho), ptr(T), ptr(P), ptr(Q), ptr(Itop), self._stream()),
                    "rts_solve_host")
        return Q, Itop

    def coefficients(self, rho, T, P):
        """Stage A alone: (kaprho, S) float32 CUDA tensors [nb][nz][ny][nx]."""
        torch = self._torch
        if self._ws is None:
            self.allocate_workspace()
        k = torch.empty((self.nbands, self.nz, self.ny, self.nx), dtype=torch.float32, device="cuda")
        s = torch.empty_like(k)
        self._check(self._lib.rts_coefficients(self._ctx, ctypes.c_void_p(rho.data_ptr()), ctypes.c_void_p(T.data_ptr()),
                                               ctypes.c_void_p(P.data_ptr()), ctypes.c_void_p(k.data_ptr()),
                                               ctypes.c_void_p(s.data_ptr()), self._stream()), "rts_coefficients")
        return k, s

    # ---- grid staggering (cells of the MHD grid <-> corner nodes of the RT grid)
    def _cell_check(self, t, nz):
        torch = self._torch
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == (nz, self.ny, self.nx)
        return ctypes.c_void_p(t.data_ptr())

    def cells_to_nodes(self, cell, node=None):
        """float32 CUDA [nz-1][ny][nx] -> [nz][ny][nx]."""
        if node is None:
            node = self._torch.empty((self.nz, self.ny, self.nx), dtype=self._torch.float32, device="cuda")
        self._check(self._lib.rts_cells_to_nodes(self._ctx, self._cell_check(cell, self.nz - 1), self._cell_check(node, self.nz),
                                                 self._stream()), "rts_cells_to_nodes")
        return node

    def nodes_to_cells(self, qn, qc=None):
        """float32 CUDA [nz][ny][nx] -> [nz-1][ny][nx]."""
        if qc is None:
            qc = self._torch.empty((self.nz - 1, self.ny, self.nx), dtype=self._torch.float32, device="cuda")
        self._check(self._lib.rts_nodes_to_cells(self._ctx, self._cell_check(qn, self.nz), self._cell_check(qc, self.nz - 1),
                                                 self._stream()), "rts_nodes_to_cells")
        return qc

    def solve_cells(self, rho_c, T_c, P_c, Qc=None, Itop=None, want_itop: bool = True):
        """Cell-centred rho, T, P (float32 CUDA [nz-1][ny][nx]) -> (Q_rad on the cells, I_top)."""
        torch = self._torch
        if self._ws is None:
            self.allocate_workspace()
        if Qc is None:
            Qc = torch.empty((self.nz - 1, self.ny, self.nx), dtype=torch.float32, device="cuda")
        if want_itop and Itop is None:
            Itop = torch.empty((self.nbands, self.num_up_rays(), self.ny, self.nx), dtype=torch.float32, device="cuda")
        ip = ctypes.c_void_p(Itop.data_ptr()) if (want_itop and Itop is not None) else None
        ncz = self.nz - 1
        self._check(self._lib.rts_solve_cells(self._ctx, self._cell_check(rho_c, ncz), self._cell_check(T_c, ncz),
                                              self._cell_check(P_c, ncz), self._cell_check(Qc, ncz), ip, self._stream()),
                    "rts_solve_cells")
        return Qc, (Itop if want_itop else None)

    def set_tolerance(self, tol: float, max_passes: int):
        """Error-controlled iteration (NEXT #3): sweep until the seam faces of every (band, ray) change by at most
        tol * max|I| on them, at most max_passes passes (0: back to the fixed pass count).  Call before
        allocate_workspace."""
        self._check(self._lib.rts_set_tolerance(self._ctx, float(tol), int(max_passes)), "rts_set_tolerance")

    def scatter_solve(self, kaprho, B, eps, niter: int, gauss_seidel: bool = True):
        """NEXT #4: S = (1 - eps) J + eps B with the source update along the ray (or as a Jacobi iteration), for one band
        (CUDA float32 [nz][ny][nx]) or several independent ones ([nb][nz][ny][nx]).  Returns (S, J CUDA float64 of the
        same shape, change per iteration: a list of floats for one band, of per-band lists for several)."""
        torch = self._torch
        shp = (self.nz, self.ny, self.nx)
        one = (kaprho.dim() == 3)
        nb = 1 if one else int(kaprho.shape[0])
        full = shp if one else (nb,) + shp
        for t in (kaprho, B, eps):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == full
        nbytes = int(self._lib.rts_scatter_workspace_bytes(self._ctx, nb, int(niter)))
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        base = (ws.data_ptr() + 255) & ~255
        S = torch.empty(full, dtype=torch.float64, device="cuda")
        J = torch.empty(full, dtype=torch.float64, device="cuda")
        change = (ctypes.c_double * max(int(niter) * nb, 1))()
        self._check(self._lib.rts_scatter_solve(self._ctx, nb, ctypes.c_void_p(kaprho.data_ptr()), ctypes.c_void_p(B.data_ptr()),
                                                ctypes.c_void_p(eps.data_ptr()), int(niter), 1 if gauss_seidel else 0,
                                                ctypes.c_void_p(base), nbytes, ctypes.c_void_p(S.data_ptr()),
                                                ctypes.c_void_p(J.data_ptr()), change, self._stream()), "rts_scatter_solve")
        if one:
            return S, J, [float(change[i]) for i in range(int(niter))]
        return S, J, [[float(change[i * nb + b]) for b in range(nb)] for i in range(int(niter))]

    def scatter_solve_static(self, kaprho, B, eps, niter: int, gauss_seidel: bool = True, S=None, J=None):
        """scatter_solve with the scratch in the library's static device array: the C call allocates nothing (pass S and
        J, CUDA float64 of the inputs' shape, to keep this wrapper from allocating them).  Small problems only
        (rts.h: RTS_SCATTER_STATIC_BYTES); calls that overlap on the GPU race."""
        torch = self._torch
        shp = (self.nz, self.ny, self.nx)
        one = (kaprho.dim() == 3)
        nb = 1 if one else int(kaprho.shape[0])
        full = shp if one else (nb,) + shp
        for t in (kaprho, B, eps):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == full
        if S is None:
            S = torch.empty(full, dtype=torch.float64, device="cuda")
        if J is None:
            J = torch.empty(full, dtype=torch.float64, device="cuda")
        for t in (S, J):
            assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == full
        change = (ctypes.c_double * max(int(niter) * nb, 1))()
        self._check(self._lib.rts_scatter_solve_static(self._ctx, nb, ctypes.c_void_p(kaprho.data_ptr()), ctypes.c_void_p(B.data_ptr()),
                                                       ctypes.c_void_p(eps.data_ptr()), int(niter), 1 if gauss_seidel else 0,
                                                       ctypes.c_void_p(S.data_ptr()), ctypes.c_void_p(J.data_ptr()), change,
                                                       self._stream()), "rts_scatter_solve_static")
        if one:
            return S, J, [float(change[i]) for i in range(int(niter))]
        return S, J, [[float(change[i * nb + b]) for b in range(nb)] for i in range(int(niter))]

    def set_warm_start(self, on: bool = True):
        self._check(self._lib.rts_set_warm_start(self._ctx, 1 if on else 0), "rts_set_warm_start")

    def passes_used(self) -> Tuple[int, float]:
        n, e = ctypes.c_int(0), ctypes.c_float(0.0)
        self._check(self._lib.rts_passes_used(self._ctx, ctypes.byref(n), ctypes.byref(e)), "rts_passes_used")
        return n.value, e.value

    def set_shard(self, rank: int, nranks: int):
        """Band x octant sharding: this context sweeps the units u with u % nranks == rank; solve() then returns
        partial Q and I_top that a sum all-reduce over the ranks completes (multi.allreduce_sum)."""
        self._check(self._lib.rts_set_shard(self._ctx, int(rank), int(nranks)), "rts_set_shard")

    def shard_info(self) -> Tuple[int, int]:
        a, b = ctypes.c_int(0), ctypes.c_int(0)
        self._check(self._lib.rts_shard_info(self._ctx, ctypes.byref(a), ctypes.byref(b)), "rts_shard_info")
        return a.value, b.value

    def set_thick_skip(self, on: bool):
        self._check(self._lib.rts_set_thick_skip(self._ctx, 1 if on else 0), "rts_set_thick_skip")

    def thick_levels(self):
        """Level pairs from the bottom found optically thick in the last solve, per band."""
        arr = (ctypes.c_int * self.nbands)()
        self._check(self._lib.rts_thick_levels(self._ctx, arr, self._stream()), "rts_thick_levels")
        return [int(v) for v in arr]

    def enable_timing(self, on: bool = True):
        self._check(self._lib.rts_enable_timing(self._ctx, 1 if on else 0), "rts_enable_timing")

    def last_timing(self) -> dict:
        arr = (ctypes.c_float * 4)()
        self._check(self._lib.rts_last_timing(self._ctx, arr), "rts_last_timing")
        return {"stage_a_ms": arr[0], "sweep_ms": arr[1], "finalize_ms": arr[2], "solve_ms": arr[3]}

    def sync_check(self):
        self._check(self._lib.rts_sync_check(self._ctx, self._stream()), "rts_sync_check")


def from_inputs(inp, tiling: Optional[dict] = None, ctas_per_sm: int = 0, exchange_interval: int = 0,
                cells: bool = False, ring_depth: int = 0, flux: bool = False, shard: Optional[Tuple[int, int]] = None,
                tolerance: Optional[Tuple[float, int]] = None) -> "RTS":
    """Create and configure a solver for an `inputs.RTSInputs` problem.  cells=True: the fields of
    `inp` are cell-centred (solve_cells); the RT node grid then has one level more."""
    r = RTS(inp.nx, inp.ny, inp.nz + (1 if cells else 0), inp.dx, inp.dy, inp.dz, inp.nbands)
    r.set_tables(inp.nT, inp.nP, inp.logT_min, inp.logT_max, inp.logP_min, inp.logP_max, inp.logkappa, inp.bandfrac)
    r.set_passes(inp.npasses)
    r.set_rays(inp.mu, inp.wq)
    if tiling:
        for march, (tu, tv) in tiling.items():
            r.set_tiling(march, tu, tv)
    if ctas_per_sm:
        r.set_ctas_per_sm(ctas_per_sm)
    if exchange_interval:
        r.set_exchange_interval(exchange_interval)
    if ring_depth:
        r.set_ring_depth(ring_depth)
    if flux:
        r.enable_flux(True)
    if shard:
        r.set_shard(*shard)
    if tolerance:
        r.set_tolerance(*tolerance)
    r.allocate_workspace()
    return r
