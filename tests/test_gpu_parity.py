"""Parity of the CUDA path (through the C-ABI) against the fp64 oracle -- needs a B200.

Tolerances are BASELINE.json's: max|dQ_rad| <= 1e-4 * max|Q_rad| over all nodes and relative
1e-5 on I_top; stage A alone: relative 1e-6 (one fp32 rounding of an fp64
evaluation is 6e-8; the margin covers exp10/log10 differences between libm and CUDA fp64).
Every case runs the same seeded inputs through both sides and compares element by element.
"""
import ctypes

import numpy as np
import pytest

from paper_2107_08145_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_Q = 1e-4
TOL_I = 1e-5
TOL_COEF = 1e-6


def _gpu():
    import torch
    from paper_2107_08145_b200 import rts
    return torch, rts


def _solve_gpu(inp, tiling=None, ctas_per_sm=0, want_itop=True):
    torch, rts = _gpu()
    s = rts.from_inputs(inp, tiling=tiling, ctas_per_sm=ctas_per_sm)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    # outputs are fully overwritten: start from garbage
    Q = torch.full(inp.shape, 1e30, dtype=torch.float32, device="cuda")
    I = torch.full((inp.nbands, inp.n_up, inp.ny, inp.nx), -1e30, dtype=torch.float32, device="cuda") if want_itop else None
    s.solve(rho, T, P, Q, I, want_itop=want_itop)
    s.sync_check()
    # inputs are never modified
    assert np.array_equal(rho.cpu().numpy(), inp.rho) and np.array_equal(T.cpu().numpy(), inp.T)
    plan = s.plan_info()
    s.close()
    return Q.cpu().numpy().astype(np.float64), (I.cpu().numpy().astype(np.float64) if want_itop else None), plan


def _errors(Q, I, Qo, Io):
    dq = np.abs(Q - Qo)
    eq = dq.max() / np.abs(Qo).max()
    where_q = np.unravel_index(dq.argmax(), dq.shape)
    if I is None or I.size == 0:
        return eq, 0.0, where_q, None
    di = np.abs(I - Io) / np.abs(Io)
    return eq, di.max(), where_q, np.unravel_index(di.argmax(), di.shape)


def _check(inp, **kw):
    import oracle
    Qo, Io = oracle.solve(inp)
    Q, I, plan = _solve_gpu(inp, **kw)
    eq, ei, wq, wi = _errors(Q, I, Qo, Io)
    msg = f"{inp.name}: dQ/maxQ = {eq:.3e} at (k,j,i)={wq}; rel dItop = {ei:.3e} at (b,r,j,i)={wi}; plan={plan}"
    print(msg)
    assert np.isfinite(Q).all() and np.isfinite(I).all(), msg
    assert eq <= TOL_Q, msg
    assert ei <= TOL_I, msg
    return eq, ei, plan


# ------------------------------------------------------------------ stage A alone
@pytest.mark.parametrize("cfg,grid", [(1, None), (3, (40, 36, 33)), (4, (20, 24, 17)), (5, (33, 47, 29))])
def test_stage_a_coefficients(cfg, grid):
    import oracle
    torch, rts = _gpu()
    inp = inputs.make_config(cfg, grid=grid)
    ko, so = oracle.coefficients(inp)
    s = rts.from_inputs(inp)
    k, S = s.coefficients(*(torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P)))
    s.sync_check()
    k = k.cpu().numpy().astype(np.float64)
    S = S.cpu().numpy().astype(np.float64)
    s.close()
    assert (np.abs(k - ko) / ko).max() <= TOL_COEF
    assert (np.abs(S - so) / so).max() <= TOL_COEF


def test_stage_a_clamps_outside_table():
    """T, P beyond the table range take the edge values (reading R8)."""
    import oracle
    torch, rts = _gpu()
    inp = inputs.make_config(1, grid=(8, 6, 5))
    inp.T[0] *= 10.0
    inp.P[1] *= 1e-6
    inp.P[2] *= 1e6
    inp.T[3] *= 0.1
    ko, so = oracle.coefficients(inp)
    s = rts.from_inputs(inp)
    k, S = s.coefficients(*(torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P)))
    k = k.cpu().numpy().astype(np.float64)
    S = S.cpu().numpy().astype(np.float64)
    s.close()
    assert (np.abs(k - ko) / ko).max() <= TOL_COEF
    assert (np.abs(S - so) / so).max() <= TOL_COEF


# ------------------------------------------------------------------ whole path, BASELINE configs
def test_config1_gray_32():
    _check(inputs.make_config(1))


def test_config2_gray_96():
    _check(inputs.make_config(2))


@pytest.mark.parametrize("cfg,grid", [
    (3, (40, 36, 33)),      # 4 bands, widths not equal, nz odd
    (3, (37, 41, 30)),      # widths not multiples of 4: ragged quads, non-TMA ring rows
    (4, (44, 40, 30)),      # 12 bands up to x1e5: exp underflow, 1/dtau
    (5, (64, 48, 40)),      # tall-box recipe: thick and thin mix, hot top
    (5, (30, 34, 61)),
])
def test_reduced_grids_of_multiband_configs(cfg, grid):
    _check(inputs.make_config(cfg, grid=grid))


# ------------------------------------------------------------------ tiles, tails, pipelines
@pytest.mark.parametrize("tv", [1, 2, 3, 5, 7, 16])
def test_many_tiles_and_ragged_tail(tv):
    """Row bands of height tv: several tiles per job with a ragged last tile, both parities."""
    inp = inputs.make_config(3, grid=(36, 44, 38), nbands=2)
    _, _, plan = _check(inp, tiling={0: (0, tv), 1: (0, tv), 2: (0, tv)})
    assert plan["tile_v_x"] == tv and plan["tasks"] > plan["units"]


def test_one_cta_per_sm():
    _check(inputs.make_config(1), ctas_per_sm=1)


@pytest.mark.parametrize("P", [1, 2, 5])
def test_pass_counts(P):
    _check(inputs.make_config(1, grid=(24, 20, 18), npasses=P))


@pytest.mark.parametrize("grid", [(2, 2, 2), (3, 2, 4), (5, 7, 2), (4, 4, 3), (2, 9, 6)])
def test_tiny_grids(grid):
    _check(inputs.make_config(1, grid=grid))


def test_more_tasks_than_resident_ctas():
    """Ticket order must keep the pipeline deadlock-free when tasks outnumber CTA slots."""
    inp = inputs.make_config(4, grid=(32, 32, 96), nbands=12)
    _, _, plan = _check(inp, tiling={0: (0, 4), 1: (0, 4), 2: (0, 2)})
    assert plan["tasks"] > plan["grid"]


# ------------------------------------------------------------------ ray sets
def test_zface_rays_only():
    mu, w = inputs.carlson24()
    sel = [r for r in range(24) if r % 3 == 2]
    inp = inputs.make_config(1, grid=(20, 24, 16))
    inp.mu = np.ascontiguousarray(mu[sel]); inp.wq = np.full(len(sel), 1.0 / len(sel))
    _check(inp)


def test_single_ray_and_unequal_weights():
    inp = inputs.make_config(2, grid=(24, 24, 20))
    inp.mu = np.array([[0.3, -0.5, 0.81]]); inp.wq = np.array([1.0])
    _check(inp)
    inp.mu = np.array([[0.3, -0.5, 0.81], [-0.9, 0.2, -0.38], [0.1, 0.95, 0.3], [0.2, 0.1, -0.97]])
    inp.wq = np.array([0.1, 0.4, 0.3, 0.2])
    _check(inp)


def test_rays_with_a_zero_component_and_lattice_aligned():
    """f = 0 (axis-parallel in one component) and f = 1 (upwind point is a corner node)."""
    inp = inputs.make_config(1, grid=(16, 12, 14))
    dz_al = inp.dx * 0.9082483 / 0.2958759        # dx/|mu_x| = dy/|mu_y| = dz/|mu_z| for the big-z rays
    inp.dz = dz_al
    inp.mu = np.array([[0.0, 0.6, 0.8], [0.6, 0.0, -0.8], [0.0, 0.0, 1.0], [0.0, 0.0, -1.0],
                       [0.2958759, 0.2958759, 0.9082483], [-0.2958759, 0.2958759, -0.9082483]])
    inp.wq = np.full(6, 1.0 / 6.0)
    _check(inp)


# ------------------------------------------------------------------ closed form straight on the GPU
def test_isothermal_closed_form_on_gpu():
    """Pin P4 evaluated by the CUDA path itself: uniform T -> upward I = S exactly (to fp32)."""
    torch, rts = _gpu()
    inp = inputs.make_config(1, grid=(16, 16, 12))
    inp.T[...] = 6000.0
    Q, I, _ = _solve_gpu(inp)
    S = 5.670374e-5 * 6000.0 ** 4 / np.pi
    assert np.abs(I / S - 1.0).max() <= 2e-6
    assert (Q <= 1e-6 * np.abs(Q).max()).all()          # only cooling (downward rays see I < S)


# ------------------------------------------------------------------ thick-plane shortcut
def test_thick_plane_shortcut_is_bit_exact_on_itop():
    """The z sweeps skip optically thick planes in the non-final passes: I_top and Q_rad must be
    bit-identical with the shortcut off."""
    torch, rts = _gpu()
    inp = inputs.make_config(4, grid=(44, 40, 60), nbands=6)      # bands up to x1e5: many thick levels
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    s = rts.from_inputs(inp, tiling={0: (16, 12), 1: (16, 12), 2: (16, 12)})
    Q1, I1 = s.solve(rho, T, P); s.sync_check()
    levels = s.thick_levels()
    Q1 = Q1.clone(); I1 = I1.clone()
    s.set_thick_skip(False)
    Q0, I0 = s.solve(rho, T, P); s.sync_check()
    assert s.thick_levels() == [0] * inp.nbands
    s.close()
    assert max(levels) >= 4 and levels == sorted(levels), levels    # opacity scale grows with the band index
    assert torch.equal(I0, I1)
    assert torch.equal(Q0, Q1)                     # no atomics on the heating path: bitwise


# ------------------------------------------------------------------ API behaviour
def test_solve_host_matches_device_solve_and_itop_optional():
    torch, rts = _gpu()
    inp = inputs.make_config(3, grid=(28, 24, 20), nbands=2)
    Qd, Id, _ = _solve_gpu(inp)
    s = rts.from_inputs(inp)
    hQ = np.empty(inp.shape, dtype=np.float32)
    hI = np.empty((inp.nbands, inp.n_up, inp.ny, inp.nx), dtype=np.float32)
    s.solve_host(inp.rho, inp.T, inp.P, hQ, hI)
    scale = np.abs(Qd).max()
    assert np.array_equal(hQ, Qd.astype(np.float32))     # fixed summation order: bitwise
    assert np.abs(hI / Id - 1).max() <= 1e-6
    hQ2 = np.empty_like(hQ)
    s.solve_host(inp.rho, inp.T, inp.P, hQ2, None)
    assert np.abs(hQ2 - Qd).max() <= 2e-6 * scale
    s.close()
    Q3, _, _ = _solve_gpu(inp, want_itop=False)
    assert np.abs(Q3 - Qd).max() <= 2e-6 * scale


def test_repeated_solves_on_one_context_agree():
    torch, rts = _gpu()
    inp = inputs.make_config(2, grid=(48, 48, 40))
    s = rts.from_inputs(inp)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    Q1, I1 = s.solve(rho, T, P)
    Q1 = Q1.clone(); I1 = I1.clone()
    for _ in range(3):
        Q2, I2 = s.solve(rho, T, P)
    s.sync_check()
    assert torch.equal(I1, I2)
    assert torch.equal(Q1, Q2)                     # deterministic accumulation: bitwise
    s.close()


def test_bad_input_does_not_reach_the_next_solve():
    """A solve fed NaN must not poison the next, valid solve on the same context.  The only state a solve inherits
    is the workspace; on planes skipped as optically thick the seam histories are still rewritten in every pass
    (hist_pass copies the carried plane, which each task starts from zeros) and no exchange strip of a skipped block
    is read, so nothing of an earlier solve is ever multiplied by the exact 0 of a thick plane."""
    torch, rts = _gpu()
    inp = inputs.make_config(4, grid=(44, 40, 60), nbands=6)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    s = rts.from_inputs(inp, tiling={0: (16, 12), 1: (16, 12), 2: (16, 12)})
    Q1, I1 = s.solve(rho, T, P); s.sync_check()
    assert max(s.thick_levels()) >= 4
    Q1 = Q1.clone(); I1 = I1.clone()
    # the bad solve: thin everywhere (no plane skipped, every seam history written) and NaN on the top plane, which
    # the downward rays carry through the whole box
    T_bad = T.clone(); T_bad[-1] = float("nan")
    Qb, _ = s.solve(rho * 1e-8, T_bad, P)
    assert not torch.isfinite(Qb).all()
    try:
        s.sync_check()
    except Exception:
        pass                                       # whatever the bad solve reports, the context stays usable
    Q2, I2 = s.solve(rho, T, P); s.sync_check()
    s.close()
    assert torch.isfinite(Q2).all() and torch.isfinite(I2).all()
    assert torch.equal(I1, I2) and torch.equal(Q1, Q2)


def test_error_codes():
    torch, rts = _gpu()
    lib = rts.load_library()
    ctx = ctypes.c_void_p()
    assert lib.rts_create(ctypes.byref(ctx), 1, 8, 8, 1.0, 1.0, 1.0, 1) == -1        # nx < 2
    assert lib.rts_create(ctypes.byref(ctx), 8, 8, 8, 1.0, -1.0, 1.0, 1) == -1       # spacing
    assert lib.rts_create(ctypes.byref(ctx), 8, 8, 8, 1.0, 1.0, 1.0, 0) == -1        # bands
    assert lib.rts_create(None, 8, 8, 8, 1.0, 1.0, 1.0, 1) == -1
    assert lib.rts_create(ctypes.byref(ctx), 8, 8, 8, 1e5, 1e5, 1e5, 1) == 0
    buf = torch.zeros(8 * 8 * 8, dtype=torch.float32, device="cuda")
    p = ctypes.c_void_p(buf.data_ptr())
    assert lib.rts_solve(ctx, p, p, p, p, None, None) == -2                          # no tables
    assert b"tables" in lib.rts_last_error(ctx)
    assert lib.rts_set_passes(ctx, 0) == -1
    mu = (ctypes.c_double * 3)(0.5, 0.5, 0.0)
    w = (ctypes.c_double * 1)(1.0)
    assert lib.rts_set_rays(ctx, 1, mu, w) == -1                                     # mu_z == 0
    tab = (ctypes.c_float * 4)(0, 0, 0, 0)
    fr = (ctypes.c_float * 2)(1, 1)
    assert lib.rts_set_tables(ctx, 1, 2, 3.0, 4.0, 2.0, 7.0, tab, fr) == -1          # nT < 2
    assert lib.rts_set_tables(ctx, 2, 2, 3.0, 4.0, 2.0, 7.0, tab, fr) == 0
    assert lib.rts_solve(ctx, p, p, p, p, None, None) == -2                          # no workspace
    n = lib.rts_workspace_bytes(ctx)
    assert n > 0
    ws = torch.empty(n + 512, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) // 256 * 256
    assert lib.rts_set_workspace(ctx, ctypes.c_void_p(base + 4), n) == -1            # misaligned
    assert lib.rts_set_workspace(ctx, ctypes.c_void_p(base), n - 1) == -1            # too small
    assert lib.rts_set_workspace(ctx, ctypes.c_void_p(base), n) == 0
    assert lib.rts_solve(ctx, None, p, p, p, None, None) == -1                       # null field
    assert lib.rts_solve(ctx, p, p, p, ctypes.c_void_p(buf.data_ptr() + 4), None, None) == -1   # Qrad not 16-byte aligned
    assert b"aligned" in lib.rts_last_error(ctx)
    assert lib.rts_solve_cells(ctx, p, p, p, None, None, None) == -1                  # null output
    assert lib.rts_set_passes(ctx, 2) == 0
    assert lib.rts_solve(ctx, p, p, p, p, None, None) == -2                          # plan changed
    assert lib.rts_destroy(ctx) == 0
    assert lib.rts_destroy(None) == -1


# ------------------------------------------------------------------ full sizes, bench launch configuration
@pytest.mark.slow
@pytest.mark.parametrize("cfg", [3, 5, 4])
def test_full_size_configs(cfg):
    """BASELINE.json configs[2], [4], [3] at full size, planner defaults (what bench.py times).

    The oracle finishes each in tens of seconds on the box's cores, so the comparison is
    over every node and every I_top element, not a sample."""
    _check(inputs.make_config(cfg))


# ------------------------------------------------------------------ protocol check without compute-sanitizer
def test_results_barely_depend_on_tiling_and_schedule():
    """Whatever the tiling, exchange interval, ring depth or CTAs per SM, a node is updated by the same
    arithmetic (one branch-free evaluator of the attenuation factors, the same stencil in a tile's core and in
    its recomputed halo), and the heating is summed per unit in ray order and over the units in unit order:
    I_top and Q_rad of all plans are BITWISE identical, and each plan is bitwise reproducible.  A race or a
    stale halo / seam / strip anywhere in the exchange protocol breaks this (compute-sanitizer is closed on the
    GPU pool; this is the stand-in, see profiles/r2_sanitizer.md)."""
    torch, rts = _gpu()
    inp = inputs.make_config(3, grid=(60, 52, 44), nbands=3)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    t168 = {0: (16, 8), 1: (16, 8), 2: (16, 8)}
    plans = [dict(), dict(tiling=t168), dict(tiling=t168, exchange_interval=1), dict(tiling=t168, exchange_interval=2),
             dict(tiling=t168, exchange_interval=3), dict(tiling=t168, ring_depth=2), dict(tiling=t168, ctas_per_sm=2),
             dict(tiling=t168, ctas_per_sm=1, ring_depth=2, exchange_interval=2),
             dict(tiling={0: (12, 5), 1: (20, 7), 2: (8, 11)}), dict(tiling={0: (40, 12), 1: (40, 12), 2: (40, 12)}),
             dict(tiling={0: (16, 6), 1: (16, 6), 2: (16, 6)}, exchange_interval=2)]
    ref = None
    for kw in plans:
        s = rts.from_inputs(inp, **kw)
        first = None
        for rep in range(3):
            Q, I = s.solve(rho, T, P)
            s.sync_check()
            if ref is None:
                ref = (Q.clone(), I.clone())
            if first is None:
                first = (Q.clone(), I.clone())
            assert torch.equal(Q, first[0]) and torch.equal(I, first[1]), (kw, rep)
            assert torch.equal(Q, ref[0]) and torch.equal(I, ref[1]), (kw, rep)
        s.close()
