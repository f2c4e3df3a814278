"""Grid staggering (paper's Interpolate) on the GPU against the
oracle's O-9: cells -> corner nodes is bit-exact (both sides form the correctly rounded mean of 8
fp32 cells), nodes -> cells and the staggered solve meet the tolerances of the main path."""
import numpy as np
import pytest

from paper_2107_08145_b200 import inputs

pytestmark = pytest.mark.gpu


def _gpu():
    import torch
    from paper_2107_08145_b200 import rts
    return torch, rts


@pytest.mark.parametrize("grid", [(2, 2, 1), (5, 3, 2), (37, 41, 30), (130, 70, 65), (288, 288, 40)])
def test_cells_to_nodes_bit_exact_and_nodes_to_cells(grid):
    import oracle
    torch, rts = _gpu()
    nx, ny, ncz = grid
    rng = np.random.default_rng(nx * 1000 + ny)
    cell = (rng.standard_normal((ncz, ny, nx)) * 10.0 ** rng.uniform(-6, 6, (ncz, 1, 1))).astype(np.float32)
    s = rts.RTS(nx, ny, ncz + 1, 1e5, 1e5, 1e5, 1)
    node = s.cells_to_nodes(torch.from_numpy(cell).cuda())
    torch.cuda.synchronize()
    assert np.array_equal(node.cpu().numpy(), oracle.cells_to_nodes(cell))          # bit-exact
    qn = rng.standard_normal((ncz + 1, ny, nx)).astype(np.float32)
    qc = s.nodes_to_cells(torch.from_numpy(qn).cuda()).cpu().numpy().astype(np.float64)
    want = oracle.nodes_to_cells(qn.astype(np.float64))
    assert np.abs(qc - want).max() <= 1e-6 * np.abs(qn).max()
    s.close()


@pytest.mark.parametrize("cfg,grid", [(1, None), (2, (48, 40, 36)), (3, (40, 36, 33)), (5, (33, 47, 29)), (2, None)])
def test_staggered_solve_matches_oracle(cfg, grid):
    """Cell-centred inputs -> Q on the cells and I_top, against oracle.solve_cells on the same cells."""
    import oracle
    torch, rts = _gpu()
    inp = inputs.make_config(cfg, grid=grid)                   # its fields are taken as cell-centred
    Qo, Io, node = oracle.solve_cells(inp)
    s = rts.from_inputs(inp, cells=True)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    Qc = torch.full(inp.shape, 1e30, dtype=torch.float32, device="cuda")
    Qc, Itop = s.solve_cells(rho, T, P, Qc)
    s.sync_check()
    Q = Qc.cpu().numpy().astype(np.float64); I = Itop.cpu().numpy().astype(np.float64)
    eq = np.abs(Q - Qo).max() / np.abs(Qo).max()
    ei = (np.abs(I - Io) / np.abs(Io)).max()
    print(f"{inp.name} staggered: dQ/maxQ = {eq:.3e}; rel dItop = {ei:.3e}")
    assert eq <= 1e-4 and ei <= 1e-5
    # the node grid solve alone agrees with the unstaggered entry point on the oracle's node fields
    Qn, _ = s.solve(*(torch.from_numpy(a).cuda() for a in (node.rho, node.T, node.P)))
    Qc2 = s.nodes_to_cells(Qn)
    assert (Qc2 - Qc).abs().max().item() <= 4e-6 * Qc.abs().max().item()        # atomics: summation order
    s.close()


@pytest.mark.slow
def test_staggered_solve_full_size_config3():
    """BASELINE.json configs[2] at full size through rts_solve_cells (planner defaults)."""
    test_staggered_solve_matches_oracle(3, None)
