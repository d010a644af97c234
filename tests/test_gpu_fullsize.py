"""Parity at BASELINE.json's full size (1024^3, the launch configuration bench.py times) on SAMPLED
outputs: 5^3 neighbourhoods are exported before a step, the oracle steps each as a tiny periodic
lattice (only the centre site is free of wrap pollution: the stencil reaches one site, diagonals
included), and the centre is compared with the GPU's value after the step."""
import gc

import numpy as np
import pytest

import inputs
from oracle import oracle as O

pytestmark = pytest.mark.gpu
DX, DTAU = 0.5, 0.1


@pytest.mark.parametrize("N", [1024])
def test_sampled_sites_full_size(N):
    import torch
    from paper_2208_01525_b200 import Lattice, Params, state_bytes, scratch_bytes
    gc.collect(); torch.cuda.empty_cache()              # lattices of earlier tests may still sit in torch's cache
    free, _ = torch.cuda.mem_get_info()
    need = state_bytes(N) + scratch_bytes(N) + (1 << 30)
    if free < need:
        pytest.skip(f"needs {need / 2**30:.0f} GiB of free HBM, have {free / 2**30:.0f}")
    lat = Lattice(N)
    prm = Params(tau_norm=256.0, friction=0.5)
    lat.init_fields(5, DX, prm)
    lat.step(6, 1.0, 0.5, 1.0)                       # damped prephase steps: links and momenta switch on
    prm.friction = 1.0
    lat.set_params(prm)
    lat.step(2, 1.6, 0.5, 1.0)
    tau = 1.8
    rng = np.random.default_rng(1024)
    corners = [(0, 0, 0), (N - 1, N - 1, N - 1), (N - 1, 0, 517), (31, 32, 33), (128, 1023, 0)]
    corners += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(27)]
    before = [lat.export_block(x - 2, y - 2, z - 2, 5, 5, 5).cpu().numpy().astype(np.float64)
              for (x, y, z) in corners]
    lat.step(1, tau, 0.5, 1.0)
    after = [lat.export_block(x, y, z, 1, 1, 1).cpu().numpy().astype(np.float64).reshape(20)
             for (x, y, z) in corners]
    K = O.Couplings()
    worst = {}
    for b, a in zip(before, after):
        ref = b.copy()
        O.step(ref, DX, K, tau, 0.5, 1.0, DTAU, tau_norm=256.0)
        for name, comps in inputs.GROUPS.items():
            scale = max(np.max(np.abs(ref[comps])), 1e-3)
            err = np.max(np.abs(a[comps] - ref[comps, 2, 2, 2])) / scale
            worst[name] = max(worst.get(name, 0.0), err)
    assert max(worst.values()) < 1e-5, worst
    # properties that hold at any size: Gauss law at roundoff (radiation, s=1), unit-ish moduli
    g = lat.gauss_violation()
    assert g[3] < 1e-5 and g[7] < 1e-5, g
    d = lat.diagnostics()
    assert d["maxW"] <= 2 and d["sumW_p"] > 0 and d["sumW_q"] > 0
    assert 0 <= d["cells_pq"] <= min(d["cells_p"], d["cells_q"])


def test_sampled_windings_full_size():
    """Winding parity at 1024^3 on sampled 6^3 blocks: the oracle evaluates the plaquettes whose four corners
    lie inside the exported block (sites 0..4 of each axis), the GPU values come from the full-size sweep."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params, state_bytes, scratch_bytes
    N = 1024
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = state_bytes(N) + scratch_bytes(N) + 9 * N ** 3 + (1 << 30)
    if free < need:
        pytest.skip(f"needs {need / 2**30:.0f} GiB of free HBM, have {free / 2**30:.0f}")
    lat = Lattice(N)
    prm = Params(tau_norm=256.0, friction=0.5)
    lat.init_fields(5, DX, prm)
    lat.step(12, 1.0, 0.5, 1.0)
    d = lat.diagnostics()
    rng = np.random.default_rng(7)
    corners = [(0, 0, 0), (N - 3, N - 3, N - 3), (N - 2, 5, 700), (30, 6, 62), (1019, 1020, 1021)]
    corners += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(20)]
    checked = flagged = nonzero = 0
    for sec in (0, 1):
        W, near, cells = lat.export_windings(sec)
        for (x, y, z) in corners:
            blk = lat.export_block(x, y, z, 6, 6, 6).cpu().numpy().astype(np.float64)
            Wr, near_r = O.windings(blk, DX, sec)
            idx = [(np.arange(c, c + 5) % N) for c in (z, y, x)]
            Wg = W[:, idx[0]][:, :, idx[1]][:, :, :, idx[2]].cpu().numpy()
            ng = near[:, idx[0]][:, :, idx[1]][:, :, :, idx[2]].cpu().numpy()
            excl = (ng > 0) | (near_r[:, :5, :5, :5] > 0)
            assert np.array_equal(Wg[~excl], Wr[:, :5, :5, :5][~excl].astype(np.int8)), (sec, x, y, z)
            checked += int((~excl).sum()); flagged += int(excl.sum()); nonzero += int(np.abs(Wg).sum())
        # cells of the sampled corners from the GPU's own windings: 6 faces of the cell at (x, y, z)
        Wc = W
        for (x, y, z) in corners[:8]:
            xp, yp, zp = (x + 1) % N, (y + 1) % N, (z + 1) % N
            c = (abs(int(Wc[0, z, y, x])) + abs(int(Wc[0, zp, y, x])) + abs(int(Wc[1, z, y, x])) + abs(int(Wc[1, z, y, xp])) +
                 abs(int(Wc[2, z, y, x])) + abs(int(Wc[2, z, yp, x])))
            assert int(cells[z, y, x]) == c
        assert d["sumW_p" if sec == 0 else "sumW_q"] == float(W.abs().sum(dtype=torch.int64))
        del W, near, cells
    assert checked > 15000 and nonzero > 0          # random-phase start: plenty of strings in any block
