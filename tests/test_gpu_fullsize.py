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
    # near-cut plaquettes are judged, not just excluded: expected 4e-5/pi of all plaquettes per sector
    assert flagged <= 1e-4 * (checked + flagged) + 3, flagged
    assert 0 < d["near_p"] <= 1e-4 * 3 * N ** 3 and 0 < d["near_q"] <= 1e-4 * 3 * N ** 3


def test_tiled_state_full_size_every_kernel():
    """A 1024^3 lattice filled with the periodic tiling of a 64^3 state evolves as the tiling of the 64^3 evolution.
    So EVERY site of the full-size run is checked at once: after the steps the full-size diagnostics (all integer
    counts, all lattice sums, the Gauss norms, the segment statistics) must equal 16^3 times / sqrt(16^3) times those
    of the small lattice, whose state is compared element by element with the oracle."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params, state_bytes, scratch_bytes
    N, n, nsteps = 1024, 64, 3
    reps = (N // n) ** 3
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = state_bytes(N) + scratch_bytes(N) + (2 << 30)
    if free < need:
        pytest.skip(f"needs {need / 2**30:.0f} GiB of free HBM, have {free / 2**30:.0f}")
    prm = Params(tau_norm=256.0)
    small = Lattice(n)
    small.init_fields(9, DX, Params(tau_norm=256.0, friction=0.5))
    small.step(40, 1.0, 0.5, 1.0)                      # a damped start: momenta, links and strings all present
    small.set_params(prm)
    s0 = small.export_state()
    big = Lattice(N)
    big.configure(DX, prm)
    big.import_state_tiled(s0)
    tau = 5.0
    small.step(nsteps, tau, 0.5, 1.0)
    big.step(nsteps, tau, 0.5, 1.0)
    # the small lattice against the oracle, element by element
    ref = s0.cpu().numpy().astype(np.float64)
    O.step(ref, DX, O.Couplings(), tau, 0.5, 1.0, DTAU, tau_norm=256.0, n=nsteps)
    sm = small.export_state().cpu().numpy().astype(np.float64)
    for name, comps in inputs.GROUPS.items():
        assert np.max(np.abs(sm[comps] - ref[comps])) / np.max(np.abs(ref[comps])) < 3e-5, name
    # sampled tiles of the big lattice are bit-identical to the small lattice (interior, boundary and wrap tiles)
    smt = small.export_state()
    for (x, y, z) in [(0, 0, 0), (960, 960, 960), (320, 0, 704), (992, 512, 64), (64, 1000, 1000)]:
        blk = big.export_block(x, y, z, 32, 24, 16)
        ix = (torch.arange(x, x + 32, device=blk.device) % n)
        iy = (torch.arange(y, y + 24, device=blk.device) % n)
        iz = (torch.arange(z, z + 16, device=blk.device) % n)
        assert torch.equal(blk, smt[:, iz][:, :, iy][:, :, :, ix]), (x, y, z)
    # every site at once: global diagnostics scale exactly with the number of tiles
    ds, db = small.diagnostics(), big.diagnostics()
    for k in ("sumW_p", "sumW_q", "cells_p", "cells_q", "cells_pq", "near_p", "near_q", "cells_pq_tol_p", "cells_pq_tol_q"):
        assert db[k] == reps * ds[k], k
    assert db["maxW"] == ds["maxW"] and ds["sumW_p"] > 0
    for k in ("sum_L", "sum_kin_L", "sum_grad_L", "sum_kin_V", "sum_grad_V", "sum_vint", "sum_kin", "sum_grad", "sum_elec",
              "sum_mag", "sum_pot"):
        assert np.isclose(db[k], reps * ds[k], rtol=1e-9, atol=1e-9 * reps * abs(ds["sum_grad"])), k
    gs, gb = small.gauss_violation(), big.gauss_violation()
    assert np.allclose(gb[[0, 1, 4, 5]], np.sqrt(reps) * gs[[0, 1, 4, 5]], rtol=1e-9)
    assert np.array_equal(gb[[2, 6]], gs[[2, 6]])                                   # max |g|
    ss, sb = small.pq_segments(1, True), big.pq_segments(1, True)
    assert sb["cells_all"] == reps * ss["cells_all"]
