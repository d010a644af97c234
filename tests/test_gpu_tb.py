"""Two leapfrog steps per pass (csrc/step_tb.cu, enabled by the aux momentum buffer) against the one-step kernel: the same
per-site function in the same order, so the states must be BIT-IDENTICAL -- and parity with the fp64 oracle follows
from the one-step kernel's (tests/test_gpu_step.py); one case is compared with the oracle directly."""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import inputs  # noqa: E402
from oracle import oracle as O  # noqa: E402
from test_gpu_step import DX, DTAU, group_errors  # noqa: E402

pytestmark = pytest.mark.gpu


def run(state64, N, params, calls, aux):
    import torch
    from paper_2208_01525_b200 import Lattice
    lat = Lattice(N, aux=aux)
    lat.configure(DX, params)
    lat.import_state(torch.from_numpy(state64.astype(np.float32)))
    l0 = lat.launch_count()
    for (n, tau, m, s) in calls:
        lat.step(n, tau, m, s)
    lat.step_launches = lat.launch_count() - l0
    return lat.export_state().cpu().numpy().astype(np.float64), lat


# flags 2048: the instances with explicit range reduction of the link phases (same bits while |theta| < 2 pi);
# 132: interior (TMA), boundary and ragged tiles, two z chunks with a ragged one; 64: no interior tile in x (cp.async
# only); 8 / 12: the lattice is smaller than a tile and the two-site halo wraps onto the tile itself; 40: ragged in x
@pytest.mark.parametrize("N,flags", [(132, 0), (132, 2), (132, 512), (64, 0), (40, 0), (12, 0), (8, 0), (96, 1024), (68, 2048)])
def test_two_steps_per_pass_bit_identical(N, flags):
    from paper_2208_01525_b200 import Params
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=41 + N))
    prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.8, eta1=1.0, eta2=1.1, kappa=0.6, friction=0.9,
                 kernel_variant=16 * flags, tau_norm=1.5)
    # 4 steps = two passes; 3 steps = one pass + a single step; then a change of era / s between calls
    calls = [(4, 2.0, 0.5, 1.0), (3, 2.4, 0.5, -1.0), (2, 2.7, 2.0 / 3.0, 0.0)]
    a, lat_a = run(s0, N, prm, calls, aux=False)
    b, lat_b = run(s0, N, prm, calls, aux=True)
    assert lat_a.step_launches == 9 and lat_b.step_launches == 5      # 9 steps: 4 passes + 1 single step
    assert np.array_equal(a, b)
    # the same diagnostics from either momentum buffer (the odd number of passes leaves them in the aux buffer)
    da, db = lat_a.diagnostics(), lat_b.diagnostics()
    assert all(da[k] == db[k] or (da[k] != da[k] and db[k] != db[k]) for k in da), {k: (da[k], db[k]) for k in da if da[k] != db[k]}
    assert np.array_equal(np.array(lat_a.gauss_violation()), np.array(lat_b.gauss_violation()))


def test_two_steps_per_pass_against_oracle():
    """BASELINE.json config 1 (64^3, radiation, s = 1): 32 steps as 16 passes, against the fp64 oracle."""
    from paper_2208_01525_b200 import Params
    N = 64
    s0 = inputs.to_f32_exact(O.init_random_phase(N, seed=1))
    ref = s0.copy()
    O.step(ref, DX, O.Couplings(), 1.0, 0.5, 1.0, DTAU, tau_norm=1.0, n=32)
    gpu, lat = run(s0, N, Params(), [(32, 1.0, 0.5, 1.0)], aux=True)
    assert lat.step_launches == 16
    err = group_errors(gpu, ref)
    assert max(err.values()) < 1e-3, err
    g = lat.gauss_violation()
    assert g[3] < 1e-5 and g[7] < 1e-5


def test_aux_attach_detach_keeps_the_state():
    """Detaching the aux buffer while it holds the current momenta copies them back; export / import work either way."""
    from paper_2208_01525_b200 import Params
    N = 48
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=5))
    a, _ = run(s0, N, Params(tau_norm=1.5), [(5, 2.0, 0.5, 1.0)], aux=False)
    b, lat = run(s0, N, Params(tau_norm=1.5), [(2, 2.0, 0.5, 1.0)], aux=True)      # momenta now in the aux buffer
    lat.set_aux(False)
    lat.step(3, 2.2, 0.5, 1.0)
    assert np.array_equal(a, lat.export_state().cpu().numpy().astype(np.float64))


def test_cooling_two_steps_per_pass_bit_identical():
    """u1u1_cool (Eq. 27-30 in the same kernels) also takes two steps per pass: the paper's IC pipeline -- random phases,
    cooling (odd count), damping, evolution -- gives the same bits with and without the aux buffer."""
    from paper_2208_01525_b200 import Lattice, Params
    N = 72
    outs = []
    for aux in (False, True):
        lat = Lattice(N, aux=aux)
        lat.init_fields(3, DX, Params(eta2=1.1, kappa=0.6))
        lat.cool(11, 1.0 / 30.0)
        lat.step(6, 1.0, 0.95, 0.0)
        lat.step(5, 1.6, 0.5, 1.0)
        outs.append((lat.export_state().cpu().numpy(), lat.diagnostics()["sumW_p"]))
    assert np.array_equal(outs[0][0], outs[1][0]) and outs[0][1] == outs[1][1]
    assert np.all(np.isfinite(outs[0][0]))


def test_full_size_two_steps_per_pass_tiled_state():
    """1024^3 in the launch configuration bench.py times: a periodic tiling of a 64^3 state evolves as the tiling of the
    64^3 evolution, so every diagnostic count / sum scales by 4096 exactly and sampled blocks are bit-identical."""
    import gc
    import torch
    from paper_2208_01525_b200 import Lattice, Params, state_bytes, scratch_bytes
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = state_bytes(1024) * 4 // 3 + scratch_bytes(1024) + (2 << 30)
    if free < need:
        pytest.skip(f"needs {need / 2**30:.0f} GiB of free HBM, have {free / 2**30:.0f}")
    n = 64
    s0 = inputs.to_f32_exact(inputs.random_state((n, n, n), seed=77)).astype(np.float32)
    prm = Params(tau_norm=256.0)
    small = Lattice(n)
    small.configure(DX, prm)
    small.import_state(torch.from_numpy(s0))
    small.step(4, 1.0, 0.5, 1.0)
    ref = small.export_state().cpu().numpy()
    dsmall = small.diagnostics()
    del small
    N = 1024
    big = Lattice(N, aux=True)
    big.configure(DX, prm)
    big.import_state_tiled(torch.from_numpy(s0).cuda())
    l0 = big.launch_count()
    big.step(4, 1.0, 0.5, 1.0)
    assert big.launch_count() - l0 == 2
    for (x0, y0, z0) in [(0, 0, 0), (1000, 1016, 1008), (30, 6, 14), (510, 250, 1020)]:
        blk = big.export_block(x0, y0, z0, 24, 8, 16).cpu().numpy()
        idx = np.ix_(range(20), [(z0 + k) % n for k in range(16)], [(y0 + k) % n for k in range(8)], [(x0 + k) % n for k in range(24)])
        assert np.array_equal(blk, ref[idx])
    dbig = big.diagnostics()
    for key in ("sumW_p", "sumW_q", "cells_p", "cells_q", "cells_pq"):
        assert dbig[key] == 4096 * dsmall[key], key
    assert abs(dbig["sum_L"] - 4096 * dsmall["sum_L"]) <= 1e-9 * 4096 * abs(dsmall["sum_grad"])
    del big
    torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------------------------------
# The two-step kernel against the ORACLE directly (Eq. 17-26), at the tight tolerance and at the size
# and launch configuration bench.py times -- not through bit-identity with the one-step kernel.
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,m,s,f", [(24, 2 / 3, 1.0, 1.0), (40, 0.5, -1.0, 0.5), (8, 0.0, 1.0, 1.0),
                                      (36, 0.9, 0.0, 1.0), (132, 0.5, 0.0, 1.0)])
def test_two_steps_per_pass_generic_state_against_oracle(N, m, s, f):
    """The five generic cases of test_gpu_step.test_generic_state_every_term (all 20 components non-trivial, unequal
    couplings, friction, ragged sizes, minimum size, every era, s in {1, 0, -1}) as ONE launch of the two-step kernel
    against two oracle steps: R-16 error below 2e-5 (twice the one-step bar)."""
    from paper_2208_01525_b200 import Params
    K = O.Couplings(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8)
    prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8, tau_norm=1.5, friction=f)
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=N))
    ref = s0.copy()
    O.step(ref, DX, K, 2.0, m, s, DTAU, tau_norm=1.5, friction=f, n=2)
    gpu, lat = run(s0, N, prm, [(2, 2.0, m, s)], aux=True)
    assert lat.step_launches == 1
    err = group_errors(gpu, ref)
    assert max(err.values()) < 2e-5, err


@pytest.mark.parametrize("N", [40, 132])
def test_cooling_two_steps_per_pass_against_oracle(N):
    """u1u1_cool through the two-step kernel (one launch for two Euler steps of Eq. 27-30) against the oracle."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    K = O.Couplings(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8)
    prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8)
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=N + 1))
    ref = s0.copy()
    O.cool(ref, DX, K, 1.0 / 30.0, n=2)
    lat = Lattice(N, aux=True)
    lat.configure(DX, prm)
    lat.import_state(torch.from_numpy(s0.astype(np.float32)))
    l0 = lat.launch_count()
    lat.cool(2, 1.0 / 30.0)
    assert lat.launch_count() - l0 == 1              # the two Euler steps were one pass of the two-step kernel
    gpu = lat.export_state().cpu().numpy().astype(np.float64)
    assert not gpu[inputs.MOM].any()
    for name in ("phi", "psi", "thetaA", "thetaB"):
        comps = inputs.GROUPS[name]
        err = np.max(np.abs(gpu[comps] - ref[comps])) / np.max(np.abs(ref[comps]))
        assert err < 2e-5, (name, err)


def test_sampled_sites_full_size_two_steps_per_pass():
    """1024^3 with the aux buffer -- the kernel and launch configuration bench.py times: 5^3 neighbourhoods are exported,
    the lattice takes ONE two-step pass, and the oracle steps each block twice as a tiny periodic lattice.  The centre's
    two-step cone of dependence is +-2 sites (diagonals included), so the centre is free of wrap pollution.  Sites sit on
    the tile seams (x = 31 | 32, y = 15 | 16), the z-chunk seams (z = 127 | 128), the periodic wrap, and at random."""
    import gc
    import torch
    from paper_2208_01525_b200 import Lattice, Params, state_bytes, scratch_bytes
    N = 1024
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = state_bytes(N) * 4 // 3 + scratch_bytes(N) + (1 << 30)
    if free < need:
        pytest.skip(f"needs {need / 2**30:.0f} GiB of free HBM, have {free / 2**30:.0f}")
    lat = Lattice(N, aux=True)
    prm = Params(tau_norm=256.0, friction=0.5)
    lat.init_fields(5, DX, prm)
    lat.step(6, 1.0, 0.5, 1.0)                       # damped prephase steps: links and momenta switch on
    prm.friction = 1.0
    lat.set_params(prm)
    lat.step(2, 1.6, 0.5, 1.0)
    tau = 1.8
    rng = np.random.default_rng(2048)
    sites = [(0, 0, 0), (N - 1, N - 1, N - 1), (N - 1, 0, 517), (1, N - 2, N - 1), (0, 1023, 1),
             (31, 15, 127), (32, 16, 128), (31, 16, 128), (32, 15, 127), (63, 31, 255), (64, 32, 256),
             (991, 1007, 895), (992, 1008, 896), (30, 14, 126), (33, 17, 129), (511, 511, 511), (512, 512, 512)]
    sites += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(19)]
    assert len(sites) >= 32
    before = [lat.export_block(x - 2, y - 2, z - 2, 5, 5, 5).cpu().numpy().astype(np.float64) for (x, y, z) in sites]
    l0 = lat.launch_count()
    lat.step(2, tau, 0.5, 1.0)
    assert lat.launch_count() - l0 == 1              # one pass of step_tb_kernel
    after = [lat.export_block(x, y, z, 1, 1, 1).cpu().numpy().astype(np.float64).reshape(20) for (x, y, z) in sites]
    K = O.Couplings()
    worst = {}
    for b, a in zip(before, after):
        ref = b.copy()
        O.step(ref, DX, K, tau, 0.5, 1.0, DTAU, tau_norm=256.0, n=2)
        for name, comps in inputs.GROUPS.items():
            scale = max(np.max(np.abs(ref[comps])), 1e-3)
            err = np.max(np.abs(a[comps] - ref[comps, 2, 2, 2])) / scale
            worst[name] = max(worst.get(name, 0.0), err)
    assert max(worst.values()) < 2e-5, worst
    g = lat.gauss_violation()
    assert g[3] < 1e-5 and g[7] < 1e-5, g
    del lat
    torch.cuda.empty_cache()
