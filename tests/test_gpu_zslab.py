"""One lattice split into z slabs (SURVEY.md 8(f)-4 "then z-slab multi-GPU"; include/u1u1.h "z slabs"): the sharded
step -- fused kernel + boundary planes stored into the neighbours' halo planes -- must be BIT-IDENTICAL to the
single-lattice run.  One GPU is all there is here, so (i) the kernel path runs as R slab contexts in one process
(SlabRing) and (ii) the multi-process path (CUDA IPC peer buffers, host barrier) as two ranks sharing the GPU."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import inputs
from oracle import oracle as O

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DX, DTAU = 0.5, 0.1


@pytest.mark.parametrize("N,world", [(128, 2), (128, 4), (64, 1), (48, 3), (132, 2)])
def test_slab_ring_is_bit_identical_to_the_single_lattice(N, world):
    """Seeded random-phase start of the GLOBAL lattice generated slab by slab, a damped phase, a parameter change, a
    free phase: the concatenated slabs equal the single-GPU lattice in every bit, whatever the number of slabs
    (interior, boundary and ragged tiles; slabs thinner and thicker than a z chunk of the kernel)."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    from paper_2208_01525_b200.zslab import SlabRing
    prm = Params(tau_norm=40.0, friction=0.5)
    ref = Lattice(N)
    ref.init_fields(5, DX, prm)
    ring = SlabRing(N, world, DX, prm)
    ring.init(5)
    assert torch.equal(ring.export_global(), ref.export_state())
    ref.step(6, 1.0, 0.5, 1.0)
    ring.step(6, 1.0, 0.5, 1.0, DTAU)
    prm.friction = 1.0
    ref.set_params(prm)
    ring.set_params(prm)
    ref.step(7, 1.6, 0.5, 1.0)
    ring.step(7, 1.6, 0.5, 1.0, DTAU)
    assert torch.equal(ring.export_global(), ref.export_state())
    assert sum(s.launch_count() for s in ring.slabs) == world * (1 + 13 + 2)       # init, 13 steps, 2 exports each


def test_slab_ring_on_a_generic_state_against_the_oracle():
    """import_slab / export_slab and every term of the kernel on a slab: all 20 components non-trivial, non-cubic
    global lattice (48 x 48 x 96 in three slabs), against the fp64 oracle."""
    import torch
    from paper_2208_01525_b200 import Params
    from paper_2208_01525_b200.zslab import SlabRing
    from test_gpu_step import group_errors
    N, NZ = 48, 96
    K = O.Couplings(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8)
    prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8, tau_norm=1.5)
    s0 = inputs.to_f32_exact(inputs.random_state((NZ, N, N), seed=12))
    ring = SlabRing(N, 3, DX, prm, nz_global=NZ)
    ring.import_global(torch.from_numpy(s0.astype(np.float32)).cuda())
    ring.step(3, 2.0, 2 / 3, 1.0, DTAU)
    gpu = ring.export_global().cpu().numpy().astype(np.float64)
    ref = s0.copy()
    O.step(ref, DX, K, 2.0, 2 / 3, 1.0, DTAU, tau_norm=1.5, n=3)
    err = group_errors(gpu, ref)
    assert max(err.values()) < 3e-5, err


@pytest.mark.parametrize("N,world,nzg", [(128, 2, None), (64, 4, None), (48, 3, 96)])
def test_slab_diagnostics_reduce_to_the_single_lattice(N, world, nzg):
    """Every slab sweeps its own planes (positions' upper halo from the step, E_z of the plane below pushed first), the
    28 raw values are reduced like the ranks' all-reduce pair does, and the result is the u1u1_diagnostics output of the
    whole lattice: integer counts identical, sums equal up to the grouping of the fp32 partial sums."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    from paper_2208_01525_b200.zslab import SlabRing
    prm = Params(tau_norm=40.0, friction=0.5)
    ring = SlabRing(N, world, DX, prm, nz_global=nzg)
    ring.init(7)
    ring.step(25, 1.0, 0.5, 1.0, DTAU)
    d = ring.diagnostics()
    if nzg is None:
        ref = Lattice(N)
        ref.init_fields(7, DX, prm)
        ref.step(25, 1.0, 0.5, 1.0)
        want = ref.diagnostics()
        ints = ("tau", "a", "c", "sumW_p", "sumW_q", "cells_p", "cells_q", "cells_pq", "near_p", "near_q", "maxW", "max_theta",
                "gauss_max_p", "gauss_max_q", "L_p", "L_q", "L_pq", "xi_p", "xi_q", "xi_pq", "xi_W", "f_total", "f_p")
        assert all(d[k] == want[k] for k in ints), {k: (d[k], want[k]) for k in ints if d[k] != want[k]}
        for k in ("sum_L", "sum_kin_L", "sum_grad_L", "sum_kin_V", "sum_grad_V", "sum_vint", "sum_kin", "sum_grad", "sum_elec",
                  "sum_mag", "sum_pot", "energy", "xi_L", "v2_L", "v2_pq", "gauss_l2_p", "gauss_rho_p", "gauss_rel_p", "gauss_rel_q"):
            assert np.isclose(d[k], want[k], rtol=2e-6, atol=1e-6 * abs(want["sum_grad"]) if k.startswith("sum_") else 0), (k, d[k], want[k])
        assert want["sumW_p"] > 0 and want["gauss_rel_p"] < 1e-5
    else:                                               # non-cubic global lattice: against the oracle on the gathered state
        snap = ring.export_global().cpu().numpy().astype(np.float64)
        _, c, _, _ = O.scalars(1.0 + 25 * DTAU, 0.5, 1.0, DTAU, 40.0)
        ref = O.diagnostics(snap, DX, O.Couplings(), c)
        assert abs(d["sumW_p"] - ref["sumW_p"]) <= d["near_p"] + ref["near_p"] and d["sumW_p"] > 0
        assert abs(d["cells_pq"] - ref["cells_pq"]) <= d["near_p"] + d["near_q"] + ref["near_p"] + ref["near_q"]
        scale = ref["sum_kin"] + ref["sum_grad"] + ref["sum_elec"] + ref["sum_mag"] + abs(ref["sum_pot"])
        for k in ("sum_kin", "sum_grad", "sum_elec", "sum_mag", "sum_pot", "sum_L"):
            assert abs(d[k] - ref[k]) < 2e-6 * scale, (k, d[k], ref[k])
        assert np.isclose(d["xi_W"], ref["xi_W"], rtol=1e-3)
    assert np.isnan(d["L_pq_tol"])                      # the tolerant overlap needs cell-array halos: not on slabs


def test_slab_calls_out_of_order():
    from paper_2208_01525_b200 import Slab, Params, U1U1Error
    s = Slab(32, 8, 0)
    with pytest.raises(U1U1Error, match="ESTATE"):
        s.init_slab(1)                                  # not configured as a slab yet
    s.configure_slab(DX, Params())
    with pytest.raises(U1U1Error, match="ESTATE"):
        s.step(1, 1.0, 0.5, 1.0)                        # no peers
    s.set_slab_peers(s.state.data_ptr(), s.state.data_ptr())
    with pytest.raises(U1U1Error, match="EINVAL"):
        s.step(2, 1.0, 0.5, 1.0)                        # one step per call: the ranks synchronise in between
    with pytest.raises(U1U1Error, match="ESTATE"):
        s._check(s.lib.u1u1_diagnostics(s._ctx, (__import__("ctypes").c_double * 48)()), "diagnostics")


def test_two_ranks_sharing_the_gpu_over_cuda_ipc(tmp_path):
    """The multi-process path of paper_2208_01525_b200.zslab (torchrun, CUDA IPC handles of the state buffers, host
    barrier between steps) with two ranks on this one GPU; their kernels never wait on one another.  The two dumped
    slabs must equal the single-lattice run bit for bit."""
    import socket
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    N, steps = 64, 9
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "-m", "paper_2208_01525_b200.zslab", "--size", str(N), "--steps", str(steps),
           "--dump", str(tmp_path)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    line = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")][-1]
    assert line["world"] == 2 and line["shared_gpu"] and line["nz_own"] == N // 2
    got = torch.cat([torch.load(os.path.join(tmp_path, f"slab_{k}.pt")) for k in range(2)], dim=1)
    ref = Lattice(N)
    ref.init_fields(5, DX, Params(tau_norm=256.0, friction=0.5))
    ref.step(steps, 1.0, 0.5, 1.0)
    assert torch.equal(got, ref.export_state().cpu())
    want = ref.diagnostics()                            # the ranks' all-reduced diagnostics
    for k, v in line["diagnostics"].items():
        assert np.isclose(v, want[k], rtol=2e-6), (k, v, want[k])
    assert line["diagnostics"]["sumW_p"] == want["sumW_p"] and line["diagnostics"]["cells_pq"] == want["cells_pq"]
