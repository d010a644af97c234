"""One lattice split into z slabs over several GPUs (SURVEY.md 8(f)-4 "then z-slab multi-GPU").

Host logic only: who owns which planes, who the neighbours are, how the ranks learn each other's state buffers (CUDA
IPC through torch) and where the per-step barrier goes.  The exchange itself is not here: the fused step kernel stores
its boundary planes straight into the neighbours' halo planes (peer memory; NVLink between GPUs).

    torchrun --nnodes=1 --nproc-per-node R -m paper_2208_01525_b200.zslab --size 1024 --steps 50

Not the default path: the benchmark workload (1024^3) fits one GPU and runs there (north_star); `bench.py --gpus N` runs
independent replicas.  Nothing in this environment has more than one GPU, so the multi-process path is exercised with
two ranks on ONE GPU (their kernels never wait on one another: the barrier is on the host) and the kernel path by R slab
contexts in one process (`SlabRing`), both bit-identical to the single-lattice run.

UNVERIFIED ON MORE THAN ONE GPU: the NCCL stream-ordered barrier and the peer stores across NVLink have never run on
real multi-GPU hardware (no node with several GPUs was available in any round).  The handle exchange relies on the private
torch calls `_share_cuda_` / `_new_shared_cuda`.
"""
from __future__ import annotations

import argparse
import json
import os
import time

from . import binding as B


def split_planes(nz_global: int, world: int, rank: int):
    """(z_first, nz_own, rank above, rank below) of `rank` in a ring of `world` equal slabs, periodic in z."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError(f"rank {rank} outside a world of {world}")
    if nz_global % world:
        raise ValueError(f"{nz_global} planes do not split into {world} equal slabs")
    nz = nz_global // world
    return rank * nz, nz, (rank + 1) % world, (rank - 1) % world


def halo_sources(nz_global: int, world: int, rank: int):
    """Global plane indices that end up in this rank's lower and upper halo plane."""
    z_first, nz, _, _ = split_planes(nz_global, world, rank)
    return (z_first - 1) % nz_global, (z_first + nz) % nz_global


class SlabRing:
    """`world` slabs of one N x N x nz_global lattice in ONE process on one device, wired as a periodic ring: the
    single-GPU stand-in for the multi-GPU run (same kernel, same peer stores, launches simply queue on one stream)."""

    def __init__(self, N: int, world: int, dx: float, params: B.Params, nz_global: int | None = None, device: str = "cuda:0"):
        from .lattice import Slab
        self.N, self.world, self.nz_global = N, world, nz_global or N
        self.slabs = []
        for r in range(world):
            z_first, nz, _, _ = split_planes(self.nz_global, world, r)
            s = Slab(N, nz, z_first, device=device)
            s.configure_slab(dx, params)
            self.slabs.append(s)
        for r, s in enumerate(self.slabs):
            _, _, up, dn = split_planes(self.nz_global, world, r)
            s.set_slab_peers(self.slabs[up].state.data_ptr(), self.slabs[dn].state.data_ptr())

    def init(self, seed: int):
        for s in self.slabs:
            s.init_slab(seed)
        for s in self.slabs:
            s.push_halos()

    def import_global(self, t):
        """t: canonical [20, nz_global, N, N]."""
        for s in self.slabs:
            s.import_slab(t[:, s.z_first:s.z_first + s.nz_own])
        for s in self.slabs:
            s.push_halos()

    def set_params(self, params: B.Params):
        for s in self.slabs:
            s.set_params(params)

    def step(self, n: int, tau: float, era_m: float, s_: float, dtau: float):
        for k in range(n):                          # every slab advances one step, then the next step: lockstep
            for s in self.slabs:
                s.step(1, tau + k * dtau, era_m, s_)

    def export_global(self):
        import torch
        return torch.cat([s.export_slab() for s in self.slabs], dim=1)

    def diagnostics(self):
        """The u1u1_diagnostics output of the whole lattice: per-slab sweeps, then the reduction the ranks would do."""
        for s in self.slabs:
            s.push_diag_halos()
        raws = [s.slab_diagnostics_partial() for s in self.slabs]
        return self.slabs[0].slab_diagnostics_finish(reduce_raw(raws), self.nz_global)


def reduce_raw(raws):
    """SUM over the first SLAB_NSUM raw values, MAX over the rest (what the all-reduce pair of the ranks computes)."""
    import numpy as np
    a = np.stack(raws)
    return np.concatenate([a[:, :B.SLAB_NSUM].sum(axis=0), a[:, B.SLAB_NSUM:].max(axis=0)])


def all_reduce_raw(raw, dist, device):
    """The same across ranks: one SUM and one MAX all-reduce of a handful of doubles."""
    import numpy as np
    import torch
    t = torch.tensor(raw, dtype=torch.float64, device=device)
    head, tail = t[:B.SLAB_NSUM].clone(), t[B.SLAB_NSUM:].clone()
    dist.all_reduce(head, op=dist.ReduceOp.SUM)
    dist.all_reduce(tail, op=dist.ReduceOp.MAX)
    return np.concatenate([head.cpu().numpy(), tail.cpu().numpy()])


def open_peer_states(state, dist, rank: int, world: int, up: int, dn: int):
    """Every rank publishes the CUDA IPC handle of its state tensor; returns tensors aliasing the state buffers of the
    ranks above and below (peer-mapped device memory; keep them alive as long as the context lives)."""
    import torch
    handles = [None] * world
    dist.all_gather_object(handles, state.untyped_storage()._share_cuda_())
    out = []
    for peer in (up, dn):
        if peer == rank:
            out.append(state)
            continue
        storage = torch.UntypedStorage._new_shared_cuda(*handles[peer])
        out.append(torch.empty(0, dtype=torch.uint8, device=state.device).set_(storage))
    return out


def run(size: int, steps: int, seed: int = 5, nz_global: int | None = None, check_every: int = 0, emit=print):
    """One rank of the multi-process run (launched by torchrun): strong scaling of one size x size x nz_global lattice."""
    import torch
    import torch.distributed as dist
    from .lattice import Slab
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    ndev = torch.cuda.device_count()
    dev = local % ndev                              # more ranks than GPUs: they share a device (testing only)
    torch.cuda.set_device(dev)
    shared_gpu = world > ndev
    # NCCL refuses two ranks on one device; the barrier and the handle exchange then go through gloo
    dist.init_process_group("gloo" if shared_gpu or world == 1 else "nccl",
                            **({} if shared_gpu or world == 1 else {"device_id": torch.device(f"cuda:{dev}")}))
    nzg = nz_global or size
    z_first, nz, up, dn = split_planes(nzg, world, rank)
    DX, DTAU, TAU0 = 0.5, 0.1, 1.0
    slab = Slab(size, nz, z_first, device=f"cuda:{dev}")
    prm = B.Params(tau_norm=256.0, friction=0.5)
    slab.configure_slab(DX, prm)
    peers = open_peer_states(slab.state, dist, rank, world, up, dn)
    slab.set_slab_peers(peers[0].data_ptr(), peers[1].data_ptr())
    slab._peers = peers                             # the context holds raw pointers into these mappings: they live as long as the slab
    token = torch.zeros(1, device=f"cuda:{dev}")

    def barrier():
        # every rank has finished the launches queued so far (their peer stores included) before anyone goes on
        if dist.get_backend() == "nccl":
            dist.all_reduce(token)                  # stream-ordered: no host synchronisation
        else:
            torch.cuda.synchronize()
            dist.barrier()

    slab.init_slab(seed)
    barrier()
    slab.push_halos()
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(steps):
        slab.step(1, TAU0 + k * DTAU, 0.5, 1.0)
        barrier()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    # diagnostics of the whole lattice: halo of E_z below, per-rank sweep, reduction of 28 doubles
    slab.push_diag_halos()
    barrier()
    raw = all_reduce_raw(slab.slab_diagnostics_partial(), dist, "cpu" if dist.get_backend() == "gloo" else f"cuda:{dev}")
    d = slab.slab_diagnostics_finish(raw, nzg)
    out = {"rank": rank, "world": world, "N": size, "nz_global": nzg, "nz_own": nz, "steps": steps, "wall_s": wall,
           "site_updates_per_s": size * size * nzg * steps / wall, "backend": dist.get_backend(), "shared_gpu": shared_gpu,
           "diagnostics": {k: d[k] for k in ("tau", "sumW_p", "sumW_q", "cells_pq", "maxW", "xi_W", "sum_L", "energy",
                                             "gauss_rel_p", "gauss_rel_q", "max_theta")}}
    if rank == 0:
        emit(json.dumps(out))
    dist.barrier()
    return slab, out


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--size", type=int, default=256)
    ap.add_argument("--nz-global", type=int, default=None)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--dump", default=None, help="directory: every rank saves its slab (canonical layout) as slab_<rank>.pt")
    a = ap.parse_args()
    slab, out = run(a.size, a.steps, nz_global=a.nz_global)
    if a.dump:
        import torch
        os.makedirs(a.dump, exist_ok=True)
        torch.save(slab.export_slab().cpu(), os.path.join(a.dump, f"slab_{out['rank']}.pt"))
    import torch.distributed as dist
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
