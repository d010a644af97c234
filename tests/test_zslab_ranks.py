"""Host logic of the z-slab split on CPU (world_size 2 and 3, gloo): ownership, neighbours and halo sources of
paper_2208_01525_b200.zslab, exercised by moving real planes between processes the way the GPU path's peer stores
do (a rank's top plane lands in the lower halo of the rank above, its bottom plane in the upper halo of the rank below)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_split_planes_and_halo_sources():
    from paper_2208_01525_b200.zslab import split_planes, halo_sources
    assert split_planes(128, 2, 0) == (0, 64, 1, 1) and split_planes(128, 2, 1) == (64, 64, 0, 0)
    assert split_planes(96, 3, 2) == (64, 32, 0, 1)
    assert split_planes(64, 1, 0) == (0, 64, 0, 0)
    assert halo_sources(128, 2, 0) == (127, 64) and halo_sources(128, 2, 1) == (63, 0)
    assert halo_sources(64, 1, 0) == (63, 0)
    owned = sorted(z for r in range(4) for z in range(split_planes(1024, 4, r)[0], sum(split_planes(1024, 4, r)[:2])))
    assert owned == list(range(1024))
    with pytest.raises(ValueError):
        split_planes(100, 3, 0)
    with pytest.raises(ValueError):
        split_planes(128, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nzg, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2208_01525_b200.zslab import split_planes, halo_sources
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    z_first, nz, up, dn = split_planes(nzg, world, rank)
    # a slab with halo planes whose plane p holds the value of the global plane it represents
    buf = torch.full((nz + 2, 4), -1.0)
    buf[1:nz + 1] = torch.arange(z_first, z_first + nz, dtype=torch.float32)[:, None]
    # what the step kernel's peer stores do: top own plane -> lower halo of `up`, bottom own plane -> upper halo of `dn`
    reqs = [dist.isend(buf[nz].clone(), up, tag=1), dist.isend(buf[1].clone(), dn, tag=2)]
    lo, hi = torch.empty(4), torch.empty(4)
    reqs += [dist.irecv(lo, dn, tag=1), dist.irecv(hi, up, tag=2)]
    for r in reqs:
        r.wait()
    buf[0], buf[nz + 1] = lo, hi
    q.put((rank, buf[:, 0].tolist(), halo_sources(nzg, world, rank)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,nzg", [(2, 16), (3, 12)])
def test_halo_planes_travel_to_the_right_ranks_gloo(world, nzg):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nzg, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, planes, (src_lo, src_hi) in out:
        nz = nzg // world
        assert planes[1:-1] == [float(z) for z in range(rank * nz, (rank + 1) * nz)]
        assert planes[0] == float(src_lo) == float((rank * nz - 1) % nzg)
        assert planes[-1] == float(src_hi) == float(((rank + 1) * nz) % nzg)
