"""Peer mode across PROCESSES: two processes share one GPU, each owns one slab, the neighbour's workspace is mapped
through CUDA IPC (torch's tensor sharing) and read by the LB kernels directly -- the multi-process plumbing of
PeerSlabRunner.distributed (handle exchange, mapping, pointer arithmetic on a foreign allocation).  The ranks are
ordered by a HOST barrier after a device synchronize between kernels (gloo), so no kernel or stream ever waits on
another process; on separate GPUs the default is a stream-ordered NCCL all-reduce instead."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, walls, q, mode="ipc-one-gpu"):
    """mode: "ipc-one-gpu"  both ranks on GPU 0, gloo, host barrier between kernels (the only way on one GPU);
             "nccl-peer"    one GPU per rank, NCCL, PeerSlabRunner.distributed with its DEFAULT signal (a one-element
                            all-reduce on the compute stream): the neighbour's memory is read over NVLink;
             "nccl-halo"    one GPU per rank, NCCL, SlabRunner.distributed: ghost planes by batch_isend_irecv"""
    try:
        os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        import torch.distributed as dist
        from paper_2012_06144_b200.slab import PeerSlabRunner, SlabRunner
        if mode == "ipc-one-gpu":
            torch.cuda.set_device(0)
            dist.init_process_group("gloo", rank=rank, world_size=world)

            def sync():
                torch.cuda.synchronize()
                dist.barrier()
        else:
            torch.cuda.set_device(rank)
            dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))

            def sync():
                torch.cuda.synchronize()
                dist.barrier()

        p = Params(nx=70, ny=6, nz=12, stencil_phase=15, stencil_hydro=19, wall_flags=walls, gravity=(1e-5, -1e-5, 2e-5))
        rng = np.random.Generator(np.random.PCG64(5))
        z, y, x = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
        phi = 0.5 + 0.35 * np.sin(2 * np.pi * (x + 0.3) / p.nx) * np.cos(2 * np.pi * (y + 0.1) / p.ny) + 0.1 * np.sin(2 * np.pi * (z + 0.7) / p.nz)
        u = rng.uniform(-0.02, 0.02, size=(3,) + p.shape)
        dev = torch.device("cuda", torch.cuda.current_device())
        if mode == "ipc-one-gpu":
            run = PeerSlabRunner.distributed(p, rank, world, sync=sync, device=dev)
        elif mode == "nccl-peer":
            run = PeerSlabRunner.distributed(p, rank, world, device=dev)          # default sync: all-reduce on the compute stream
        else:
            run = SlabRunner.distributed(p, rank, world, device=dev)
        run.init(torch.from_numpy(phi).cuda(), torch.from_numpy(u).cuda())
        run.step(4)
        c, uu, pr = run.fields()
        h, g = run.get_pdfs()
        mine = [t.cpu().numpy() for t in (c, uu, pr, h, g)]
        gathered = [None] * world
        dist.all_gather_object(gathered, mine)
        ok = True
        if mode == "nccl-peer":
            nb = (rank + 1) % world
            assert torch.cuda.can_device_access_peer(rank, nb), f"no peer access {rank} -> {nb}"
        if rank == 0:
            from paper_2012_06144_b200.binding import ACM
            a = ACM.from_params(p)
            a.init(torch.from_numpy(phi).cuda(), torch.from_numpy(u).cuda())
            a.step(4)
            ref = [t.cpu().numpy() for t in a.fields() + a.get_pdfs()]
            for k in range(5):
                got = np.concatenate([gathered[r][k] for r in range(world)], axis=-3)
                ok = ok and np.array_equal(got, ref[k])
        sync()
        dist.destroy_process_group()
        q.put((rank, "ok" if ok else "mismatch"))
    except Exception:  # pragma: no cover
        import traceback
        q.put((rank, traceback.format_exc()))
        raise


@pytest.mark.parametrize("walls", [0, inputs.WALL_Z])
def test_two_processes_one_gpu_peer_mode_over_cuda_ipc(walls):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, walls, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    try:
        out = sorted(q.get(timeout=240) for _ in procs)
    finally:
        for pr in procs:
            pr.join(timeout=60)
            if pr.is_alive():
                pr.kill()
    assert [o[1] for o in out] == ["ok", "ok"], out


@pytest.mark.parametrize("mode", ["nccl-peer", "nccl-halo"])
@pytest.mark.parametrize("walls", [0, inputs.WALL_Z])
def test_two_gpus_over_nccl(mode, walls):
    """The transports that one GPU cannot exercise: one slab per GPU, NCCL process group.  "nccl-peer": the LB kernels
    read the neighbour GPU's boundary planes over NVLink (CUDA-IPC mapped workspace), ordered by the default
    one-element all-reduce; "nccl-halo": ghost planes travel by batch_isend_irecv on the comm stream.  Both must
    reproduce the single-domain run bit for bit.  Skipped on a single-GPU box."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, walls, q, mode)) for r in range(2)]
    for pr in procs:
        pr.start()
    try:
        out = sorted(q.get(timeout=300) for _ in procs)
    finally:
        for pr in procs:
            pr.join(timeout=60)
            if pr.is_alive():
                pr.kill()
    assert [o[1] for o in out] == ["ok", "ok"], out
