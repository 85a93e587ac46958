"""Slab decomposition, host side (no GPU): the halo plan of libacm (which planes of which directions
cross a z face) and the exchange protocol of paper_2012_06144_b200/slab.py over gloo with 2 and 3 ranks.

acm_create_slab / acm_halo_plan are host-only calls, so the real plan is used here with CPU tensors as
stand-ins for the workspaces; the kernels' use of the ghost planes is covered on the GPU
(tests/test_gpu_slab.py)."""
import ctypes as C
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp

import bruteforce
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

HALO_H, HALO_G, HALO_PHI = 0, 1, 2


class CpuPort:
    """A slab context created against a fake workspace pointer (no device call is made) plus a CPU tensor of
    the same size: halo_views() slices it at the offsets of the real acm_halo_plan."""

    def __init__(self, p, rank, nranks):
        from paper_2012_06144_b200 import binding
        from paper_2012_06144_b200.slab import halo_plan, slab_range
        self.lib = binding.load()
        self.rank, self.nranks = rank, nranks
        self.z0, self.nzl = slab_range(p.nz, rank, nranks)
        self.nbytes = self.lib.acm_workspace_bytes_slab(p.nx, p.ny, p.nz, p.stencil_phase, p.stencil_hydro, 0, rank, nranks)
        assert self.nbytes > 0
        g = (C.c_double * 3)(*p.gravity)
        self.h = C.c_void_p()
        rc = self.lib.acm_create_slab(C.byref(self.h), p.nx, p.ny, p.nz, p.stencil_phase, p.stencil_hydro, p.rho_H, p.rho_L,
                                      p.sigma, p.xi, p.M, p.nu_H, p.nu_L, g, p.wall_flags, 0, 0, rank, nranks,
                                      C.c_void_p(256 * 4096), None)
        assert rc == 0, self.lib.acm_last_error()
        self._plan = halo_plan
        # every 8-byte word of the "workspace" names its owner and its position
        self.ws = (torch.arange(self.nbytes // 8, dtype=torch.float64) + rank * 1e12).view(torch.uint8)

    def plan(self, what, side, recv):
        return self._plan(self.lib, self.h, what, side, recv)

    def halo_views(self, what, side, recv):
        return [self.ws[o:o + n] for o, n in self.plan(what, side, recv)]

    def close(self):
        self.lib.acm_destroy(self.h)


def _align256(v):
    return (v + 255) & ~255


@pytest.mark.parametrize("Qh,Qg", [(15, 19), (27, 27), (19, 15)])
def test_halo_plan_lists_the_crossing_directions(Qh, Qg):
    """Layout contract of DESIGN.md section 4 (H[2][Qh][N], G[2][Qg][N], C[2][N], each 256-byte aligned) lets the
    offsets be decoded into (direction, plane); compared with the lattices typed in tests/bruteforce.py:
    a cell pulls slot i from z - e_iz, so the low ghost plane must receive the e_z = +1 slots, etc."""
    nx, ny, nzg, R = 12, 5, 17, 3
    p = Params(nx=nx, ny=ny, nz=nzg, stencil_phase=Qh, stencil_hydro=Qg)
    covered = 0
    for rank in range(R):
        port = CpuPort(p, rank, R)
        nzl = port.nzl
        covered += nzl
        assert port.z0 == sum(CpuPort(p, r, R).nzl for r in range(rank))
        N = nx * ny * (nzl + 2)
        plane = nx * ny * 8
        offH0 = 0
        offH1 = _align256(offH0 + Qh * N * 8)
        offG0 = _align256(offH1 + Qh * N * 8)
        offG1 = _align256(offG0 + Qg * N * 8)
        offC0 = _align256(offG1 + Qg * N * 8)
        for what, Q, base in ((HALO_H, Qh, offH0), (HALO_G, Qg, offG0)):
            e, _ = bruteforce.lattice(Q)
            for side in (0, 1):
                for recv in (False, True):
                    chunks = port.plan(what, side, recv)
                    dirs = [(o - base) // (N * 8) for o, _ in chunks]
                    planes = {((o - base) % (N * 8)) // plane for o, _ in chunks}
                    assert all(n == plane for _, n in chunks)
                    assert all(((o - base) % (N * 8)) % plane == 0 for o, _ in chunks)
                    want_sign = +1 if (side == 0) == recv else -1
                    assert dirs == [i for i in range(Q) if e[i][2] == want_sign]
                    want_plane = (0 if recv else 1) if side == 0 else (nzl + 1 if recv else nzl)
                    assert planes == {want_plane}
        for side in (0, 1):
            for recv in (False, True):
                (o, n), = port.plan(HALO_PHI, side, recv)
                want_plane = (0 if recv else 1) if side == 0 else (nzl + 1 if recv else nzl)
                assert (o, n) == (offC0 + want_plane * plane, plane)
        port.close()
    assert covered == nzg


def test_slab_range_and_argument_checks():
    from paper_2012_06144_b200 import binding
    from paper_2012_06144_b200.slab import slab_range
    assert [slab_range(10, r, 4) for r in range(4)] == [(0, 3), (3, 3), (6, 2), (8, 2)]
    assert slab_range(7, 0, 1) == (0, 7)
    for bad in ((4, 0, 5), (4, 4, 4), (4, -1, 2), (0, 0, 1)):
        with pytest.raises(binding.AcmError):
            slab_range(*bad)
    lib = binding.load()
    assert lib.acm_workspace_bytes_slab(16, 8, 8, 15, 19, 0, 0, 9) == 0
    # in-place / unfused are refused for slabs; acm_step is refused on a slab
    p = Params(nx=8, ny=4, nz=8)
    g = (C.c_double * 3)(0, 0, 0)
    h = C.c_void_p()
    args = [p.nx, p.ny, p.nz, 15, 19, p.rho_H, p.rho_L, p.sigma, p.xi, p.M, p.nu_H, p.nu_L, g, 0, 0]
    assert lib.acm_create_slab(C.byref(h), *args, 1, 0, 2, C.c_void_p(4096), None) == binding.ACM_EINVAL
    assert lib.acm_create_slab(C.byref(h), *args, 4, 0, 2, C.c_void_p(4096), None) == binding.ACM_EINVAL
    assert lib.acm_create_slab(C.byref(h), *args, 0, 0, 2, C.c_void_p(4096), None) == binding.ACM_OK
    info = (C.c_int * 6)()
    assert lib.acm_slab_info(h, info) == 0 and list(info) == [0, 2, 0, 4, 6, 1]
    assert lib.acm_phase_launch(h, 0, 4) == binding.ACM_ESTATE          # before acm_init
    lib.acm_destroy(h)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _expected(sender_rank, chunks):
    """what the sender's workspace holds at these chunks"""
    return [(torch.arange(o // 8, (o + n) // 8, dtype=torch.float64) + sender_rank * 1e12) for o, n in chunks]


def _worker(rank, world, port, wall_z, q):
    try:
        os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        import torch.distributed as dist
        from paper_2012_06144_b200.slab import HaloExchanger
        dist.init_process_group("gloo", rank=rank, world_size=world)
        p = Params(nx=12, ny=5, nz=4 * world + 1, stencil_phase=15, stencil_hydro=27,
                   wall_flags=inputs.WALL_Z if wall_z else 0)
        me = CpuPort(p, rank, world)
        others = {r: CpuPort(p, r, world) for r in range(world)}       # only their PLANS are used below
        ex = HaloExchanger([me], world, wall_z)
        pristine = me.ws.clone()
        touched = torch.zeros(me.nbytes, dtype=torch.bool)
        for what in (HALO_PHI, HALO_H, HALO_G):
            HaloExchanger.finish(ex.exchange(what))
            lo, hi = (rank - 1) % world, (rank + 1) % world
            faces = []
            if not (wall_z and rank == 0):
                faces.append((0, lo, 1))       # my low ghost <- the low neighbour's HIGH face
            if not (wall_z and rank == world - 1):
                faces.append((1, hi, 0))       # my high ghost <- the high neighbour's LOW face
            for side, nb, nb_side in faces:
                got = me.halo_views(what, side, True)
                want = _expected(nb, others[nb].plan(what, nb_side, False))
                assert len(got) == len(want) > 0
                for gt, wt in zip(got, want):
                    assert torch.equal(gt.view(torch.float64), wt), (what, side)
                for o, n in me.plan(what, side, True):
                    touched[o:o + n] = True
        # nothing outside the ghost chunks changed
        assert torch.equal(me.ws[~touched], pristine[~touched])
        dist.barrier()
        dist.destroy_process_group()
        q.put((rank, "ok"))
    except Exception as e:  # pragma: no cover
        import traceback
        q.put((rank, traceback.format_exc()))
        raise


@pytest.mark.parametrize("world,wall_z", [(2, False), (2, True), (3, False)])
def test_halo_exchange_over_gloo(world, wall_z):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, wall_z, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    out = sorted(q.get(timeout=180) for _ in procs)
    for pr in procs:
        pr.join(timeout=60)
    assert [o[1] for o in out] == ["ok"] * world, out
    assert all(pr.exitcode == 0 for pr in procs)


def test_local_exchange_single_process_two_and_one_slab():
    """all slabs in one process: neighbours reached by copies; one slab wraps onto itself"""
    from paper_2012_06144_b200.slab import HaloExchanger
    for world in (1, 2):
        p = Params(nx=12, ny=5, nz=6, stencil_phase=19, stencil_hydro=19)
        ports = [CpuPort(p, r, world) for r in range(world)]
        ex = HaloExchanger(ports, world)
        for what in (HALO_PHI, HALO_H, HALO_G):
            assert ex.exchange(what) == []
            for r, me in enumerate(ports):
                for side, nb, nb_side in ((0, (r - 1) % world, 1), (1, (r + 1) % world, 0)):
                    for gt, wt in zip(me.halo_views(what, side, True), _expected(nb, ports[nb].plan(what, nb_side, False))):
                        assert torch.equal(gt.view(torch.float64), wt)
