"""Slab decomposition of the coupled ACM step along z over several GPUs.

The paper distributes the domain in blocks with one ghost layer and hides the communication behind an
inner / outer split of each LB step (Alg. 2 and Fig. 3).  Here: one process per
GPU, one z-slab per process (`acm_create_slab`), `torch.distributed` point-to-point transfers (NCCL over
NVLink) of exactly the planes `acm_halo_plan` lists -- the e_z != 0 populations of the outermost owned
plane and one phi plane per face -- straight from and into the population arrays (a z plane of one
direction is contiguous: no pack / unpack kernels).  The schedule of `SlabRunner.step`:

    phase kernel (all planes)                         compute stream
    exchange phi_new, then h                          comm stream   (h is needed by the NEXT phase step)
    hydro kernel on the inner planes                  compute stream, overlaps the exchange
    hydro kernel on the two outer planes              after phi_new (and the g of the previous step) arrived
    exchange g                                        comm stream, overlaps the next phase kernel

This module only moves bytes and orders launches: every step of the method runs in libacm's kernels.
The same code drives several slabs inside ONE process (neighbours reached by device copies), which is how
the kernels' ghost-plane logic is tested on a single GPU, and the exchanger alone runs on CPU tensors over
gloo (tests/test_slab_gloo.py).
"""
from __future__ import annotations

import ctypes as C
from typing import List, Optional, Sequence

import torch

from . import binding
from .binding import ACM, ACM_EINVAL, ACM_F32, ACM_F64, AcmError, _check

HALO_H, HALO_G, HALO_PHI = 0, 1, 2
MAX_CHUNKS = 16


def slab_range(nz_global: int, rank: int, nranks: int):
    """(first plane, number of planes) of the global grid owned by `rank` (acm_slab_range)."""
    lib = binding.load()
    z0, cnt = C.c_int(), C.c_int()
    _check(lib, lib.acm_slab_range(int(nz_global), int(rank), int(nranks), C.byref(z0), C.byref(cnt)))
    return z0.value, cnt.value


def halo_plan(lib, handle, what: int, side: int, recv: bool):
    """[(byte offset in the workspace, bytes)] of acm_halo_plan."""
    off = (C.c_size_t * MAX_CHUNKS)()
    nb = (C.c_size_t * MAX_CHUNKS)()
    n = lib.acm_halo_plan(handle, int(what), int(side), int(bool(recv)), MAX_CHUNKS, off, nb)
    if n < 0:
        raise AcmError(-n, lib.acm_last_error().decode())
    return [(off[k], nb[k]) for k in range(n)]


def pad_planes(a: torch.Tensor, z0: int, cnt: int) -> torch.Tensor:
    """Planes z0-1 .. z0+cnt of a global (..., nz, ny, nx) array (periodic wrap in z): the padded local
    array of a slab, ghost planes first and last."""
    nz = a.shape[-3]
    idx = torch.arange(z0 - 1, z0 + cnt + 1, device=a.device) % nz
    return a.index_select(a.dim() - 3, idx).contiguous()


class SlabACM(ACM):
    """One z-slab of a decomposed domain (acm_create_slab).  Field arrays have nz_local + 2 planes."""

    def __init__(self, p, rank: int, nranks: int, precision="f64", device="cuda:0", stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2012_06144_b200 needs a CUDA device (no CPU fallback)")
        self._lib = binding.load()
        self.device = torch.device(device)
        self.rank, self.nranks = int(rank), int(nranks)
        self.z0, self.nzl = slab_range(p.nz, rank, nranks)
        self.nx, self.ny, self.nz = int(p.nx), int(p.ny), self.nzl + 2
        self.nz_global = int(p.nz)
        self.Qh, self.Qg = int(p.stencil_phase), int(p.stencil_hydro)
        self.N = self.nx * self.ny * self.nz
        self.shape = (self.nz, self.ny, self.nx)
        self.precision = {"f64": ACM_F64, "f32": ACM_F32}[precision]
        self.dtype = torch.float64 if precision == "f64" else torch.float32
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.options = binding.ACM_OPT_PHASE_SRT if getattr(p, "phase_srt", False) else 0
        self.wall_z = bool(p.wall_flags & binding.ACM_WALL_Z)
        nbytes = self._lib.acm_workspace_bytes_slab(self.nx, self.ny, self.nz_global, self.Qh, self.Qg, self.precision,
                                                    self.rank, self.nranks)
        if nbytes == 0:
            raise AcmError(ACM_EINVAL, "invalid grid size / stencil / precision / decomposition")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        self.base = ((self.workspace.data_ptr() + 255) & ~255) - self.workspace.data_ptr()
        g = (C.c_double * 3)(*[float(v) for v in p.gravity])
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = self._lib.acm_create_slab(C.byref(h), self.nx, self.ny, self.nz_global, self.Qh, self.Qg, p.rho_H, p.rho_L,
                                           p.sigma, p.xi, p.M, p.nu_H, p.nu_L, g, int(p.wall_flags), self.precision,
                                           self.options, self.rank, self.nranks,
                                           C.c_void_p(self.workspace.data_ptr() + self.base),
                                           C.c_void_p(self.stream.cuda_stream))
        _check(self._lib, rc)
        self._h = h

    # ---- pieces of a step -------------------------------------------------------------------
    def phase_launch(self, z0, z1):
        self._call(self._lib.acm_phase_launch, int(z0), int(z1))

    def phase_commit(self):
        self._call(self._lib.acm_phase_commit)

    def hydro_launch(self, z0, z1):
        self._call(self._lib.acm_hydro_launch, int(z0), int(z1))

    def hydro_commit(self):
        self._call(self._lib.acm_hydro_commit)

    def bubble_sums(self):
        out = (C.c_double * 7)()
        self._call(self._lib.acm_bubble_sums, out)
        return list(out)

    # ---- halo views ---------------------------------------------------------------------------
    def halo_views(self, what, side, recv) -> List[torch.Tensor]:
        """uint8 views of the workspace for the planes acm_halo_plan lists."""
        return [self.workspace[self.base + off: self.base + off + nb]
                for off, nb in halo_plan(self._lib, self._h, what, side, recv)]

    def owned(self, t: torch.Tensor) -> torch.Tensor:
        """strip the ghost planes of a field array of this slab"""
        return t[..., 1:-1, :, :]


class HaloExchanger:
    """Fills the ghost planes of the local slabs for one stage (HALO_H, HALO_G or HALO_PHI).

    `ports` are the slabs this process holds: objects with `.rank` and
    `.halo_views(what, side, recv) -> [uint8 tensors]` (SlabACM, or a stand-in on CPU tensors in the
    gloo test).  Either this process holds ALL `nranks` slabs (neighbours are reached by `copy_`), or it
    holds exactly one and slab r lives in process r of `group` (neighbours are reached by isend / irecv).

    Message order (NCCL matches sends and receives per peer in issue order; with two ranks both faces
    talk to the same peer): every rank SENDS low face then high face, and RECEIVES high ghost then low
    ghost -- what my high ghost receives is what the neighbour sent through its low face.
    Faces on a z wall of the global domain exchange nothing.
    """

    def __init__(self, ports: Sequence, nranks: int, wall_z: bool = False, group=None):
        self.ports = {int(p.rank): p for p in ports}
        self.nranks, self.wall_z, self.group = int(nranks), bool(wall_z), group
        if len(self.ports) != len(ports):
            raise ValueError("two local slabs with the same rank")
        self.local_only = len(self.ports) == self.nranks
        if not self.local_only and len(self.ports) != 1:
            raise ValueError("a process holds either all slabs or exactly one")

    def _faces(self, r):
        has_lo = not (self.wall_z and r == 0)
        has_hi = not (self.wall_z and r == self.nranks - 1)
        return has_lo, has_hi, (r - 1) % self.nranks, (r + 1) % self.nranks

    def exchange(self, what: int):
        """Enqueues the transfers on the current stream (device copies) / the backend's stream (P2P) and
        returns the list of outstanding `dist` works (empty for local copies); call `finish` on it."""
        works = []
        if self.local_only:
            for r, port in self.ports.items():
                has_lo, has_hi, lo, hi = self._faces(r)
                if has_lo:      # my low face -> low neighbour's high ghost
                    for dst, src in zip(self.ports[lo].halo_views(what, 1, True), port.halo_views(what, 0, False)):
                        dst.copy_(src, non_blocking=True)
                if has_hi:      # my high face -> high neighbour's low ghost
                    for dst, src in zip(self.ports[hi].halo_views(what, 0, True), port.halo_views(what, 1, False)):
                        dst.copy_(src, non_blocking=True)
            return works
        import torch.distributed as dist
        (r, port), = self.ports.items()
        has_lo, has_hi, lo, hi = self._faces(r)
        peer = (lambda k: dist.get_global_rank(self.group, k)) if self.group is not None else (lambda k: k)
        ops = []
        if has_lo:
            ops += [dist.P2POp(dist.isend, t, peer(lo), self.group) for t in port.halo_views(what, 0, False)]
        if has_hi:
            ops += [dist.P2POp(dist.isend, t, peer(hi), self.group) for t in port.halo_views(what, 1, False)]
        if has_hi:
            ops += [dist.P2POp(dist.irecv, t, peer(hi), self.group) for t in port.halo_views(what, 1, True)]
        if has_lo:
            ops += [dist.P2POp(dist.irecv, t, peer(lo), self.group) for t in port.halo_views(what, 0, True)]
        if ops:
            works = dist.batch_isend_irecv(ops)
        return works

    @staticmethod
    def finish(works):
        for w in works:
            w.wait()


class SlabRunner:
    """Advances the slabs held by this process with the overlapped schedule of the module docstring.

    single process:  SlabRunner.local(p, nranks)            all slabs on one GPU (testing, memory studies)
    distributed:     SlabRunner.distributed(p, rank, world) one slab per process / GPU, torch.distributed
    """

    def __init__(self, slabs: Sequence[SlabACM], nranks: int, wall_z: bool, group=None, overlap: Optional[bool] = None):
        self.slabs = list(slabs)
        self.nranks = nranks
        self.ex = HaloExchanger(self.slabs, nranks, wall_z, group)
        dev = self.slabs[0].device
        self.compute = self.slabs[0].stream
        # overlap: the exchanges run on a second stream behind events (default for the distributed run; local
        # copies between slabs of one process are ordered by the one compute stream unless it is asked for)
        if overlap is None:
            overlap = not self.ex.local_only
        self.comm = torch.cuda.Stream(dev) if overlap else None
        self._ev_h = self._ev_g = None
        self.steps = 0

    @classmethod
    def local(cls, p, nranks: int, precision="f64", device="cuda:0", overlap: Optional[bool] = None):
        slabs = [SlabACM(p, r, nranks, precision, device) for r in range(nranks)]
        return cls(slabs, nranks, bool(p.wall_flags & binding.ACM_WALL_Z), None, overlap)

    @classmethod
    def distributed(cls, p, rank: int, world: int, precision="f64", device="cuda:0", group=None, overlap: Optional[bool] = None):
        return cls([SlabACM(p, rank, world, precision, device)], world, bool(p.wall_flags & binding.ACM_WALL_Z), group, overlap)

    # ---- exchange helpers -------------------------------------------------------------------------
    def _exchange_now(self, stages):
        """blocking (stream-ordered) exchange on the compute stream"""
        for what in stages:
            HaloExchanger.finish(self.ex.exchange(what))

    def _exchange_async(self, stages):
        """exchange on the comm stream after everything enqueued on the compute stream so far; returns one
        event per stage that the compute stream can wait for"""
        start = torch.cuda.Event()
        start.record(self.compute)
        events = []
        with torch.cuda.stream(self.comm):
            self.comm.wait_event(start)
            for what in stages:
                HaloExchanger.finish(self.ex.exchange(what))      # work.wait() orders the comm stream, not the host
                ev = torch.cuda.Event()
                ev.record(self.comm)
                events.append(ev)
        return events

    # ---- life cycle ---------------------------------------------------------------------------------
    def init(self, phi_global: torch.Tensor, u_global: torch.Tensor):
        """phi_global (nz, ny, nx), u_global (3, nz, ny, nx): device tensors of the GLOBAL fields; every slab
        takes its planes plus one ghost plane on each side."""
        for s in self.slabs:
            s.init(pad_planes(phi_global, s.z0, s.nzl).to(s.dtype), pad_planes(u_global, s.z0, s.nzl).to(s.dtype))
        self.refresh_halos()

    def refresh_halos(self):
        """ghost planes of h, g and phi from the neighbours (after init / set_pdfs)"""
        self._exchange_now((HALO_PHI, HALO_H, HALO_G))
        self._ev_h = self._ev_g = None

    def step(self, n: int = 1):
        for _ in range(int(n)):
            if self._ev_h is not None:
                self.compute.wait_event(self._ev_h)               # h ghosts of the previous step
            for s in self.slabs:
                s.phase_launch(0, s.nzl)
                s.phase_commit()
            if self.comm is None:
                self._exchange_now((HALO_PHI, HALO_H))
                ev_phi = None
            else:
                ev_phi, self._ev_h = self._exchange_async((HALO_PHI, HALO_H))
            for s in self.slabs:
                if s.nzl > 2:
                    s.hydro_launch(1, s.nzl - 1)                  # inner planes read no ghost plane
            if ev_phi is not None:
                self.compute.wait_event(ev_phi)
            if self._ev_g is not None:
                self.compute.wait_event(self._ev_g)               # g ghosts of the previous step
            for s in self.slabs:
                s.hydro_launch(0, min(1, s.nzl))
                if s.nzl > 1:
                    s.hydro_launch(s.nzl - 1, s.nzl)
                s.hydro_commit()
            if self.comm is None:
                self._exchange_now((HALO_G,))
            else:
                self._ev_g, = self._exchange_async((HALO_G,))
            self.steps += 1

    def sync_halos(self):
        """make the compute stream wait for the outstanding exchanges (before reading fields / populations)"""
        for ev in (self._ev_h, self._ev_g):
            if ev is not None:
                self.compute.wait_event(ev)

    # ---- results (owned planes of the local slabs, in rank order) -------------------------------------
    def fields(self, want_p=True):
        self.sync_halos()
        out = [s.fields(want_p) for s in self.slabs]
        cat = lambda k: None if out[0][k] is None else torch.cat([s.owned(o[k]) for s, o in zip(self.slabs, out)], dim=-3)
        return cat(0), cat(1), cat(2)

    def get_pdfs(self):
        self.sync_halos()
        out = [s.get_pdfs() for s in self.slabs]
        return tuple(torch.cat([s.owned(o[k]) for s, o in zip(self.slabs, out)], dim=-3) for k in (0, 1))

    def set_pdfs(self, h_global, g_global):
        """GLOBAL population arrays (Q, nz, ny, nx) in the ABI's conventions"""
        for s in self.slabs:
            s.set_pdfs(pad_planes(h_global, s.z0, s.nzl), pad_planes(g_global, s.z0, s.nzl))
        self.refresh_halos()

    def phi_mass_local(self):
        return sum(s.phi_mass() for s in self.slabs)

    def bubble_sums_local(self):
        tot = [0.0] * 7
        for s in self.slabs:
            tot = [a + b for a, b in zip(tot, s.bubble_sums())]
        return tot


class PeerSlabRunner(SlabRunner):
    """Slabs in PEER MODE (acm_set_peers): the LB kernels read the neighbour slabs' boundary planes straight from
    the neighbours' workspaces -- the same GPU, or a peer GPU's memory mapped over NVLink (CUDA IPC) -- so a step is
    just  phase kernel, signal, hydro kernel, signal  with no halo copies, no pack / unpack and no inner / outer
    split; what crosses NVLink per step are the loads of the 5 + 5 (+ 2 phi) boundary planes themselves.

    `peer_ws[r]` = (uint8 tensor over slab r's workspace allocation, byte offset of its 256-byte-aligned base) for
    the neighbours of the local slabs; `sync()` must order kernel n of every rank after kernel n-1 of its
    neighbours (nothing to do when all slabs share one stream).  Slabs must have equal heights.
    """

    def __init__(self, slabs, nranks, wall_z, peer_ws, sync=None, group=None):
        super().__init__(slabs, nranks, wall_z, group, overlap=False)
        self.peer_ws = dict(peer_ws)
        self.sync = sync if sync is not None else (lambda: None)
        self._wall_z = wall_z
        for s in self.slabs:
            lo, hi = self._neighbours(s.rank)
            s._call(s._lib.acm_set_peers, self._ptr(lo), self._ptr(hi))
        self.check_consistency()

    def check_consistency(self):
        """A slab reads its neighbours' arrays at its OWN offsets and buffer parity (peers_at in acm.cu): layout,
        current buffers, step count, slab height and fp32 reference phase must agree on all ranks.  Compared
        across the local slabs and, for one slab per process, across the group (host-side all_gather)."""
        sigs = {s.rank: s.state_signature() for s in self.slabs}
        if not self.ex.local_only:
            import torch.distributed as dist
            gathered = [None] * self.nranks
            dist.all_gather_object(gathered, sigs, group=self.ex.group)
            sigs = {r: v for d in gathered for r, v in d.items()}
        ref = next(iter(sigs.values()))
        bad = {r: v for r, v in sigs.items() if v != ref}
        if bad or ref[6]:
            raise RuntimeError(f"peer mode: the slabs are out of step (workspace bytes, offsets of the current h/g/phi, steps, "
                               f"planes, partly launched, reference phase): {sigs}")

    def _neighbours(self, r):
        lo = None if (self._wall_z and r == 0) else (r - 1) % self.nranks
        hi = None if (self._wall_z and r == self.nranks - 1) else (r + 1) % self.nranks
        return lo, hi

    def _ptr(self, r):
        if r is None:
            return None
        t, base = self.peer_ws[r]
        return C.c_void_p(t.data_ptr() + base)

    @classmethod
    def local(cls, p, nranks: int, precision="f64", device="cuda:0"):
        slabs = [SlabACM(p, r, nranks, precision, device) for r in range(nranks)]
        return cls(slabs, nranks, bool(p.wall_flags & binding.ACM_WALL_Z), {s.rank: (s.workspace, s.base) for s in slabs})

    @classmethod
    def distributed(cls, p, rank: int, world: int, precision="f64", device="cuda:0", group=None, sync=None):
        """One slab per process.  The workspaces are shared through CUDA IPC (torch's own tensor sharing), gathered
        with all_gather_object; default `sync`: a one-element all-reduce on the compute stream (NCCL), which makes
        every rank's next kernel wait for all ranks' previous kernel without blocking the host."""
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        slab = SlabACM(p, rank, world, precision, device)
        mine = (reduce_tensor(slab.workspace), slab.base)
        gathered = [None] * world
        dist.all_gather_object(gathered, mine, group=group)
        peer_ws = {rank: (slab.workspace, slab.base)}
        for r in {(rank - 1) % world, (rank + 1) % world} - {rank}:
            (rebuild, args), base = gathered[r]
            peer_ws[r] = (rebuild(*args), base)
        if sync is None:
            token = torch.zeros(1, device=device)

            def sync():
                dist.all_reduce(token, group=group)
        return cls([slab], world, bool(p.wall_flags & binding.ACM_WALL_Z), peer_ws, sync, group)

    # ---- a step: two kernels, two signals -----------------------------------------------------------------------
    def step(self, n: int = 1):
        for _ in range(int(n)):
            for s in self.slabs:
                s.phase_launch(0, s.nzl)
                s.phase_commit()
            self.sync()
            for s in self.slabs:
                s.hydro_launch(0, s.nzl)
                s.hydro_commit()
            self.sync()
            self.steps += 1

    def init(self, phi_global, u_global):
        super().init(phi_global, u_global)
        self.check_consistency()

    def refresh_halos(self):
        """Ghost planes are not used for stepping in peer mode; the exports (acm_get_pdfs, pressure) still read them:
        pull them from the neighbours' workspaces.  Equal layouts: the neighbour's planes sit at the offsets of this
        slab's own plan for the opposite face."""
        self.check_consistency()
        self.sync()
        for s in self.slabs:
            lo, hi = self._neighbours(s.rank)
            for what in (HALO_PHI, HALO_H, HALO_G):
                for nb, my_side, nb_side in ((lo, 0, 1), (hi, 1, 0)):
                    if nb is None:
                        continue
                    t, base = self.peer_ws[nb]
                    for dst, (off, nbytes) in zip(s.halo_views(what, my_side, True), halo_plan(s._lib, s._h, what, nb_side, False)):
                        dst.copy_(t[base + off: base + off + nbytes], non_blocking=True)
        self.sync()

    def sync_halos(self):
        self.refresh_halos()
