"""Slab decomposition on ONE GPU: all slabs of a z-decomposed domain live in one process, their halo planes
travel by device copies through the same plan / exchanger / schedule code as the distributed run
(paper_2012_06144_b200/slab.py).  The decomposed run must reproduce the oracle at the bars of the
single-domain path, and the single-domain CUDA path bit for bit (same kernels, same arithmetic per cell).
The launches are sequential on one stream: no rank waits on another."""
import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _runner(p, nranks, **kw):
    from paper_2012_06144_b200.slab import SlabRunner
    return SlabRunner.local(p, nranks, **kw)


def _acm(p, **kw):
    from paper_2012_06144_b200.binding import ACM
    return ACM.from_params(p, **kw)


@pytest.mark.parametrize("nranks", [1, 2, 3, 5])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls", [(70, 6, 11, 15, 19, 0), (33, 5, 10, 27, 27, inputs.WALL_Y),
                                                  (40, 4, 9, 19, 27, inputs.WALL_Z | inputs.WALL_X), (128, 3, 7, 15, 15, 0)])
def test_slab_steps_match_oracle_and_single_domain(nx, ny, nz, Qh, Qg, walls, nranks):
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -1e-5, 2e-5),
               nu_H=0.02, nu_L=0.05)
    phi, u, h, g = random_state(p, seed=41)
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    r = _runner(p, nranks)
    r.init(_dev(phi), _dev(u))
    r.set_pdfs(_dev(h), _dev(g))
    for _ in range(3):
        o.step(1)
        a.step(1)
        r.step(1)
        ho, go = o.get_pdfs()
        hr, gr = r.get_pdfs()
        ha, ga = a.get_pdfs()
        po, uo, pro = o.fields()
        pr, ur, prr = r.fields()
        pa, ua, pra = a.fields()
        assert np.abs(hr.cpu().numpy() - ho).max() <= 1e-13
        assert np.abs(gr.cpu().numpy() - go).max() <= 1e-13
        assert np.abs(pr.cpu().numpy() - po).max() <= 1e-13
        assert np.abs(ur.cpu().numpy() - uo).max() <= 1e-13
        assert np.abs(prr.cpu().numpy() - pro).max() <= 1e-13
        for x, y in ((hr, ha), (gr, ga), (pr, pa), (ur, ua), (prr, pra)):
            assert torch.equal(x, y)


def test_slab_init_matches_single_domain():
    """equilibrium initialiser on slabs (the pre-shifted g needs u of the neighbour planes)"""
    p, phi, u = inputs.scaled_config3(24)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    r = _runner(p, 3)
    r.init(_dev(phi), _dev(u))
    for x, y in zip(r.get_pdfs() + r.fields(), a.get_pdfs() + a.fields()):
        assert torch.equal(x, y)
    assert abs(r.phi_mass_local() - a.phi_mass()) <= 1e-9


@pytest.mark.parametrize("overlap", [False, True])
def test_slab_config3_scaled_100_steps(overlap):
    """overlap=True runs the exchanges on the second stream behind the events of the distributed schedule"""
    p, phi, u = inputs.scaled_config3(40)
    o = Oracle.from_params(p)
    o.init(phi, u)
    r = _runner(p, 4, overlap=overlap)
    r.init(_dev(phi), _dev(u))
    m0 = r.phi_mass_local()
    o.step(100)
    r.step(100)
    po, uo, pro = o.fields()
    pr, ur, prr = r.fields()
    assert np.abs(pr.cpu().numpy() - po).max() <= 1e-10
    assert np.abs(ur.cpu().numpy() - uo).max() <= 1e-10
    assert np.abs(prr.cpu().numpy() - pro).max() <= 1e-10
    assert abs(r.phi_mass_local() - m0) / m0 < 1e-12


def test_slab_walls_in_z_gravity_40_steps_and_diagnostics():
    """config-2-like set-up turned so that the walls are the faces the decomposition cuts across"""
    p = Params(nx=24, ny=24, nz=48, gravity=(0.0, 0.0, -1e-6), wall_flags=inputs.WALL_Z)
    phi = inputs.sphere_phi(p, (12.0, 12.0, 14.0), 6.0, heavy_inside=False)
    u = inputs.zeros_u(p)
    o = Oracle.from_params(p)
    o.init(phi, u)
    r = _runner(p, 3)
    r.init(_dev(phi), _dev(u))
    o.step(40)
    r.step(40)
    po, uo, _ = o.fields(False)
    pr, ur, _ = r.fields(False)
    assert np.abs(pr.cpu().numpy() - po).max() <= 1e-10
    assert np.abs(ur.cpu().numpy() - uo).max() <= 1e-10
    s = r.bubble_sums_local()
    Vo, Xo, Uo = o.bubble_diag()
    assert abs(s[0] / Vo - 1) < 1e-12
    assert np.abs(np.array(s[1:4]) / s[0] - Xo).max() < 1e-10          # z in global coordinates
    assert np.abs(np.array(s[4:7]) / s[0] - Uo).max() < 1e-12


def test_slab_fp32_and_state_errors():
    from paper_2012_06144_b200.binding import AcmError, ACM_ESTATE
    p = Params(nx=40, ny=6, nz=9, stencil_phase=27, stencil_hydro=27)
    phi, u, h, g = random_state(p, seed=4)
    phi, u, h, g = (np.asarray(x, dtype=np.float32) for x in (phi, u, h, g))
    a = _acm(p, precision="f32")
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    r = _runner(p, 2, precision="f32")
    r.init(_dev(phi), _dev(u))
    r.set_pdfs(_dev(h), _dev(g))
    a.step(3)
    r.step(3)
    for x, y in zip(r.get_pdfs(), a.get_pdfs()):
        assert torch.equal(x, y)
    with pytest.raises(AcmError) as e:
        r.slabs[0].step(1)
    assert e.value.code == ACM_ESTATE


# ------------------------------------------------------------------------------------------------------------
# peer mode: the kernels read the neighbour slabs' boundary planes directly (acm_set_peers), no halo copies
# ------------------------------------------------------------------------------------------------------------
def _peer_runner(p, nranks, **kw):
    from paper_2012_06144_b200.slab import PeerSlabRunner
    return PeerSlabRunner.local(p, nranks, **kw)


@pytest.mark.parametrize("nranks", [1, 2, 3, 4])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls,srt", [(70, 6, 12, 15, 19, 0, False), (33, 5, 12, 27, 27, inputs.WALL_Y, True),
                                                      (40, 4, 12, 19, 27, inputs.WALL_Z | inputs.WALL_X, False), (128, 3, 24, 15, 15, 0, False)])
def test_peer_mode_steps_match_oracle_and_single_domain(nx, ny, nz, Qh, Qg, walls, srt, nranks):
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -1e-5, 2e-5),
               nu_H=0.02, nu_L=0.05, phase_srt=srt)
    phi, u, h, g = random_state(p, seed=43)
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    r = _peer_runner(p, nranks)
    r.init(_dev(phi), _dev(u))
    r.set_pdfs(_dev(h), _dev(g))
    for _ in range(3):
        o.step(1)
        a.step(1)
        r.step(1)
        ho, go = o.get_pdfs()
        hr, gr = r.get_pdfs()
        ha, ga = a.get_pdfs()
        po, uo, pro = o.fields()
        pr, ur, prr = r.fields()
        pa, ua, pra = a.fields()
        assert np.abs(hr.cpu().numpy() - ho).max() <= 1e-13
        assert np.abs(gr.cpu().numpy() - go).max() <= 1e-13
        assert np.abs(ur.cpu().numpy() - uo).max() <= 1e-13
        assert np.abs(prr.cpu().numpy() - pro).max() <= 1e-13
        for x, y in ((hr, ha), (gr, ga), (pr, pa), (ur, ua), (prr, pra)):
            assert torch.equal(x, y)


def test_peer_mode_never_reads_ghost_planes_while_stepping():
    """poison the ghost planes of every array: the steps must not notice (ghosts are only refreshed for the exports)"""
    p, phi, u = inputs.scaled_config3(24)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    r = _peer_runner(p, 3)
    r.init(_dev(phi), _dev(u))
    from paper_2012_06144_b200.slab import HALO_G, HALO_H, HALO_PHI
    for k in range(4):
        for s in r.slabs:
            for what in (HALO_PHI, HALO_H, HALO_G):
                for side in (0, 1):
                    for v in s.halo_views(what, side, True):
                        v.view(torch.float64).fill_(float("nan"))
        r.step(1)
        a.step(1)
    for x, y in zip(r.get_pdfs() + r.fields(), a.get_pdfs() + a.fields()):
        assert torch.equal(x, y)


def test_peer_mode_100_steps_fp32_and_argument_checks():
    from paper_2012_06144_b200.binding import AcmError, ACM_EINVAL
    from paper_2012_06144_b200.slab import PeerSlabRunner
    p = Params(nx=40, ny=6, nz=10, stencil_phase=27, stencil_hydro=27)
    with pytest.raises(AcmError) as e:
        PeerSlabRunner.local(p, 3)                       # 10 planes over 3 slabs: unequal heights
    assert e.value.code == ACM_EINVAL
    p, phi, u = inputs.scaled_config3(40)
    o = Oracle.from_params(p)
    o.init(phi, u)
    r = _peer_runner(p, 4)
    r.init(_dev(phi), _dev(u))
    m0 = r.phi_mass_local()
    o.step(100)
    r.step(100)
    po, uo, pro = o.fields()
    pr, ur, prr = r.fields()
    assert np.abs(pr.cpu().numpy() - po).max() <= 1e-10
    assert np.abs(ur.cpu().numpy() - uo).max() <= 1e-10
    assert abs(r.phi_mass_local() - m0) / m0 < 1e-12
    # fp32 slabs in peer mode against the fp32 single domain (reference phase: heavy for slabs; force the same)
    q = Params(nx=40, ny=6, nz=8, stencil_phase=15, stencil_hydro=19)
    phi, u, h, g = random_state(q, seed=4)
    phi, u, h, g = (np.asarray(x, dtype=np.float32) for x in (phi, u, h, g))
    a = _acm(q, precision="f32")
    a.set_reference_phase(1)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    r = _peer_runner(q, 2, precision="f32")
    r.init(_dev(phi), _dev(u))
    r.set_pdfs(_dev(h), _dev(g))
    a.step(3)
    r.step(3)
    for x, y in zip(r.get_pdfs(), a.get_pdfs()):
        assert torch.equal(x, y)
