"""The two-cells-per-thread LB kernels (pair.cuh, vec2.cuh: 8 / 16-byte accesses, packed fp32 arithmetic) and the
single-cell kernels against the oracle, selected explicitly with acm_set_cells_per_thread -- the library's default
picks one or the other by precision, lattice and the parity of nx, so both are forced here on the same grids.
Bars as in test_gpu_parity.py / test_gpu_fp32.py."""
import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu

TOL_PDF_1STEP = 1e-13
TOL_FIELD_100 = 1e-10


def _acm(p, cpt, **kw):
    from paper_2012_06144_b200.binding import ACM
    a = ACM.from_params(p, **kw)
    a.set_cells_per_thread(*cpt)
    return a


def _dev(a, dtype=np.float64):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


GRIDS = [
    # nx (even), ny, nz, Qh, Qg, walls, block
    (150, 7, 5, 15, 19, 0, None),                                              # 75 pairs per row: one ragged block
    (70, 9, 6, 15, 19, inputs.WALL_Y, (32, 2, 2)),
    (36, 6, 11, 27, 27, inputs.WALL_X | inputs.WALL_Z, (16, 4, 2)),             # x walls: per-cell bounce-back flags inside a pair
    (260, 5, 4, 19, 27, inputs.WALL_X, None),                                  # 130 pairs: linear launch
    (20, 12, 9, 27, 19, inputs.WALL_X | inputs.WALL_Y | inputs.WALL_Z, (8, 2, 1)),
    (2, 6, 5, 15, 19, 0, None),                                                # one pair per row: both x neighbours wrap onto the pair itself
    (64, 10, 1, 9, 9, inputs.WALL_Y, None),                                    # D2Q9
]


@pytest.mark.parametrize("cpt", [(1, 1), (2, 2), (2, 1)])
@pytest.mark.parametrize("opts", [dict(), dict(inplace=True), dict(phase_srt=True), dict(bulk_one=True, subiter=2)])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls,block", GRIDS)
def test_one_step_fp64(nx, ny, nz, Qh, Qg, walls, block, opts, cpt):
    grav = (1e-5, -1e-5, 0.0 if nz == 1 else 2e-5)
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=grav, rho_L=0.05, sigma=2e-3,
               nu_H=0.05, nu_L=0.2)
    phi, u, h, g = random_state(p, seed=31)
    if nz == 1:
        u[2] = 0.0
    okw = {k: v for k, v in opts.items() if k != "inplace"}
    o = Oracle.from_params(p, **okw)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, cpt, **opts)
    if block:
        a.set_block(*block)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    for _ in range(2):          # two steps: both kernels of the in-place pattern
        o.step(1)
        a.step(1)
        ho, go = o.get_pdfs()
        ha, ga = a.get_pdfs()
        po, uo, pro = o.fields()
        pa, ua, pra = a.fields()
        assert np.abs(ha.cpu().numpy() - ho).max() <= TOL_PDF_1STEP
        assert np.abs(ga.cpu().numpy() - go).max() <= TOL_PDF_1STEP
        assert np.abs(pa.cpu().numpy() - po).max() <= TOL_PDF_1STEP
        assert np.abs(ua.cpu().numpy() - uo).max() <= TOL_PDF_1STEP
        assert np.abs(pra.cpu().numpy() - pro).max() <= TOL_PDF_1STEP


@pytest.mark.parametrize("cpt", [(1, 1), (2, 2)])
@pytest.mark.parametrize("Qh,Qg", [(15, 19), (27, 27)])
def test_100_steps_fp64(Qh, Qg, cpt):
    p, phi, u = inputs.scaled_config3(40, stencil_phase=Qh, stencil_hydro=Qg)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p, cpt)
    a.init(_dev(phi), _dev(u))
    m0 = a.phi_mass()
    o.step(100)
    a.step(100)
    po, uo, pro = o.fields()
    pa, ua, pra = a.fields()
    assert np.abs(pa.cpu().numpy() - po).max() <= TOL_FIELD_100
    assert np.abs(ua.cpu().numpy() - uo).max() <= TOL_FIELD_100
    assert np.abs(pra.cpu().numpy() - pro).max() <= TOL_FIELD_100
    assert abs(a.phi_mass() - m0) / m0 < 1e-12


@pytest.mark.parametrize("cpt", [(1, 1), (2, 2), (1, 2)])
@pytest.mark.parametrize("opts", [dict(), dict(inplace=True), dict(phase_srt=True)])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls,block", GRIDS[:5])
def test_one_step_fp32(nx, ny, nz, Qh, Qg, walls, block, opts, cpt):
    """fp32 instance from an fp32-representable state against the fp64 oracle (bars of test_gpu_fp32.py)."""
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -1e-5, 2e-5))
    phi, u, h, g = [np.asarray(x, dtype=np.float32) for x in random_state(p, seed=7)]
    o = Oracle.from_params(p, phase_srt=opts.get("phase_srt", False))
    o.init(phi.astype(np.float64), u.astype(np.float64))
    o.set_pdfs(h.astype(np.float64), g.astype(np.float64))
    a = _acm(p, cpt, precision="f32", **opts)
    if block:
        a.set_block(*block)
    a.init(_dev(phi, np.float32), _dev(u, np.float32))
    a.set_pdfs(_dev(h, np.float32), _dev(g, np.float32))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    po, uo, _ = o.fields(False)
    pa, ua, _ = a.fields(False)
    # populations up to 0.11: ulp/2 = 3.7e-9 per rounding; the SRT form adds (1 - omega) h_i to the six-term sum: a few more
    tol_h = 1e-7 if opts.get("phase_srt") else 5e-8
    assert np.abs(ga.cpu().numpy().astype(np.float64) - go).max() <= 5e-8
    assert np.abs(ha.cpu().numpy().astype(np.float64)[1:] - ho[1:]).max() <= tol_h
    assert np.abs(ha.cpu().numpy().astype(np.float64)[0] - ho[0]).max() <= 4e-7      # rest population by subtraction: Q - 1 roundings
    assert np.abs(pa.cpu().numpy().astype(np.float64) - po).max() <= 5e-7
    assert np.abs(ua.cpu().numpy().astype(np.float64) - uo).max() <= 2e-6          # F/(2 rho) with rho down to 1e-3


def test_default_rule_and_argument_checks():
    from paper_2012_06144_b200 import binding
    from paper_2012_06144_b200.binding import ACM
    p = Params(nx=33, ny=4, nz=4)
    a = ACM.from_params(p)
    assert a._lib.acm_set_cells_per_thread(a._h, 2, 2) == binding.ACM_EINVAL          # odd nx
    assert a._lib.acm_set_cells_per_thread(a._h, 1, 0) == binding.ACM_OK
    assert a._lib.acm_set_cells_per_thread(a._h, 3, 1) == binding.ACM_EINVAL
    b = ACM.from_params(Params(nx=32, ny=4, nz=4), unfused=True)
    assert b._lib.acm_set_cells_per_thread(b._h, 2, 2) == binding.ACM_EINVAL          # Algorithm 1 has single-cell kernels only


def test_pair_against_single_cell_on_seeded_random_shapes():
    """Differential check on 16 seeded random grids / lattices / walls / options / blocks: the pair kernels against the
    single-cell kernels over 3 steps (both are tied to the oracle above; this sweeps shapes no table lists)."""
    rng = np.random.Generator(np.random.PCG64(2012))
    for case in range(16):
        nx = 2 * int(rng.integers(1, 90))
        ny, nz = int(rng.integers(1, 9)), int(rng.integers(1, 9))
        Qh, Qg = int(rng.choice([15, 19, 27])), int(rng.choice([15, 19, 27]))
        walls = int(rng.integers(0, 8))
        opts = dict(inplace=bool(rng.integers(0, 2)), phase_srt=bool(rng.integers(0, 2)), bulk_one=bool(rng.integers(0, 2)),
                    subiter=int(rng.integers(1, 4)))
        bx = int(rng.choice([8, 32, 64, 128]))
        by = int(rng.choice([1, 2]))
        p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -2e-5, 1e-5),
                   rho_L=0.05, sigma=2e-3, nu_H=0.05, nu_L=0.2)
        phi, u, h, g = random_state(p, seed=100 + case)
        out = []
        for cpt in ((1, 1), (2, 2)):
            a = _acm(p, cpt, **opts)
            a.set_block(bx, by, 1)
            a.init(_dev(phi), _dev(u))
            a.set_pdfs(_dev(h), _dev(g))
            a.step(3)
            out.append(a.get_pdfs() + a.fields())
        for x, y in zip(*out):
            assert float((x - y).abs().max()) <= 3 * TOL_PDF_1STEP, (case, nx, ny, nz, Qh, Qg, walls, opts, bx, by)
