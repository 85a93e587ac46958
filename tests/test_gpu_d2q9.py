"""Two-dimensional instance (D2Q9 for both LB steps, nz = 1; paper Fig. 5) against the oracle, at the bars
of the 3-D path: 1e-13 on populations after one step, 1e-10 on fields after 100 steps."""
import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu


def _acm(p, **kw):
    from paper_2012_06144_b200.binding import ACM
    return ACM.from_params(p, **kw)


def _dev(a, dtype=np.float64):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


@pytest.mark.parametrize("mode", [dict(), dict(inplace=True), dict(unfused=True)])
@pytest.mark.parametrize("nx,ny,walls,srt", [(150, 37, 0, False), (70, 9, inputs.WALL_Y, True), (33, 20, inputs.WALL_X | inputs.WALL_Y, False),
                                             (256, 3, 0, False)])
def test_d2q9_steps(nx, ny, walls, srt, mode):
    p = Params(nx=nx, ny=ny, nz=1, stencil_phase=9, stencil_hydro=9, wall_flags=walls, gravity=(1e-5, -1e-5, 0.0),
               nu_H=0.02, nu_L=0.05, phase_srt=srt)
    phi, u, h, g = random_state(p, seed=51)
    u[2] = 0.0
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, **mode)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    for _ in range(2):
        o.step(1)
        a.step(1)
        ho, go = o.get_pdfs()
        ha, ga = a.get_pdfs()
        po, uo, pro = o.fields()
        pa, ua, pra = a.fields()
        assert np.abs(ha.cpu().numpy() - ho).max() <= 1e-13
        assert np.abs(ga.cpu().numpy() - go).max() <= 1e-13
        assert np.abs(pa.cpu().numpy() - po).max() <= 1e-13
        assert np.abs(ua.cpu().numpy() - uo).max() <= 1e-13
        assert np.abs(pra.cpu().numpy() - pro).max() <= 1e-13
        assert float(ua[2].abs().max()) == 0.0


def test_d2q9_discs_100_steps_init_and_mass():
    p, phi, u = inputs.disc2d(n=96, count=5, r_min=6.0, r_max=12.0)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    h0o, g0o = o.get_pdfs()
    h0a, g0a = a.get_pdfs()
    assert np.abs(h0a.cpu().numpy() - h0o).max() <= 1e-15 and np.abs(g0a.cpu().numpy() - g0o).max() <= 1e-15
    m0 = a.phi_mass()
    o.step(100)
    a.step(100)
    po, uo, pro = o.fields()
    pa, ua, pra = a.fields()
    assert np.abs(pa.cpu().numpy() - po).max() <= 1e-10
    assert np.abs(ua.cpu().numpy() - uo).max() <= 1e-10
    assert np.abs(pra.cpu().numpy() - pro).max() <= 1e-10
    assert abs(a.phi_mass() - m0) / m0 < 1e-12


def test_d2q9_fp32_and_argument_checks():
    from paper_2012_06144_b200.binding import ACM, AcmError, ACM_EINVAL
    for bad in (dict(nz=2), dict(stencil_hydro=19), dict(gravity=(0.0, 0.0, 1e-6))):
        kw = dict(nx=16, ny=8, nz=1, stencil_phase=9, stencil_hydro=9)
        kw.update(bad)
        with pytest.raises(AcmError) as e:
            ACM(**kw)
        assert e.value.code == ACM_EINVAL
    p = Params(nx=70, ny=40, nz=1, stencil_phase=9, stencil_hydro=9, wall_flags=inputs.WALL_Y)
    phi, u, h, g = random_state(p, seed=4)
    u[2] = 0.0
    phi, u, h, g = (np.asarray(x, dtype=np.float32).astype(np.float64) for x in (phi, u, h, g))
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, precision="f32")
    a.init(_dev(phi, np.float32), _dev(u, np.float32))
    a.set_pdfs(_dev(h, np.float32), _dev(g, np.float32))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    assert np.abs(ha.cpu().numpy() - ho).max() < 3e-7
    assert np.abs(ga.cpu().numpy() - go).max() < 2e-7
