"""Algorithm 1 (six unfused kernels, ACM_OPT_UNFUSED) against the same oracle and at the same
bars as the fused path: 1e-13 on populations after one step, 1e-10 on fields after 100 steps.  It is a
measured comparison for the paper's fusion claim, so it must compute the same thing."""
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


@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls,srt", [
    (150, 7, 5, 15, 19, 0, False), (70, 9, 6, 15, 27, inputs.WALL_Y, True),
    (37, 6, 11, 27, 27, inputs.WALL_X | inputs.WALL_Z, False), (128, 4, 3, 19, 19, inputs.WALL_X | inputs.WALL_Y | inputs.WALL_Z, False)])
def test_unfused_steps_match_oracle(nx, ny, nz, Qh, Qg, walls, srt):
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -1e-5, 2e-5),
               nu_H=0.02, nu_L=0.05, phase_srt=srt)
    phi, u, h, g = random_state(p, seed=31)
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, unfused=True)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    n0 = a.launch_count
    for k in range(3):          # three steps: both u buffers, both grids
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


def test_unfused_launches_six_kernels_per_step():
    p, phi, u = inputs.scaled_config3(24)
    a = _acm(p, unfused=True)
    a.init(_dev(phi), _dev(u))
    n0 = a.launch_count
    a.step(5)
    assert a.launch_count - n0 == 30
    b = _acm(p)
    b.init(_dev(phi), _dev(u))
    n0 = b.launch_count
    b.step(5)
    assert b.launch_count - n0 == 10


def test_unfused_config3_scaled_100_steps_and_equals_fused():
    p, phi, u = inputs.scaled_config3(40)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p, unfused=True)
    a.init(_dev(phi), _dev(u))
    f = _acm(p)
    f.init(_dev(phi), _dev(u))
    m0 = a.phi_mass()
    o.step(100)
    a.step(100)
    f.step(100)
    po, uo, pro = o.fields()
    pa, ua, pra = a.fields()
    pf, uf, _ = f.fields()
    assert np.abs(pa.cpu().numpy() - po).max() <= 1e-10
    assert np.abs(ua.cpu().numpy() - uo).max() <= 1e-10
    assert np.abs(pra.cpu().numpy() - pro).max() <= 1e-10
    assert float((pa - pf).abs().max()) <= 1e-12 and float((ua - uf).abs().max()) <= 1e-12
    assert abs(a.phi_mass() - m0) / m0 < 1e-12


def test_unfused_fp32_and_option_checks():
    from paper_2012_06144_b200.binding import AcmError, ACM_EINVAL
    p = Params(nx=70, ny=9, nz=6, stencil_phase=27, stencil_hydro=27)
    with pytest.raises(AcmError) as e:
        _acm(p, unfused=True, inplace=True)
    assert e.value.code == ACM_EINVAL
    phi, u, h, g = random_state(p, seed=4)
    phi, u, h, g = (np.asarray(x, dtype=np.float32).astype(np.float64) for x in (phi, u, h, g))
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, unfused=True, precision="f32")
    a.init(_dev(phi, np.float32), _dev(u, np.float32))
    a.set_pdfs(_dev(h, np.float32), _dev(g, np.float32))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    assert np.abs(ha.cpu().numpy() - ho).max() < 3e-7
    assert np.abs(ga.cpu().numpy() - go).max() < 2e-7
