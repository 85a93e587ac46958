"""CUDA path vs oracle for the operator variants and diagnostics of SURVEY.md 8(f)-2:
SRT phase-field collision (ACM_OPT_PHASE_SRT), the viscosity contrast mu* = 100 of section 6
(nu_H != nu_L, eq. 20), and the rising-bubble diagnostics (acm_bubble_diag, A24).  Same bars as
test_gpu_parity.py: 1e-13 on populations after one step, 1e-10 on fields after 100 steps."""
import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from oracle import oracle as om
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu

TOL_PDF_1STEP = 1e-13
TOL_FIELD_100 = 1e-10


def _acm(p, **kw):
    from paper_2012_06144_b200.binding import ACM
    return ACM.from_params(p, **kw)


def _dev(a, dtype=np.float64):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls", [(150, 7, 5, 15, 27, 0), (70, 9, 6, 15, 19, inputs.WALL_Y),
                                                  (37, 6, 11, 27, 27, inputs.WALL_X | inputs.WALL_Z), (33, 5, 4, 19, 19, 0)])
def test_srt_one_step(nx, ny, nz, Qh, Qg, walls, inplace):
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(1e-5, -1e-5, 0.0))
    phi, u, h, g = random_state(p, seed=21)
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, phase_srt=True, inplace=inplace)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    for _ in range(2):          # two steps: both kernels of the in-place pattern
        o.step(1)
        a.step(1)
        ho, go = o.get_pdfs()
        ha, ga = a.get_pdfs()
        assert np.abs(ha.cpu().numpy() - ho).max() <= TOL_PDF_1STEP
        assert np.abs(ga.cpu().numpy() - go).max() <= TOL_PDF_1STEP
    # the option really selects another operator
    b = _acm(p)
    b.init(_dev(phi), _dev(u))
    b.set_pdfs(_dev(h), _dev(g))
    b.step(2)
    assert float((b.get_pdfs()[0] - ha).abs().max()) > 1e-5


def test_srt_paper_benchmark_setup_100_steps():
    """The paper's benchmark scheme: D3Q15 SRT phase field + D3Q27 MRT hydrodynamics, one light
    bubble in the middle of a periodic box (P:283 scaled from 260^3, R=65 to 40^3, R=10)."""
    p = Params(nx=40, ny=40, nz=40, stencil_phase=15, stencil_hydro=27)
    phi = inputs.sphere_phi(p, (20.0, 20.0, 20.0), 10.0, heavy_inside=False)
    u = inputs.zeros_u(p)
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, u)
    a = _acm(p, phase_srt=True)
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


def test_srt_fp32_one_step():
    p = Params(nx=70, ny=9, nz=6, stencil_phase=15, stencil_hydro=27, wall_flags=inputs.WALL_Y)
    phi, u, h, g = random_state(p, seed=4)
    phi, u, h, g = (np.asarray(x, dtype=np.float32).astype(np.float64) for x in (phi, u, h, g))
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, phase_srt=True, precision="f32")
    a.init(_dev(phi, np.float32), _dev(u, np.float32))
    a.set_pdfs(_dev(h, np.float32), _dev(g, np.float32))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    assert np.abs(ha.cpu().numpy() - ho).max() < 3e-7
    assert np.abs(ga.cpu().numpy() - go).max() < 2e-7
    assert abs(a.phi_mass() / o.phi_mass() - 1) < 2e-7      # rest population by subtraction: phi = sum h exactly


def test_rising_bubble_section6_setup_scaled():
    """Section 6.1 set-up on a scale model: walls in y, gravity, rho* = 1000, mu* = 100 (so nu_L = 10 nu_H:
    tau and s_nu vary across the interface, eqs. 20-21), parameters from Re_Gr / Eo through eqs. 31-33,
    D3Q19 + D3Q19 MRT, M = 0.04.  40 steps at 1e-10; the bubble diagnostics agree."""
    from paper_2012_06144_b200 import binding
    D = 12.0
    q = binding.bubble_params(35.0, 10.0, D, 600.0)
    qo = om.bubble_params(35.0, 10.0, D, 600.0)
    assert all(abs(q[k] - qo[k]) <= 1e-15 * abs(qo[k]) for k in qo)
    p = Params(nx=24, ny=48, nz=24, stencil_phase=19, stencil_hydro=19, rho_H=1.0, rho_L=q["rho_L"], sigma=q["sigma"],
               M=0.04, nu_H=q["nu_H"], nu_L=q["nu_L"], gravity=(0.0, -q["gy"], 0.0), wall_flags=inputs.WALL_Y)
    assert abs(p.nu_L / p.nu_H - 10.0) < 1e-9
    # a light bulk next to the walls keeps the step well conditioned: the
    # bubble sits in a heavy-liquid column that ends 6 cells before each wall
    phi = inputs.sphere_phi(p, (12.0, 16.0, 12.0), D / 2, heavy_inside=False)
    y = (np.arange(p.ny) + 0.5)[None, :, None]
    phi = phi * 0.25 * (1 + np.tanh(2 * (y - 6.0) / p.xi)) * (1 - np.tanh(2 * (y - 42.0) / p.xi))
    phi = np.ascontiguousarray(np.broadcast_to(phi, p.shape))
    u = inputs.zeros_u(p)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    o.step(40)
    a.step(40)
    po, uo, _ = o.fields(False)
    pa, ua, _ = a.fields(False)
    assert np.abs(pa.cpu().numpy() - po).max() <= TOL_FIELD_100
    assert np.abs(ua.cpu().numpy() - uo).max() <= TOL_FIELD_100
    Vo, Xo, Uo = o.bubble_diag()
    Va, Xa, Ua = a.bubble_diag()
    assert abs(Va / Vo - 1) < 1e-12
    assert np.abs(np.array(Xa) - Xo).max() < 1e-10
    assert np.abs(np.array(Ua) - Uo).max() < 1e-12
    assert np.isfinite(binding.drag_lbm(q["gy"], p.rho_H, p.rho_L, D, max(abs(Ua[1]), 1e-12)))


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_bubble_diag_matches_oracle_and_is_deterministic(precision):
    """Ragged size spanning many reduction blocks; random phi, u; bitwise equal on repetition."""
    p = Params(nx=150, ny=37, nz=29)
    phi, u, _, _ = random_state(p, seed=9)
    dt = np.float64 if precision == "f64" else np.float32
    phi, u = (np.asarray(x, dtype=dt).astype(np.float64) for x in (phi, u))
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p, precision=precision)
    a.init(_dev(phi, dt), _dev(u, dt))
    Vo, Xo, Uo = o.bubble_diag()
    r1 = a.bubble_diag()
    r2 = a.bubble_diag()
    assert r1 == r2
    assert abs(r1[0] / Vo - 1) < 1e-12
    assert np.abs(np.array(r1[1]) - Xo).max() < 1e-10
    assert np.abs(np.array(r1[2]) - Uo).max() < 1e-13


def test_bubble_diag_errors():
    from paper_2012_06144_b200.binding import AcmError, ACM_ESTATE, ACM_EUNSTABLE
    p = Params(nx=16, ny=8, nz=8)
    a = _acm(p)
    with pytest.raises(AcmError) as e:
        a.bubble_diag()
    assert e.value.code == ACM_ESTATE
    a.init(_dev(np.ones(p.shape)), _dev(inputs.zeros_u(p)))     # no light phase at all: V = 0
    with pytest.raises(AcmError) as e:
        a.bubble_diag()
    assert e.value.code == ACM_EUNSTABLE
