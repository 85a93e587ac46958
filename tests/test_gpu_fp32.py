"""fp32 instance (config 5 of BASELINE.json, reading A22) against the fp64 oracle.

Tolerance from BASELINE.json: 1e-5 on phi and u after 500 steps.  One step: fp32 rounding of O(1)
populations, a few 1e-7.
"""
import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu


def _acm32(p):
    from paper_2012_06144_b200.binding import ACM
    return ACM.from_params(p, precision="f32")


def _dev32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.mark.parametrize("Qh,Qg,walls", [(27, 27, 0), (15, 19, inputs.WALL_Y)])
def test_fp32_one_step(Qh, Qg, walls):
    p = Params(nx=70, ny=9, nz=6, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=(0.0, -1e-5, 0.0))
    phi, u, h, g = random_state(p, seed=4)
    # start both sides from the SAME fp32-representable state
    phi, u, h, g = (np.asarray(x, dtype=np.float32).astype(np.float64) for x in (phi, u, h, g))
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm32(p)
    a.init(_dev32(phi), _dev32(u))
    a.set_pdfs(_dev32(h), _dev32(g))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    dh = np.abs(ha.cpu().numpy() - ho)
    assert dh[1:].max() < 5e-8                 # a few ulp of 0.07
    # rest population by subtraction (A22): Q-1 roundings of ulp(0.07)/2 = 3.7e-9 each, the same again in phi = sum h,
    # and the un-shifting h' + ref w_0 (ulp(0.3)/2 = 1.5e-8)
    assert dh[0].max() < 4e-7
    assert np.abs(ga.cpu().numpy() - go).max() < 2e-8
    po, uo, _ = o.fields(False)
    pa, ua, _ = a.fields(False)
    assert np.abs(pa.cpu().numpy() - po).max() < 5e-7
    assert np.abs(ua.cpu().numpy() - uo).max() < 2e-6          # F/(2 rho) with rho down to 1e-3


def test_fp32_config5_scaled_500_steps():
    """Config 5 on a 32^3 scale model (D3Q27+D3Q27), 500 steps: |d phi|, |d u| <= 1e-5 vs the fp64 oracle;
    the rest-population-by-subtraction keeps sum(phi) within 1e-6 relative."""
    p, phi, u = inputs.scaled_config3(32, stencil_phase=27, stencil_hydro=27)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm32(p)
    a.init(_dev32(phi), _dev32(u))
    m0 = a.phi_mass()
    o.step(500)
    a.step(500)
    po, uo, _ = o.fields(False)
    pa, ua, _ = a.fields(False)
    assert np.abs(pa.cpu().numpy() - po).max() <= 1e-5
    assert np.abs(ua.cpu().numpy() - uo).max() <= 1e-5
    assert abs(a.phi_mass() - m0) / m0 < 1e-6


def test_fp32_full_size_sampled_256():
    """Config 5 fp32 at 256^3: one step checked on sampled 14^3 sub-boxes recomputed by the fp64 oracle
    from the fp32 state (inner 8^3 exact dependence cone)."""
    p, phi, u = inputs.config5()
    a = _acm32(p)
    a.init(_dev32(phi), _dev32(u))
    a.step(2)
    h0, g0 = a.get_pdfs()
    c0, u0, _ = a.fields(False)
    B, n = 14, p.nx
    starts = [(0, 0, 0), (n - 7, n - 7, n - 7), (37, 201, 118), (200, 13, n - 4)]
    subs = []
    for (z, y, x) in starts:
        iz = (torch.arange(z, z + B, device="cuda") % n)[:, None, None]
        iy = (torch.arange(y, y + B, device="cuda") % n)[None, :, None]
        ix = (torch.arange(x, x + B, device="cuda") % n)[None, None, :]
        subs.append((iz, iy, ix) + tuple(t.cpu().numpy().astype(np.float64) for t in
                                         (h0[:, iz, iy, ix], g0[:, iz, iy, ix], c0[iz, iy, ix], u0[:, iz, iy, ix])))
    del h0, g0
    a.step(1)
    h1, g1 = a.get_pdfs()
    c1, u1, _ = a.fields(False)
    pb = p.replace(nx=B, ny=B, nz=B)
    inner = (slice(3, -3),) * 3
    sl = (slice(None),) + inner
    for (iz, iy, ix, hs, gs, cs, us) in subs:
        o = Oracle.from_params(pb)
        o.init(cs, us)
        o.set_pdfs(hs, gs)
        o.step(1)
        ho, go = o.get_pdfs()
        po, uo, _ = o.fields(False)
        assert np.abs(h1[:, iz, iy, ix].cpu().numpy()[sl] - ho[sl]).max() < 1e-6      # rest population: 26 subtractions
        assert np.abs(g1[:, iz, iy, ix].cpu().numpy()[sl] - go[sl]).max() < 2e-7
        assert np.abs(c1[iz, iy, ix].cpu().numpy()[inner] - po[inner]).max() < 5e-7
        assert np.abs(u1[:, iz, iy, ix].cpu().numpy()[sl] - uo[sl]).max() < 2e-6
