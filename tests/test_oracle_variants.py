"""Pins of the oracle's operator variants and rising-bubble diagnostics, CPU only.

  A23  SRT phase-field collision: brute force on 4x5x3, the omega = 1 special case where
       SRT and MRT coincide, the diffusion limit (diffusivity = M), sum(phi) conservation.
  A24  bubble volume / centroid / velocity over phi < 1/2 weighted with 1 - phi: symmetry, translation,
       continuum integral of the tanh-profile volume, brute force with numpy.
  eqs. 31-35: parameters from the dimensionless groups and back; limits of eq. 35.
"""
import math

import numpy as np
import pytest

import bruteforce
from helpers import random_state
from oracle import Oracle
from oracle import oracle as om
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params


@pytest.mark.parametrize("case", [dict(stencil_phase=15, stencil_hydro=19, wall_flags=0),
                                  dict(stencil_phase=27, stencil_hydro=27, wall_flags=inputs.WALL_Y),
                                  dict(stencil_phase=19, stencil_hydro=19, wall_flags=inputs.WALL_X | inputs.WALL_Z, M=0.08)])
def test_srt_bruteforce_one_step(case):
    p = Params(nx=4, ny=5, nz=3, rho_H=1.0, rho_L=0.05, sigma=2e-3, xi=3.0, gravity=(1e-4, -1e-4, 0.0), **case)
    phi, u, h, g = random_state(p, seed=11)
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, u)
    o.set_pdfs(h, g)
    o.step(1)
    ho, go = o.get_pdfs()
    po, uo, _ = o.fields(False)
    Hb, Gb, Cb, Ub = bruteforce.step(p, list(h), list(g), phi, list(u), phase_srt=True)
    assert np.abs(ho - np.array(Hb)).max() < 1e-14
    assert np.abs(go - np.array(Gb)).max() < 1e-14
    assert np.abs(po - Cb).max() < 1e-14
    assert np.abs(uo - np.array(Ub)).max() < 1e-14
    # and the flag does something: the MRT operator gives different populations
    o2 = Oracle.from_params(p)
    o2.init(phi, u)
    o2.set_pdfs(h, g)
    o2.step(1)
    assert np.abs(o2.get_pdfs()[0] - ho).max() > 1e-4


def test_srt_equals_mrt_at_omega_one():
    """M = 1/6 gives tau_phi = 1/2, omega_phi = 1: every moment relaxes with 1 in both operators."""
    p = Params(nx=6, ny=5, nz=4, M=1.0 / 6.0, rho_L=0.05, sigma=2e-3, xi=3.0)
    phi, u, h, g = random_state(p, seed=3)
    out = []
    for srt in (False, True):
        o = Oracle.from_params(p, phase_srt=srt)
        o.init(phi, u)
        o.set_pdfs(h, g)
        o.step(3)
        out.append(o.get_pdfs()[0])
    assert np.abs(out[0] - out[1]).max() < 1e-15


@pytest.mark.parametrize("Mob", [0.02, 0.08])
def test_srt_mobility_sine_decay(Mob):
    """Diffusion limit of the SRT operator: diffusivity c_s^2 (1/omega - 1/2) = M (eq. 2, A2)."""
    L = 64
    p = Params(nx=L, ny=1, nz=1, rho_H=1.0, rho_L=1.0, sigma=0.0, xi=1e300, M=Mob)
    x = np.arange(L) + 0.5
    k = 2 * np.pi / L
    phi = (0.5 + 0.1 * np.sin(k * x)).reshape(p.shape)
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, inputs.zeros_u(p))
    o.step(200)
    a0 = 2 * np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1]) / L
    o.step(800)
    a1 = 2 * np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1]) / L
    D = -math.log(a1 / a0) / (k * k * 800)
    assert abs(D / Mob - 1) < 2e-3


def test_srt_mass_conservation_and_uniform_state():
    p, phi, u = inputs.scaled_config3(16)
    o = Oracle.from_params(p, phase_srt=True)
    o.init(phi, u)
    m0 = o.phi_mass()
    o.step(30)
    assert abs(o.phi_mass() - m0) / m0 < 1e-13
    q = Params(nx=6, ny=6, nz=6)
    o = Oracle.from_params(q, phase_srt=True)
    o.init(np.full(q.shape, 0.3), inputs.zeros_u(q))
    o.step(20)
    c = o.fields(False)[0]
    assert (c == c.flat[0]).all()


# ------------------------------------------------------------------------------------------
# bubble diagnostics (A24)
# ------------------------------------------------------------------------------------------
def test_bubble_diag_sphere_symmetry_translation_volume():
    R, xi = 8.0, 5.0
    p = Params(nx=40, ny=48, nz=40, xi=xi)
    c0 = (20.0, 24.0, 20.0)
    o = Oracle.from_params(p)
    o.init(inputs.sphere_phi(p, c0, R, heavy_inside=False), inputs.zeros_u(p))
    V, X, Ub = o.bubble_diag()
    assert np.abs(X - np.array(c0)).max() < 1e-11            # mirror symmetry about the centre
    assert np.abs(Ub).max() == 0.0
    # the definition integrated in the continuum: V = int_0^R (1/2)(1 - tanh(2 (r-R)/xi)) 4 pi r^2 dr (phi < 1/2 <=> r < R)
    from scipy.integrate import quad
    V_exact = quad(lambda r: 0.5 * (1.0 - math.tanh(2.0 * (r - R) / xi)) * 4.0 * math.pi * r * r, 0.0, R)[0]
    assert 0.70 * 4.0 / 3.0 * math.pi * R ** 3 < V_exact < 4.0 / 3.0 * math.pi * R ** 3
    assert abs(V / V_exact - 1) < 1e-2
    # integer shift of the sphere shifts the centroid by that much and keeps V (thin interface, so
    # that the tails cut by the box, 1 - phi ~ exp(-4 (d-R)/xi) < 1e-9, do not matter)
    pt = p.replace(xi=2.0)
    res = []
    for c in (c0, (23.0, 19.0, 21.0)):
        o2 = Oracle.from_params(pt)
        o2.init(inputs.sphere_phi(pt, c, R, heavy_inside=False), inputs.zeros_u(pt))
        res.append(o2.bubble_diag())
    assert np.abs(res[1][1] - res[0][1] - np.array([3.0, -5.0, 1.0])).max() < 1e-8
    assert abs(res[1][0] / res[0][0] - 1) < 1e-9


def test_bubble_diag_velocity_weighting():
    p = Params(nx=12, ny=10, nz=8)
    phi, u, _, _ = random_state(p, seed=5)
    o = Oracle.from_params(p)
    # uniform velocity: the weighted mean is that velocity
    uu = np.empty((3,) + p.shape)
    uu[0], uu[1], uu[2] = 0.01, -0.02, 0.005
    o.init(phi, uu)
    _, _, Ub = o.bubble_diag()
    assert np.abs(Ub - np.array([0.01, -0.02, 0.005])).max() < 1e-16
    # general field: the definition written with numpy
    o.init(phi, u)
    V, X, Ub = o.bubble_diag()
    w = np.where(phi < 0.5, 1.0 - phi, 0.0)
    z, y, x = np.meshgrid(np.arange(p.nz) + 0.5, np.arange(p.ny) + 0.5, np.arange(p.nx) + 0.5, indexing="ij")
    assert abs(V - w.sum()) < 1e-10
    assert np.abs(X - np.array([(w * x).sum(), (w * y).sum(), (w * z).sum()]) / w.sum()).max() < 1e-12
    assert np.abs(Ub - (w[None] * u).sum(axis=(1, 2, 3)) / w.sum()).max() < 1e-15


# ------------------------------------------------------------------------------------------
# eqs. 31-35
# ------------------------------------------------------------------------------------------
def test_bubble_params_round_trip_and_worked_value():
    """Section 6.1: D = 32 (R = 16), t_ref = 18 000, rho* = 1000, mu* = 100."""
    D, t_ref, Re, Eo = 32.0, 18000.0, 35.0, 30.0
    q = om.bubble_params(Re, Eo, D, t_ref)
    assert abs(q["gy"] - 32.0 / 18000.0 ** 2) < 1e-22          # eq. 33: g_y = D / t_ref^2 = 9.8765e-8
    assert abs(q["gy"] - 9.876543209876543e-08) < 1e-20
    rho_H = 1.0
    mu_H = q["nu_H"] * rho_H
    assert abs(rho_H * math.sqrt(q["gy"] * D ** 3) / mu_H - Re) < 1e-12        # eq. 31
    assert abs(q["gy"] * rho_H * D ** 2 / q["sigma"] - Eo) < 1e-12             # eq. 32
    assert abs(math.sqrt(D / q["gy"]) - t_ref) < 1e-8                          # eq. 33
    assert abs(rho_H / q["rho_L"] - 1000.0) < 1e-9
    assert abs(mu_H / (q["nu_L"] * q["rho_L"]) - 100.0) < 1e-9
    assert abs(q["nu_L"] / q["nu_H"] - 10.0) < 1e-9                            # rho*/mu*
    with pytest.raises(ValueError):
        om.bubble_params(0.0, Eo, D, t_ref)


def test_drag_formulas():
    # eq. 35 limits: Re -> inf gives 2.67, Re -> 0 gives 16/Re; monotone decreasing in Re
    assert abs(om.drag_exp(1e12) - 2.67) < 1e-6
    assert abs(om.drag_exp(1e-9) * 1e-9 / 16.0 - 1) < 1e-6
    v = [om.drag_exp(r) for r in (1, 5, 10, 35, 100, 1000)]
    assert all(a > b for a, b in zip(v, v[1:]))
    # at Re = 16 the two terms are 2.67^0.9 and 1
    assert abs(om.drag_exp(16.0) - (2.67 ** 0.9 + 1.0) ** (10.0 / 9.0)) < 1e-14
    # eq. 34: a bubble whose drag balances buoyancy at u_t: C_D u_t^2 = 4/3 g (1 - rho_L/rho_H) D
    cd = om.drag_lbm(1e-7, 1.0, 1e-3, 32.0, 2e-3)
    assert abs(cd * (2e-3) ** 2 - 4.0 / 3.0 * 1e-7 * 0.999 * 32.0) < 1e-20
    assert abs(om.drag_lbm(1e-7, 1.0, 1e-3, 32.0, 4e-3) / cd - 0.25) < 1e-14
