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


# ------------------------------------------------------------------------------------------
# A26: bulk moment relaxed with 1 (the other reading of P:152-156)
# ------------------------------------------------------------------------------------------
def _one_step(p, phi, u, h, g, n=1, **variant):
    o = Oracle.from_params(p, **variant)
    o.init(phi, u)
    o.set_pdfs(h, g)
    o.step(n)
    return o.get_pdfs() + o.fields(False)[:2]


@pytest.mark.parametrize("case", [dict(stencil_phase=15, stencil_hydro=19, wall_flags=0),
                                  dict(stencil_phase=27, stencil_hydro=27, wall_flags=inputs.WALL_Y),
                                  dict(stencil_phase=19, stencil_hydro=15, wall_flags=inputs.WALL_X | inputs.WALL_Z, nu_H=0.3, nu_L=0.03),
                                  dict(stencil_phase=9, stencil_hydro=9, nz=1, wall_flags=inputs.WALL_Y)])
def test_bulk_one_bruteforce_one_step(case):
    """Omega^g = I - (1 - s_nu)(P_2 - P_trace): the second-order projector of the default operator minus the
    w-orthogonal projector on the trace moment |e|^2 - D/3, hand-expanded per direction pair."""
    case = dict(case)
    nz = case.pop("nz", 3)
    grav = (1e-4, -1e-4, 0.0)
    p = Params(nx=4, ny=5, nz=nz, rho_H=1.0, rho_L=0.05, sigma=2e-3, xi=3.0, gravity=grav, **case)
    phi, u, h, g = random_state(p, seed=21)
    if nz == 1:
        u[2] = 0.0
    ho, go, po, uo = _one_step(p, phi, u, h, g, bulk_one=True)
    Hb, Gb, Cb, Ub = bruteforce.step(p, list(h), list(g), phi, list(u), bulk_one=True)
    assert np.abs(ho - np.array(Hb)).max() < 1e-14
    assert np.abs(go - np.array(Gb)).max() < 1e-14
    assert np.abs(po - Cb).max() < 1e-14
    assert np.abs(uo - np.array(Ub)).max() < 1e-14
    # the flag does something: the default operator (trace at s_nu, A4) gives different g, and a different u through F_mu
    hd, gd, pd, ud = _one_step(p, phi, u, h, g)
    assert np.abs(gd - go).max() > 1e-6
    assert np.abs(ud - uo).max() > 1e-9
    assert np.abs(hd - ho).max() == 0.0          # the phase-field step does not know about it


@pytest.mark.parametrize("Q", [9, 15, 19, 27])
def test_bulk_split_basis(Q):
    """The basis of the variant: one row proportional to |e|^2 - D/3 (order ORDER_BULK), five (2-D: two) second-order
    rows that are trace-free in the w-inner product, everything still weighted-orthogonal, M^-1 M = 1; and the
    operator M^-1 S M equals the hand-written projector form."""
    e, w, opp, M, Minv, order = om.lattice(Q, bulk_split=True)
    D = 2 if Q == 9 else 3
    G = (M * w[None, :]) @ M.T
    assert np.abs(G - np.diag(np.diag(G))).max() < 1e-13
    assert np.abs(Minv @ M - np.eye(Q)).max() < 1e-12
    bulk = np.where(order == om.ORDER_BULK)[0]
    assert len(bulk) == 1
    t = (e * e).sum(1) - D / 3.0
    row = M[bulk[0]]
    assert np.abs(row / row[np.argmax(np.abs(row))] - t / t[np.argmax(np.abs(row))]).max() < 1e-13
    assert (order == 2).sum() == (5 if D == 3 else 2)
    # the other orders are as in the default basis
    order0 = om.lattice(Q)[5]
    assert sorted(order0[order0 != 2]) == sorted(order[(order != 2) & (order != om.ORDER_BULK)])
    s = 1.37
    S = np.where(order == 2, s, 1.0)
    Omega = Minv @ np.diag(S) @ M
    eg, wg = bruteforce.lattice(Q)
    og = bruteforce.hydro_operator(eg, wg, s, bulk_one=True)
    Ob = np.array([[og(i, j) for j in range(Q)] for i in range(Q)])
    assert np.abs(Omega - Ob).max() < 1e-13


def test_bulk_one_equals_default_at_s_nu_one():
    """nu = 1/6 gives tau = 1/2, s_nu = 1: every moment relaxes with 1 in both operators."""
    p = Params(nx=6, ny=5, nz=4, nu_H=1.0 / 6.0, nu_L=1.0 / 6.0, rho_L=0.05, sigma=2e-3, xi=3.0)
    phi, u, h, g = random_state(p, seed=4)
    a = _one_step(p, phi, u, h, g, n=3)
    b = _one_step(p, phi, u, h, g, n=3, bulk_one=True)
    for x, y in zip(a, b):
        assert np.abs(x - y).max() < 2e-15


def _single_phase(L, nu, bulk_one, **kw):
    p = Params(nx=L, ny=1, nz=1, stencil_phase=19, stencil_hydro=19, rho_H=1.0, rho_L=1.0, sigma=0.0, nu_H=nu, nu_L=nu, **kw)
    o = Oracle.from_params(p, bulk_one=bulk_one)
    return p, o


@pytest.mark.parametrize("bulk_one", [False, True])
def test_bulk_one_shear_viscosity_unchanged(bulk_one):
    """A transverse wave u_y = A sin(k x) decays with nu = c_s^2 (1/s_nu - 1/2) whatever the bulk moment does."""
    L, nu = 64, 1.0 / 60.0
    p, o = _single_phase(L, nu, bulk_one)
    k = 2 * np.pi / L
    u = inputs.zeros_u(p)
    u[1] = 1e-3 * np.sin(k * (np.arange(L) + 0.5)).reshape(p.shape)
    o.init(np.ones(p.shape), u)
    o.step(100)
    a0 = np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1])
    o.step(400)
    a1 = np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1])
    assert abs(-math.log(a1 / a0) / (k * k * 400) / nu - 1) < 2e-3


@pytest.mark.parametrize("bulk_one,nu", [(False, 1.0 / 60.0), (True, 1.0 / 60.0), (True, 0.1)])
def test_bulk_one_sound_attenuation(bulk_one, nu):
    """A longitudinal wave u_x = A sin(k x) is a standing sound wave; its energy u^2 + c_s^2 p*^2 decays as
    exp(-2 Gamma k^2 t) with Gamma = (4/3 nu + zeta)/2.  The bulk moment relaxed with rate s_b gives the bulk
    viscosity zeta = (2/9)(1/s_b - 1/2) on these lattices: (2/3) nu for the default (s_b = s_nu, A4), 1/9 for the
    variant (s_b = 1).  Distinguishes the two readings of P:152-156 by an O(1) factor."""
    L = 64
    p, o = _single_phase(L, nu, bulk_one)
    k = 2 * np.pi / L
    u = inputs.zeros_u(p)
    u[0] = 1e-4 * np.sin(k * (np.arange(L) + 0.5)).reshape(p.shape)
    o.init(np.ones(p.shape), u)

    def energy():
        _, uu, pr = o.fields()
        uk = np.abs(np.fft.rfft(uu[0].ravel())[1])
        pk = np.abs(np.fft.rfft(pr.ravel())[1]) * 3.0        # p* = p / (rho c_s^2), rho = 1
        return uk * uk + pk * pk / 3.0
    o.step(60)
    t, E = [], []
    for _ in range(40):
        o.step(10)
        t.append(10 * (len(t) + 1))
        E.append(energy())
    slope = np.polyfit(np.array(t, dtype=float), np.log(np.array(E)), 1)[0]
    zeta = (1.0 / 9.0) if bulk_one else (2.0 / 3.0) * nu
    gamma = 0.5 * (4.0 / 3.0 * nu + zeta)
    assert abs(-slope / (2 * k * k) / gamma - 1) < 0.03


# ------------------------------------------------------------------------------------------
# A27: sub-iterated velocity (fixed point of eq. 22)
# ------------------------------------------------------------------------------------------
def _subiter_case():
    p = Params(nx=4, ny=5, nz=3, stencil_phase=15, stencil_hydro=27, rho_H=1.0, rho_L=0.05, sigma=2e-3, xi=3.0,
               gravity=(1e-4, -1e-4, 0.0), nu_H=0.05, nu_L=0.2, wall_flags=inputs.WALL_Y)
    return (p,) + random_state(p, seed=31)


def test_subiter_one_is_the_default_bit_for_bit():
    p, phi, u, h, g = _subiter_case()
    a = _one_step(p, phi, u, h, g, n=3)
    b = _one_step(p, phi, u, h, g, n=3, subiter=1)
    for x, y in zip(a, b):
        assert (x == y).all()


@pytest.mark.parametrize("k", [2, 3])
def test_subiter_bruteforce_one_step(k):
    p, phi, u, h, g = _subiter_case()
    ho, go, po, uo = _one_step(p, phi, u, h, g, subiter=k)
    Hb, Gb, Cb, Ub = bruteforce.step(p, list(h), list(g), phi, list(u), subiter=k)
    assert np.abs(go - np.array(Gb)).max() < 1e-14
    assert np.abs(uo - np.array(Ub)).max() < 1e-14
    assert np.abs(ho - np.array(Hb)).max() < 1e-14
    # differs from the single evaluation (A10) where grad rho and u are not small
    _, gd, _, ud = _one_step(p, phi, u, h, g)
    assert np.abs(ud - uo).max() > 1e-8


def test_subiter_fixed_point_satisfies_eq22():
    """After enough sweeps the stored velocity solves u = sum g e + F(u)/(2 rho) with F_mu evaluated at that same u
    (eq. 22 with eq. 18): residual from the brute-force force at rounding level; the single
    evaluation of reading A10 leaves a residual orders of magnitude larger."""
    p, phi, u, h, g = _subiter_case()
    grid = bruteforce.Grid(p.nx, p.ny, p.nz, p.wall_flags)
    eg, wg = bruteforce.lattice(p.stencil_hydro)

    def residual(k):
        _, _, cn, un = _one_step(p, phi, u, h, g, subiter=k)
        worst = 0.0
        for zyx in grid.cells():
            gc = [g[i][zyx] for i in range(p.stencil_hydro)]
            uc = [un[a][zyx] for a in range(3)]
            F, rho, j, _ = bruteforce.hydro_force(p, grid, eg, wg, gc, cn, zyx, uc)
            worst = max(worst, max(abs(uc[a] - (j[a] + F[a] / (2.0 * rho))) for a in range(3)))
        return worst
    r1, r2, r12 = residual(1), residual(2), residual(12)
    assert r12 < 1e-15
    assert r1 > 1e3 * max(r12, 1e-16) and r2 < r1
