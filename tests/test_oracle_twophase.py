"""Physics pins of the oracle's hydrodynamic forces under TWO-PHASE conditions (grad rho != 0), CPU only.

The single-phase pins (shear wave, Poiseuille) run with rho_H = rho_L, where F_mu (eq. 18) and F_p
(eq. 14) vanish; Laplace and the tanh slab are at rest.  These cases make both forces carry the result:

  * layered two-fluid Poiseuille flow: walls in y, uniform acceleration g_x, a flat interface, rho_H/rho_L = 10.
    The steady state of eq. 9 is  d/dy( mu(y) du/dy ) = -rho(y) g_x  with mu = rho(phi) nu(phi):
    two parabolas with a KINK at the interface (continuous shear stress mu du/dy).  It is F_mu that turns the
    velocity-based LBE's  rho nu lap u  into  div( mu (grad u + grad u^T) ); without it (or with a wrong sign or
    factor) the profile is the single parabola g/(2 nu) y (L - y) or worse -- an O(1) difference in the light layer.
  * two-layer hydrostatics: gravity g_y, heavy liquid below, interface off-centre so that the pressure at the
    interface is not zero.  At rest  grad p = rho g  with p = p* rho c_s^2, and p is continuous across the
    interface only because F_p = -p* c_s^2 grad rho completes  -c_s^2 grad p*  to  -grad p / rho.

Expected values: the sharp-interface analytic solution (2 x 2 linear system for the two parabolas) away from the
interface, and the diffuse-interface momentum balance solved by finite volumes on the oracle's own phi profile
(which is itself checked against eq. 3).
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

NY, H, XI = 48, 16.0, 4.0


def _column(rho_L, nu_H, nu_L, gravity, sigma, steps):
    """one column of NY cells between walls (x, z periodic with one cell), heavy liquid in 0 < y < H"""
    p = Params(nx=1, ny=NY, nz=1, stencil_phase=19, stencil_hydro=19, rho_H=1.0, rho_L=rho_L, sigma=sigma, xi=XI,
               M=0.02, nu_H=nu_H, nu_L=nu_L, gravity=gravity, wall_flags=inputs.WALL_Y)
    y = np.arange(NY) + 0.5
    phi0 = 0.5 - 0.5 * np.tanh(2.0 * (y - H) / XI)
    o = Oracle.from_params(p)
    o.init(phi0.reshape(p.shape), inputs.zeros_u(p))
    o.step(steps)
    c, u, pr = o.fields()
    return p, y, phi0, c.ravel(), u[:, 0, :, 0], pr.ravel()


def _two_parabolas(y, L, h, rho1, mu1, rho2, mu2, g):
    """sharp interface: mu_k u_k'' = -rho_k g, u(0) = u(L) = 0, u and mu u' continuous at y = h"""
    a1, a2 = rho1 * g / (2 * mu1), rho2 * g / (2 * mu2)
    # u1 = -a1 y^2 + A y,  u2 = -a2 (L-y)^2 + B (L-y)
    A, B = np.linalg.solve(np.array([[h, -(L - h)], [mu1, mu2]]),
                           np.array([a1 * h * h - a2 * (L - h) ** 2, 2 * mu1 * a1 * h + 2 * mu2 * a2 * (L - h)]))
    return np.where(y < h, -a1 * y * y + A * y, -a2 * (L - y) ** 2 + B * (L - y))


def _diffuse_balance(rho, mu, g):
    """finite volumes for d/dy(mu du/dy) = -rho g on the cell centres; walls half a cell outside the first / last cell"""
    n = len(rho)
    mf = 0.5 * (mu[1:] + mu[:-1])
    A = np.zeros((n, n))
    for i in range(n):
        lo = mf[i - 1] if i > 0 else 2.0 * mu[0]
        hi = mf[i] if i < n - 1 else 2.0 * mu[-1]
        A[i, i] = -(lo + hi)
        if i > 0:
            A[i, i - 1] = lo
        if i < n - 1:
            A[i, i + 1] = hi
    return np.linalg.solve(A, -rho * g)


@pytest.mark.parametrize("nu_H,nu_L", [(0.1, 0.1), (0.1, 0.25)])
def test_layered_poiseuille_viscous_force(nu_H, nu_L):
    rho_L, gx = 0.1, 1e-6
    steps = int(12 * NY * NY / (math.pi ** 2 * min(nu_H, nu_L)))
    p, y, phi0, c, u, _ = _column(rho_L, nu_H, nu_L, (gx, 0.0, 0.0), 1e-3, steps)
    ux = u[0]
    # the flow is along x (what is left in u_y is the staggered (-1)^y mode that streaming with bounce-back at both
    # ends conserves on a one-cell-wide column; it was excited by the start-up and does not couple to u_x)
    assert np.abs(u[1:]).max() < 5e-3 * ux.max()
    assert np.abs(c - phi0).max() < 0.02                      # the interface stayed where it was (eq. 3)
    rho = rho_L + c * (1.0 - rho_L)
    mu = rho * (nu_L + c * (nu_H - nu_L))                     # nu = tau c_s^2, tau linear in phi (eqs. 19, 20)
    # (i) the diffuse-interface momentum balance on the oracle's own phi: everywhere
    ud = _diffuse_balance(rho, mu, gx)
    assert np.abs(ux - ud).max() < 0.015 * ud.max()
    # (ii) the sharp-interface solution away from the interface: the heavy layer closely, the light layer within the
    #      shift the smeared viscosity causes (mu linear in phi moves the effective interface into the light side)
    us = _two_parabolas(y, NY, H, 1.0, nu_H, rho_L, rho_L * nu_L, gx)
    heavy, light = y < H - 1.5 * XI, y > H + 1.5 * XI
    assert np.abs(ux - us)[heavy].max() < 0.01 * us.max()
    assert np.abs(ux - us)[light].max() < 0.08 * us.max()
    # (iii) the kink: the slope changes across the interface by about the viscosity ratio (continuous shear stress)
    s_heavy = (ux[9] - ux[8])
    s_light = (ux[23] - ux[22])
    e_heavy = (us[9] - us[8])
    e_light = (us[23] - us[22])
    assert abs(s_heavy / e_heavy - 1) < 0.05 and abs(s_light / e_light - 1) < 0.15
    # (iv) and it is NOT what comes out without the viscous force: rho nu u'' = -rho g, one parabola per layer
    #      with continuous slope (for nu_H = nu_L the single parabola g/(2 nu) y (L-y))
    if nu_H == nu_L:
        single = gx / (2 * nu_H) * y * (NY - y)
        assert np.abs(ux - single).max() > 0.25 * us.max()


def test_two_layer_hydrostatics_pressure_force():
    rho_L, gy = 0.1, -1e-5
    p, y, phi0, c, u, pr = _column(rho_L, 0.1, 0.1, (0.0, gy, 0.0), 0.0, 20000)
    assert np.abs(u).max() < 1e-6                              # at rest
    assert np.abs(c - phi0).max() < 0.02
    rho = rho_L + c * (1.0 - rho_L)
    rho_f = 0.5 * (rho[1:] + rho[:-1])
    ratio = np.diff(pr) / (rho_f * gy)
    bulk = (y[:-1] < H - 2.5 * XI) | (y[:-1] > H + 2.5 * XI)
    assert np.abs(ratio[bulk][1:-1] - 1).max() < 2e-3          # dp/dy = rho g in both layers (first/last face: wall)
    assert np.abs(ratio - 1).max() < 0.25                      # and within the discretisation error inside the interface
    # pressure difference between the two bulks = weight of the column in between (p continuous across the interface)
    j0, j1 = 6, 30
    assert abs((pr[j0] - pr[j1]) / (-gy * rho_f[j0:j1].sum()) - 1) < 0.015
    # the pressure at the interface is not zero (else F_p would be idle): sum p* is conserved at its initial 0, so
    # p_I follows from the off-centre interface
    pstar = 3.0 * pr / rho
    assert abs(pstar.sum()) < 1e-10
    assert abs(pr[15]) > 0.1 * abs(pr[j0] - pr[j1])
