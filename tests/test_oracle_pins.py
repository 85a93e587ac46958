"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Each test names the passage (PAPER.md "P:<line>") or the DESIGN.md reading it pins.
None of the expected values comes from the CUDA path.
"""
import itertools
import math

import numpy as np
import pytest

import bruteforce
from helpers import random_state
from oracle import Oracle, lattice
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params


# --------------------------------------------------------------------------------------
# lattices and moment bases
# --------------------------------------------------------------------------------------

@pytest.mark.parametrize("Q", [15, 19, 27])
def test_lattice_identities(Q):
    """Textbook lattices: sum w = 1, sum w e = 0, sum w e e = c_s^2 I,
    fourth-order isotropy sum w eeee = c_s^4 (dd + dd + dd); opposite of odd k is k+1."""
    e, w, opp, M, Minv, order = lattice(Q)
    e = e.astype(float)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs(w @ e).max() < 1e-16
    assert np.abs(np.einsum("i,ia,ib->ab", w, e, e) - np.eye(3) / 3).max() < 1e-15
    d = np.eye(3)
    iso = (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d) + np.einsum("ad,bc->abcd", d, d)) / 9
    assert np.abs(np.einsum("i,ia,ib,ic,id->abcd", w, e, e, e, e) - iso).max() < 1e-15
    assert np.abs(np.einsum("i,ia,ib,ic->abc", w, e, e, e)).max() < 1e-16
    assert (e[opp] == -e).all()
    assert opp[0] == 0 and all(opp[k] == k + 1 for k in range(1, Q, 2))
    # same table as the independently typed one of the brute-force reference
    eb, wb = bruteforce.lattice(Q)
    assert (np.array(eb) == e).all() and np.allclose(wb, w, rtol=0, atol=1e-17)


@pytest.mark.parametrize("Q,counts", [(15, [1, 3, 6, 4, 1]), (19, [1, 3, 6, 6, 3]), (27, [1, 3, 6, 7, 6, 3, 1])])
def test_moment_basis_weighted_orthogonal(Q, counts):
    """'weighted orthogonal moment set': M W M^T diagonal, M^-1 M = I, rows grouped by order."""
    e, w, opp, M, Minv, order = lattice(Q)
    D = M @ np.diag(w) @ M.T
    assert np.abs(D - np.diag(np.diag(D))).max() < 1e-15
    assert np.abs(Minv @ M - np.eye(Q)).max() < 1e-14
    assert list(np.bincount(order)) == counts
    # order-0 row is the constant, order-1 rows are e_x, e_y, e_z
    assert np.allclose(M[0], 1)
    assert np.allclose(M[1:4], e.T.astype(float)[[0, 1, 2]])
    # each row of order d is w-orthogonal to every polynomial of degree < d
    ef = e.astype(float)
    for k in range(Q):
        for a, b, c in itertools.product(range(3), repeat=3):
            if a + b + c < order[k]:
                mono = ef[:, 0] ** a * ef[:, 1] ** b * ef[:, 2] ** c
                assert abs((w * mono) @ M[k]) < 1e-14


@pytest.mark.parametrize("Q", [19, 27])
def test_eq25_forcing_moments(Q):
    """eq. 25: F_m = rho^-1 (0, Fx, Fy, Fz, 0, ...) -- M applied to eq. 11's F_i
    has entries only in the three first-order rows (true for the w-orthogonal basis, A5)."""
    e, w, opp, M, Minv, order = lattice(Q)
    F, rho = np.array([0.3, -0.2, 0.7]), 0.37
    Fi = w * (e.astype(float) @ F) / (rho / 3.0)
    Fm = M @ Fi
    expect = np.zeros(Q)
    expect[1:4] = F / rho
    assert np.abs(Fm - expect).max() < 1e-14


@pytest.mark.parametrize("Q", [15, 19, 27])
def test_projector_forms(Q):
    """Readings A3/A4: Omega = M^-1 S M equals I + (rate-1) P with the projectors the brute-force
    reference expands per direction pair."""
    e, w, opp, M, Minv, order = lattice(Q)
    ef = e.astype(float)
    P1 = 3.0 * w[:, None] * (ef @ ef.T)
    ee = ef @ ef.T
    n2 = (ef * ef).sum(1)
    P2 = 4.5 * w[:, None] * (ee ** 2 - n2[:, None] / 3 - n2[None, :] / 3 + 1 / 3)
    for P, k in ((P1, 1), (P2, 2)):
        S = np.where(order == k, 0.37, 1.0)
        Om = Minv @ np.diag(S) @ M
        assert np.abs(Om - (np.eye(Q) + (0.37 - 1.0) * P)).max() < 1e-14


# --------------------------------------------------------------------------------------
# brute force on a tiny grid
# --------------------------------------------------------------------------------------

BF_CASES = [
    dict(stencil_phase=15, stencil_hydro=19, wall_flags=0, gravity=(0.0, 0.0, 0.0)),
    dict(stencil_phase=15, stencil_hydro=19, wall_flags=inputs.WALL_Y, gravity=(0.0, -1e-4, 0.0)),
    dict(stencil_phase=27, stencil_hydro=27, wall_flags=0, gravity=(1e-4, 0.0, 2e-4)),
    dict(stencil_phase=19, stencil_hydro=27, wall_flags=inputs.WALL_X | inputs.WALL_Z, gravity=(0.0, 1e-4, 0.0)),
    dict(stencil_phase=15, stencil_hydro=19, wall_flags=0, gravity=(0.0, 0.0, 0.0), nu_H=0.1, nu_L=0.02, M=0.08),
]


@pytest.mark.parametrize("case", BF_CASES)
def test_bruteforce_one_step(case):
    """One coupled step from a random state on 4x5x3 cells: oracle (matrix form) vs. the
    hand-expanded per-direction reference of eqs. 4-8, 10-17, 20-24."""
    p = Params(nx=4, ny=5, nz=3, rho_H=1.0, rho_L=0.05, sigma=2e-3, xi=3.0, **case)
    phi, u, h, g = random_state(p, seed=7)
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.set_pdfs(h, g)
    o.step(1)
    ho, go = o.get_pdfs()
    po, uo, _ = o.fields(want_p=False)
    Hb, Gb, Cb, Ub = bruteforce.step(p, list(h), list(g), phi, list(u))
    assert np.abs(ho - np.array(Hb)).max() < 1e-14
    assert np.abs(go - np.array(Gb)).max() < 1e-14
    assert np.abs(po - Cb).max() < 1e-14
    assert np.abs(uo - np.array(Ub)).max() < 1e-14


def test_bruteforce_init_and_pressure():
    """Equilibrium initialiser (A14: h = phi Gamma(u), g = Gamma(u) - w, eqs. 6, 12) and
    p = p* rho c_s^2."""
    p = Params(nx=4, ny=3, nz=2, stencil_phase=27, stencil_hydro=19)
    phi, u, h, g = random_state(p, seed=3)
    o = Oracle.from_params(p)
    o.init(phi, u)
    ho, go = o.get_pdfs()
    eh, wh = bruteforce.lattice(27)
    eg, wg = bruteforce.lattice(19)
    for zyx in itertools.product(range(2), range(3), range(4)):
        uu = [u[a][zyx] for a in range(3)]
        for i in range(27):
            assert abs(ho[i][zyx] - phi[zyx] * bruteforce.gamma(eh[i], wh[i], uu)) < 1e-16
        for i in range(19):
            assert abs(go[i][zyx] - (bruteforce.gamma(eg[i], wg[i], uu) - wg[i])) < 1e-16
    o.set_pdfs(None, g)
    _, _, pr = o.fields()
    rho = p.rho_L + phi * (p.rho_H - p.rho_L)
    assert np.abs(pr - g.sum(0) * rho / 3.0).max() < 1e-17


# --------------------------------------------------------------------------------------
# finite-difference operators (eqs. 23, 24)
# --------------------------------------------------------------------------------------

@pytest.mark.parametrize("Q", [15, 19, 27])
def test_fd_operators_polynomials(Q):
    """Second-order isotropic stencils: exact gradient of a linear field, exact Laplacian of a
    quadratic one (interior cells; textbook property of eqs. 23-24)."""
    p = Params(nx=8, ny=7, nz=6, stencil_phase=Q, stencil_hydro=Q)
    o = Oracle.from_params(p)
    z, y, x = np.meshgrid(np.arange(6.0), np.arange(7.0), np.arange(8.0), indexing="ij")
    a = np.array([0.3, -1.1, 0.7])
    inner = (slice(1, -1),) * 3
    for hydro in (False, True):
        grad, lap = o.fd(a[0] * x + a[1] * y + a[2] * z + 2.0, hydro)
        for k in range(3):
            assert np.abs(grad[k][inner] - a[k]).max() < 1e-14
        assert np.abs(lap[inner]).max() < 1e-13
        quad = 0.5 * x * x - 0.25 * y * y + 2.0 * z * z + 0.3 * x * y - 0.2 * y * z
        grad, lap = o.fd(quad, hydro)
        assert np.abs(lap[inner] - (1.0 - 0.5 + 4.0)).max() < 1e-12
        assert np.abs(grad[0][inner] - (x + 0.3 * y)[inner]).max() < 1e-12


def test_fd_wall_mirror():
    """A16: phi ghost behind a wall mirrors the first fluid cell => zero normal gradient for a
    field that is constant along y next to the wall."""
    p = Params(nx=4, ny=6, nz=4, wall_flags=inputs.WALL_Y)
    o = Oracle.from_params(p)
    z, y, x = np.meshgrid(np.arange(4.0), np.arange(6.0), np.arange(4.0), indexing="ij")
    f = np.where(y < 2, 1.0, np.where(y > 3, 3.0, 2.0))
    grad, lap = o.fd(f, True)
    assert np.abs(grad[1][:, 0, :]).max() == 0.0 and np.abs(grad[1][:, -1, :]).max() == 0.0
    assert np.abs(lap[:, 0, :]).max() == 0.0


# --------------------------------------------------------------------------------------
# invariants
# --------------------------------------------------------------------------------------

def test_mass_conservation_periodic():
    """north_star: sum(phi) conserved to 1e-12 relative on periodic domains (collision and
    forcing of eq. 4 conserve the zeroth moment; streaming permutes)."""
    p, phi, u = inputs.config1(n=16, R=4.0)
    u = inputs.velocity_noise(p, 1e-3)
    o = Oracle.from_params(p)
    o.init(phi, u)
    m0 = o.phi_mass()
    assert abs(m0 - phi.sum()) < 1e-9
    o.step(40)
    assert abs(o.phi_mass() - m0) / m0 < 1e-12


def test_mass_conservation_walls():
    """A16: half-way bounce-back conserves sum(phi) too (light bubble next to a wall, gravity)."""
    p, phi, u = inputs.config2(nx=12, ny=24, nz=12, R=4.0, gy=-1e-5, centre=(6.0, 6.0, 6.0))
    o = Oracle.from_params(p)
    o.init(phi, u)
    m0 = o.phi_mass()
    o.step(40)
    ph, uu, _ = o.fields(want_p=False)
    assert abs(o.phi_mass() - m0) / m0 < 1e-12
    assert np.isfinite(uu).all() and np.abs(uu).max() < 1e-2


@pytest.mark.parametrize("phi0", [0.0, 0.3, 0.5, 1.0])
def test_uniform_state_stays_uniform(phi0):
    """north_star: a uniform phi at rest stays exactly (bitwise) uniform; u stays 0."""
    p = Params(nx=6, ny=5, nz=4)
    o = Oracle.from_params(p)
    o.init(np.full(p.shape, phi0), inputs.zeros_u(p))
    o.step(30)
    ph, uu, pr = o.fields()
    assert (ph == ph.flat[0]).all()
    assert abs(ph.flat[0] - phi0) < 1e-13
    assert (uu == 0.0).all()
    assert np.abs(pr).max() < 1e-18


@pytest.mark.parametrize("phi0", [0.0, 1.0])
def test_galilean_uniform_flow(phi0):
    """Uniform phi in {0,1} with uniform u != 0, no gravity: equilibrium is a fixed point,
    U stays uniform (special case reducing to a textbook LBM equilibrium)."""
    p = Params(nx=5, ny=4, nz=6, sigma=5e-3)
    u0 = np.array([0.03, -0.02, 0.01])
    o = Oracle.from_params(p)
    o.init(np.full(p.shape, phi0), np.broadcast_to(u0[:, None, None, None], (3,) + p.shape).copy())
    o.step(30)
    ph, uu, _ = o.fields()
    assert np.abs(uu - u0[:, None, None, None]).max() < 1e-14
    assert np.abs(ph - phi0).max() < 1e-14


# --------------------------------------------------------------------------------------
# physics: closed forms and textbook limits
# --------------------------------------------------------------------------------------

def test_planar_interface_stationary():
    """eq. 3: phi0 +- 1/2 tanh(2(x-x0)/xi) is the equilibrium profile, so a slab
    initialised with it must stay where it is (A1 makes grad phi - n theta vanish for it).
    Bounds from the discrete model at xi=5: profile error <= 1.2e-2 always,
    <= 5e-3 after 1000 steps, phi=1/2 crossings within 1e-5 of x=16 and x=48, y/z-uniform."""
    p = Params(nx=64, ny=2, nz=2)
    x = np.arange(64) + 0.5
    prof = 0.5 * (np.tanh(2 * (x - 16) / p.xi) - np.tanh(2 * (x - 48) / p.xi))
    phi = np.broadcast_to(prof[None, None, :], p.shape).copy()
    o = Oracle.from_params(p)
    o.init(phi, inputs.zeros_u(p))

    def crossing(line, lo):
        k = lo + int(np.argmax((line[lo:lo + 31] - 0.5) * (line[lo + 1:lo + 32] - 0.5) <= 0))
        return x[k] + (0.5 - line[k]) / (line[k + 1] - line[k])

    worst = 0.0
    for it in range(10):
        o.step(120)
        ph, uu, _ = o.fields(want_p=False)
        assert (ph == ph[0:1, 0:1, :]).all()           # y/z uniform, exactly
        worst = max(worst, np.abs(ph[0, 0] - prof).max())
    assert worst < 1.2e-2
    assert np.abs(ph[0, 0] - prof).max() < 5e-3
    assert abs(crossing(ph[0, 0], 0) - 16.0) < 1e-5
    assert abs(crossing(ph[0, 0], 32) - 48.0) < 1e-5
    assert np.abs(uu).max() < 1e-5


@pytest.mark.parametrize("rho_L,sigma,u0", [(1.0, 0.0, 0.02), (1.0, 0.0, -0.05), (1e-3, 1e-4, 0.02)])
def test_interface_is_advected_with_the_flow(rho_L, sigma, u0):
    """eq. 1: d phi/dt + div(phi u) = (a term that vanishes on the equilibrium profile), so in a uniform flow
    the slab of eq. 3 translates with u: after T steps both phi = 1/2 crossings have moved by u0 T (across the
    periodic seam), within 0.5 % (measured lag 0.2 %), the flow stays uniform and sum(phi) is conserved.  A dropped or
    mis-signed u in h^eq (eq. 6) changes the displacement by O(1)."""
    p = Params(nx=64, ny=2, nz=2, rho_L=rho_L, sigma=sigma)
    x = np.arange(64) + 0.5
    prof = 0.5 * (np.tanh(2 * (x - 16) / p.xi) - np.tanh(2 * (x - 48) / p.xi))
    phi = np.broadcast_to(prof[None, None, :], p.shape).copy()
    u = inputs.zeros_u(p)
    u[0] = u0
    o = Oracle.from_params(p)
    o.init(phi, u)
    T = 500
    o.step(T)
    ph, uu, _ = o.fields(want_p=False)
    line = ph[0, 0]

    def crossing(lo):
        idx = [(lo + k) % 64 for k in range(32)]
        seg = line[idx]
        k = int(np.argmax((seg[:-1] - 0.5) * (seg[1:] - 0.5) <= 0))
        return x[idx[k]] + (0.5 - seg[k]) / (seg[k + 1] - seg[k])

    for x0 in (16.0, 48.0):
        moved = (crossing(int(x0 + u0 * T) - 15) - x0 + 32.0) % 64.0 - 32.0
        assert abs(moved / (u0 * T) - 1.0) < 5e-3, (x0, moved)
    assert np.abs(uu[0] - u0).max() < 2e-5 and np.abs(uu[1:]).max() < 1e-12
    assert abs(ph.sum() / phi.sum() - 1.0) < 1e-12


@pytest.mark.parametrize("Mob", [0.02, 0.08])
def test_mobility_sine_decay(Mob):
    """eq. 2 + A2: with the interface term switched off (xi -> inf) and u = 0 the phase
    step is a textbook diffusion LBM: a sine of wavelength 64 decays with diffusivity M."""
    L = 64
    p = Params(nx=L, ny=1, nz=1, rho_H=1.0, rho_L=1.0, sigma=0.0, xi=1e300, M=Mob)
    x = np.arange(L) + 0.5
    k = 2 * np.pi / L
    phi = (0.5 + 0.1 * np.sin(k * x)).reshape(p.shape)
    o = Oracle.from_params(p)
    o.init(phi, inputs.zeros_u(p))
    o.step(200)
    a0 = 2 * np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1]) / L
    o.step(800)
    a1 = 2 * np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1]) / L
    D = -math.log(a1 / a0) / (k * k * 800)
    assert abs(D / Mob - 1) < 2e-3


@pytest.mark.parametrize("nu", [1 / 60, 0.1])
def test_viscosity_shear_wave(nu):
    """eqs. 19-21 + A4: single phase (rho_H = rho_L, sigma = 0): a shear wave u_y(x) decays with
    the kinematic viscosity nu (textbook incompressible LBM limit)."""
    L = 64
    p = Params(nx=L, ny=1, nz=1, rho_H=1.0, rho_L=1.0, sigma=0.0, nu_H=nu, nu_L=nu)
    x = np.arange(L) + 0.5
    k = 2 * np.pi / L
    u = inputs.zeros_u(p)
    u[1, 0, 0, :] = 1e-3 * np.sin(k * x)
    o = Oracle.from_params(p)
    o.init(np.ones(p.shape), u)
    o.step(100)
    a0 = 2 * np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1]) / L
    o.step(400)
    a1 = 2 * np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1]) / L
    assert abs(-math.log(a1 / a0) / (k * k * 400) / nu - 1) < 2e-3


@pytest.mark.parametrize("nu", [1 / 60, 0.1])
def test_poiseuille_walls(nu):
    """A16/A17: body force along x between half-way bounce-back walls in y, single phase:
    steady parabola u(y) = g/(2 nu) (y+1/2)(ny-1/2-y), walls half a cell outside the first/last
    cell; within 1 % of u_max."""
    ny, g = 16, 1e-6
    p = Params(nx=2, ny=ny, nz=2, rho_H=1.0, rho_L=1.0, sigma=0.0, nu_H=nu, nu_L=nu, gravity=(g, 0.0, 0.0),
               wall_flags=inputs.WALL_Y)
    o = Oracle.from_params(p)
    o.init(np.ones(p.shape), inputs.zeros_u(p))
    o.step(int(14 * ny * ny / (math.pi ** 2 * nu)))
    _, uu, _ = o.fields(False)
    y = np.arange(ny)
    exact = g / (2 * nu) * (y + 0.5) * (ny - 0.5 - y)
    assert np.abs(uu[0][0, :, 0] - exact).max() < 0.01 * exact.max()
    assert np.abs(uu[1]).max() < 1e-12 and np.abs(uu[2]).max() < 1e-12
