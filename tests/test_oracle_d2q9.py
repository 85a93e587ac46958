"""Pins of the oracle's two-dimensional instance (D2Q9 for both LB steps, one plane; the paper measures it in
Fig. 5).  Same kinds of pins as for the 3-D lattices: lattice identities, weighted-orthogonal basis,
projector forms, brute force on a tiny grid, FD operators on polynomials, invariants, transport coefficients."""
import itertools
import math

import numpy as np
import pytest

import bruteforce
from helpers import random_state
from oracle import Oracle, lattice
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params


def test_d2q9_lattice_identities_and_basis():
    e, w, opp, M, Minv, order = lattice(9)
    ef = e.astype(float)
    assert (e[:, 2] == 0).all()
    assert abs(w.sum() - 1) < 1e-15 and np.abs(w @ ef).max() < 1e-16
    d = np.diag([1.0, 1.0, 0.0])                                  # unit tensor of the plane
    assert np.abs(np.einsum("i,ia,ib->ab", w, ef, ef) - d / 3).max() < 1e-15
    iso = (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d) + np.einsum("ad,bc->abcd", d, d)) / 9
    assert np.abs(np.einsum("i,ia,ib,ic,id->abcd", w, ef, ef, ef, ef) - iso).max() < 1e-15
    assert (e[opp] == -e).all() and all(opp[k] == k + 1 for k in range(1, 9, 2))
    eb, wb = bruteforce.lattice(9)
    assert (np.array(eb) == e).all() and np.allclose(wb, w, rtol=0, atol=1e-17)
    # weighted-orthogonal basis: 1, 2, 3, 2, 1 rows of order 0..4
    D = M @ np.diag(w) @ M.T
    assert np.abs(D - np.diag(np.diag(D))).max() < 1e-15
    assert np.abs(Minv @ M - np.eye(9)).max() < 1e-14
    assert list(np.bincount(order)) == [1, 2, 3, 2, 1]
    # projector forms with the 2-D unit tensor (trace 2)
    ee = ef @ ef.T
    n2 = (ef * ef).sum(1)
    P1 = 3.0 * w[:, None] * ee
    P2 = 4.5 * w[:, None] * (ee ** 2 - n2[:, None] / 3 - n2[None, :] / 3 + 2 / 9)
    for P, k in ((P1, 1), (P2, 2)):
        Om = Minv @ np.diag(np.where(order == k, 0.37, 1.0)) @ M
        assert np.abs(Om - (np.eye(9) + (0.37 - 1.0) * P)).max() < 1e-14
    # eq. 25: the forcing of eq. 11 has first-order moments only
    F, rho = np.array([0.3, -0.2, 0.0]), 0.37
    Fm = M @ (w * (ef @ F) / (rho / 3.0))
    expect = np.zeros(9)
    expect[1:3] = F[:2] / rho
    assert np.abs(Fm - expect).max() < 1e-14


@pytest.mark.parametrize("case", [dict(wall_flags=0, gravity=(0.0, 0.0, 0.0)), dict(wall_flags=inputs.WALL_Y, gravity=(1e-4, -1e-4, 0.0)),
                                  dict(wall_flags=inputs.WALL_X, gravity=(0.0, 1e-4, 0.0), nu_H=0.1, nu_L=0.02, M=0.08)])
@pytest.mark.parametrize("srt", [False, True])
def test_d2q9_bruteforce_one_step(case, srt):
    p = Params(nx=5, ny=4, nz=1, stencil_phase=9, stencil_hydro=9, rho_H=1.0, rho_L=0.05, sigma=2e-3, xi=3.0, **case)
    phi, u, h, g = random_state(p, seed=7)
    u[2] = 0.0
    o = Oracle.from_params(p, phase_srt=srt)
    o.init(phi, u)
    o.set_pdfs(h, g)
    o.step(1)
    ho, go = o.get_pdfs()
    po, uo, _ = o.fields(False)
    Hb, Gb, Cb, Ub = bruteforce.step(p, list(h), list(g), phi, list(u), phase_srt=srt)
    assert np.abs(ho - np.array(Hb)).max() < 1e-14
    assert np.abs(go - np.array(Gb)).max() < 1e-14
    assert np.abs(po - Cb).max() < 1e-14
    assert np.abs(uo - np.array(Ub)).max() < 1e-14
    assert np.abs(uo[2]).max() == 0.0


def test_d2q9_argument_checks():
    with pytest.raises(ValueError):
        Oracle(8, 8, 2, 9, 9)                       # more than one plane
    with pytest.raises(ValueError):
        Oracle(8, 8, 1, 9, 19)                      # mixed 2-D / 3-D lattices
    with pytest.raises(ValueError):
        Oracle(8, 8, 1, 9, 9, gravity=(0.0, 0.0, 1e-6))


def test_d2q9_fd_operators_polynomials():
    p = Params(nx=8, ny=7, nz=1, stencil_phase=9, stencil_hydro=9)
    o = Oracle.from_params(p)
    _, y, x = np.meshgrid(np.arange(1.0), np.arange(7.0), np.arange(8.0), indexing="ij")
    inner = (slice(None), slice(1, -1), slice(1, -1))
    grad, lap = o.fd(0.3 * x - 1.1 * y + 2.0, True)
    assert np.abs(grad[0][inner] - 0.3).max() < 1e-14 and np.abs(grad[1][inner] + 1.1).max() < 1e-14
    assert np.abs(grad[2]).max() == 0.0 and np.abs(lap[inner]).max() < 1e-13
    grad, lap = o.fd(0.5 * x * x - 0.25 * y * y + 0.3 * x * y, False)
    assert np.abs(lap[inner] - 0.5).max() < 1e-12
    assert np.abs(grad[0][inner] - (x + 0.3 * y)[inner]).max() < 1e-12


def test_d2q9_invariants_and_transport():
    # sum(phi) conserved, uniform state stays uniform
    p = Params(nx=24, ny=20, nz=1, stencil_phase=9, stencil_hydro=9)
    phi = inputs.sphere_phi(p, (12.0, 10.0, 0.5), 5.0, heavy_inside=False)       # a disc
    o = Oracle.from_params(p)
    o.init(phi, inputs.zeros_u(p))
    m0 = o.phi_mass()
    o.step(50)
    assert abs(o.phi_mass() - m0) / m0 < 1e-13
    q = Params(nx=6, ny=6, nz=1, stencil_phase=9, stencil_hydro=9)
    o = Oracle.from_params(q)
    o.init(np.full(q.shape, 0.3), inputs.zeros_u(q))
    o.step(20)
    c = o.fields(False)[0]
    assert (c == c.flat[0]).all()
    # shear-wave viscosity and sine-wave mobility (textbook limits, as for the 3-D lattices)
    L, nu, Mob = 64, 1 / 60, 0.02
    k = 2 * np.pi / L
    x = np.arange(L) + 0.5
    p = Params(nx=L, ny=1, nz=1, stencil_phase=9, stencil_hydro=9, rho_H=1.0, rho_L=1.0, sigma=0.0, nu_H=nu, nu_L=nu)
    u = inputs.zeros_u(p)
    u[1, 0, 0, :] = 1e-3 * np.sin(k * x)
    o = Oracle.from_params(p)
    o.init(np.full(p.shape, 0.5), u)
    o.step(200)
    a0 = np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1])
    o.step(800)
    a1 = np.abs(np.fft.rfft(o.fields(False)[1][1].ravel())[1])
    assert abs(-math.log(a1 / a0) / (k * k * 800) / nu - 1) < 2e-3
    p = Params(nx=L, ny=1, nz=1, stencil_phase=9, stencil_hydro=9, rho_H=1.0, rho_L=1.0, sigma=0.0, xi=1e300, M=Mob)
    o = Oracle.from_params(p)
    o.init((0.5 + 0.1 * np.sin(k * x)).reshape(p.shape), inputs.zeros_u(p))
    o.step(200)
    a0 = np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1])
    o.step(800)
    a1 = np.abs(np.fft.rfft(o.fields(False)[0].ravel())[1])
    assert abs(-math.log(a1 / a0) / (k * k * 800) / Mob - 1) < 2e-3
