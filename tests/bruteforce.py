"""Third, independent statement of ONE coupled ACM step for tiny grids (pin for the oracle).

Pure-Python scalar loops, written from PAPER.md eqs. 4-8, 10-17, 20-24 with the
collision operators expanded per direction pair (no moment matrices, no
Gram-Schmidt).  The operators follow from the readings A3/A4 of DESIGN.md:

  phase:  Omega^h_ij = delta_ij + (omega_phi - 1) * 3 w_i (e_i . e_j)
          (the w-orthogonal projector on the first-order moments is 3 w_i e_i.e_j)
  hydro:  Omega^g_ij = delta_ij + (s_nu - 1) * 9/2 w_i [ (e_i.e_j)^2 - |e_i|^2/3 - |e_j|^2/3 + 1/3 ]
          (projector on the six second-order moments x^2-1/3, y^2-1/3, z^2-1/3, xy, xz, yz;
           for D2Q9 the last constant is 2/9: three moments x^2-1/3, y^2-1/3, xy)

Variants (A26, A27):
  bulk_one: the trace moment t_i = |e_i|^2 - D/3 (D = dimension) is taken out of the second-order projector,
          Omega^g_ij = delta_ij + (s_nu - 1) * [ 9/2 w_i (...) - w_i t_i t_j / sum_k w_k t_k^2 ]
  subiter: the velocity of eq. 22 by k sweeps of u <- j + F(u)/(2 rho)

Shares nothing with oracle/ or with the CUDA sources; lattices are re-typed here.
"""
import itertools
import math

CS2 = 1.0 / 3.0


def lattice(Q):
    """Directions in the canonical order (rest, axis pairs, edge pairs, corner pairs) and weights."""
    axis = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    edge = [(1, 1, 0), (-1, -1, 0), (1, -1, 0), (-1, 1, 0), (1, 0, 1), (-1, 0, -1), (1, 0, -1), (-1, 0, 1),
            (0, 1, 1), (0, -1, -1), (0, 1, -1), (0, -1, 1)]
    corner = [(1, 1, 1), (-1, -1, -1), (1, 1, -1), (-1, -1, 1), (1, -1, 1), (-1, 1, -1), (-1, 1, 1), (1, -1, -1)]
    if Q == 9:      # D2Q9: the x-y plane
        e = [(0, 0, 0)] + axis[:4] + edge[:4]
        w = [4 / 9] + [1 / 9] * 4 + [1 / 36] * 4
    elif Q == 15:
        e = [(0, 0, 0)] + axis + corner
        w = [2 / 9] + [1 / 9] * 6 + [1 / 72] * 8
    elif Q == 19:
        e = [(0, 0, 0)] + axis + edge
        w = [1 / 3] + [1 / 18] * 6 + [1 / 36] * 12
    elif Q == 27:
        e = [(0, 0, 0)] + axis + edge + corner
        w = [8 / 27] + [2 / 27] * 6 + [1 / 54] * 12 + [1 / 216] * 8
    else:
        raise ValueError(Q)
    return e, w


def dot(a, b):
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]


def gamma(e, w, u):
    eu = dot(e, u)
    return w * (1.0 + eu / CS2 + eu * eu / (2 * CS2 * CS2) - dot(u, u) / (2 * CS2))


def opposite(e, i):
    return e.index((-e[i][0], -e[i][1], -e[i][2]))


class Grid:
    def __init__(self, nx, ny, nz, walls):
        self.n = (nx, ny, nz)
        self.walls = (bool(walls & 1), bool(walls & 2), bool(walls & 4))

    def cells(self):
        nx, ny, nz = self.n
        return itertools.product(range(nz), range(ny), range(nx))  # (z,y,x), matches numpy (nz,ny,nx)

    def nb(self, zyx, e, s):
        """(z,y,x) of x + s e, or None if beyond a wall."""
        c = [zyx[2] + s * e[0], zyx[1] + s * e[1], zyx[0] + s * e[2]]
        for a in range(3):
            if c[a] < 0 or c[a] >= self.n[a]:
                if self.walls[a]:
                    return None
                c[a] %= self.n[a]
        return (c[2], c[1], c[0])

    def mirror(self, zyx, e, s):
        """(z,y,x) of x + s e with periodic wrap, clamped at walls (phi mirror ghost)."""
        c = [zyx[2] + s * e[0], zyx[1] + s * e[1], zyx[0] + s * e[2]]
        for a in range(3):
            if c[a] < 0 or c[a] >= self.n[a]:
                c[a] = min(max(c[a], 0), self.n[a] - 1) if self.walls[a] else c[a] % self.n[a]
        return (c[2], c[1], c[0])


def grad(grid, e, w, C, zyx):
    g = [0.0, 0.0, 0.0]
    for i in range(1, len(e), 2):
        d = C[grid.mirror(zyx, e[i], 1)] - C[grid.mirror(zyx, e[i], -1)]
        for a in range(3):
            g[a] += w[i] * e[i][a] * d
    return [3.0 * v for v in g]


def laplacian(grid, e, w, C, zyx):
    return 6.0 * sum(w[i] * (C[grid.mirror(zyx, e[i], 1)] - C[zyx]) for i in range(1, len(e)))


def hydro_operator(eg, wg, s, bulk_one=False):
    """Omega^g(i, j) for the relaxation rate s of the second-order moments (see the module docstring)."""
    Qg = len(eg)
    D = 2 if Qg == 9 else 3
    t = [dot(e, e) - D / 3.0 for e in eg]
    tnorm = sum(w * v * v for w, v in zip(wg, t))

    def omega_g(i, j):
        ei, ej = eg[i], eg[j]
        # (e_i e_i - I/3) : (e_j e_j - I/3) with I the unit tensor of the lattice's dimension (trace 3, or 2 for D2Q9)
        p2 = dot(ei, ej) ** 2 - dot(ei, ei) / 3.0 - dot(ej, ej) / 3.0 + D / 9.0
        proj = 4.5 * wg[i] * p2
        if bulk_one:
            proj -= wg[i] * t[i] * t[j] / tnorm
        return (1.0 if i == j else 0.0) + (s - 1.0) * proj
    return omega_g


def hydro_force(par, grid, eg, wg, g, Cn, zyx, u_eq, bulk_one=False):
    """F = F_s + F_p + F_mu + F_b (eqs. 13-18, 30) at one cell, with g^eq(u_eq) inside F_mu.
    Returns (F, rho, j = sum g e, gradient of phi)."""
    Qg = len(eg)
    beta, kappa = 12.0 * par.sigma / par.xi, 1.5 * par.sigma * par.xi
    drho = par.rho_H - par.rho_L
    pstar = sum(g)
    phi = Cn[zyx]
    rho = par.rho_L + phi * drho
    gp = grad(grid, eg, wg, Cn, zyx)
    lap = laplacian(grid, eg, wg, Cn, zyx)
    mu = 4.0 * beta * phi * (phi - 1.0) * (phi - 0.5) - kappa * lap
    gr = [drho * v for v in gp]
    tau = par.nu_L / CS2 + phi * (par.nu_H / CS2 - par.nu_L / CS2)
    omega_g = hydro_operator(eg, wg, 1.0 / (tau + 0.5), bulk_one)
    neq = [g[i] - (pstar * wg[i] + gamma(eg[i], wg[i], u_eq) - wg[i]) for i in range(Qg)]
    relaxed = [sum(omega_g(i, j) * neq[j] for j in range(Qg)) for i in range(Qg)]
    Fmu = [0.0, 0.0, 0.0]
    for a in range(3):
        for b in range(3):
            Pi = sum(eg[k][a] * eg[k][b] * relaxed[k] for k in range(Qg))
            Fmu[a] -= tau * Pi * gr[b]                     # nu/(c_s^2 dt) = tau
    F = [mu * gp[a] - pstar * CS2 * gr[a] + Fmu[a] + rho * par.gravity[a] for a in range(3)]
    j = [sum(g[i] * eg[i][a] for i in range(Qg)) for a in range(3)]
    return F, rho, j, gp


def step(par, H, G, C, U, phase_srt=False, bulk_one=False, subiter=1):
    """One coupled step.  phase_srt: Omega^h = omega_phi I (eq. 4 with a single relaxation time).
     H[Qh], G[Qg]: lists of numpy (nz,ny,nx) arrays; C: array; U: list of 3 arrays.
    Returns new (H, G, C, U) in the oracle's storage convention."""
    import numpy as np
    grid = Grid(par.nx, par.ny, par.nz, par.wall_flags)
    eh, wh = lattice(par.stencil_phase)
    eg, wg = lattice(par.stencil_hydro)
    Qh, Qg = len(eh), len(eg)
    omega = 1.0 / (par.M / CS2 + 0.5)
    beta, kappa = 12.0 * par.sigma / par.xi, 1.5 * par.sigma * par.xi
    tauH, tauL = par.nu_H / CS2, par.nu_L / CS2
    drho = par.rho_H - par.rho_L

    # ---------------- phase-field LB step: pull, phi, forcing, collide ----------------
    Hn = [np.zeros_like(C) for _ in range(Qh)]
    Cn = np.zeros_like(C)
    for zyx in grid.cells():
        ht = []
        for i in range(Qh):
            src = grid.nb(zyx, eh[i], -1)
            ht.append(H[opposite(eh, i)][zyx] if src is None else H[i][src])
        phin = sum(ht)
        g = grad(grid, eh, wh, C, zyx)
        nrm = math.sqrt(dot(g, g))
        n = [v / nrm for v in g] if nrm > 0 else [0.0, 0.0, 0.0]
        theta = (1.0 - 4.0 * (C[zyx] - 0.5) ** 2) / par.xi
        u = [U[a][zyx] for a in range(3)]
        F = [theta * wh[i] * dot(eh[i], n) for i in range(Qh)]
        d = [phin * gamma(eh[i], wh[i], u) - ht[i] - 0.5 * F[i] for i in range(Qh)]
        for i in range(Qh):
            coll = 0.0
            for j in range(Qh):
                if phase_srt:
                    om = omega if i == j else 0.0
                else:
                    om = (1.0 if i == j else 0.0) + (omega - 1.0) * 3.0 * wh[i] * dot(eh[i], eh[j])
                coll += om * d[j]
            Hn[i][zyx] = coll + ht[i] + F[i]
        Cn[zyx] = phin

    # ---------------- hydrodynamic LB step: collide, push ----------------
    Gn = [np.zeros_like(C) for _ in range(Qg)]
    Un = [np.zeros_like(C) for _ in range(3)]
    for zyx in grid.cells():
        g = [G[i][zyx] for i in range(Qg)]
        pstar = sum(g)
        phi = Cn[zyx]
        tau = tauL + phi * (tauH - tauL)
        omega_g = hydro_operator(eg, wg, 1.0 / (tau + 0.5), bulk_one)
        un = [U[a][zyx] for a in range(3)]
        for _ in range(subiter):
            F, rho, j, _ = hydro_force(par, grid, eg, wg, g, Cn, zyx, un, bulk_one)
            un = [j[a] + F[a] / (2.0 * rho) for a in range(3)]
        Fi = [wg[i] * dot(eg[i], F) / (rho * CS2) for i in range(Qg)]
        d = [pstar * wg[i] + gamma(eg[i], wg[i], un) - wg[i] - g[i] - 0.5 * Fi[i] for i in range(Qg)]
        for i in range(Qg):
            post = g[i] + sum(omega_g(i, j) * d[j] for j in range(Qg)) + Fi[i]
            dst = grid.nb(zyx, eg[i], 1)
            if dst is None:
                Gn[opposite(eg, i)][zyx] = post
            else:
                Gn[i][dst] = post
        for a in range(3):
            Un[a][zyx] = un[a]
    return Hn, Gn, Cn, Un
