"""The seeded input generators (paper_2012_06144_b200/inputs.py): deterministic, the shapes / layout the ABI expects,
and the structure DESIGN.md section 3 states (non-overlapping bubbles with 2 xi clearance, volume fraction of a few
per cent, velocity noise within its amplitude).  No arithmetic of the method lives there."""
import numpy as np

from paper_2012_06144_b200 import inputs


def test_generators_are_deterministic_and_well_formed():
    for make in (lambda: inputs.config1(), lambda: inputs.scaled_config3(32), lambda: inputs.scaled_config3(24, 27, 27),
                 lambda: inputs.config2(nx=16, ny=64, nz=16, R=4.0, centre=(8.0, 12.0, 8.0)), lambda: inputs.paper_benchmark(n=20),
                 lambda: inputs.disc2d(n=64, count=4, r_min=4.0, r_max=7.0)):
        p, phi, u = make()
        p2, phi2, u2 = make()
        assert p == p2 and np.array_equal(phi, phi2) and np.array_equal(u, u2)
        assert phi.shape == (p.nz, p.ny, p.nx) and u.shape == (3, p.nz, p.ny, p.nx)
        assert phi.dtype == np.float64 and u.dtype == np.float64 and phi.flags.c_contiguous and u.flags.c_contiguous
        assert 0.0 <= phi.min() and phi.max() <= 1.0 and np.abs(u).max() <= 1e-3


def test_bubble_set_structure():
    p = inputs.Params(nx=96, ny=96, nz=96)
    c, r = inputs.bubble_set(p, 12, 4.0, 7.0)
    assert c.shape == (12, 3) and r.shape == (12,) and (r >= 4.0).all() and (r <= 7.0).all()
    L = np.array([p.nx, p.ny, p.nz], dtype=float)
    for i in range(12):
        for j in range(i):
            d = np.abs(c[i] - c[j])
            d = np.minimum(d, L - d)
            assert np.sqrt((d * d).sum()) >= r[i] + r[j] + 2.0 * p.xi
    phi = inputs.bubbles_phi(p, c, r)
    frac = (phi < 0.5).mean()
    assert abs(frac / (4.0 / 3.0 * np.pi * (r ** 3).sum() / p.ncells) - 1) < 0.05      # light volume = the spheres'
    # the fast per-bubble evaluation equals the plain definition phi = 1/2 + 1/2 tanh(2 min_b(d_b - R_b)/xi)
    x, y, z = inputs.cell_centres(p)
    dmin = np.full(p.shape, np.inf)
    for cb, rb in zip(c, r):
        dd = [np.minimum(np.abs(q - v), n - np.abs(q - v)) for q, v, n in ((x, cb[0], p.nx), (y, cb[1], p.ny), (z, cb[2], p.nz))]
        dmin = np.minimum(dmin, np.sqrt(dd[0] ** 2 + dd[1] ** 2 + dd[2] ** 2) - rb)
    assert np.abs(phi - (0.5 + 0.5 * np.tanh(2.0 * dmin / p.xi))).max() < 1e-15      # same up to the order of the sum under the root


def test_headline_workload_recipe():
    """config 3 at the benchmark size: 64 bubbles, R in [8, 14], about 2 % light phase, noise of 1e-3 (only shape and
    statistics are checked here; building the 256^3 field takes a second)."""
    p, phi, u = inputs.config3()
    assert (p.nx, p.ny, p.nz, p.stencil_phase, p.stencil_hydro, p.wall_flags) == (256, 256, 256, 15, 19, 0)
    assert 0.01 < (phi < 0.5).mean() < 0.04
    assert 0.9e-3 < np.abs(u).max() <= 1e-3 and abs(u.mean()) < 1e-6
