"""ACM_OPT_MOMENTS: the two fused kernels in moment representation (the workspace holds the coefficients
A, b (, T) of the post-collision state instead of the populations; include/acm.h) against the CPU oracle, at
the bars of the population path: max|d pdf| <= 1e-13 per step, max|d phi|, |d u|, |d p| <= 1e-10 after 100
steps.  acm_set_pdfs does not exist in this mode (arbitrary populations have no such representation), so the
one-step comparisons start from acm_init on a rough state (wavy phi, velocity noise of 0.02) and follow the
populations over the first steps: step 1 runs the LOCAL instance of the hydrodynamic kernel (g is defined
pre-collision at its cell, A13 / A14), the later ones the pulling instance."""
import dataclasses

import numpy as np
import pytest
import torch

from helpers import random_state
from oracle import Oracle
from paper_2012_06144_b200 import inputs
from paper_2012_06144_b200.inputs import Params

pytestmark = pytest.mark.gpu

TOL_PDF_1STEP = 1e-13
TOL_FIELD_100 = 1e-10


def _acm(p, **kw):
    from paper_2012_06144_b200.binding import ACM
    kw.setdefault("moments", True)
    return ACM.from_params(p, **kw)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _fields_diff(o, a):
    po, uo, pro = o.fields()
    pa, ua, pra = a.fields()
    return (np.abs(pa.cpu().numpy() - po).max(), np.abs(ua.cpu().numpy() - uo).max(), np.abs(pra.cpu().numpy() - pro).max())


def _pdf_diff(o, a):
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    return np.abs(ha.cpu().numpy() - ho).max(), np.abs(ga.cpu().numpy() - go).max()


SHAPES = [
    # (nx, ny, nz, Qh, Qg, walls, gravity, block)   -- ragged sizes spanning several blocks
    (150, 7, 5, 15, 19, 0, (0.0, 0.0, 0.0), (128, 1, 1)),
    (70, 9, 6, 15, 19, inputs.WALL_Y, (0.0, -1e-5, 0.0), (32, 2, 2)),
    (37, 6, 11, 27, 27, 0, (1e-5, 0.0, 2e-5), (32, 4, 2)),
    (33, 5, 4, 19, 27, inputs.WALL_X | inputs.WALL_Z, (0.0, 1e-5, 0.0), (64, 1, 1)),
    (20, 12, 9, 27, 19, inputs.WALL_X | inputs.WALL_Y | inputs.WALL_Z, (0.0, 0.0, -1e-5), (32, 2, 1)),
    (16, 8, 8, 15, 15, 0, (0.0, 0.0, 0.0), (16, 4, 4)),
    (3, 2, 2, 27, 27, 0, (0.0, 0.0, 0.0), (32, 1, 1)),
    (1, 1, 1, 15, 19, 0, (0.0, 0.0, 0.0), (32, 1, 1)),
    (2, 5, 1, 19, 19, inputs.WALL_X | inputs.WALL_Y | inputs.WALL_Z, (1e-5, 0.0, 0.0), (32, 1, 1)),
]


@pytest.mark.parametrize("march", [0, 1, 3], ids=["direct", "march", "march-zchunk3"])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls,grav,block", SHAPES)
def test_first_steps_pdf_parity(nx, ny, nz, Qh, Qg, walls, grav, block, march):
    """march: the tiled kernels (marching phase-field kernel, pushing / marching hydrodynamic kernel; shared-memory
    window) forced on these small ragged grids -- one tile wider than the grid, several tiles with a ragged last one, z
    ranges of one chunk and of chunks of 3 planes with a ragged last one.  (Odd nx: the direct kernels run.)"""
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=grav,
               rho_H=1.0, rho_L=1e-3, sigma=1e-4, nu_H=0.05, nu_L=1 / 60)
    phi, u, _, _ = random_state(p, seed=11)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p)
    a.set_block(*block)
    a.set_moment_kernels(1 if march else 0, march if march > 1 else 0)
    a.init(_dev(phi), _dev(u))
    dh, dg = _pdf_diff(o, a)
    assert dh <= 1e-15 and dg <= 1e-15, (dh, dg)
    pa, ua, _ = a.fields()
    assert (pa.cpu().numpy() == phi).all() and (ua.cpu().numpy() == u).all()
    for k in (1, 2, 3, 4):
        o.step(1)
        a.step(1)
        dh, dg = _pdf_diff(o, a)
        assert dh <= k * TOL_PDF_1STEP and dg <= k * TOL_PDF_1STEP, (k, dh, dg)
        assert max(_fields_diff(o, a)) <= k * TOL_PDF_1STEP


@pytest.mark.parametrize("march", [0, 1], ids=["direct", "march"])
@pytest.mark.parametrize("case", ["config1", "walls", "config3", "config5", "mu100"])
def test_100_steps(case, march):
    """phi, u, p within 1e-10 of the oracle after 99 and 100 steps; sum(phi) conserved."""
    if case == "config1":
        p, phi, u = inputs.config1()
    elif case == "walls":
        p = Params(nx=24, ny=20, nz=28, gravity=(0.0, -1e-6, 0.0), wall_flags=inputs.WALL_X | inputs.WALL_Y | inputs.WALL_Z)
        phi, u = inputs.sphere_phi(p, (12.0, 9.0, 14.0), 6.0, heavy_inside=True), inputs.zeros_u(p)
    elif case == "config3":
        p, phi, u = inputs.scaled_config3(40)
    elif case == "config5":
        p, phi, u = inputs.scaled_config3(32, stencil_phase=27, stencil_hydro=27)
    else:      # viscosity contrast of section 6 (mu* = 100)
        p, phi, u = inputs.scaled_config3(32)
        p = dataclasses.replace(p, nu_H=1 / 60, nu_L=1 / 6)
    o = Oracle.from_params(p)
    o.init(phi, u)
    a = _acm(p)
    a.set_moment_kernels(march, 0)
    a.init(_dev(phi), _dev(u))
    o.step(99)
    a.step(99)
    assert max(_fields_diff(o, a)) <= TOL_FIELD_100
    o.step(1)
    a.step(1)
    assert max(_fields_diff(o, a)) <= TOL_FIELD_100
    assert max(_pdf_diff(o, a)) <= TOL_FIELD_100
    m0 = phi.sum()
    assert abs(a.phi_mass() - m0) / m0 < 1e-12
    assert abs(a.phi_mass() - o.phi_mass()) / m0 < 1e-13


@pytest.mark.parametrize("march", [0, 1], ids=["direct", "march"])
def test_d2q9_100_steps(march):
    p = Params(nx=48, ny=40, nz=1, stencil_phase=9, stencil_hydro=9, wall_flags=inputs.WALL_Y, gravity=(1e-6, 0.0, 0.0))
    phi = inputs.sphere_phi(p, (24.0, 17.0, 0.5), 9.0, heavy_inside=True)
    o = Oracle.from_params(p)
    o.init(phi, inputs.zeros_u(p))
    a = _acm(p)
    a.set_moment_kernels(march, 0)
    a.init(_dev(phi), _dev(inputs.zeros_u(p)))
    for n in (1, 1, 98):
        o.step(n)
        a.step(n)
        assert max(_pdf_diff(o, a)) <= TOL_FIELD_100
    assert max(_fields_diff(o, a)) <= TOL_FIELD_100


@pytest.mark.parametrize("variant", ["bulk_one", "subiter3", "both"])
def test_operator_variants(variant):
    """A26 (bulk moment relaxed with 1) and A27 (sub-iterated velocity) in moment representation."""
    p, phi, u = inputs.scaled_config3(24)
    kw = dict(bulk_one=variant in ("bulk_one", "both"), subiter=3 if variant in ("subiter3", "both") else 1)
    o = Oracle.from_params(p, **kw)
    o.init(phi, u)
    a = _acm(p, **kw)
    a.set_moment_kernels(1, 7)
    a.init(_dev(phi), _dev(u))
    o.step(1)
    a.step(1)
    assert max(_pdf_diff(o, a)) <= TOL_PDF_1STEP
    o.step(49)
    a.step(49)
    assert max(_fields_diff(o, a)) <= TOL_FIELD_100


def test_uniform_state_exact():
    """north_star invariant: uniform phi at rest stays bitwise uniform, u = 0."""
    p = Params(nx=64, ny=6, nz=5)
    a = _acm(p)
    a.init(_dev(np.full(p.shape, 0.3)), _dev(inputs.zeros_u(p)))
    a.step(30)
    pa, ua, _ = a.fields()
    pa = pa.cpu().numpy()
    assert (pa == pa.flat[0]).all() and abs(pa.flat[0] - 0.3) < 1e-13
    assert (ua.cpu().numpy() == 0).all()


def test_graph_replay_is_bit_identical():
    """acm_step through the CUDA graph of 16 steps (the state right after acm_init differs from the one every
    completed step leaves: LOCAL first hydrodynamic kernel, both velocity buffers equal) equals plain launches."""
    p, phi, u = inputs.scaled_config3(24)
    res = []
    for mode in (0, 1):
        a = _acm(p)
        a.set_graph(mode)
        a.init(_dev(phi), _dev(u))
        a.step(37)          # 2 replays + 5 plain steps (graph), or 37 plain steps
        a.step(16)
        a.step(1)
        assert (a.graph_replays > 0) == (mode == 1)
        pa, ua, pra = a.fields()
        h, g = a.get_pdfs()
        res.append([t.cpu().numpy() for t in (pa, ua, pra, h, g)])
    for x, y in zip(*res):
        assert (x == y).all()


def test_same_trajectory_as_the_population_kernels():
    """Both storage forms follow the same time step: after 100 steps they differ by rounding only, whichever kernels
    advance the moment representation (walls on one axis, ragged tiles).  The chunking of the z range matters in the last
    place only (the first plane of a chunk is expanded by a second inlined copy of the same expressions, in which the
    compiler contracts multiply-adds differently: measured 1e-19 on u after 3 steps, confined to the chunk boundaries)."""
    p, phi, u = inputs.scaled_config3(36)
    p = dataclasses.replace(p, wall_flags=inputs.WALL_Z, gravity=(0.0, 0.0, -1e-6))
    out = []
    for moments, tiled, zchunk in ((False, 0, 0), (True, 0, 0), (True, 1, 0), (True, 1, 5)):
        a = _acm(p, moments=moments)
        if moments:
            a.set_moment_kernels(tiled, zchunk)
        a.init(_dev(phi), _dev(u))
        a.step(100)
        out.append([t.cpu().numpy() for t in a.fields()] + [t.cpu().numpy() for t in a.get_pdfs()])
    for other in out[1:]:
        for x, y in zip(out[0], other):
            assert np.abs(x - y).max() <= 1e-12
    for x, y in zip(out[2], out[3]):
        assert np.abs(x - y).max() <= 1e-13


def test_workspace_and_errors():
    from paper_2012_06144_b200 import binding
    lib = binding.load()
    n = 32
    full = lib.acm_workspace_bytes_opt(n, n, n, 15, 19, 0, 0)
    mom = lib.acm_workspace_bytes_opt(n, n, n, 15, 19, 0, binding.ACM_OPT_MOMENTS)
    # 2 (4 + 10) + 2 + 6 planes instead of 2 (15 + 19) + 2 + 3, the same for every lattice
    assert full - mom == (2 * (15 + 19 - 14) - 3) * n ** 3 * 8
    assert lib.acm_workspace_bytes_opt(n, n, n, 27, 27, 0, binding.ACM_OPT_MOMENTS) == mom
    # fp64 only; not with in-place streaming, Algorithm 1 or the SRT phase-field collision
    assert lib.acm_workspace_bytes_opt(n, n, n, 15, 19, 1, binding.ACM_OPT_MOMENTS) == 0
    for other in (binding.ACM_OPT_INPLACE, binding.ACM_OPT_UNFUSED, binding.ACM_OPT_PHASE_SRT):
        assert lib.acm_workspace_bytes_opt(n, n, n, 15, 19, 0, binding.ACM_OPT_MOMENTS | other) == 0
    p, phi, u = inputs.config1(n=8, R=2.0)
    with pytest.raises(binding.AcmError) as e:
        _acm(p, inplace=True)
    assert e.value.code == binding.ACM_EINVAL
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    h, g = a.get_pdfs()
    with pytest.raises(binding.AcmError) as e:
        a.set_pdfs(h, g)
    assert e.value.code == binding.ACM_EINVAL
    for fn in (lib.acm_phase_launch, lib.acm_hydro_launch):
        assert fn(a._h, 0, p.nz) == binding.ACM_ESTATE
    with pytest.raises(binding.AcmError) as e:
        a.set_cells_per_thread(2, 2)
    assert e.value.code == binding.ACM_EINVAL
    a.step(3)       # still usable after the refused calls
    assert np.isfinite(a.phi_mass())


def test_run_host_matches_step():
    p, phi, u = inputs.scaled_config3(24)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    a.step(7)
    ref = [t.cpu().numpy() for t in a.fields()]
    b = _acm(p)
    outs = [torch.empty(p.shape, dtype=torch.float64).pin_memory(), torch.empty((3,) + p.shape, dtype=torch.float64).pin_memory(),
            torch.empty(p.shape, dtype=torch.float64).pin_memory()]
    b.run_host(torch.from_numpy(phi).pin_memory(), torch.from_numpy(u).pin_memory(), 7, *outs)
    for x, y in zip(ref, outs):
        assert (x == y.numpy()).all()
