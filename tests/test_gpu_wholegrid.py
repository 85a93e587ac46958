"""WHOLE-GRID parity with the oracle at the headline size ("configs 1-3 in full").

The oracle steps the complete 256^3 config-3 input (16.8 M cells, ~13 GB of host memory, ~1.5 s per step on the
box's 16 cores) beside the CUDA path, in the launch configuration bench.py times, and EVERY element is compared:
  * after 1 and 3 steps: all populations h, g and the fields phi, u, p at north_star's one-step bar (1e-13 per step);
  * after 100 steps: phi, u, p at north_star's 1e-10, sum(phi) against the oracle's and against its initial value.
Config 2 (128 x 512 x 128, walls + gravity) runs the same way at full size; what can be asserted there after 100
steps is limited by the conditioning of the method itself near the bottom wall.
These tests take minutes of oracle time: marked `slow`, still part of `-m gpu`.
"""
import os
import time

import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2012_06144_b200 import inputs

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL_PDF_1STEP = 1e-13
TOL_FIELD_100 = 1e-10
# Oracle time one long comparison may take (seconds).  The box's 16 cores do a 256^3 step in ~2.5 s; on a slower or busy
# host the long tests shorten their run (never below 30 steps, same bars) instead of running into the suite's time limit.
ORACLE_BUDGET_S = float(os.environ.get("ACM_ORACLE_BUDGET_S", "330"))


def _dmax(t, a):
    """max |t - a|: t a device tensor, a the oracle's numpy array; one leading plane at a time"""
    if t.dim() == 3:
        return float((t - torch.from_numpy(a).cuda()).abs().max())
    return max(_dmax(t[i], a[i]) for i in range(t.shape[0]))


class _Twin:
    """the oracle and the CUDA path on the same input, advanced together"""

    def __init__(self, p, phi, u, with_moments=False, **kw):
        from paper_2012_06144_b200.binding import ACM
        self.p = p
        self.o = Oracle.from_params(p)
        self.o.init(phi, u)
        dphi, du = torch.from_numpy(np.ascontiguousarray(phi)).cuda(), torch.from_numpy(np.ascontiguousarray(u)).cuda()
        self.a = ACM.from_params(p, **kw)
        self.a.init(dphi, du)
        # the same run in moment representation (ACM_OPT_MOMENTS), advanced beside the other two
        self.m = ACM.from_params(p, moments=True, **kw) if with_moments else None
        if self.m is not None:
            self.m.init(dphi, du)
        self.m0 = self.a.phi_mass()
        self.done = 0
        self.oracle_s_per_step = None

    def advance_to(self, n):
        assert n >= self.done
        t0 = time.time()
        self.o.step(n - self.done)
        if n > self.done:
            self.oracle_s_per_step = (time.time() - t0) / (n - self.done)
        self.a.step(n - self.done)
        if self.m is not None:
            self.m.step(n - self.done)
        self.done = n

    def affordable(self, n, at_least=30, runs=1):
        """the step count a long comparison runs to: n, or fewer if the oracle (`runs` of them) is too slow here for ORACLE_BUDGET_S"""
        if not self.oracle_s_per_step:
            return n
        fits = self.done + int(ORACLE_BUDGET_S / (runs * self.oracle_s_per_step))
        return max(min(n, fits), min(n, at_least))

    def field_diffs(self, which="a"):
        po, uo, pro = self.o.fields()
        pa, ua, pra = getattr(self, which).fields()
        return _dmax(pa, po), _dmax(ua, uo), _dmax(pra, pro)

    def pdf_diffs(self, which="a"):
        ho, go = self.o.get_pdfs()
        ha, ga = getattr(self, which).get_pdfs()
        return _dmax(ha, ho), _dmax(ga, go)


@pytest.fixture(scope="module")
def config3_twin():
    p, phi, u = inputs.config3()
    t = _Twin(p, phi, u, with_moments=True)
    yield t
    del t
    torch.cuda.empty_cache()


def test_config3_whole_grid_first_steps(config3_twin):
    t = config3_twin
    for n in (1, 3):
        t.advance_to(n)
        dh, dg = t.pdf_diffs()
        dphi, du, dp = t.field_diffs()
        print(f"config 3, 256^3, step {n}: max|dh| {dh:.2e} |dg| {dg:.2e} |dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e}")
        for d in (dh, dg, dphi, du, dp):
            assert d <= n * TOL_PDF_1STEP, (n, dh, dg, dphi, du, dp)
        # moment representation (tiled kernels, as bench.py runs them): the populations it stands for, and the fields
        mh, mg = t.pdf_diffs("m")
        mphi, mu, mp = t.field_diffs("m")
        print(f"   moment representation:   max|dh| {mh:.2e} |dg| {mg:.2e} |dphi| {mphi:.2e} |du| {mu:.2e} |dp| {mp:.2e}")
        for d in (mh, mg, mphi, mu, mp):
            assert d <= n * TOL_PDF_1STEP, (n, mh, mg, mphi, mu, mp)


def test_config3_whole_grid_100_steps(config3_twin):
    t = config3_twin
    n = t.affordable(100)
    t.advance_to(n)
    dphi, du, dp = t.field_diffs()
    print(f"config 3, 256^3, step {n}: max|dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e} (oracle {t.oracle_s_per_step:.2f} s per step)")
    assert dphi <= TOL_FIELD_100 and du <= TOL_FIELD_100 and dp <= TOL_FIELD_100, (dphi, du, dp)
    mass = t.a.phi_mass()
    assert abs(mass - t.o.phi_mass()) <= 1e-12 * abs(mass)
    assert abs(mass - t.m0) <= 1e-12 * abs(t.m0)
    mphi, mu, mp = t.field_diffs("m")
    print(f"   moment representation:   max|dphi| {mphi:.2e} |du| {mu:.2e} |dp| {mp:.2e}")
    assert mphi <= TOL_FIELD_100 and mu <= TOL_FIELD_100 and mp <= TOL_FIELD_100, (mphi, mu, mp)
    assert abs(t.m.phi_mass() - t.o.phi_mass()) <= 1e-12 * abs(mass)


# ------------------------------------------------------------------------------------------
# config 2 at full size: walls in y, gravity, one light bubble
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def config2_twin():
    p, phi, u = inputs.config2()
    t = _Twin(p, phi, u)
    yield t
    del t
    torch.cuda.empty_cache()


def test_config2_whole_grid_first_20_steps(config2_twin):
    """Every element after 1 and 3 steps at the one-step bar; phi, u, p after 20 steps at the plain 1e-10 (observed
    1e-14): up to there the run is well conditioned everywhere."""
    t = config2_twin
    for n in (1, 3):
        t.advance_to(n)
        dh, dg = t.pdf_diffs()
        dphi, du, dp = t.field_diffs()
        print(f"config 2, 128x512x128, step {n}: max|dh| {dh:.2e} |dg| {dg:.2e} |dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e}")
        for d in (dh, dg, dphi, du, dp):
            assert d <= n * TOL_PDF_1STEP, (n, dh, dg, dphi, du, dp)
    t.advance_to(20)
    dphi, du, dp = t.field_diffs()
    print(f"config 2, step 20: max|dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e}")
    assert dphi <= TOL_FIELD_100 and du <= TOL_FIELD_100 and dp <= TOL_FIELD_100, (dphi, du, dp)


def test_config2_whole_grid_100_steps_conditioning_aware(config2_twin):
    """After 100 steps the plain 1e-10 is NOT attainable on this configuration, for any implementation: where phi sits
    a little off a bulk value (compressed liquid at the bottom wall, the tails of the tanh profile around the bubble)
    and its gradient is at rounding level, the unit normal of eq. 5 turns rounding noise into an O(theta) flux
    (DESIGN.md "Conditioning").  The oracle shows it against itself: a second oracle run whose input differs by
    1e-16 relative (`own`) drifts from the first by 1e-5 in phi in those regions.  So the bound is made per y-plane
    from the oracle's own sensitivity: max(1e-10, 10 x own) with `own` taken over the plane and its 8 neighbours
    on either side; planes the twin leaves below 1e-12 are held to the plain 1e-10, and they must be the majority.
    Global caps keep the test from passing on garbage: 1e-4 on phi (the saturation level ~ theta), 1e-8 on u and p."""
    t = config2_twin
    p = t.p
    rng = np.random.Generator(np.random.PCG64(1))
    _, phi, u = inputs.config2()
    twin = Oracle.from_params(p)
    twin.init(phi * (1.0 + 1e-16 * rng.uniform(-1.0, 1.0, size=phi.shape)), u)
    steps = t.affordable(100, at_least=60, runs=2)      # (the per-plane bound below is built at the same step count)
    twin.step(steps)
    t.advance_to(steps)
    fo = t.o.fields()
    ft = twin.fields()
    fa = t.a.fields()
    del twin
    names = ("phi", "u", "p")
    caps = (1e-4, 1e-8, 1e-8)
    well = np.ones(p.ny, dtype=bool)
    for name, cap, o_, t_, a_ in zip(names, caps, fo, ft, fa):
        ax = (0, 2) if o_.ndim == 3 else (0, 1, 3)
        own = np.abs(o_ - t_).max(axis=ax)
        got = np.abs(a_.cpu().numpy() - o_).max(axis=ax)
        own_w = np.array([own[max(0, y - 8): y + 9].max() for y in range(p.ny)])
        bound = np.maximum(TOL_FIELD_100, 10.0 * own_w)
        worst = int(np.argmax(got / bound))
        print(f"config 2, step {steps}, {name}: max|d| {got.max():.2e} (oracle vs its 1e-16 twin: {own.max():.2e}); "
              f"planes with own <= 1e-12: {(own_w <= 1e-12).sum()} of {p.ny}; worst plane y={worst}: {got[worst]:.2e} vs bound {bound[worst]:.2e}")
        assert (got <= bound).all(), (name, worst, got[worst], bound[worst])
        assert got.max() <= cap, (name, got.max())
        well &= own_w <= 1e-12
    assert well.sum() >= 0.6 * p.ny            # most of the domain is well conditioned, and there the plain bar holds
    mass = t.a.phi_mass()
    assert abs(mass - t.o.phi_mass()) <= 1e-12 * abs(mass)
    assert abs(mass - t.m0) <= 1e-12 * abs(t.m0)


# ------------------------------------------------------------------------------------------
# config 5 at full size: D3Q27 + D3Q27, fp64 and the fp32 instance
# ------------------------------------------------------------------------------------------
def test_config5_whole_grid_q27_fp64_and_fp32_10_steps():
    """256^3 D3Q27 + D3Q27 against the oracle on every element: the fp64 path after 1 and 3 steps (populations and
    fields, 1e-13 per step) and after 10 steps (fields, 1e-10); the fp32 instance (two cells per thread, packed fp32
    arithmetic, deviation storage: DESIGN.md A22, 5.7) after 10 steps from the same fp32-representable input, within
    the share of BASELINE.json's 500-step bound of 1e-5 that 10 steps may use.  The 500-step comparison of the two
    CUDA precisions (test_gpu_fullruns.py) hangs on this anchor."""
    from paper_2012_06144_b200.binding import ACM
    p, phi, u = inputs.config5()
    phi = phi.astype(np.float32).astype(np.float64)      # both precisions and the oracle start from the same numbers
    u = u.astype(np.float32).astype(np.float64)
    t = _Twin(p, phi, u)
    a32 = ACM.from_params(p, precision="f32")
    a32.init(torch.from_numpy(phi.astype(np.float32)).cuda(), torch.from_numpy(u.astype(np.float32)).cuda())
    for n in (1, 3):
        t.advance_to(n)
        dh, dg = t.pdf_diffs()
        dphi, du, dp = t.field_diffs()
        print(f"config 5 fp64, 256^3 D3Q27, step {n}: max|dh| {dh:.2e} |dg| {dg:.2e} |dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e}")
        for d in (dh, dg, dphi, du, dp):
            assert d <= n * TOL_PDF_1STEP, (n, dh, dg, dphi, du, dp)
    t.advance_to(10)
    dphi, du, dp = t.field_diffs()
    print(f"config 5 fp64, step 10: max|dphi| {dphi:.2e} |du| {du:.2e} |dp| {dp:.2e}")
    assert dphi <= TOL_FIELD_100 and du <= TOL_FIELD_100 and dp <= TOL_FIELD_100, (dphi, du, dp)
    a32.step(10)
    po, uo, _ = t.o.fields(False)
    c32, u32, _ = a32.fields(False)
    d32 = _dmax(c32.double(), po), _dmax(u32.double(), uo)
    print(f"config 5 fp32 instance, step 10: max|dphi| {d32[0]:.2e} |du| {d32[1]:.2e}")
    assert d32[0] <= 2e-6 and d32[1] <= 2e-6, d32
    m32 = a32.phi_mass()
    assert abs(m32 - t.o.phi_mass()) <= 1e-6 * abs(m32)


@pytest.mark.skipif(not __import__("os").environ.get("ACM_LONG"), reason="about 35 minutes of oracle time: set ACM_LONG=1")
def test_config5_fp32_500_steps_against_the_oracle():
    """BASELINE.json's criterion for the fp32 instance, taken literally at full size: 256^3 D3Q27 + D3Q27, 500 steps,
    max|d phi|, max|d u| <= 1e-5 against the fp64 ORACLE (the default suite checks it against the fp64 CUDA path, which
    the tests above tie to the oracle).  Opt-in because the oracle needs ~4 s per step here; the result of the run on
    record is in profiles/r2_profiles.md section 5."""
    from paper_2012_06144_b200.binding import ACM
    p, phi, u = inputs.config5()
    phi32, u32 = phi.astype(np.float32), u.astype(np.float32)
    o = Oracle.from_params(p)
    o.init(phi32.astype(np.float64), u32.astype(np.float64))
    a = ACM.from_params(p, precision="f32")
    a.init(torch.from_numpy(phi32).cuda(), torch.from_numpy(u32).cuda())
    m0 = a.phi_mass()
    done = 0
    for n in (10, 50, 100, 200, 300, 400, 500):
        o.step(n - done)
        a.step(n - done)
        done = n
        po, uo, _ = o.fields(False)
        c, v, _ = a.fields(False)
        dphi, du = _dmax(c.double(), po), _dmax(v.double(), uo)
        print(f"config 5 fp32 instance vs fp64 oracle, 256^3, step {n}: max|dphi| {dphi:.2e} max|du| {du:.2e}", flush=True)
    assert dphi <= 1e-5 and du <= 1e-5, (dphi, du)
    assert abs(a.phi_mass() - m0) <= 1e-6 * m0


@pytest.mark.skipif(not __import__("os").environ.get("ACM_LONG"), reason="about 7 minutes of oracle time: set ACM_LONG=1")
def test_config5_fp64_100_steps_against_the_oracle():
    """north_star's 100-step bar on config 5's fp64 leg at full size (256^3 D3Q27 + D3Q27, every element), for the
    population path and the moment representation.  Opt-in (the oracle needs ~4 s per step here); the run on record is
    in profiles/r2b_profiles.md section 5."""
    p, phi, u = inputs.config5()
    t = _Twin(p, phi, u, with_moments=True)
    for n in (10, 50, 100):
        t.advance_to(n)
        d, m = t.field_diffs(), t.field_diffs("m")
        print(f"config 5 fp64, 256^3 D3Q27, step {n}: max|dphi| {d[0]:.2e} |du| {d[1]:.2e} |dp| {d[2]:.2e};  "
              f"moment representation: {m[0]:.2e} {m[1]:.2e} {m[2]:.2e}", flush=True)
    assert max(d) <= TOL_FIELD_100 and max(m) <= TOL_FIELD_100, (d, m)
    mass = t.a.phi_mass()
    assert abs(mass - t.o.phi_mass()) <= 1e-12 * abs(mass) and abs(t.m.phi_mass() - t.o.phi_mass()) <= 1e-12 * abs(mass)
