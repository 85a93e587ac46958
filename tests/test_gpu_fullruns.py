"""The BASELINE.json configurations run for their full step counts on the GPU (the oracle cannot follow at
these sizes; its parity is covered by the scale models and the sampled sub-boxes).  Checked: properties
that hold at any size -- sum(phi) conserved to 1e-12 relative (north_star), fields finite and bounded, phi
stays within the two phases up to the interface overshoot -- and the physics the set-up is about."""
import numpy as np
import pytest
import torch

from paper_2012_06144_b200 import inputs

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run(p, phi, u, steps, **kw):
    from paper_2012_06144_b200.binding import ACM
    a = ACM.from_params(p, **kw)
    a.init(_dev(phi), _dev(u))
    m0 = a.phi_mass()
    a.step(steps)
    m1 = a.phi_mass()
    c, uu, pr = a.fields()
    assert abs(m1 - m0) / m0 < 1e-12
    assert bool(torch.isfinite(c).all() and torch.isfinite(uu).all() and torch.isfinite(pr).all())
    assert float(c.min()) > -0.05 and float(c.max()) < 1.05
    assert float(uu.abs().max()) < 0.1          # far below the lattice speed of sound
    return a, c, uu, pr


def test_config2_rising_bubble_2000_steps():
    """128 x 512 x 128, walls in y, g_y = -1e-6: after 2000 steps the light bubble has started to rise (+y),
    symmetrically in x and z, and its volume is unchanged."""
    p, phi, u = inputs.config2()
    from paper_2012_06144_b200.binding import ACM
    a0 = ACM.from_params(p)
    a0.init(_dev(phi), _dev(u))
    V0, X0, U0 = a0.bubble_diag()
    del a0
    a, c, uu, pr = _run(p, phi, u, 2000)
    V1, X1, U1 = a.bubble_diag()
    assert abs(V1 / V0 - 1) < 0.1            # sum(phi) is conserved exactly; this weighted volume follows the relaxing interface
    assert U1[1] > 1e-4                                           # rising against gravity
    print("config2 after 2000 steps: V", V0, V1, "X", X0, X1, "U", U1)
    assert 0.5 < X1[1] - X0[1] < 4.0                              # about u_b * t: a couple of cells
    assert abs(X1[0] - X0[0]) < 1e-3 and abs(X1[2] - X0[2]) < 1e-3          # mirror symmetry in x and z (up to the noise of "Conditioning")
    assert abs(U1[0]) < 1e-3 * U1[1] and abs(U1[2]) < 1e-3 * U1[1]
    # hydrostatic pressure builds up in the heavy liquid: higher at the bottom than at the top
    assert float(pr[64, 5, 10] - pr[64, 500, 10]) > 0


def test_config3_headline_500_steps():
    p, phi, u = inputs.config3()
    a, c, uu, pr = _run(p, phi, u, 500)
    # the velocity noise (1e-3) has been damped by viscosity; the 64 bubbles are still there
    assert float(uu.abs().max()) < 1e-3
    assert abs(float((c < 0.5).double().mean()) / float((torch.from_numpy(phi) < 0.5).double().mean()) - 1) < 0.02


def test_config5_q27_500_steps_fp64_and_fp32_agree():
    """config 5 at full size: the fp32 run against the fp64 run of the CUDA path (which is tied to the oracle
    elsewhere) after 500 steps, 1e-5 on phi and u as BASELINE.json asks.  This needs the deviation storage of the
    fp32 instance (A22): with phi and h stored as they are the bulk of the heavy liquid (phi = 1 - 1e-4)
    carries 6e-8 of rounding noise per step, which the ill-conditioned interface normal there (DESIGN.md
    "Conditioning") amplifies to 2.4e-5 in 500 steps; forcing the light phase as reference reproduces that."""
    from paper_2012_06144_b200.binding import ACM
    p, phi, u = inputs.config5()
    phi32, u32 = phi.astype(np.float32), u.astype(np.float32)
    a64, c64, v64, _ = _run(p, phi, u, 500)
    out = {}
    for ref in (-1, 0):
        a32 = ACM.from_params(p, precision="f32")
        a32.set_reference_phase(ref)
        a32.init(_dev(phi32), _dev(u32))
        m0 = a32.phi_mass()
        a32.step(500)
        c32, v32, _ = a32.fields(False)
        out[ref] = (float((c32.double() - c64).abs().max()), float((v32.double() - v64).abs().max()))
        assert abs(a32.phi_mass() - m0) / m0 < 1e-6
        assert bool(torch.isfinite(c32).all() and torch.isfinite(v32).all())
        del a32, c32, v32
    print("config5 fp32 vs fp64 after 500 steps (max |dphi|, max |du|): reference phase automatic (heavy)", out[-1], " light", out[0])
    assert out[-1][0] <= 1e-5 and out[-1][1] <= 1e-5
    assert out[0][0] > out[-1][0]           # the plain storage is the worse one on this workload


def test_config4_512_100_steps():
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info()[0] < 110e9:
        pytest.skip("needs 110 GB of free device memory")
    p, phi, u = inputs.config4()
    _run(p, phi, u, 100)
