"""CUDA path vs oracle for the two remaining operator variants of SURVEY.md 8(f)-2 (A26, A27), for the
CUDA-graph replay of acm_step on launch-bound grids, and for the commit guards of the split launches.
Bars as in test_gpu_parity.py: 1e-13 on populations after one step, 1e-10 on fields after 100 steps."""
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
    return ACM.from_params(p, **kw)


def _dev(a, dtype=np.float64):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


CASES = [(150, 7, 5, 15, 27, 0), (70, 9, 6, 15, 19, inputs.WALL_Y), (37, 6, 11, 27, 27, inputs.WALL_X | inputs.WALL_Z),
         (33, 5, 4, 19, 15, 0), (40, 13, 1, 9, 9, inputs.WALL_Y)]


@pytest.mark.parametrize("variant", [dict(bulk_one=True), dict(subiter=3), dict(bulk_one=True, subiter=2, phase_srt=True)])
@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("nx,ny,nz,Qh,Qg,walls", CASES)
def test_variant_one_step(nx, ny, nz, Qh, Qg, walls, inplace, variant):
    grav = (1e-5, -1e-5, 0.0)
    p = Params(nx=nx, ny=ny, nz=nz, stencil_phase=Qh, stencil_hydro=Qg, wall_flags=walls, gravity=grav, rho_L=0.05, sigma=2e-3,
               nu_H=0.05, nu_L=0.2)
    phi, u, h, g = random_state(p, seed=23)
    if nz == 1:
        u[2] = 0.0
    o = Oracle.from_params(p, **variant)
    o.init(phi, u)
    o.set_pdfs(h, g)
    a = _acm(p, inplace=inplace, **variant)
    a.init(_dev(phi), _dev(u))
    a.set_pdfs(_dev(h), _dev(g))
    for _ in range(2):          # two steps: both kernels of the in-place pattern
        o.step(1)
        a.step(1)
        ho, go = o.get_pdfs()
        ha, ga = a.get_pdfs()
        assert np.abs(ha.cpu().numpy() - ho).max() <= TOL_PDF_1STEP
        assert np.abs(ga.cpu().numpy() - go).max() <= TOL_PDF_1STEP
        assert np.abs(a.fields(False)[1].cpu().numpy() - o.fields(False)[1]).max() <= TOL_PDF_1STEP
    # the variant really selects other arithmetic than the default
    b = _acm(p, inplace=inplace, phase_srt=variant.get("phase_srt", False))
    b.init(_dev(phi), _dev(u))
    b.set_pdfs(_dev(h), _dev(g))
    b.step(2)
    assert float((b.get_pdfs()[1] - ga).abs().max()) > 1e-9


@pytest.mark.parametrize("variant", [dict(bulk_one=True), dict(subiter=4)])
def test_variant_100_steps_and_difference_to_default(variant):
    """config-3-like scale model, 100 steps at the plain 1e-10; the measured distance to the default operators is
    what DESIGN.md A4 / A10 quote (it shows the readings are distinguishable, and by how much)."""
    p, phi, u = inputs.scaled_config3(40)
    o = Oracle.from_params(p, **variant)
    o.init(phi, u)
    a = _acm(p, **variant)
    a.init(_dev(phi), _dev(u))
    d = _acm(p)
    d.init(_dev(phi), _dev(u))
    m0 = a.phi_mass()
    o.step(100)
    a.step(100)
    d.step(100)
    po, uo, pro = o.fields()
    pa, ua, pra = a.fields()
    assert np.abs(pa.cpu().numpy() - po).max() <= TOL_FIELD_100
    assert np.abs(ua.cpu().numpy() - uo).max() <= TOL_FIELD_100
    assert np.abs(pra.cpu().numpy() - pro).max() <= TOL_FIELD_100
    assert abs(a.phi_mass() - m0) / m0 < 1e-12
    pd, ud, _ = d.fields(False)
    print("variant", variant, "vs default after 100 steps: max|dphi|", float((pd - pa).abs().max()), "max|du|", float((ud - ua).abs().max()))
    assert float((ud - ua).abs().max()) > 1e-9


def test_variant_fp32_one_step():
    p = Params(nx=70, ny=9, nz=6, stencil_phase=15, stencil_hydro=27, wall_flags=inputs.WALL_Y, rho_L=0.05, sigma=2e-3)
    phi, u, h, g = random_state(p, seed=4)
    f32 = lambda x: np.asarray(x, dtype=np.float32)
    phi, u, h, g = f32(phi), f32(u), f32(h), f32(g)
    o = Oracle.from_params(p, bulk_one=True, subiter=3)
    o.init(phi.astype(np.float64), u.astype(np.float64))
    o.set_pdfs(h.astype(np.float64), g.astype(np.float64))
    a = _acm(p, precision="f32", bulk_one=True, subiter=3)
    a.init(_dev(phi, np.float32), _dev(u, np.float32))
    a.set_pdfs(_dev(h, np.float32), _dev(g, np.float32))
    o.step(1)
    a.step(1)
    ho, go = o.get_pdfs()
    ha, ga = a.get_pdfs()
    assert np.abs(ga.cpu().numpy().astype(np.float64) - go).max() <= 5e-8
    assert np.abs(ha.cpu().numpy().astype(np.float64)[1:] - ho[1:]).max() <= 5e-8


# ------------------------------------------------------------------------------------------
# CUDA graph replay of acm_step
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kw", [dict(), dict(inplace=True), dict(unfused=True), dict(precision="f32")])
def test_graph_replay_is_bit_identical(kw):
    """config 1 (32^3, launch-bound): 100 steps = 6 graph replays of 16 steps + 4 plain steps, against the same
    run with graphs off, bit for bit; odd step counts exercise the second buffer parity."""
    p, phi, u = inputs.config1()
    dt = np.float32 if kw.get("precision") == "f32" else np.float64
    res = []
    for mode in (0, -1):
        a = _acm(p, **kw)
        a.set_graph(mode)
        a.init(_dev(phi, dt), _dev(u, dt))
        l0 = a.launch_count
        for n in (37, 16, 47):
            a.step(n)
        per_step = 6 if kw.get("unfused") else 2
        assert a.launch_count - l0 == 100 * per_step
        assert a.graph_replays == (0 if mode == 0 else 2 + 1 + 2)
        res.append(a.get_pdfs() + a.fields())
    for x, y in zip(*res):
        assert torch.equal(x, y)
    # and against the oracle at the usual bar
    if "precision" not in kw:
        o = Oracle.from_params(p)
        o.init(phi, u)
        o.step(100)
        po, uo, pro = o.fields()
        assert np.abs(res[1][2].cpu().numpy() - po).max() <= TOL_FIELD_100
        assert np.abs(res[1][3].cpu().numpy() - uo).max() <= TOL_FIELD_100


def test_graph_on_a_side_stream_and_after_reinit():
    p, phi, u = inputs.config1()
    s = torch.cuda.Stream()
    from paper_2012_06144_b200.binding import ACM
    with torch.cuda.stream(s):
        a = ACM.from_params(p, stream=s)
        a.init(_dev(phi), _dev(u))
        a.step(40)
        c1 = a.fields(False)[0].clone()
        a.init(_dev(phi), _dev(u))          # graphs are dropped and captured again
        a.step(40)
        c2 = a.fields(False)[0]
        s.synchronize()
    assert a.graph_replays == 4
    assert torch.equal(c1, c2)
    b = _acm(p)
    b.set_graph(0)
    b.init(_dev(phi), _dev(u))
    b.step(40)
    assert torch.equal(b.fields(False)[0], c2)


def test_profile_switches_graphs_off_and_times_every_kernel():
    p, phi, u = inputs.config1()
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    a.profile(True)
    a.step(40)
    a.step(3)
    ph, hy, n = a.profile_read()
    assert n == 43 and ph > 0 and hy > 0 and a.graph_replays == 0
    a.profile(False)
    a.step(32)
    assert a.graph_replays == 2


# ------------------------------------------------------------------------------------------
# split launches: commit guards (Alg. 2 inner / outer order)
# ------------------------------------------------------------------------------------------
def test_commit_guards():
    from paper_2012_06144_b200 import binding
    p, phi, u = inputs.scaled_config3(24)
    a = _acm(p)
    a.init(_dev(phi), _dev(u))
    lib, h = a._lib, a._h
    assert lib.acm_phase_commit(h) == binding.ACM_ESTATE                  # nothing launched
    assert lib.acm_phase_launch(h, 0, 10) == binding.ACM_OK
    assert lib.acm_phase_commit(h) == binding.ACM_ESTATE                  # 10 of 24 planes
    assert lib.acm_hydro_launch(h, 0, 24) == binding.ACM_ESTATE           # phase step not committed
    assert lib.acm_set_block(h, 64, 1, 1) == binding.ACM_ESTATE           # step partly launched
    assert lib.acm_phase_launch(h, 10, 25) == binding.ACM_EINVAL
    assert lib.acm_phase_launch(h, 5, 24) == binding.ACM_ESTATE           # 10 + 19 > 24 planes
    assert lib.acm_phase_launch(h, 10, 24) == binding.ACM_OK
    assert lib.acm_phase_commit(h) == binding.ACM_OK
    assert lib.acm_phase_commit(h) == binding.ACM_ESTATE                  # a second commit
    assert lib.acm_hydro_launch(h, 1, 23) == binding.ACM_OK
    assert lib.acm_hydro_launch(h, 0, 1) == binding.ACM_OK
    assert lib.acm_hydro_commit(h) == binding.ACM_ESTATE
    assert lib.acm_hydro_launch(h, 23, 24) == binding.ACM_OK
    assert lib.acm_hydro_commit(h) == binding.ACM_OK
    # the guarded sequence was one full step: identical to acm_step(1)
    b = _acm(p)
    b.init(_dev(phi), _dev(u))
    b.step(1)
    for x, y in zip(a.get_pdfs() + a.fields(), b.get_pdfs() + b.fields()):
        assert torch.equal(x, y)


def test_context_on_a_side_stream_while_the_caller_uses_another():
    """libacm enqueues on the stream given to acm_create; the caller's tensors live on torch's current stream.  The
    binding orders the two (inputs complete before the library reads them, outputs complete before the caller does)."""
    from paper_2012_06144_b200.binding import ACM
    p, phi, u = inputs.scaled_config3(32)
    side = torch.cuda.Stream()
    a = ACM.from_params(p, stream=side)                 # current stream stays the default one
    big = torch.randn(4096, 4096, device="cuda")
    for _ in range(3):
        big = big @ big * 1e-4                          # keep the current stream busy while the inputs are produced on it
    phi_d = _dev(phi) + 0.0 * big[0, 0].double()
    u_d = _dev(u) + 0.0 * big[1, 1].double()
    a.init(phi_d, u_d)
    del phi_d, u_d
    a.step(10)
    c, uu, pr = a.fields()
    h, g = a.get_pdfs()
    got = [t.clone() for t in (c, uu, pr, h, g)]        # reads on the current stream
    b = _acm(p)
    b.init(_dev(phi), _dev(u))
    b.step(10)
    for x, y in zip(got, b.fields() + b.get_pdfs()):
        assert torch.equal(x, y)
