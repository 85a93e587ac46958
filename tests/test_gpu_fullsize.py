"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot step 8..134 million cells in a test, so one step of the CUDA path is checked on
sampled sub-boxes that the oracle recomputes one by one: the new h, g, phi, u of a cell depend on
the old state within 3 cells (h pulled from 1 cell away, its collision reads phi within 1 cell;
the hydrodynamic kernel reads the NEW phi within 1 cell, which itself came from h 1 cell further),
so the cells of a B^3 sub-box that are at least 3 cells away from its artificial faces are exact.
A sub-box that starts at a real wall keeps that wall (the oracle gets the wall flag), and its cells
next to the wall are compared too.  Plus properties that hold at any size: sum(phi) conserved,
everything finite.
"""
import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2012_06144_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_PDF_1STEP = 1e-13
B = 14


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gather(t, idx):
    return t[(slice(None),) * (t.dim() - 3) + idx].cpu().numpy()


def _boxes(p, starts):
    """index tuples (iz, iy, ix) of the sub-boxes and the slices of each that are exact"""
    n = (p.nz, p.ny, p.nx)
    wall = (p.wall_flags & inputs.WALL_Z, p.wall_flags & inputs.WALL_Y, p.wall_flags & inputs.WALL_X)
    out = []
    for s in starts:
        idx, trust = [], []
        for a in range(3):
            r = torch.arange(s[a], s[a] + B, device="cuda")
            if wall[a]:
                assert 0 <= s[a] <= n[a] - B, "a sub-box must not wrap across a wall"
                lo = 0 if s[a] == 0 else 3
                hi = B if s[a] == n[a] - B else B - 3
            else:
                r = r % n[a]
                lo, hi = 3, B - 3
            idx.append(r)
            trust.append(slice(lo, hi))
        out.append(((idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :]), tuple(trust)))
    return out


def _check_one_step_sampled(p, phi, u, starts, presteps=2, **kw):
    from paper_2012_06144_b200.binding import ACM
    a = ACM.from_params(p, **kw)
    a.init(_dev(phi), _dev(u))
    m0 = a.phi_mass()
    a.step(presteps)
    h0, g0 = a.get_pdfs()
    c0, u0, _ = a.fields(False)
    boxes = _boxes(p, starts)
    olds = [(_gather(h0, ix), _gather(g0, ix), _gather(c0, ix), _gather(u0, ix)) for ix, _ in boxes]
    del h0, g0, c0, u0
    torch.cuda.empty_cache()
    a.step(1)
    h1, g1 = a.get_pdfs()
    c1, u1, _ = a.fields(False)
    pb = p.replace(nx=B, ny=B, nz=B)
    worst = 0.0
    for (ix, trust), (hs, gs, cs, us) in zip(boxes, olds):
        o = Oracle.from_params(pb)
        o.init(cs, us)
        o.set_pdfs(hs, gs)
        o.step(1)
        ho, go = o.get_pdfs()
        po, uo, _ = o.fields(False)
        sl = (slice(None),) + trust
        for got, want, s in ((_gather(h1, ix), ho, sl), (_gather(g1, ix), go, sl), (_gather(c1, ix), po, trust),
                             (_gather(u1, ix), uo, sl)):
            d = float(np.abs(got[s] - want[s]).max())
            worst = max(worst, d)
            assert d <= TOL_PDF_1STEP, d
    assert abs(a.phi_mass() - m0) / m0 < 1e-12
    assert bool(torch.isfinite(c1).all() and torch.isfinite(u1).all())
    return worst


@pytest.mark.parametrize("moments", [False, True], ids=["populations", "moments"])
def test_config2_full_size_walls_gravity(moments):
    """128 x 512 x 128, half-way bounce-back walls in y, gravity: sub-boxes on both walls, on the
    bubble's interface (centre (64,64,64), R=16), across the periodic x/z seams.  moments: the same in moment
    representation (ACM_OPT_MOMENTS, tiled kernels; the populations compared are the ones acm_get_pdfs rebuilds)."""
    p, phi, u = inputs.config2()
    starts = [(0, 0, 0), (p.nz - 7, p.ny - B, p.nx - 7), (57, 0, 57), (57, 41, 57), (57, 73, 57), (57, 57, 73),
              (120, 300, 3), (57, p.ny - B, 57)]
    # z, y, x order
    _check_one_step_sampled(p, phi, u, starts, moments=moments)


@pytest.mark.parametrize("moments", [False, True], ids=["populations", "moments"])
def test_config5_full_size_q27_fp64(moments):
    """256^3 D3Q27 + D3Q27 fp64 (the fp64 leg of config 5)."""
    p, phi, u = inputs.config5()
    cs, rs = inputs.bubble_set(p, 64, 8.0, 14.0)
    starts = [(0, 0, 0), (p.nz - 7, p.ny - 7, p.nx - 7), (37, 201, 118),
              tuple(int(v) - 7 for v in (cs[3] + np.array([0.0, 0.0, rs[3]]))[::-1])]
    _check_one_step_sampled(p, phi, u, starts, moments=moments)


@pytest.mark.parametrize("inplace", [False, True, "moments"])
def test_config4_full_size_512(inplace):
    """512^3 (134 M cells, 64-bit plane offsets: the last h plane starts at element 14*2^27): needs
    ~125 GB of the 180 GB for the two-grid layout plus the exported populations."""
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 150e9:
        pytest.skip("needs a GPU with 150 GB free")
    p, phi, u = inputs.config4()
    cs, rs = inputs.bubble_set(p, 512, 10.0, 16.0)
    n = p.nx
    starts = [(0, 0, 0), (n - 7, n - 7, n - 7), (n - 5, 300, 3), (411, 77, 250),
              tuple(int(v) - 7 for v in (cs[0] + np.array([rs[0], 0.0, 0.0]))[::-1]),
              tuple(int(v) - 7 for v in (cs[100] + np.array([0.0, -rs[100], 0.0]))[::-1])]
    # the in-place pattern alternates two kernels: 2 pre-steps then an odd..even pair is covered by presteps 2 and 3
    if inplace == "moments":      # moment representation: 38.6 GB of workspace instead of 79.5
        _check_one_step_sampled(p, phi, u, starts, moments=True)
    else:
        _check_one_step_sampled(p, phi, u, starts, presteps=3 if inplace else 2, inplace=inplace)
