"""The C-ABI library builds, loads and exports every symbol include/acm.h declares (no GPU needed)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "acm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(acm_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported():
    from paper_2012_06144_b200 import binding, build
    path = build.build_lib()
    lib = ctypes.CDLL(path)
    names = _declared()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_workspace_bytes_and_argument_checks():
    """Host-only entry points: size arithmetic and acm_create argument validation (no kernel runs)."""
    from paper_2012_06144_b200 import binding
    lib = binding.load()
    N = 32 ** 3
    b = lib.acm_workspace_bytes(32, 32, 32, 15, 19, 0)
    payload = (2 * (15 + 19) + 2 + 3 + 5) * N * 8
    assert payload <= b <= payload + 16 * 256 + 7 * 593 * 8 + 256      # + reduction scratch
    assert lib.acm_workspace_bytes(32, 32, 32, 15, 19, 1) < b
    assert lib.acm_workspace_bytes(0, 32, 32, 15, 19, 0) == 0
    assert lib.acm_workspace_bytes(32, 32, 32, 13, 19, 0) == 0
    assert lib.acm_workspace_bytes(2048, 2048, 2048, 15, 19, 0) == 0      # >= 2^31 cells
    h = ctypes.c_void_p()
    g = (ctypes.c_double * 3)(0, 0, 0)
    fake_ws = ctypes.c_void_p(256 * 1000)

    def create(**kw):
        a = dict(nx=8, ny=8, nz=8, qh=15, qg=19, rho_H=1.0, rho_L=1e-3, sigma=1e-4, xi=5.0, M=0.02, nu_H=1 / 60,
                 nu_L=1 / 60, walls=0, prec=0, ws=fake_ws)
        a.update(kw)
        return lib.acm_create(ctypes.byref(h), a["nx"], a["ny"], a["nz"], a["qh"], a["qg"], a["rho_H"], a["rho_L"],
                              a["sigma"], a["xi"], a["M"], a["nu_H"], a["nu_L"], g, a["walls"], a["prec"], a["ws"], None)

    for bad in (dict(nx=0), dict(qh=9), dict(rho_L=0.0), dict(rho_H=1e-4), dict(xi=0.0), dict(M=0.0), dict(nu_L=-1.0),
                dict(walls=8), dict(prec=2), dict(ws=None), dict(ws=ctypes.c_void_p(8)), dict(sigma=-1.0)):
        assert create(**bad) == binding.ACM_EINVAL, bad
        assert h.value is None
        assert len(lib.acm_last_error()) > 0
    assert create() == binding.ACM_OK and h.value
    assert lib.acm_step(h, 1) == binding.ACM_ESTATE          # before acm_init
    assert lib.acm_step(h, -1) == binding.ACM_EINVAL
    assert lib.acm_launch_count(h) == 0
    # a commit without the launches of a full step is refused (Alg. 2's inner / outer order)
    assert lib.acm_phase_commit(h) == binding.ACM_ESTATE and b"0 of 8" in lib.acm_last_error()
    assert lib.acm_hydro_commit(h) == binding.ACM_ESTATE
    assert lib.acm_phase_launch(h, 0, 8) == binding.ACM_ESTATE        # before acm_init
    # operator variants and CUDA-graph switch: argument checks
    assert lib.acm_set_subiter(h, 0) == binding.ACM_EINVAL and lib.acm_set_subiter(h, 65) == binding.ACM_EINVAL
    assert lib.acm_set_subiter(h, 3) == binding.ACM_OK and lib.acm_set_subiter(h, 1) == binding.ACM_OK
    assert lib.acm_set_graph(h, 2) == binding.ACM_EINVAL and lib.acm_set_graph(h, -1) == binding.ACM_OK
    assert lib.acm_graph_replays(h) == 0
    lib.acm_destroy(h)
    h2 = ctypes.c_void_p()

    def create_opt(options):
        return lib.acm_create_opt(ctypes.byref(h2), 8, 8, 8, 15, 19, 1.0, 1e-3, 1e-4, 5.0, 0.02, 1 / 60, 1 / 60, g, 0, 0, options,
                                  fake_ws, None)
    assert create_opt(binding.ACM_OPT_BULK_ONE | binding.ACM_OPT_UNFUSED) == binding.ACM_EINVAL
    assert create_opt(32) == binding.ACM_EINVAL                       # unknown option bit
    # moment representation: fp64 two-grid fused kernels with the MRT phase-field collision only
    for other in (binding.ACM_OPT_INPLACE, binding.ACM_OPT_UNFUSED, binding.ACM_OPT_PHASE_SRT):
        assert create_opt(binding.ACM_OPT_MOMENTS | other) == binding.ACM_EINVAL
    assert lib.acm_workspace_bytes_opt(8, 8, 8, 15, 19, 1, binding.ACM_OPT_MOMENTS) == 0
    assert create_opt(binding.ACM_OPT_MOMENTS | binding.ACM_OPT_BULK_ONE) == binding.ACM_OK
    assert lib.acm_set_moment_kernels(h2, 2, 0) == binding.ACM_EINVAL and lib.acm_set_moment_kernels(h2, 1, -1) == binding.ACM_EINVAL
    assert lib.acm_set_moment_kernels(h2, 1, 16) == binding.ACM_OK and lib.acm_set_moment_kernels(h2, -1, 0) == binding.ACM_OK
    assert lib.acm_set_cells_per_thread(h2, 2, 2) == binding.ACM_EINVAL
    lib.acm_destroy(h2)
    assert create_opt(binding.ACM_OPT_BULK_ONE | binding.ACM_OPT_INPLACE | binding.ACM_OPT_PHASE_SRT) == binding.ACM_OK
    lib.acm_destroy(h2)
    assert create_opt(binding.ACM_OPT_UNFUSED) == binding.ACM_OK
    assert lib.acm_set_subiter(h2, 2) == binding.ACM_EINVAL           # Algorithm 1 evaluates the forces in two kernels
    assert lib.acm_set_moment_kernels(h2, 1, 0) == binding.ACM_ESTATE  # not a moment-representation context
    lib.acm_destroy(h2)


def test_host_only_bubble_helpers_match_oracle():
    """acm_bubble_params / acm_drag_* are host functions (eqs. 31-35): compared with the oracle's
    own statement of the same equations; argument checks."""
    from oracle import oracle as om
    from paper_2012_06144_b200 import binding
    for Re, Eo, D, t_ref, rs, ms in ((35.0, 30.0, 32.0, 18000.0, 1000.0, 100.0), (50.0, 50.0, 32.0, 18000.0, 1000.0, 100.0),
                                     (5.0, 1.0, 20.0, 6000.0, 10.0, 1.0)):
        a = binding.bubble_params(Re, Eo, D, t_ref, 1.0, rs, ms)
        o = om.bubble_params(Re, Eo, D, t_ref, 1.0, rs, ms)
        for k in o:
            assert abs(a[k] - o[k]) <= 1e-15 * abs(o[k]), k
        assert abs(binding.drag_exp(Re) - om.drag_exp(Re)) < 1e-14
        assert abs(binding.drag_lbm(a["gy"], 1.0, a["rho_L"], D, 1e-3) / om.drag_lbm(o["gy"], 1.0, o["rho_L"], D, 1e-3) - 1) < 1e-15
    lib = binding.load()
    out = (ctypes.c_double * 5)()
    assert lib.acm_bubble_params(0.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0, out) == binding.ACM_EINVAL
    assert lib.acm_bubble_params(1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0, None) == binding.ACM_EINVAL
