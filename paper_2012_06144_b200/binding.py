"""Thin Python binding of libacm.so (include/acm.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the
library's CUDA kernels.  There is no fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os

import torch

from . import build as _build

ACM_OK, ACM_EINVAL, ACM_ESTATE, ACM_ECUDA, ACM_EUNSTABLE = 0, 1, 2, 3, 4
ACM_F64, ACM_F32 = 0, 1
ACM_WALL_X, ACM_WALL_Y, ACM_WALL_Z = 1, 2, 4
ACM_OPT_INPLACE, ACM_OPT_PHASE_SRT, ACM_OPT_UNFUSED, ACM_OPT_BULK_ONE, ACM_OPT_MOMENTS = 1, 2, 4, 8, 16

EXPORTS = ["acm_workspace_bytes", "acm_workspace_bytes_opt", "acm_create", "acm_create_opt", "acm_init", "acm_step", "acm_fields", "acm_phi_mass", "acm_get_pdfs",
           "acm_set_pdfs", "acm_run_host", "acm_set_reference_phase", "acm_bubble_diag", "acm_bubble_sums", "acm_slab_range", "acm_workspace_bytes_slab", "acm_create_slab", "acm_slab_info",
           "acm_halo_plan", "acm_set_peers", "acm_state_signature", "acm_phase_launch", "acm_phase_commit", "acm_hydro_launch", "acm_hydro_commit", "acm_bubble_params", "acm_drag_lbm", "acm_drag_exp", "acm_set_block", "acm_set_cells_per_thread", "acm_set_subiter", "acm_set_moment_kernels", "acm_set_graph", "acm_graph_replays", "acm_profile", "acm_profile_read", "acm_launch_count", "acm_destroy", "acm_last_error"]

_lib = None


class AcmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libacm error {code}: {msg}")
        self.code = code


def lib_path() -> str:
    """In-tree libacm.so, or the build named by $ACM_LIB (kernel tuning experiments)."""
    return os.environ.get("ACM_LIB") or _build.LIB


def load(build_if_missing: bool = True):
    """Loads libacm.so (building it with nvcc if it is absent and nvcc exists)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        if not build_if_missing:
            raise RuntimeError(f"{path} is missing: run `python -m paper_2012_06144_b200.build`")
        _build.build_lib()
    lib = C.CDLL(path)
    vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
    lib.acm_workspace_bytes.restype = C.c_size_t
    lib.acm_workspace_bytes.argtypes = [i32] * 6
    lib.acm_create.argtypes = [C.POINTER(vp)] + [i32] * 5 + [dbl] * 7 + [C.POINTER(dbl), C.c_uint, i32, vp, vp]
    lib.acm_workspace_bytes_opt.restype = C.c_size_t
    lib.acm_workspace_bytes_opt.argtypes = [i32] * 6 + [C.c_uint]
    lib.acm_create_opt.argtypes = [C.POINTER(vp)] + [i32] * 5 + [dbl] * 7 + [C.POINTER(dbl), C.c_uint, i32, C.c_uint, vp, vp]
    lib.acm_init.argtypes = [vp, vp, vp]
    lib.acm_step.argtypes = [vp, i32]
    lib.acm_fields.argtypes = [vp, vp, vp, vp]
    lib.acm_phi_mass.argtypes = [vp, C.POINTER(dbl)]
    lib.acm_get_pdfs.argtypes = [vp, vp, vp]
    lib.acm_set_pdfs.argtypes = [vp, vp, vp]
    lib.acm_run_host.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    lib.acm_bubble_diag.argtypes = [vp, C.POINTER(dbl)]
    lib.acm_set_reference_phase.argtypes = [vp, i32]
    lib.acm_bubble_sums.argtypes = [vp, C.POINTER(dbl)]
    lib.acm_slab_range.argtypes = [i32, i32, i32, C.POINTER(i32), C.POINTER(i32)]
    lib.acm_workspace_bytes_slab.restype = C.c_size_t
    lib.acm_workspace_bytes_slab.argtypes = [i32] * 8
    lib.acm_create_slab.argtypes = [C.POINTER(vp)] + [i32] * 5 + [dbl] * 7 + [C.POINTER(dbl), C.c_uint, i32, C.c_uint, i32, i32, vp, vp]
    lib.acm_slab_info.argtypes = [vp, C.POINTER(i32)]
    lib.acm_halo_plan.argtypes = [vp, i32, i32, i32, i32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    lib.acm_set_peers.argtypes = [vp, vp, vp]
    lib.acm_state_signature.argtypes = [vp, C.POINTER(C.c_ulonglong)]
    lib.acm_phase_launch.argtypes = [vp, i32, i32]
    lib.acm_phase_commit.argtypes = [vp]
    lib.acm_hydro_launch.argtypes = [vp, i32, i32]
    lib.acm_hydro_commit.argtypes = [vp]
    lib.acm_bubble_params.argtypes = [dbl] * 7 + [C.POINTER(dbl)]
    lib.acm_drag_lbm.argtypes = [dbl] * 5
    lib.acm_drag_lbm.restype = dbl
    lib.acm_drag_exp.argtypes = [dbl]
    lib.acm_drag_exp.restype = dbl
    lib.acm_set_block.argtypes = [vp, i32, i32, i32]
    lib.acm_set_subiter.argtypes = [vp, i32]
    lib.acm_set_cells_per_thread.argtypes = [vp, i32, i32]
    lib.acm_set_graph.argtypes = [vp, i32]
    lib.acm_set_moment_kernels.argtypes = [vp, i32, i32]
    lib.acm_graph_replays.argtypes = [vp]
    lib.acm_graph_replays.restype = C.c_longlong
    lib.acm_profile.argtypes = [vp, i32]
    lib.acm_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(C.c_longlong)]
    lib.acm_launch_count.argtypes = [vp]
    lib.acm_launch_count.restype = C.c_longlong
    lib.acm_destroy.argtypes = [vp]
    lib.acm_destroy.restype = None
    lib.acm_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _check(lib, rc):
    if rc != ACM_OK:
        raise AcmError(rc, lib.acm_last_error().decode())


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def bubble_params(Re_Gr, Eo, D, t_ref, rho_H=1.0, rho_star=1000.0, mu_star=100.0):
    """acm_bubble_params: lattice parameters from the dimensionless groups of section 6.1."""
    lib = load()
    out = (C.c_double * 5)()
    _check(lib, lib.acm_bubble_params(Re_Gr, Eo, D, t_ref, rho_H, rho_star, mu_star, out))
    return dict(gy=out[0], sigma=out[1], nu_H=out[2], nu_L=out[3], rho_L=out[4])


def drag_lbm(gy, rho_H, rho_L, D, u_t):
    return load().acm_drag_lbm(gy, rho_H, rho_L, D, u_t)


def drag_exp(Re_Gr):
    return load().acm_drag_exp(Re_Gr)


class ACM:
    """One simulation context: acm_create / acm_init / acm_step / acm_fields / acm_phi_mass."""

    def __init__(self, nx, ny, nz, stencil_phase=15, stencil_hydro=19, rho_H=1.0, rho_L=1e-3, sigma=1e-4, xi=5.0,
                 M=0.02, nu_H=1 / 60, nu_L=1 / 60, gravity=(0.0, 0.0, 0.0), wall_flags=0, precision="f64",
                 device="cuda:0", stream=None, inplace=False, phase_srt=False, unfused=False, bulk_one=False, subiter=1,
                 guard_bytes=0, moments=False):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2012_06144_b200 needs a CUDA device (no CPU fallback)")
        self._lib = load()
        self.device = torch.device(device)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.Qh, self.Qg = int(stencil_phase), int(stencil_hydro)
        self.N = self.nx * self.ny * self.nz
        self.shape = (self.nz, self.ny, self.nx)
        self.precision = {"f64": ACM_F64, "f32": ACM_F32}[precision]
        self.dtype = torch.float64 if precision == "f64" else torch.float32
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.options = ((ACM_OPT_INPLACE if inplace else 0) | (ACM_OPT_PHASE_SRT if phase_srt else 0) | (ACM_OPT_UNFUSED if unfused else 0)
                        | (ACM_OPT_BULK_ONE if bulk_one else 0) | (ACM_OPT_MOMENTS if moments else 0))
        nbytes = self._lib.acm_workspace_bytes_opt(self.nx, self.ny, self.nz, self.Qh, self.Qg, self.precision,
                                                   self.options)
        if nbytes == 0:
            raise AcmError(ACM_EINVAL, "invalid grid size / stencil / precision")
        # guard_bytes (debugging aid): canary regions before and after the workspace, see guards_intact()
        self._guard = (int(guard_bytes) + 255) & ~255
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256 + 2 * self._guard, dtype=torch.uint8, device=self.device)
            if self._guard:
                self.workspace.fill_(0xA5)
        base = ((self.workspace.data_ptr() + 255) & ~255) + self._guard
        self._ws_span = (base - self.workspace.data_ptr(), nbytes)
        g = (C.c_double * 3)(*[float(v) for v in gravity])
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = self._lib.acm_create_opt(C.byref(h), self.nx, self.ny, self.nz, self.Qh, self.Qg, rho_H, rho_L, sigma,
                                          xi, M, nu_H, nu_L, g, int(wall_flags), self.precision, self.options,
                                          C.c_void_p(base), C.c_void_p(self.stream.cuda_stream))
        _check(self._lib, rc)
        self._h = h
        if subiter != 1:
            self.set_subiter(subiter)

    @classmethod
    def from_params(cls, p, **kw):
        kw.setdefault("phase_srt", getattr(p, "phase_srt", False))
        return cls(p.nx, p.ny, p.nz, p.stencil_phase, p.stencil_hydro, p.rho_H, p.rho_L, p.sigma, p.xi, p.M, p.nu_H,
                   p.nu_L, p.gravity, p.wall_flags, **kw)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.acm_destroy(self._h)
            self._h = None

    __del__ = close

    def _call(self, fn, *args):
        with torch.cuda.device(self.device):
            _check(self._lib, fn(self._h, *args))

    @contextlib.contextmanager
    def _on_stream(self, *inputs):
        """libacm enqueues on self.stream; torch allocates and the caller computes on torch's CURRENT stream.  When the
        two differ: self.stream first waits for the current stream (inputs are complete before the library reads
        them; their memory is not recycled while it does: record_stream), outputs are allocated under self.stream,
        and the current stream waits for self.stream afterwards (outputs are complete before the caller reads them)."""
        cur = torch.cuda.current_stream(self.device)
        same = cur.cuda_stream == self.stream.cuda_stream
        if not same:
            self.stream.wait_stream(cur)
            for t in inputs:
                if t is not None:
                    t.record_stream(self.stream)
        outputs = []
        with torch.cuda.stream(self.stream):
            yield outputs
        if not same:
            cur.wait_stream(self.stream)
            for t in outputs:          # allocated under self.stream, read by the caller on `cur`
                if t is not None:
                    t.record_stream(cur)

    def _dev(self, t, shape):
        assert t.is_cuda and t.dtype == self.dtype and t.is_contiguous() and tuple(t.shape) == tuple(shape), \
            (t.device, t.dtype, t.shape, shape)
        return _ptr(t)

    def guards_intact(self):
        """True if no byte outside the workspace handed to acm_create was written (needs guard_bytes > 0)."""
        off, n = self._ws_span
        torch.cuda.synchronize(self.device)
        return bool((self.workspace[:off] == 0xA5).all() and (self.workspace[off + n:] == 0xA5).all())

    def set_block(self, bx, by=1, bz=1):
        self._call(self._lib.acm_set_block, int(bx), int(by), int(bz))

    def set_cells_per_thread(self, phase, hydro=None):
        """cells per thread of the phase / hydro kernel: 1, 2 = pair kernels (8/16-byte accesses, packed fp32
        arithmetic), 0 = the library's default (2 for fp32 and for fp64 lattices up to D3Q19, when nx is even)"""
        self._call(self._lib.acm_set_cells_per_thread, int(phase), int(phase if hydro is None else hydro))

    def set_subiter(self, sweeps):
        """sweeps of the fixed point of eq. 22 (1 = single evaluation of F_mu with the previous velocity)"""
        self._call(self._lib.acm_set_subiter, int(sweeps))

    def set_moment_kernels(self, mode=-1, zchunk=0):
        self._call(self._lib.acm_set_moment_kernels, int(mode), int(zchunk))

    def set_graph(self, mode):
        """CUDA graphs of 16 steps in acm_step: -1 automatic (small grids), 0 never, 1 always"""
        self._call(self._lib.acm_set_graph, int(mode))

    @property
    def graph_replays(self):
        return int(self._lib.acm_graph_replays(self._h))

    def set_reference_phase(self, phase):
        """fp32 instance: reference phase of the deviation storage (-1 automatic, 0 light, 1 heavy); before init"""
        self._call(self._lib.acm_set_reference_phase, int(phase))

    def init(self, phi, u):
        with self._on_stream(phi, u):
            self._call(self._lib.acm_init, self._dev(phi, self.shape), self._dev(u, (3,) + self.shape))

    def step(self, n=1):
        self._call(self._lib.acm_step, int(n))

    def fields(self, want_p=True):
        with self._on_stream() as outs:
            phi = torch.empty(self.shape, dtype=self.dtype, device=self.device)
            u = torch.empty((3,) + self.shape, dtype=self.dtype, device=self.device)
            p = torch.empty(self.shape, dtype=self.dtype, device=self.device) if want_p else None
            self._call(self._lib.acm_fields, _ptr(phi), _ptr(u), _ptr(p))
            outs += [phi, u, p]
        return phi, u, p

    def phi_mass(self):
        t = C.c_double()
        self._call(self._lib.acm_phi_mass, C.byref(t))
        return t.value

    def bubble_diag(self):
        """(V, centroid (x,y,z), velocity) of the light phase, weighted with 1 - phi."""
        out = (C.c_double * 7)()
        self._call(self._lib.acm_bubble_diag, out)
        return out[0], tuple(out[1:4]), tuple(out[4:7])

    def get_pdfs(self):
        with self._on_stream() as outs:
            h = torch.empty((self.Qh,) + self.shape, dtype=self.dtype, device=self.device)
            g = torch.empty((self.Qg,) + self.shape, dtype=self.dtype, device=self.device)
            self._call(self._lib.acm_get_pdfs, _ptr(h), _ptr(g))
            outs += [h, g]
        return h, g

    def set_pdfs(self, h=None, g=None):
        hp = None if h is None else self._dev(h, (self.Qh,) + self.shape)
        gp = None if g is None else self._dev(g, (self.Qg,) + self.shape)
        with self._on_stream(h, g):
            self._call(self._lib.acm_set_pdfs, hp, gp)

    def run_host(self, phi_host, u_host, n, phi_out=None, u_out=None, p_out=None):
        """Host buffers in (CPU tensors, ideally pinned), host buffers out; transfers inside."""
        for t in (phi_host, u_host, phi_out, u_out, p_out):
            assert t is None or (not t.is_cuda and t.dtype == self.dtype and t.is_contiguous())
        self._call(self._lib.acm_run_host, _ptr(phi_host), _ptr(u_host), int(n), _ptr(phi_out), _ptr(u_out), _ptr(p_out))

    def profile(self, enable=True):
        self._call(self._lib.acm_profile, int(bool(enable)))

    def profile_read(self):
        """(phase_ms, hydro_ms, steps) summed over the acm_step calls since profile(True)."""
        a, b, n = C.c_double(), C.c_double(), C.c_longlong()
        self._call(self._lib.acm_profile_read, C.byref(a), C.byref(b), C.byref(n))
        return a.value, b.value, n.value

    def state_signature(self):
        """acm_state_signature: what must agree between the slabs of a decomposition in peer mode"""
        out = (C.c_ulonglong * 8)()
        self._call(self._lib.acm_state_signature, out)
        return tuple(out)

    @property
    def launch_count(self):
        return int(self._lib.acm_launch_count(self._h))
