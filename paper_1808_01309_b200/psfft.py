"""Thin Python binding of libpsfft (include/psfft.h).  Argument marshalling only.

Same names as the C ABI (``plan_query``, ``plan_create``, ``fft3d_r2c``, ``fft3d_c2r``, ``hd_rhs``,
``mhd_rhs``, ...).  PyTorch supplies device memory and streams and nothing else: every step of the
path runs in the library's own kernels.  There is no fallback: if ``libpsfft.so`` is missing or a
call returns a non-zero code, this module raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

F32, F64 = 0, 1
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpsfft.so")

EXPORTS = [
    "psfft_plan_query", "psfft_plan_create", "psfft_plan_query3", "psfft_plan_create3", "psfft_plan_destroy",
    "psfft_plan_layout", "psfft_plan_set_box",
    "psfft_fft3d_r2c", "psfft_fft3d_c2r", "psfft_fft3d_c2r_static", "psfft_hd_rhs", "psfft_mhd_rhs", "psfft_boussinesq_rhs", "psfft_gpe_rhs",
    "psfft_rk_work_bytes", "psfft_rk_step",
    "psfft_hd_rhs_unfused", "psfft_mhd_rhs_unfused",
    "psfft_slab_query", "psfft_slab_r2c_xy", "psfft_slab_z", "psfft_slab_c2r_yx",
    "psfft_fft3d_r2c_host", "psfft_fft3d_c2r_host", "psfft_hd_rhs_host",
    "psfft_hd_rhs_host_box", "psfft_host_box_bytes",
    "psfft_profile_enable", "psfft_profile_reset", "psfft_profile_count", "psfft_profile_get",
    "psfft_kernel_name", "psfft_last_launch_count", "psfft_strerror", "psfft_version",
]


class PsfftError(RuntimeError):
    pass


class Layout(ctypes.Structure):
    """Mirror of ``psfft_layout``."""
    _fields_ = [("N", ctypes.c_int), ("dtype", ctypes.c_int), ("batch", ctypes.c_int), ("ldk", ctypes.c_int),
                ("real_elems", ctypes.c_size_t), ("spec_elems", ctypes.c_size_t),
                ("real_bytes", ctypes.c_size_t), ("spec_bytes", ctypes.c_size_t),
                ("table_bytes", ctypes.c_size_t), ("work_bytes_fft", ctypes.c_size_t),
                ("work_bytes_hd", ctypes.c_size_t), ("work_bytes_mhd", ctypes.c_size_t),
                ("work_bytes_boussinesq", ctypes.c_size_t), ("Ny", ctypes.c_int), ("Nz", ctypes.c_int),
                ("work_bytes_gpe", ctypes.c_size_t)]


MAX_RANKS = 16


class SlabLayout(ctypes.Structure):
    """Mirror of ``psfft_slab_layout``."""
    _fields_ = [("P", ctypes.c_int), ("rank", ctypes.c_int), ("Mz", ctypes.c_int), ("z0", ctypes.c_int),
                ("w", ctypes.c_int), ("x0", ctypes.c_int * (MAX_RANKS + 1)),
                ("real_elems", ctypes.c_size_t), ("real_bytes", ctypes.c_size_t),
                ("zspec_elems", ctypes.c_size_t), ("zspec_bytes", ctypes.c_size_t),
                ("xslab_elems", ctypes.c_size_t), ("xslab_bytes", ctypes.c_size_t)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libpsfft.so (built in-tree by ``paper_1808_01309_b200.build``).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PsfftError(f"{LIB_PATH} not found: run `python -m paper_1808_01309_b200.build` "
                             "(there is no CPU or PyTorch fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        L.psfft_plan_query.argtypes = [ci, ci, ci, ctypes.POINTER(Layout)]
        L.psfft_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, vp, sz, vp]
        L.psfft_plan_query3.argtypes = [ci, ci, ci, ci, ci, ctypes.POINTER(Layout)]
        L.psfft_plan_create3.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, vp, sz, vp]
        L.psfft_plan_destroy.argtypes = [vp]
        L.psfft_plan_layout.argtypes = [vp, ctypes.POINTER(Layout)]
        L.psfft_plan_set_box.argtypes = [vp, cd, cd, cd]
        L.psfft_fft3d_r2c.argtypes = [vp, vp, vp, vp, vp]
        L.psfft_fft3d_c2r.argtypes = [vp, vp, vp, vp, vp]
        L.psfft_fft3d_c2r_static.argtypes = [vp, vp, vp, vp]
        L.psfft_hd_rhs.argtypes = [vp, vp, vp, cd, vp, vp]
        L.psfft_mhd_rhs.argtypes = [vp, vp, vp, vp, vp, cd, cd, vp, vp]
        L.psfft_boussinesq_rhs.argtypes = [vp, vp, vp, vp, vp, cd, cd, cd, vp, vp]
        L.psfft_gpe_rhs.argtypes = [vp, vp, vp, cd, cd, vp, vp]
        L.psfft_rk_work_bytes.argtypes = [vp, ci]
        L.psfft_rk_work_bytes.restype = sz
        L.psfft_rk_step.argtypes = [vp, ci, vp, vp, ci, cd, ctypes.POINTER(cd), vp, vp]
        L.psfft_hd_rhs_unfused.argtypes = [vp, vp, vp, cd, vp, vp]
        L.psfft_mhd_rhs_unfused.argtypes = [vp, vp, vp, vp, vp, cd, cd, vp, vp]
        cl = ctypes.c_long
        L.psfft_slab_query.argtypes = [vp, ci, ci, ctypes.POINTER(SlabLayout)]
        L.psfft_slab_r2c_xy.argtypes = [vp, ci, ci, vp, vp, ctypes.POINTER(vp), cl, vp]
        L.psfft_slab_z.argtypes = [vp, ci, ci, ci, vp, vp]
        L.psfft_slab_c2r_yx.argtypes = [vp, ci, ci, ctypes.POINTER(vp), cl, vp, vp, vp]
        L.psfft_fft3d_r2c_host.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.psfft_fft3d_c2r_host.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.psfft_hd_rhs_host.argtypes = [vp, vp, vp, cd, vp, vp, vp, vp]
        L.psfft_hd_rhs_host_box.argtypes = [vp, vp, vp, cd, vp, vp, vp, vp]
        L.psfft_host_box_bytes.argtypes = [vp]
        L.psfft_host_box_bytes.restype = sz
        L.psfft_profile_enable.argtypes = [vp, ci]
        L.psfft_profile_reset.argtypes = [vp]
        L.psfft_profile_count.argtypes = [vp]
        L.psfft_profile_get.argtypes = [vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd), ctypes.POINTER(cd)]
        L.psfft_kernel_name.argtypes = [ci]
        L.psfft_kernel_name.restype = ctypes.c_char_p
        L.psfft_last_launch_count.argtypes = [vp]
        L.psfft_strerror.argtypes = [ci]
        L.psfft_strerror.restype = ctypes.c_char_p
        L.psfft_version.restype = ctypes.c_char_p
        for name in EXPORTS:
            if getattr(L, name).restype is None:
                getattr(L, name).restype = ci
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().psfft_strerror(int(code)).decode()


def _check(code: int, what: str) -> None:
    if code != 0:
        raise PsfftError(f"{what} failed with code {code}: {strerror(code)}")


def _ptr(t) -> int:
    if t is None:
        return 0
    if isinstance(t, torch.Tensor):
        return t.data_ptr()
    return int(t)


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


# ---- the C ABI, one function per entry point ------------------------------------------------------

def plan_query(N: int, dtype: int, batch: int = 1) -> Layout:
    lay = Layout()
    _check(lib().psfft_plan_query(N, dtype, batch, ctypes.byref(lay)), "psfft_plan_query")
    return lay


def plan_create(N: int, dtype: int, batch: int, d_tables, table_bytes: int, stream=None) -> int:
    h = ctypes.c_void_p()
    _check(lib().psfft_plan_create(ctypes.byref(h), N, dtype, batch, _ptr(d_tables), table_bytes, _stream(stream)),
           "psfft_plan_create")
    return h.value


def plan_query3(Nx: int, Ny: int, Nz: int, dtype: int, batch: int = 1) -> Layout:
    lay = Layout()
    _check(lib().psfft_plan_query3(Nx, Ny, Nz, dtype, batch, ctypes.byref(lay)), "psfft_plan_query3")
    return lay


def plan_create3(Nx: int, Ny: int, Nz: int, dtype: int, batch: int, d_tables, table_bytes: int, stream=None) -> int:
    h = ctypes.c_void_p()
    _check(lib().psfft_plan_create3(ctypes.byref(h), Nx, Ny, Nz, dtype, batch, _ptr(d_tables), table_bytes,
                                    _stream(stream)), "psfft_plan_create3")
    return h.value


def plan_set_box(plan: int, Lx: float, Ly: float, Lz: float) -> None:
    _check(lib().psfft_plan_set_box(plan, float(Lx), float(Ly), float(Lz)), "psfft_plan_set_box")


def plan_destroy(plan: int) -> None:
    _check(lib().psfft_plan_destroy(plan), "psfft_plan_destroy")


def fft3d_r2c(plan: int, d_real, d_spec, d_work=None, stream=None) -> None:
    _check(lib().psfft_fft3d_r2c(plan, _ptr(d_real), _ptr(d_spec), _ptr(d_work), _stream(stream)), "psfft_fft3d_r2c")


def fft3d_c2r(plan: int, d_spec, d_real, d_work, stream=None) -> None:
    _check(lib().psfft_fft3d_c2r(plan, _ptr(d_spec), _ptr(d_real), _ptr(d_work), _stream(stream)), "psfft_fft3d_c2r")


STATIC_SCRATCH_BYTES = 32 << 20      # PSFFT_STATIC_SCRATCH_BYTES
E_SCRATCH = -9                       # PSFFT_E_SCRATCH


def fft3d_c2r_static(plan: int, d_spec, d_real, stream=None) -> None:
    """``psfft_fft3d_c2r`` without a caller workspace, for callers that cannot allocate device memory: the
    workspace is a 32 MiB array inside libpsfft.so (one per GPU, shared by all calls -- calls that overlap on the
    GPU race; plans with work_bytes_fft above the limit are refused with code -9).  See include/psfft.h."""
    _check(lib().psfft_fft3d_c2r_static(plan, _ptr(d_spec), _ptr(d_real), _stream(stream)), "psfft_fft3d_c2r_static")


def hd_rhs(plan: int, d_uhat, d_rhs, nu: float, d_work, stream=None) -> None:
    _check(lib().psfft_hd_rhs(plan, _ptr(d_uhat), _ptr(d_rhs), float(nu), _ptr(d_work), _stream(stream)),
           "psfft_hd_rhs")


def mhd_rhs(plan: int, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu: float, eta: float, d_work, stream=None) -> None:
    _check(lib().psfft_mhd_rhs(plan, _ptr(d_uhat), _ptr(d_bhat), _ptr(d_rhs_u), _ptr(d_rhs_b), float(nu), float(eta),
                               _ptr(d_work), _stream(stream)), "psfft_mhd_rhs")


def boussinesq_rhs(plan: int, d_uhat, d_thhat, d_rhs_u, d_rhs_th, nu: float, kappa: float, nbv: float, d_work,
                   stream=None) -> None:
    _check(lib().psfft_boussinesq_rhs(plan, _ptr(d_uhat), _ptr(d_thhat), _ptr(d_rhs_u), _ptr(d_rhs_th), float(nu),
                                      float(kappa), float(nbv), _ptr(d_work), _stream(stream)), "psfft_boussinesq_rhs")


SYS_HD, SYS_MHD, SYS_BOUSSINESQ, SYS_GPE = 0, 1, 2, 3


def gpe_rhs(plan: int, d_psihat, d_rhs, alpha: float, beta: float, d_work, stream=None) -> None:
    _check(lib().psfft_gpe_rhs(plan, _ptr(d_psihat), _ptr(d_rhs), float(alpha), float(beta), _ptr(d_work),
                               _stream(stream)), "psfft_gpe_rhs")


def rk_work_bytes(plan: int, system: int) -> int:
    return int(lib().psfft_rk_work_bytes(plan, system))


def rk_step(plan: int, system: int, d_y_in, d_y_out, ord: int, dt: float, params, d_work, stream=None) -> None:
    """params = (nu, eta | kappa, N_bv), passed as a host array of 3 doubles."""
    par = (ctypes.c_double * 3)(*[float(x) for x in params])
    _check(lib().psfft_rk_step(plan, system, _ptr(d_y_in), _ptr(d_y_out), ord, float(dt), par, _ptr(d_work),
                               _stream(stream)), "psfft_rk_step")


def hd_rhs_unfused(plan: int, d_uhat, d_rhs, nu: float, d_work, stream=None) -> None:
    _check(lib().psfft_hd_rhs_unfused(plan, _ptr(d_uhat), _ptr(d_rhs), float(nu), _ptr(d_work), _stream(stream)),
           "psfft_hd_rhs_unfused")


def mhd_rhs_unfused(plan: int, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu: float, eta: float, d_work, stream=None) -> None:
    _check(lib().psfft_mhd_rhs_unfused(plan, _ptr(d_uhat), _ptr(d_bhat), _ptr(d_rhs_u), _ptr(d_rhs_b), float(nu),
                                       float(eta), _ptr(d_work), _stream(stream)), "psfft_mhd_rhs_unfused")


def slab_query(plan: int, P: int, rank: int) -> SlabLayout:
    sl = SlabLayout()
    _check(lib().psfft_slab_query(plan, P, rank, ctypes.byref(sl)), "psfft_slab_query")
    return sl


def _ptr_array(blocks):
    return (ctypes.c_void_p * len(blocks))(*[_ptr(b) for b in blocks])


def slab_r2c_xy(plan: int, P: int, rank: int, d_real_slab, d_zspec, d_blocks, zoff: int, stream=None) -> None:
    """d_blocks: P tensors / device pointers, the block of each rank (see psfft.h)."""
    _check(lib().psfft_slab_r2c_xy(plan, P, rank, _ptr(d_real_slab), _ptr(d_zspec), _ptr_array(d_blocks), int(zoff),
                                   _stream(stream)), "psfft_slab_r2c_xy")


def slab_z(plan: int, P: int, rank: int, direction: int, d_xslab, stream=None) -> None:
    _check(lib().psfft_slab_z(plan, P, rank, int(direction), _ptr(d_xslab), _stream(stream)), "psfft_slab_z")


def slab_c2r_yx(plan: int, P: int, rank: int, d_blocks, zoff: int, d_zspec, d_real_slab, stream=None) -> None:
    _check(lib().psfft_slab_c2r_yx(plan, P, rank, _ptr_array(d_blocks), int(zoff), _ptr(d_zspec), _ptr(d_real_slab),
                                   _stream(stream)), "psfft_slab_c2r_yx")


def fft3d_r2c_host(plan: int, h_real, h_spec, d_in, d_out, d_work=None, stream=None) -> None:
    _check(lib().psfft_fft3d_r2c_host(plan, _ptr(h_real), _ptr(h_spec), _ptr(d_in), _ptr(d_out), _ptr(d_work),
                                      _stream(stream)), "psfft_fft3d_r2c_host")


def fft3d_c2r_host(plan: int, h_spec, h_real, d_in, d_out, d_work, stream=None) -> None:
    _check(lib().psfft_fft3d_c2r_host(plan, _ptr(h_spec), _ptr(h_real), _ptr(d_in), _ptr(d_out), _ptr(d_work),
                                      _stream(stream)), "psfft_fft3d_c2r_host")


def hd_rhs_host(plan: int, h_uhat, h_rhs, nu: float, d_in, d_out, d_work, stream=None) -> None:
    _check(lib().psfft_hd_rhs_host(plan, _ptr(h_uhat), _ptr(h_rhs), float(nu), _ptr(d_in), _ptr(d_out), _ptr(d_work),
                                   _stream(stream)), "psfft_hd_rhs_host")


def hd_rhs_host_box(plan: int, h_uhat, h_rhs, nu: float, d_in, d_out, d_work, stream=None) -> None:
    """hd_rhs_host copying only the index box around the retained modes (about 30 % of the dense bytes each way).
    h_rhs must have been zeroed once: only the box is written (include/psfft.h)."""
    _check(lib().psfft_hd_rhs_host_box(plan, _ptr(h_uhat), _ptr(h_rhs), float(nu), _ptr(d_in), _ptr(d_out),
                                       _ptr(d_work), _stream(stream)), "psfft_hd_rhs_host_box")


def host_box_bytes(plan: int) -> int:
    """Bytes per spectral field and direction that hd_rhs_host_box copies."""
    return int(lib().psfft_host_box_bytes(plan))


def profile_enable(plan: int, on: bool) -> None:
    _check(lib().psfft_profile_enable(plan, int(bool(on))), "psfft_profile_enable")


def profile_reset(plan: int) -> None:
    _check(lib().psfft_profile_reset(plan), "psfft_profile_reset")


def profile_records(plan: int):
    """[(kernel name, ms, algorithmic bytes)] for every launch recorded since the last reset."""
    out = []
    kind, ms, by = ctypes.c_int(), ctypes.c_double(), ctypes.c_double()
    for i in range(int(lib().psfft_profile_count(plan))):
        _check(lib().psfft_profile_get(plan, i, ctypes.byref(kind), ctypes.byref(ms), ctypes.byref(by)),
               "psfft_profile_get")
        out.append((lib().psfft_kernel_name(kind.value).decode(), ms.value, by.value))
    return out


def last_launch_count(plan: int) -> int:
    return int(lib().psfft_last_launch_count(plan))


def version() -> str:
    return lib().psfft_version().decode()


# ---- convenience: a plan that owns its torch-allocated tables and workspace -----------------------

def _on_plan_device(method):
    """Plan methods run with the plan's device current (so that the stream resolved for the launch and every
    buffer the method allocates belong to it) and refuse tensors that live elsewhere."""
    import functools

    @functools.wraps(method)
    def wrapper(self, *args, **kwargs):
        for t in list(args) + list(kwargs.values()):
            if isinstance(t, torch.Tensor) and t.device != self.device:
                raise PsfftError(f"tensor on {t.device}, plan on {self.device}")
        with torch.cuda.device(self.device):
            return method(self, *args, **kwargs)
    return wrapper


class Plan:
    """Plan + its caller-owned device buffers (allocated with torch; the library allocates nothing).

    >>> p = Plan(512, torch.float64, batch=3)
    >>> spec = p.r2c(real)          # real: [3, 512, 512, 512] cuda float64 -> [3, 512, 512, 257] complex128
    >>> back = p.c2r(spec)
    >>> rhs = p.hd_rhs(uhat)        # uhat: [3, N, N, N/2+1] complex
    """

    def __init__(self, N, dtype=torch.float64, batch: int = 1, device="cuda:0", work: str = "fft", box=None):
        if not torch.cuda.is_available():
            raise PsfftError("no CUDA device: libpsfft has no CPU fallback")
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self.rdtype = dtype
        self.cdtype = torch.complex128 if dtype == torch.float64 else torch.complex64
        code = F64 if dtype == torch.float64 else F32
        # N: one size (cubic grid) or (Nx, Ny, Nz) for an anisotropic grid; box = (Lx, Ly, Lz), default 2 pi each
        Nx, Ny, Nz = (N, N, N) if isinstance(N, int) else tuple(N)
        self.layout = plan_query3(Nx, Ny, Nz, code, batch)
        self.N, self.Ny, self.Nz, self.batch, self.ldk = Nx, Ny, Nz, batch, self.layout.ldk
        with torch.cuda.device(self.device):
            self.tables = torch.empty(self.layout.table_bytes, dtype=torch.uint8, device=self.device)
            self.handle = plan_create3(Nx, Ny, Nz, code, batch, self.tables, self.layout.table_bytes)
        if box is not None:
            plan_set_box(self.handle, *box)
        self._work = None
        self._work_kind = None
        self.ensure_work(work)

    @_on_plan_device
    def ensure_work(self, kind: str):
        need = {"fft": self.layout.work_bytes_fft, "hd": self.layout.work_bytes_hd,
                "mhd": self.layout.work_bytes_mhd, "boussinesq": self.layout.work_bytes_boussinesq,
                "rk_hd": 3 * self.layout.spec_bytes + self.layout.work_bytes_hd,
                "rk_mhd": 6 * self.layout.spec_bytes + self.layout.work_bytes_mhd,
                "rk_boussinesq": 4 * self.layout.spec_bytes + self.layout.work_bytes_boussinesq,
                "gpe": self.layout.work_bytes_gpe, "rk_gpe": 2 * self.layout.spec_bytes + self.layout.work_bytes_gpe}[kind]
        if self._work is None or self._work.numel() < need:
            self._work = None
            self._work = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._work

    def close(self):
        if getattr(self, "handle", None):
            plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def spec_shape(self, fields: int):
        return (fields, self.Nz, self.Ny, self.ldk)

    @_on_plan_device
    def r2c(self, real: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert real.is_cuda and real.dtype == self.rdtype and real.is_contiguous()
        assert real.numel() == self.batch * self.layout.real_elems
        if out is None:
            out = torch.empty(self.spec_shape(self.batch), dtype=self.cdtype, device=self.device)
        fft3d_r2c(self.handle, real, out, self.ensure_work("fft"))
        return out

    @_on_plan_device
    def c2r(self, spec: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert spec.is_cuda and spec.dtype == self.cdtype and spec.is_contiguous()
        assert spec.numel() == self.batch * self.layout.spec_elems
        if out is None:
            out = torch.empty((self.batch, self.Nz, self.Ny, self.N), dtype=self.rdtype, device=self.device)
        fft3d_c2r(self.handle, spec, out, self.ensure_work("fft"))
        return out

    @_on_plan_device
    def c2r_static(self, spec: torch.Tensor, out: torch.Tensor) -> torch.Tensor:
        """``c2r`` through ``psfft_fft3d_c2r_static``: the library's built-in 32 MiB workspace instead of this
        plan's.  ``out`` is required -- this method exists for callers that must not allocate, so it does not."""
        assert spec.is_cuda and spec.dtype == self.cdtype and spec.is_contiguous()
        assert spec.numel() == self.batch * self.layout.spec_elems
        assert out.is_cuda and out.dtype == self.rdtype and out.is_contiguous()
        assert out.numel() == self.batch * self.layout.real_elems
        fft3d_c2r_static(self.handle, spec, out)
        return out

    @_on_plan_device
    def hd_rhs(self, uhat: torch.Tensor, nu: float = 0.0, out: torch.Tensor | None = None) -> torch.Tensor:
        assert uhat.is_cuda and uhat.dtype == self.cdtype and uhat.is_contiguous()
        assert tuple(uhat.shape) == self.spec_shape(3)
        if out is None:
            out = torch.empty_like(uhat)
        hd_rhs(self.handle, uhat, out, nu, self.ensure_work("hd"))
        return out

    @_on_plan_device
    def mhd_rhs(self, uhat: torch.Tensor, bhat: torch.Tensor, nu: float = 0.0, eta: float = 0.0):
        for t in (uhat, bhat):
            assert t.is_cuda and t.dtype == self.cdtype and t.is_contiguous() and tuple(t.shape) == self.spec_shape(3)
        ru, rb = torch.empty_like(uhat), torch.empty_like(bhat)
        mhd_rhs(self.handle, uhat, bhat, ru, rb, nu, eta, self.ensure_work("mhd"))
        return ru, rb

    @_on_plan_device
    def boussinesq_rhs(self, uhat: torch.Tensor, thhat: torch.Tensor, nu: float = 0.0, kappa: float = 0.0,
                       nbv: float = 0.0):
        assert uhat.is_cuda and uhat.dtype == self.cdtype and uhat.is_contiguous()
        assert thhat.is_cuda and thhat.dtype == self.cdtype and thhat.is_contiguous()
        assert tuple(uhat.shape) == self.spec_shape(3) and thhat.numel() == self.layout.spec_elems
        ru, rt = torch.empty_like(uhat), torch.empty_like(thhat)
        boussinesq_rhs(self.handle, uhat, thhat, ru, rt, nu, kappa, nbv, self.ensure_work("boussinesq"))
        return ru, rt

    @_on_plan_device
    def rk_step(self, system: int, y: torch.Tensor, ord: int, dt: float, nu: float = 0.0, c2: float = 0.0,
                nbv: float = 0.0, out: torch.Tensor | None = None) -> torch.Tensor:
        """One Runge-Kutta step; y: [3 | 6 | 4, N, N, N/2+1] complex (HD | MHD u,b | Boussinesq u,theta)."""
        nf = {SYS_HD: 3, SYS_MHD: 6, SYS_BOUSSINESQ: 4, SYS_GPE: 2}[system]
        assert y.is_cuda and y.dtype == self.cdtype and y.is_contiguous() and tuple(y.shape) == self.spec_shape(nf)
        if out is None:
            out = torch.empty_like(y)
        work = self.ensure_work({SYS_HD: "rk_hd", SYS_MHD: "rk_mhd", SYS_BOUSSINESQ: "rk_boussinesq",
                                 SYS_GPE: "rk_gpe"}[system])
        assert rk_work_bytes(self.handle, system) <= work.numel()
        rk_step(self.handle, system, y, out, ord, dt, (nu, c2, nbv), work)
        return out

    @_on_plan_device
    def gpe_rhs(self, psihat: torch.Tensor, alpha: float, beta: float) -> torch.Tensor:
        """psihat: [2, N, N, N/2+1] = (p^, q^) of psi = p + i q."""
        assert psihat.is_cuda and psihat.dtype == self.cdtype and psihat.is_contiguous()
        assert tuple(psihat.shape) == self.spec_shape(2)
        out = torch.empty_like(psihat)
        gpe_rhs(self.handle, psihat, out, alpha, beta, self.ensure_work("gpe"))
        return out
