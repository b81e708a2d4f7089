"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes front end of ``oracle/psfft_oracle.c`` (plain C, fp64).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It imports nothing from ``paper_1808_01309_b200`` and the CUDA path
imports nothing from here.

Every function cites the passage of PAPER.md (arxiv 1808.01309) it follows; see the C file for
the definitions themselves.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "psfft_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over pencils).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB,
                               _SRC, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_set_threads.restype = ctypes.c_int
        _lib.orc_get_threads.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n: int) -> int:
    """Set the OpenMP thread count; returns the count in effect."""
    return int(_load().orc_set_threads(ctypes.c_int(int(n))))


def get_threads() -> int:
    return int(_load().orc_get_threads())


def dft1d_direct(x, sign: int) -> np.ndarray:
    """O1: X[p] = sum_j x[j] exp(sign 2 pi i p j / n)  (Eq. 8, one axis)."""
    x = _c128(x)
    X = np.empty_like(x)
    _load().orc_dft1d_direct(ctypes.c_int(x.size), ctypes.c_int(sign), _p(x), ctypes.c_long(1), _p(X),
                             ctypes.c_long(1))
    return X


def fft1d(x, sign: int) -> np.ndarray:
    """O2: recursive mixed-radix decimation in time (north_star: "naive radix-2/mixed-radix FFT")."""
    x = _c128(x)
    X = np.empty_like(x)
    _load().orc_fft1d(ctypes.c_int(x.size), ctypes.c_int(sign), _p(x), ctypes.c_long(1), _p(X),
                      ctypes.c_long(1))
    return X


def r2c3d(x) -> np.ndarray:
    """O3: unnormalised forward 3D DFT of a real field [z][y][x] -> [kz][ky][kx<=Nx/2]."""
    x = _f64(x)
    Nz, Ny, Nx = x.shape
    X = np.empty((Nz, Ny, Nx // 2 + 1), dtype=np.complex128)
    _load().orc_r2c3d(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(x), _p(X))
    return X


def c2r3d(X, Nx: int | None = None) -> np.ndarray:
    """O4: inverse (sign +, scaled 1/(Nx Ny Nz)) of a half spectrum -> real field."""
    X = _c128(X)
    Nz, Ny, H = X.shape
    if Nx is None:
        Nx = 2 * (H - 1)
    assert Nx // 2 + 1 == H
    x = np.empty((Nz, Ny, Nx), dtype=np.float64)
    _load().orc_c2r3d(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(X), _p(x))
    return x


def dft3d_bruteforce(x) -> np.ndarray:
    """O5: the O(N^6) triple sum of Eq. 8 for every output; FULL spectrum [r][q][p]."""
    x = _f64(x)
    Nz, Ny, Nx = x.shape
    X = np.empty((Nz, Ny, Nx), dtype=np.complex128)
    _load().orc_dft3d_bruteforce(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(x), _p(X))
    return X


def r2c3d_mode(x, r: int, q: int, p: int) -> complex:
    """O5 for ONE output mode (sampled parity at sizes where O3 over the whole grid is too slow)."""
    x = _f64(x)
    Nz, Ny, Nx = x.shape
    out = np.zeros(2)
    _load().orc_r2c3d_mode(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(x), ctypes.c_int(r),
                           ctypes.c_int(q), ctypes.c_int(p), _p(out))
    return complex(out[0], out[1])


def idft3d_point(Xfull, k: int, j: int, i: int) -> complex:
    """Brute-force inverse (Eq. 8 with the sign changed, x 1/N^3) for one grid point from a FULL spectrum."""
    Xfull = _c128(Xfull)
    Nz, Ny, Nx = Xfull.shape
    out = np.zeros(2)
    _load().orc_idft3d_point(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(Xfull),
                             ctypes.c_int(k), ctypes.c_int(j), ctypes.c_int(i), _p(out))
    return complex(out[0], out[1])


def _grid(a, ncomp_axes: int = 1):
    """(Nz, Ny, Nx) of a half-spectrum array [...][kz][ky][kx <= Nx/2]."""
    Nz, Ny, H = a.shape[-3:]
    return int(Nz), int(Ny), 2 * (int(H) - 1)


def _box(box):
    """box = (Lx, Ly, Lz), the physical box lengths of PAPER.md:64; None = 2 pi each."""
    if box is None:
        box = (2.0 * np.pi,) * 3
    assert len(box) == 3
    return (ctypes.c_double * 3)(*[float(b) for b in box])


def _dims(a):
    Nz, Ny, Nx = _grid(a)
    return ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx)


def dealias_mask(N, Ny: int | None = None, Nz: int | None = None) -> np.ndarray:
    """a9: 2/3-rule truncation in integers.  Cubic: keep iff 9|n|^2 < N^2.  General grid
    (Nx, Ny, Nz): the ellipsoid sum (n_i/N_i)^2 < 1/9 as 9 sum (n_i L/N_i)^2 < L^2, L = lcm (G25)."""
    Nx = int(N)
    Ny = Nx if Ny is None else int(Ny)
    Nz = Nx if Nz is None else int(Nz)
    m = np.empty((Nz, Ny, Nx // 2 + 1), dtype=np.uint8)
    _load().orc_dealias_mask3(ctypes.c_int(Nz), ctypes.c_int(Ny), ctypes.c_int(Nx), _p(m))
    return m.astype(bool)


def apply_mask(f) -> np.ndarray:
    f = _c128(f).copy()
    N = f.shape[-2]
    assert f.shape[-3] == N and f.shape[-1] == N // 2 + 1
    _load().orc_apply_mask(ctypes.c_int(N), ctypes.c_int(f.shape[0]), _p(f))
    return f


def curl(uhat, box=None) -> np.ndarray:
    """a7: i k x uhat, k_i = n_i 2 pi / L_i (PAPER.md:66: derivatives are taken in spectral space; :64 box)."""
    u = _c128(uhat)
    w = np.empty_like(u)
    _load().orc_curl3(*_dims(u), _box(box), _p(u), _p(w))
    return w


def project(f, box=None) -> np.ndarray:
    """a10: f - k (k.f)/|k|^2, identity at k = 0 ("projecting ... onto a divergence-free space")."""
    f = _c128(f).copy()
    _load().orc_project3(*_dims(f), _box(box), _p(f))
    return f


def _cubic(a, box) -> bool:
    Nz, Ny, Nx = _grid(a)
    return box is None and Nz == Ny == Nx


def hd_rhs(uhat, nu: float = 0.0, box=None) -> np.ndarray:
    """O6: M P F[F^-1(M u) x F^-1(i k x M u)] - nu |k|^2 M u (PAPER.md:36 Eq. 1, :66); any grid (Nx, Ny, Nz)
    and box (Lx, Ly, Lz)."""
    u = _c128(uhat)
    assert u.ndim == 4 and u.shape[0] == 3
    out = np.empty_like(u)
    if _cubic(u, box):
        _load().orc_hd_rhs(ctypes.c_int(u.shape[-2]), _p(u), ctypes.c_double(nu), _p(out))
    else:
        _load().orc_hd_rhs3(*_dims(u), _box(box), _p(u), ctypes.c_double(nu), _p(out))
    return out


def mhd_rhs(uhat, bhat, nu: float = 0.0, eta: float = 0.0, box=None):
    """O7: (R_u, R_b) of PAPER.md:48-52 Eqs. 4-6."""
    u, b = _c128(uhat), _c128(bhat)
    assert u.shape == b.shape and u.ndim == 4 and u.shape[0] == 3
    ru, rb = np.empty_like(u), np.empty_like(u)
    if _cubic(u, box):
        _load().orc_mhd_rhs(ctypes.c_int(u.shape[-2]), _p(u), _p(b), ctypes.c_double(nu), ctypes.c_double(eta),
                            _p(ru), _p(rb))
    else:
        _load().orc_mhd_rhs3(*_dims(u), _box(box), _p(u), _p(b), ctypes.c_double(nu), ctypes.c_double(eta),
                             _p(ru), _p(rb))
    return ru, rb


def boussinesq_rhs(uhat, thhat, nu: float = 0.0, kappa: float = 0.0, nbv: float = 0.0, box=None):
    """O8: (R_u, R_theta) of the Boussinesq equations, Eqs. 1-3:
    R_u = M P (F[u x w] - N_bv theta^ z^) - nu |k|^2 M u^,  R_th = -M F[u . grad theta] + N_bv M u^_z - kappa |k|^2 M theta^."""
    u, t = _c128(uhat), _c128(thhat)
    assert u.ndim == 4 and u.shape[0] == 3 and t.shape == u.shape[1:]
    ru, rt = np.empty_like(u), np.empty_like(t)
    args = (_p(u), _p(t), ctypes.c_double(nu), ctypes.c_double(kappa), ctypes.c_double(nbv), _p(ru), _p(rt))
    if _cubic(u, box):
        _load().orc_boussinesq_rhs(ctypes.c_int(u.shape[-2]), *args)
    else:
        _load().orc_boussinesq_rhs3(*_dims(u), _box(box), *args)
    return ru, rt


def rk_step(sys: int, y, ord: int, dt: float, nu: float = 0.0, c2: float = 0.0, nbv: float = 0.0, box=None) -> np.ndarray:
    """O9: one low-storage Runge-Kutta step of `ord` stages (reading G21):
    y^(ord) = y_n; y^(o-1) = M y_n + (dt/o) R(y^(o)), o = ord..1.  sys 0 = HD (y: 3 fields), 1 = MHD (u^, b^: 6
    fields; c2 = eta), 2 = Boussinesq (u^, theta^: 4 fields; c2 = kappa), 3 = GPE (p^, q^; nu = alpha, c2 = beta)."""
    y = _c128(y)
    assert y.ndim == 4 and y.shape[0] == {0: 3, 1: 6, 2: 4, 3: 2}[sys]
    out = np.empty_like(y)
    par = (ctypes.c_double * 3)(nu, c2, nbv)
    args = (ctypes.c_int(sys), ctypes.c_int(ord), ctypes.c_double(dt), par, _p(y), _p(out))
    if _cubic(y, box):
        _load().orc_rk_step(ctypes.c_int(y.shape[-2]), *args)
    else:
        _load().orc_rk_step3(*_dims(y), _box(box), *args)
    return out


def gpe_rhs(psihat, alpha: float, beta: float, box=None) -> np.ndarray:
    """O10: right-hand side of the Gross-Pitaevskii equation (Eq. 7) for psi = p + i q carried as
    the two real fields (p, q): psihat, result = [2][kz][ky][kx]; alpha = hbar/(2m), beta = g/hbar."""
    y = _c128(psihat)
    assert y.ndim == 4 and y.shape[0] == 2
    out = np.empty_like(y)
    if _cubic(y, box):
        _load().orc_gpe_rhs(ctypes.c_int(y.shape[-2]), _p(y), ctypes.c_double(alpha), ctypes.c_double(beta), _p(out))
    else:
        _load().orc_gpe_rhs3(*_dims(y), _box(box), _p(y), ctypes.c_double(alpha), ctypes.c_double(beta), _p(out))
    return out
