"""Seeded synthetic inputs (numpy only).

This module is DATA, not method: it holds none of the transform / right-hand-side
arithmetic.  It is the one module that both the CPU oracle's tests and the CUDA
path's tests / bench draw their inputs from.

The paper's workloads are its own turbulence runs (HD 256^3; HD/MHD at
512^3) whose initial conditions are not stated; BASELINE.json's configs
define the synthetic stand-ins generated here:

* ``uniform_field``        -- values uniform in [-1, 1) from a counter-based generator
                              (BASELINE.json configs 1 and 3).
* ``solenoidal_spectrum``  -- 3-component divergence-free random-phase field with
                              E(k) ~ k^4 exp(-2 (k/k0)^2), unit energy (configs 2, 4, 5).
* ``broadband_spectrum`` / ``broadband_scalar`` -- the same construction with a power-law shell
                              spectrum filled to the Nyquist planes (developed-turbulence stand-in; the
                              full-size parity inputs).
* ``aniso_spectrum``       -- the broadband construction on an anisotropic grid (Nx, Ny, Nz) in a box
                              (Lx, Ly, Lz) (the paper's 1024 x 1024 x 256 Boussinesq runs).
* ``taylor_green`` / ``abc_flow`` / ``single_mode`` -- closed-form physical-space fields
                              used by the oracle's pins.

Layouts: real field ``[z][y][x]`` (x contiguous; the paper's
``rarr(Nx,Ny,k)`` column-major); half spectrum ``[kz][ky][kx]`` with
``kx in [0, N/2]``, value = N^3 x Fourier coefficient (Eq. 8 is
unnormalised).
"""
from __future__ import annotations

import numpy as np

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix64(z: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = np.asarray(z, dtype=np.uint64)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def counter_bits(seed: int, idx: np.ndarray) -> np.ndarray:
    """64 random bits for counter ``idx`` under ``seed``: mix64(seed + (idx+1)*odd)."""
    with np.errstate(over="ignore"):
        idx = np.asarray(idx, dtype=np.uint64)
        return _mix64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (idx + np.uint64(1)) * _GOLD)


def uniform01(seed: int, idx: np.ndarray, bits: int = 53) -> np.ndarray:
    """Uniform variate in [0,1) with ``bits`` random bits (53 for fp64, 24 for fp32)."""
    r = counter_bits(seed, idx)
    return (r >> np.uint64(64 - bits)).astype(np.float64) * (2.0 ** -bits)


def uniform_field(N: int, batch: int = 1, seed: int = 1234, dtype=np.float64) -> np.ndarray:
    """``x[b][z][y][x] = 2 U(idx) - 1`` with idx the linear index over [b][z][y][x].

    fp32 draws 24 bits so the value is exact in fp32 and stays in [-1, 1).
    """
    dtype = np.dtype(dtype)
    bits = 53 if dtype == np.float64 else 24
    n = batch * N * N * N
    out = np.empty(n, dtype=dtype)
    chunk = 1 << 24
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        idx = np.arange(s, e, dtype=np.uint64)
        out[s:e] = (2.0 * uniform01(seed, idx, bits) - 1.0).astype(dtype)
    return out.reshape(batch, N, N, N)


def _key(seed: int, tag: int, kx, ky, kz) -> np.ndarray:
    """Per-wavevector key: nested mixes of (seed, tag, kx, ky, kz); offsets keep negatives distinct."""
    off = np.int64(1 << 20)
    with np.errstate(over="ignore"):
        h = _mix64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + np.uint64(tag + 1) * _GOLD)
        h = _mix64(h + (np.asarray(kx, np.int64) + off).astype(np.uint64) * _GOLD)
        h = _mix64(h + (np.asarray(ky, np.int64) + off).astype(np.uint64) * _GOLD)
        h = _mix64(h + (np.asarray(kz, np.int64) + off).astype(np.uint64) * _GOLD)
    return h


def _variate(key: np.ndarray, j: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        r = _mix64(key + np.uint64(j + 1) * _GOLD)
    return (r >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def solenoidal_coefficients(k0: float, kcut: int, seed: int = 1234, tag: int = 0):
    """Grid-independent Fourier coefficients a_k of a random-phase solenoidal field.

    Returns ``(kx, ky, kz, a)``: integer wavevectors (canonical half: kx > 0, or kx == 0 and
    (ky > 0 or (ky == 0 and kz > 0))) and complex coefficients ``a[3, nmodes]`` scaled so that
    the field has unit energy, 1/2 <|u|^2> = 1.  Keying the
    variates on the integer wavevector (not a sequential stream) makes the same physical
    field available on any grid (pin P12).
    """
    r = np.arange(-kcut, kcut + 1)
    kx, ky, kz = np.meshgrid(np.arange(0, kcut + 1), r, r, indexing="ij")
    kx, ky, kz = kx.ravel(), ky.ravel(), kz.ravel()
    k2 = kx * kx + ky * ky + kz * kz
    canon = (kx > 0) | ((kx == 0) & ((ky > 0) | ((ky == 0) & (kz > 0))))
    sel = canon & (k2 >= 1) & (k2 <= kcut * kcut)
    kx, ky, kz, k2 = kx[sel], ky[sel], kz[sel], k2[sel].astype(np.float64)
    kk = np.sqrt(k2)
    key = _key(seed, tag, kx, ky, kz)
    th1 = 2.0 * np.pi * _variate(key, 0)
    th2 = 2.0 * np.pi * _variate(key, 1)
    phi = 2.0 * np.pi * _variate(key, 2)
    # e1 = (k x zhat)/|k x zhat| = (ky, -kx, 0)/sqrt(kx^2+ky^2), xhat when kx = ky = 0
    kh = np.sqrt((kx * kx + ky * ky).astype(np.float64))
    axis = kh == 0
    khs = np.where(axis, 1.0, kh)
    e1 = np.stack([np.where(axis, 1.0, ky / khs), np.where(axis, 0.0, -kx / khs), np.zeros_like(kk)])
    kvec = np.stack([kx, ky, kz]).astype(np.float64)
    e2 = np.cross(kvec, e1, axis=0) / kk
    amp = np.sqrt(k2 * k2 * np.exp(-2.0 * k2 / (k0 * k0)) / (4.0 * np.pi * k2))
    a = amp * (np.cos(phi) * np.exp(1j * th1) * e1 + np.sin(phi) * np.exp(1j * th2) * e2)
    # energy: each canonical mode stands for itself and its conjugate partner -> 1/2 * 2 * |a|^2
    energy = np.sum(np.abs(a) ** 2)
    a = a / np.sqrt(energy)
    return kx, ky, kz, a


def solenoidal_spectrum(N: int, k0: float = 4.0, kcut: int | None = None, seed: int = 1234,
                        tag: int = 0, dtype=np.complex128) -> np.ndarray:
    """Half spectrum ``uhat[3][kz][ky][kx]`` (= N^3 a_k) of the random solenoidal field."""
    if kcut is None:
        kcut = int(8 * k0)
    if kcut >= N // 2:
        raise ValueError("kcut must be below the Nyquist wavenumber")
    iz, iy, ix, v = solenoidal_modes(N, k0, kcut, seed, tag)
    u = np.zeros((3, N, N, N // 2 + 1), dtype=np.complex128)
    u[:, iz, iy, ix] = v
    return u.astype(dtype)


def solenoidal_modes(N: int, k0: float = 4.0, kcut: int | None = None, seed: int = 1234, tag: int = 0):
    """The non-zero entries of ``solenoidal_spectrum`` as a list: indices ``(iz, iy, ix)`` into
    ``[kz][ky][kx]`` and values ``v[3, n]`` (= N^3 a_k, conjugate partners of the kx = 0 plane included).
    For callers that scatter the few thousand modes into a zero-initialised DEVICE array instead of building
    the dense host array (bench.py at 1024^3)."""
    if kcut is None:
        kcut = int(8 * k0)
    if kcut >= N // 2:
        raise ValueError("kcut must be below the Nyquist wavenumber")
    kx, ky, kz, a = solenoidal_coefficients(k0, kcut, seed, tag)
    scale = float(N) ** 3
    on0 = kx == 0
    iz = np.concatenate([kz % N, (-kz[on0]) % N])
    iy = np.concatenate([ky % N, (-ky[on0]) % N])
    ix = np.concatenate([kx, np.zeros(int(on0.sum()), dtype=kx.dtype)])
    v = np.concatenate([a * scale, np.conj(a[:, on0]) * scale], axis=1)
    return iz, iy, ix, v


def scalar_coefficients(k0: float, kcut: int, seed: int = 1234, tag: int = 7):
    """Grid-independent Fourier coefficients of a random-phase real SCALAR field (the temperature
    fluctuation theta of the Boussinesq runs): same shell amplitude as the
    velocity recipe, one uniform phase per canonical wavevector keyed on ``(seed, tag, kx, ky, kz)``,
    scaled to unit variance-energy 1/2 <theta^2> = 1.  Returns ``(kx, ky, kz, a)``."""
    r = np.arange(-kcut, kcut + 1)
    kx, ky, kz = np.meshgrid(np.arange(0, kcut + 1), r, r, indexing="ij")
    kx, ky, kz = kx.ravel(), ky.ravel(), kz.ravel()
    k2 = kx * kx + ky * ky + kz * kz
    canon = (kx > 0) | ((kx == 0) & ((ky > 0) | ((ky == 0) & (kz > 0))))
    sel = canon & (k2 >= 1) & (k2 <= kcut * kcut)
    kx, ky, kz, k2 = kx[sel], ky[sel], kz[sel], k2[sel].astype(np.float64)
    ph = 2.0 * np.pi * _variate(_key(seed, tag, kx, ky, kz), 0)
    amp = np.sqrt(k2 * k2 * np.exp(-2.0 * k2 / (k0 * k0)) / (4.0 * np.pi * k2))
    a = amp * np.exp(1j * ph)
    return kx, ky, kz, a / np.sqrt(np.sum(np.abs(a) ** 2))


def scalar_spectrum(N: int, k0: float = 4.0, kcut: int | None = None, seed: int = 1234, tag: int = 7,
                    dtype=np.complex128) -> np.ndarray:
    """Half spectrum ``thhat[kz][ky][kx]`` (= N^3 a_k) of the random scalar field."""
    if kcut is None:
        kcut = int(8 * k0)
    if kcut >= N // 2:
        raise ValueError("kcut must be below the Nyquist wavenumber")
    kx, ky, kz, a = scalar_coefficients(k0, kcut, seed, tag)
    t = np.zeros((N, N, N // 2 + 1), dtype=np.complex128)
    scale = float(N) ** 3
    t[kz % N, ky % N, kx] = a * scale
    on0 = kx == 0
    t[(-kz[on0]) % N, (-ky[on0]) % N, 0] = np.conj(a[on0]) * scale
    return t.astype(dtype)


def _shell_amplitude(k2: np.ndarray, slope: float) -> np.ndarray:
    """Per-mode amplitude of a power-law shell spectrum E(k) ~ k^slope: sqrt(E(k) / (4 pi k^2))."""
    return np.sqrt(k2 ** (0.5 * slope) / (4.0 * np.pi * k2))


def _canonical_plane(kx: int, kcut: int):
    """Canonical wavevectors (kx, ky, kz) of one kx plane with 1 <= |k| <= kcut (see solenoidal_coefficients)."""
    r = np.arange(-kcut, kcut + 1)
    ky, kz = np.meshgrid(r, r, indexing="ij")
    ky, kz = ky.ravel(), kz.ravel()
    k2 = kx * kx + ky * ky + kz * kz
    canon = (kx > 0) | ((ky > 0) | ((ky == 0) & (kz > 0)))
    sel = canon & (k2 >= 1) & (k2 <= kcut * kcut)
    return np.full(int(sel.sum()), kx), ky[sel], kz[sel], k2[sel].astype(np.float64)


def _map_planes(fn, n: int) -> list:
    """fn(0..n-1) on a small thread pool (numpy releases the GIL; the planes write disjoint slices).  The
    results come back in plane order, so sums over them do not depend on the scheduling."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    workers = max(1, min(16, os.cpu_count() or 1))
    if workers == 1 or n < 8:
        return [fn(i) for i in range(n)]
    with ThreadPoolExecutor(workers) as ex:
        return list(ex.map(fn, range(n)))


def broadband_spectrum(N: int, slope: float = -5.0 / 3.0, kcut: int | None = None, seed: int = 1234, tag: int = 0,
                       dtype=np.complex128) -> np.ndarray:
    """Half spectrum ``uhat[3][kz][ky][kx]`` of a random-phase solenoidal field whose shell spectrum is the
    power law E(k) ~ k^slope on 1 <= |k| <= kcut (default: N/2 - 1, every shell below the Nyquist planes), unit
    energy.  The stand-in for a developed turbulent state (the paper's production runs):
    every mode of the 2/3-rule sphere carries an O(1) share of its shell, and modes OUTSIDE the sphere are
    populated too, so the input mask, the pruned column ranges and the outermost retained shell all see data.
    Same per-wavevector keys and polarisation construction as ``solenoidal_spectrum`` (grid independent);
    generated one kx plane at a time so that 1024^3 stays within a few GB of host memory."""
    if kcut is None:
        kcut = N // 2 - 1
    if kcut >= N // 2:
        raise ValueError("kcut must be below the Nyquist wavenumber")
    u = np.zeros((3, N, N, N // 2 + 1), dtype=dtype)

    def plane(kx0: int) -> float:
        kx, ky, kz, k2 = _canonical_plane(kx0, kcut)
        if kx.size == 0:
            return 0.0
        kk = np.sqrt(k2)
        key = _key(seed, tag, kx, ky, kz)
        th1 = 2.0 * np.pi * _variate(key, 0)
        th2 = 2.0 * np.pi * _variate(key, 1)
        phi = 2.0 * np.pi * _variate(key, 2)
        kh = np.sqrt((kx * kx + ky * ky).astype(np.float64))
        axis = kh == 0
        khs = np.where(axis, 1.0, kh)
        e1 = np.stack([np.where(axis, 1.0, ky / khs), np.where(axis, 0.0, -kx / khs), np.zeros_like(kk)])
        e2 = np.cross(np.stack([kx, ky, kz]).astype(np.float64), e1, axis=0) / kk
        a = _shell_amplitude(k2, slope) * (np.cos(phi) * np.exp(1j * th1) * e1 + np.sin(phi) * np.exp(1j * th2) * e2)
        u[:, kz % N, ky % N, kx0] = a
        if kx0 == 0:
            u[:, (-kz) % N, (-ky) % N, 0] = np.conj(a)
        return float(np.sum(np.abs(a) ** 2))

    energy = sum(_map_planes(plane, kcut + 1))
    u *= np.asarray(float(N) ** 3 / np.sqrt(energy)).astype(u.real.dtype)
    return u


def broadband_scalar(N: int, slope: float = -5.0 / 3.0, kcut: int | None = None, seed: int = 1234, tag: int = 7,
                     dtype=np.complex128) -> np.ndarray:
    """Half spectrum ``thhat[kz][ky][kx]`` of a random-phase real scalar field with the power-law shell
    spectrum of ``broadband_spectrum`` (one uniform phase per canonical wavevector), unit variance-energy."""
    if kcut is None:
        kcut = N // 2 - 1
    if kcut >= N // 2:
        raise ValueError("kcut must be below the Nyquist wavenumber")
    t = np.zeros((N, N, N // 2 + 1), dtype=dtype)

    def plane(kx0: int) -> float:
        kx, ky, kz, k2 = _canonical_plane(kx0, kcut)
        if kx.size == 0:
            return 0.0
        ph = 2.0 * np.pi * _variate(_key(seed, tag, kx, ky, kz), 0)
        a = _shell_amplitude(k2, slope) * np.exp(1j * ph)
        t[kz % N, ky % N, kx0] = a
        if kx0 == 0:
            t[(-kz) % N, (-ky) % N, 0] = np.conj(a)
        return float(np.sum(np.abs(a) ** 2))

    energy = sum(_map_planes(plane, kcut + 1))
    t *= np.asarray(float(N) ** 3 / np.sqrt(energy)).astype(t.real.dtype)
    return t


def aniso_spectrum(shape, box=None, slope: float = -5.0 / 3.0, seed: int = 1234, tag: int = 0, ncomp: int = 3,
                   fill: float = 0.5, dtype=np.complex128) -> np.ndarray:
    """Random-phase field on an ANISOTROPIC grid ``shape = (Nx, Ny, Nz)`` in the box ``box = (Lx, Ly, Lz)``
    (grid points and box lengths independent per direction; default box 2 pi each): half spectrum
    ``[ncomp][kz][ky][kx]``, value = Nx Ny Nz x Fourier coefficient.  The stand-in for the paper's flat-box
    Boussinesq runs (1024 x 1024 x 256).

    Every integer index vector n inside the ellipsoid sum (n_i / N_i)^2 < fill^2 (fill = 1/2: up to the Nyquist
    planes, so the 2/3-rule mask of the right-hand side has something to remove) carries a mode keyed on
    ``(seed, tag, nx, ny, nz)`` -- the same physical field on any grid that holds it -- with the power-law shell
    amplitude of ``broadband_spectrum`` in the PHYSICAL wavenumber |k|, k_i = 2 pi n_i / L_i.  ncomp = 3: solenoidal
    (k . a = 0 with the physical k), same polarisation construction as ``solenoidal_coefficients``; ncomp = 1: a real
    scalar (returned with the leading axis dropped).  Unit energy, 1/2 <|u|^2> = 1."""
    Nx, Ny, Nz = (int(v) for v in shape)
    kf = [1.0, 1.0, 1.0] if box is None else [2.0 * np.pi / float(b) for b in box]
    u = np.zeros((ncomp, Nz, Ny, Nx // 2 + 1), dtype=dtype)
    ry = np.arange(-(Ny // 2) + 1, Ny // 2)
    rz = np.arange(-(Nz // 2) + 1, Nz // 2)
    ny_, nz_ = (a.ravel() for a in np.meshgrid(ry, rz, indexing="ij"))

    def plane(nx0: int) -> float:
        rho2 = (nx0 / Nx) ** 2 + (ny_ / Ny) ** 2 + (nz_ / Nz) ** 2
        canon = (nx0 > 0) | ((ny_ > 0) | ((ny_ == 0) & (nz_ > 0)))
        sel = canon & (rho2 < fill * fill) & ((nx0 != 0) | (ny_ != 0) | (nz_ != 0))
        ny, nz = ny_[sel], nz_[sel]
        if ny.size == 0:
            return 0.0
        nx = np.full(ny.size, nx0)
        kx, ky, kz = nx * kf[0], ny * kf[1], nz * kf[2]
        k2 = kx * kx + ky * ky + kz * kz
        kk = np.sqrt(k2)
        key = _key(seed, tag, nx, ny, nz)
        if ncomp == 1:
            a = (_shell_amplitude(k2, slope) * np.exp(2j * np.pi * _variate(key, 0)))[None]
        else:
            th1 = 2.0 * np.pi * _variate(key, 0)
            th2 = 2.0 * np.pi * _variate(key, 1)
            phi = 2.0 * np.pi * _variate(key, 2)
            kh = np.sqrt(kx * kx + ky * ky)
            axis = kh == 0
            khs = np.where(axis, 1.0, kh)
            e1 = np.stack([np.where(axis, 1.0, ky / khs), np.where(axis, 0.0, -kx / khs), np.zeros_like(kk)])
            e2 = np.cross(np.stack([kx, ky, kz]), e1, axis=0) / kk
            a = _shell_amplitude(k2, slope) * (np.cos(phi) * np.exp(1j * th1) * e1 + np.sin(phi) * np.exp(1j * th2) * e2)
        u[:, nz % Nz, ny % Ny, nx0] = a
        if nx0 == 0:
            u[:, (-nz) % Nz, (-ny) % Ny, 0] = np.conj(a)
        return float(np.sum(np.abs(a) ** 2))

    nxmax = int(np.ceil(fill * Nx))
    energy = sum(_map_planes(plane, min(nxmax, Nx // 2 - 1) + 1))
    u *= np.asarray(float(Nx) * Ny * Nz / np.sqrt(energy)).astype(u.real.dtype)
    return u[0] if ncomp == 1 else u


def box_axes(shape, box=None):
    """Physical coordinates of the grid ``shape = (Nx, Ny, Nz)`` in the box ``(Lx, Ly, Lz)``: x_i = L_x i / N_x ...
    as broadcastable [z][y][x] arrays (returns x, y, z)."""
    Nx, Ny, Nz = shape
    Lx, Ly, Lz = (2.0 * np.pi,) * 3 if box is None else box
    return (Lx * np.arange(Nx) / Nx)[None, None, :], (Ly * np.arange(Ny) / Ny)[None, :, None], \
        (Lz * np.arange(Nz) / Nz)[:, None, None]


def grid_axes(N: int):
    """Physical coordinates X_i = 2 pi i / N as broadcastable [z][y][x] arrays (returns x, y, z)."""
    t = 2.0 * np.pi * np.arange(N) / N
    return t[None, None, :], t[None, :, None], t[:, None, None]


def taylor_green(N: int) -> np.ndarray:
    """u = (sin x cos y cos z, -cos x sin y cos z, 0), shape [3][z][y][x]."""
    x, y, z = grid_axes(N)
    u = np.zeros((3, N, N, N))
    u[0] = np.sin(x) * np.cos(y) * np.cos(z)
    u[1] = -np.cos(x) * np.sin(y) * np.cos(z)
    return u


def taylor_green_spectrum(N: int, m: int = 1, dtype=np.complex128) -> np.ndarray:
    """Half spectrum (= N^3 x Fourier coefficient) of the Taylor-Green vortex at wavenumber m,
    u = (sin mx cos my cos mz, -cos mx sin my cos mz, 0), written down mode by mode (no transform): eight
    entries, u^_x[+-m][+-m][m] = -i N^3/8 and u^_y[+-m][s m][m] = i s N^3/8.  Needs no N^3 physical array, so the
    closed-form pin reaches the last retained shell of the large grids."""
    u = np.zeros((3, N, N, N // 2 + 1), dtype=dtype)
    a = float(N) ** 3 / 8.0
    for kz in (m, N - m):
        for ky, sy in ((m, 1.0), (N - m, -1.0)):
            u[0, kz, ky, m] = -1j * a
            u[1, kz, ky, m] = 1j * sy * a
    return u


def abc_flow(N: int, A: float = 1.0, B: float = 0.7, C: float = 0.43, k: int = 1) -> np.ndarray:
    """Beltrami flow u = (B cos ky + C sin kz, C cos kz + A sin kx, A cos kx + B sin ky): curl u = k u."""
    x, y, z = grid_axes(N)
    u = np.zeros((3, N, N, N))
    u[0] = B * np.cos(k * y) + C * np.sin(k * z)
    u[1] = C * np.cos(k * z) + A * np.sin(k * x)
    u[2] = A * np.cos(k * x) + B * np.sin(k * y)
    return u


def single_mode(N: int, p: int, q: int, r: int) -> np.ndarray:
    """x[k][j][i] = cos(2 pi (p i + q j + r k)/N), shape [z][y][x]."""
    i = np.arange(N)
    ph = (p * i[None, None, :] + q * i[None, :, None] + r * i[:, None, None]) % N
    return np.cos(2.0 * np.pi * ph / N)
