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
    kx, ky, kz, a = solenoidal_coefficients(k0, kcut, seed, tag)
    u = np.zeros((3, N, N, N // 2 + 1), dtype=np.complex128)
    scale = float(N) ** 3
    u[:, kz % N, ky % N, kx] = a * scale
    on0 = kx == 0
    u[:, (-kz[on0]) % N, (-ky[on0]) % N, 0] = np.conj(a[:, on0]) * scale
    return u.astype(dtype)


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
