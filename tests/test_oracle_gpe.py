"""Pins for the oracle's Gross-Pitaevskii right-hand side (O10, Eq. 7) -- CPU only.

psi = p + i q is carried as two real fields ("1 complex (or 2 real)").  A plausible mistake (sign of
the dispersion or of the interaction term, p and q swapped, a missing factor in |psi|^2, a missing mask) fails at
least one of: the exact plane-wave solution, the uniform condensate, the linear (beta = 0) dispersion relation,
mass and energy conservation, the numpy re-statement.
"""
import numpy as np
import pytest

import oracle
from paper_1808_01309_b200 import synth


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


def pack(psi):
    """complex physical field -> (p^, q^) half spectra"""
    return np.stack([oracle.r2c3d(np.ascontiguousarray(psi.real)), oracle.r2c3d(np.ascontiguousarray(psi.imag))])


def random_psi(N, kcut, seed):
    """band-limited smooth complex field from two random-phase scalar spectra (synth recipe, tags 11 / 12)"""
    p = oracle.c2r3d(synth.scalar_spectrum(N, 2.0, kcut, seed, tag=11), N)
    q = oracle.c2r3d(synth.scalar_spectrum(N, 2.0, kcut, seed, tag=12), N)
    return 1.0 + 0.3 * (p + 1j * q)            # condensate plus fluctuations


def half_weights(N):
    w = np.full(N // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    return w[None, None, :]


@pytest.mark.parametrize("k", [(2, 1, -3), (0, 0, 0), (1, 0, 0), (-2, 3, 1)])
def test_plane_wave_is_an_exact_solution(k):
    """psi = A exp(i k.x): |psi|^2 = A^2, so d_t psi = -i (alpha |k|^2 + beta A^2) psi exactly (k = 0: the
    uniform condensate rotating at the chemical potential beta A^2)."""
    N, A, alpha, beta = 16, 0.7, 0.3, 1.1
    x, y, z = synth.grid_axes(N)
    psi = A * np.exp(1j * (k[0] * x + k[1] * y + k[2] * z + 0 * x * y * z))
    k2 = sum(c * c for c in k)
    got = oracle.gpe_rhs(pack(psi), alpha, beta)
    assert rel(got, pack(-1j * (alpha * k2 + beta * A * A) * psi)) < 1e-14


def test_linear_limit_is_the_free_particle_dispersion():
    """beta = 0: R_p = alpha |k|^2 q^, R_q = -alpha |k|^2 p^ mode by mode (omega = alpha |k|^2)."""
    N = 16
    y0 = pack(random_psi(N, 4, 3))
    got = oracle.gpe_rhs(y0, 0.25, 0.0)
    kk = np.arange(N)
    kk = np.where(kk < N // 2, kk, kk - N)
    k2 = (np.arange(N // 2 + 1)[None, None, :] ** 2 + kk[None, :, None] ** 2 + kk[:, None, None] ** 2).astype(float)
    ym = oracle.apply_mask(y0)
    assert rel(got[0], 0.25 * k2 * ym[1]) < 1e-14 and rel(got[1], -0.25 * k2 * ym[0]) < 1e-14


def test_mass_and_energy_are_conserved():
    """d/dt int |psi|^2 = 2 Re <psi, R> = 0 and dE/dt = 2 Re <alpha (-Lap psi) + beta |psi|^2 psi, R> = 0 for a
    field inside the truncation sphere (both exact: <psi, i H psi> is imaginary for a Hermitian H)."""
    N, alpha, beta = 24, 0.4, 0.9
    psi = random_psi(N, 3, 5)                      # |k| <= 3: the cubic term reaches 9 > N/3 = 8, so the mask acts
    y0 = pack(psi)
    R = oracle.gpe_rhs(y0, alpha, beta)
    w = half_weights(N)
    dot = lambda a, b: float(np.sum(w * (np.conj(a) * b).real))
    norm = dot(y0[0], y0[0]) + dot(y0[1], y0[1])
    assert abs(dot(y0[0], R[0]) + dot(y0[1], R[1])) / (norm * max(alpha, beta)) < 1e-13
    # energy gradient dE/dpsi* = alpha |k|^2 psi + beta |psi|^2 psi, taken with the SAME truncation
    kk = np.arange(N)
    kk = np.where(kk < N // 2, kk, kk - N)
    k2 = (np.arange(N // 2 + 1)[None, None, :] ** 2 + kk[None, :, None] ** 2 + kk[:, None, None] ** 2).astype(float)
    rho = np.abs(psi) ** 2
    g = alpha * k2 * y0 + beta * oracle.apply_mask(pack(rho * psi))
    assert abs(dot(g[0], R[0]) + dot(g[1], R[1])) / (np.sqrt(dot(g[0], g[0]) + dot(g[1], g[1])) *
                                                     np.sqrt(dot(R[0], R[0]) + dot(R[1], R[1]))) < 1e-13


def test_numpy_restatement_and_mask():
    N, alpha, beta = 12, 0.3, 1.7
    y0 = np.stack([synth.scalar_spectrum(N, 2.0, 5, 9, tag=11), synth.scalar_spectrum(N, 2.0, 5, 9, tag=12)])
    M = oracle.dealias_mask(N)
    ym = y0 * M
    p, q = np.fft.irfftn(ym[0], s=(N, N, N), axes=(0, 1, 2)), np.fft.irfftn(ym[1], s=(N, N, N), axes=(0, 1, 2))
    rho = p * p + q * q
    kk = np.fft.fftfreq(N, 1.0 / N)
    k2 = np.arange(N // 2 + 1)[None, None, :] ** 2 + kk[None, :, None] ** 2 + kk[:, None, None] ** 2
    want = np.stack([beta * np.fft.rfftn(rho * q) * M + alpha * k2 * ym[1],
                     -beta * np.fft.rfftn(rho * p) * M - alpha * k2 * ym[0]])
    got = oracle.gpe_rhs(y0, alpha, beta)
    assert rel(got, want) < 1e-13
    assert np.all(got[:, ~M] == 0)


def test_rk_step_on_a_plane_wave_is_the_truncated_exponential():
    """O9 with sys = 3: |psi| stays A along the exact solution, so the RK polynomial of -i omega dt multiplies psi
    only to first order in the nonlinearity; for beta = 0 (linear) it is exact: psi_1 = P_ord(-i alpha k^2 dt) psi_0."""
    N, alpha, dt, ord = 16, 0.3, 0.05, 4
    x, y, z = synth.grid_axes(N)
    psi = 0.7 * np.exp(1j * (2 * x + y - z + 0 * x * y * z))
    w = -1j * alpha * 6 * dt
    poly = 1 + w + w ** 2 / 2 + w ** 3 / 6 + w ** 4 / 24
    got = oracle.rk_step(3, pack(psi), ord, dt, alpha, 0.0)
    assert rel(got, pack(poly * psi)) < 1e-14
