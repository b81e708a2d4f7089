"""Pins for the oracle's Boussinesq right-hand side (O8, Eqs. 1-3) -- CPU only.

A plausible mistake anywhere in it (sign of the buoyancy or of N_bv w, buoyancy outside the projection,
a dropped gradient component, wrong diffusion factor, missing mask) fails at least one of these.
"""
import numpy as np
import pytest

import oracle
from paper_1808_01309_b200 import synth


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


def wavenumbers(N):
    k = np.arange(N)
    k = np.where(k < N // 2, k, k - N)
    return np.arange(N // 2 + 1)[None, None, :], k[None, :, None], k[:, None, None]


def half_weights(N):
    w = np.full(N // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    return w[None, None, :]


def spec3(fields):
    return np.stack([oracle.r2c3d(f) for f in fields])


def test_theta_zero_reduces_to_hd():
    """theta = 0: R_u is the Navier-Stokes right-hand side (Eq. 1 with theta = 0), R_theta = N_bv M w^."""
    N = 16
    uh = synth.solenoidal_spectrum(N, 2.0, 5, 7)
    ru, rt = oracle.boussinesq_rhs(uh, np.zeros((N, N, N // 2 + 1), complex), nu=0.3, kappa=0.1, nbv=2.5)
    assert rel(ru, oracle.hd_rhs(uh, 0.3)) < 1e-14
    assert rel(rt, 2.5 * oracle.apply_mask(uh)[2]) < 1e-14


@pytest.mark.parametrize("N", [16, 24])
def test_taylor_green_with_sin_x_temperature_closed_form(N):
    """u = Taylor-Green, theta = sin x (hand derivation):
         u . grad theta = u_x cos x = 1/2 sin 2x cos y cos z,   w = 0,   Lap theta = -theta
         => R_theta = -1/2 sin 2x cos y cos z - kappa sin x
         buoyancy -N_bv sin x z^ has k = (+-1,0,0) perpendicular to z^: the projection leaves it unchanged
         => R_u = P[u x w] - 3 nu u + (0, 0, -N_bv sin x),  P[u x w] = (-1/8 sin2x cos2z, -1/8 sin2y cos2z,
            1/8 (cos2x + cos2y) sin2z)."""
    nu, kappa, nbv = 0.2, 0.7, 1.5
    x, y, z = synth.grid_axes(N)
    one = np.ones((N, N, N))
    u = synth.taylor_green(N)
    th = np.sin(x) * one
    ru, rt = oracle.boussinesq_rhs(spec3(u), oracle.r2c3d(th), nu, kappa, nbv)
    want_t = -0.5 * np.sin(2 * x) * np.cos(y) * np.cos(z) - kappa * np.sin(x) * one
    want_u = np.stack([-0.125 * np.sin(2 * x) * np.cos(2 * z) * one, -0.125 * np.sin(2 * y) * np.cos(2 * z) * one,
                       0.125 * (np.cos(2 * x) + np.cos(2 * y)) * np.sin(2 * z)]) - 3.0 * nu * u
    want_u[2] += -nbv * np.sin(x) * one
    assert np.abs(oracle.c2r3d(rt) - want_t).max() < 5e-14
    for c in range(3):
        assert np.abs(oracle.c2r3d(ru[c]) - want_u[c]).max() < 5e-14
    # the same statement in spectral entries: -1/2 sin2x cos y cos z -> +i N^3/16 at (kx, ky, kz) = (2, +-1, +-1)
    for kz in (1, -1):
        for ky in (1, -1):
            assert abs(rt[kz % N, ky % N, 2] / N**3 - 1j / 16) < 1e-15
    assert abs(rt[0, 0, 1] / N**3 - (-kappa) * (-0.5j)) < 1e-15


def test_buoyancy_is_inside_the_projection():
    """theta = sin z, u = 0: -N_bv theta z^ is a pure gradient (k parallel to z^) and the pressure removes it
    entirely (hydrostatic balance): R_u = 0.  With theta = sin(x + z) half of it survives:
    P[-N sin(x+z) z^] = -N sin(x+z) (z^ - k k_z/|k|^2) = -N sin(x+z) (-1/2, 0, 1/2)."""
    N, nbv = 12, 3.0
    x, y, z = synth.grid_axes(N)
    one = np.ones((N, N, N))
    zero3 = np.zeros((3, N, N, N // 2 + 1), complex)
    ru, rt = oracle.boussinesq_rhs(zero3, oracle.r2c3d(np.sin(z) * one), 0.0, 0.0, nbv)
    assert np.abs(ru).max() < 1e-12 and np.abs(rt).max() < 1e-12
    ru, rt = oracle.boussinesq_rhs(zero3, oracle.r2c3d(np.sin(x + z) * one), 0.0, 0.0, nbv)
    s = np.sin(x + z) * one
    assert np.abs(oracle.c2r3d(ru[0]) - 0.5 * nbv * s).max() < 1e-13
    assert np.abs(oracle.c2r3d(ru[1])).max() < 1e-13
    assert np.abs(oracle.c2r3d(ru[2]) + 0.5 * nbv * s).max() < 1e-13


def test_internal_wave_coupling_signs():
    """Linear terms only (one small-amplitude mode each, products are O(eps^2) and removed by choosing
    u along z^ uniform in z so that u.grad theta = 0 and u x w is a gradient):
    u = (0, 0, cos x), theta = 0  =>  R_theta = +N_bv cos x (Eq. 2 source N_bv w)."""
    N, nbv = 12, 0.8
    x, y, z = synth.grid_axes(N)
    one = np.ones((N, N, N))
    u = np.stack([0 * one, 0 * one, np.cos(x) * one])
    ru, rt = oracle.boussinesq_rhs(spec3(u), np.zeros((N, N, N // 2 + 1), complex), 0.0, 0.0, nbv)
    assert np.abs(oracle.c2r3d(rt) - nbv * np.cos(x) * one).max() < 1e-14
    # u x w = (0,0,cos x) x (0, sin x, 0) = (-cos x sin x, 0, 0) = grad(...): projected away
    assert np.abs(ru).max() / N**3 < 1e-14


@pytest.mark.parametrize("N", [24, 32])
def test_invariants_random_fields(N):
    """nu = kappa = 0: total energy 1/2<|u|^2 + theta^2> is conserved (advection conserves both parts, the
    buoyancy exchange -N theta w + N theta w cancels), theta-variance alone is conserved when N_bv = 0,
    R_u is solenoidal, both outputs vanish exactly outside the mask and are Hermitian on kx = 0."""
    kc = N // 3 - 1
    uh = synth.solenoidal_spectrum(N, 3.0, kc, 11)
    th = synth.scalar_spectrum(N, 3.0, kc, 11)
    w = half_weights(N)
    kx, ky, kz = wavenumbers(N)
    ru, rt = oracle.boussinesq_rhs(uh, th, 0.0, 0.0, 1.7)
    scale = float(np.sum(w * np.abs(uh) ** 2))
    e = np.sum(w * (np.conj(uh) * ru).real) + np.sum(w * (np.conj(th) * rt).real)
    assert abs(e) / scale < 1e-13
    assert abs(np.sum(w * (np.conj(uh) * ru).real)) / scale > 1e-4      # ...but not each part alone
    assert np.abs(kx * ru[0] + ky * ru[1] + kz * ru[2]).max() / np.abs(ru).max() < 1e-12
    m = oracle.dealias_mask(N)
    assert np.all(ru[:, ~m] == 0) and np.all(rt[~m] == 0)
    idx = (-np.arange(N)) % N
    assert rel(rt[:, :, 0], np.conj(rt[idx][:, idx][:, :, 0])) < 1e-12
    ru0, rt0 = oracle.boussinesq_rhs(uh, th, 0.0, 0.0, 0.0)
    assert abs(np.sum(w * (np.conj(th) * rt0).real)) / scale < 1e-13
    assert rel(ru0, oracle.hd_rhs(uh, 0.0)) < 1e-13                     # N_bv = 0: theta is passive


def test_diffusion_terms():
    N = 16
    uh = synth.solenoidal_spectrum(N, 2.0, 4, 3)
    th = synth.scalar_spectrum(N, 2.0, 4, 3)
    kx, ky, kz = wavenumbers(N)
    k2 = kx**2 + ky**2 + kz**2
    a_u, a_t = oracle.boussinesq_rhs(uh, th, 0.0, 0.0, 0.4)
    b_u, b_t = oracle.boussinesq_rhs(uh, th, 0.5, 0.25, 0.4)
    assert rel(b_u - a_u, -0.5 * k2 * uh) < 1e-13
    assert rel(b_t - a_t, -0.25 * k2 * th) < 1e-13


def test_against_independent_numpy_restatement():
    """The nine steps written again with numpy's pocketfft (rfftn / irfftn) and array expressions."""
    N, nu, kappa, nbv = 20, 0.1, 0.05, 2.0
    kc = 6
    uh = synth.solenoidal_spectrum(N, 2.5, kc, 5)
    th = synth.scalar_spectrum(N, 2.5, kc, 5)
    # unmasked content on purpose: add modes outside the sphere that the mask-on-load must remove
    uh[0, 0, 0, N // 2 - 1] = 3.0 * N**3
    th[1, 2, N // 2 - 2] = (1 - 2j) * N**3
    kx, ky, kz = wavenumbers(N)
    k2 = kx**2 + ky**2 + kz**2
    M = 9 * k2 < N * N
    um, tm = uh * M, th * M
    inv = lambda f: np.fft.irfftn(f, s=(N, N, N), axes=(0, 1, 2))
    fwd = lambda f: np.fft.rfftn(f, axes=(0, 1, 2))
    u = [inv(um[c]) for c in range(3)]
    wh = [1j * (ky * um[2] - kz * um[1]), 1j * (kz * um[0] - kx * um[2]), 1j * (kx * um[1] - ky * um[0])]
    w = [inv(f) for f in wh]
    g = [inv(1j * kk * tm) for kk in (kx, ky, kz)]
    n = [u[1] * w[2] - u[2] * w[1], u[2] * w[0] - u[0] * w[2], u[0] * w[1] - u[1] * w[0]]
    s = u[0] * g[0] + u[1] * g[1] + u[2] * g[2]
    nh = np.stack([fwd(f) for f in n]) * M
    nh[2] -= nbv * tm
    k2s = np.where(k2 == 0, 1, k2)
    d = (kx * nh[0] + ky * nh[1] + kz * nh[2]) / k2s
    want_u = nh - np.stack([kx * d, ky * d, kz * d]) * (k2 != 0) - nu * k2 * um
    want_t = -fwd(s) * M + nbv * um[2] - kappa * k2 * tm
    ru, rt = oracle.boussinesq_rhs(uh, th, nu, kappa, nbv)
    assert rel(ru, want_u) < 1e-13 and rel(rt, want_t) < 1e-13
