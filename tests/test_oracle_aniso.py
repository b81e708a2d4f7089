"""Pins for the oracle on anisotropic grids (Nx, Ny, Nz) and boxes (Lx, Ly, Lz) -- CPU only.

PAPER.md:64 (Sec. 2, below Eq. 8): "both the physical box size, L_i, and the number of physical space points,
N_i, may be specified independently in each direction".  Readings (G24, G25): k_i = 2 pi n_i / L_i, and
the 2/3 rule as the index-space ellipsoid sum (n_i / N_i)^2 < 1/9.

What fixes the general code (the cubic 2 pi box stays pinned by tests/test_oracle_rhs.py etc., which now run
through the same functions): closed forms in a stretched box (derivative, projection of a gradient, the
Taylor-Green vortex with three different wavenumbers, the Boussinesq scalar terms, the Gross-Pitaevskii plane
wave, the uniform-field induction term), the exact scaling law of an isotropic dilation, covariance under a
cyclic relabelling of the axes, embedding into the cubic grid, conservation laws, integer mask properties.
"""
import numpy as np
import pytest

import oracle
from paper_1808_01309_b200 import synth

TWO_PI = 2.0 * np.pi
SHAPE = (16, 12, 24)          # Nx, Ny, Nz
BOX = (TWO_PI, 3.0, 9.5)      # Lx, Ly, Lz


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


def spec(fields):
    return np.stack([oracle.r2c3d(f) for f in fields])


def phys(spectra):
    return np.stack([oracle.c2r3d(s) for s in spectra])


def indices(shape):
    Nx, Ny, Nz = shape
    f = lambda n: np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
    return np.arange(Nx // 2 + 1)[None, None, :], f(Ny)[None, :, None], f(Nz)[:, None, None]


def wavenumbers(shape, box):
    nx, ny, nz = indices(shape)
    return nx * (TWO_PI / box[0]), ny * (TWO_PI / box[1]), nz * (TWO_PI / box[2])


def half_weights(shape):
    w = np.full(shape[0] // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    return w[None, None, :]


# ---- a9 on a general grid (G25) -------------------------------------------------------------------------

@pytest.mark.parametrize("shape", [(16, 12, 24), (32, 32, 8), (24, 8, 16), (12, 48, 16)])
def test_mask_is_the_cubic_mask_of_the_lcm_grid_sampled(shape):
    """sum (n_i/N_i)^2 < 1/9 does not know the grid: mode n of (Nx, Ny, Nz) is kept iff mode (n_i L / N_i) of the
    cubic L^3 grid, L = lcm, is kept by the cubic rule (itself pinned by the golden mask counts)."""
    Nx, Ny, Nz = shape
    L = int(np.lcm.reduce(shape))
    m = oracle.dealias_mask(Nx, Ny, Nz)
    assert m.shape == (Nz, Ny, Nx // 2 + 1)
    big = oracle.dealias_mask(L)
    nx, ny, nz = indices(shape)
    want = big[np.broadcast_to((nz * (L // Nz)) % L, m.shape), np.broadcast_to((ny * (L // Ny)) % L, m.shape),
               np.broadcast_to(nx * (L // Nx), m.shape)]
    assert np.array_equal(m, want)


@pytest.mark.parametrize("shape", [(16, 12, 24), (32, 32, 8), (48, 24, 12)])
def test_mask_axis_extents_and_symmetry(shape):
    """Along each axis the last kept index is the largest n with 3 n < N_i (strict, G4); the mask is even in ny, nz;
    every Nyquist plane is out; the kept fraction approaches the ellipsoid volume (4 pi / 3) / 27 / 2."""
    Nx, Ny, Nz = shape
    m = oracle.dealias_mask(Nx, Ny, Nz)
    for axis_mask, n in ((m[0, 0, :], Nx), (m[0, :Ny // 2, 0], Ny), (m[:Nz // 2, 0, 0], Nz)):
        kept = np.nonzero(axis_mask)[0]
        assert kept.max() == (n - 1) // 3 and np.array_equal(kept, np.arange(kept.max() + 1))
    assert np.array_equal(m[:, 1:], m[:, 1:][:, ::-1]) and np.array_equal(m[1:], m[1:][::-1])
    assert not m[Nz // 2].any() and not m[:, Ny // 2].any() and not m[:, :, Nx // 2].any()
    frac = m.sum() / m.size
    assert abs(frac - 4 * np.pi / 3 / 27) < 0.04


# ---- a7, a10 with physical wavenumbers (G24) --------------------------------------------------------------

def test_curl_closed_form_in_a_stretched_box():
    """u = (0, 0, sin(a X) cos(b Y)), a = 3 (2 pi/Lx), b = 2 (2 pi/Ly): curl u = (-b sin aX sin bY, -a cos aX cos bY, 0);
    and u = (sin(c Z), 0, 0), c = 5 (2 pi/Lz): curl u = (0, c cos cZ, 0) -- each axis with its own box length."""
    x, y, z = synth.box_axes(SHAPE, BOX)
    one = np.ones(SHAPE[::-1])
    a, b, c = 3 * TWO_PI / BOX[0], 2 * TWO_PI / BOX[1], 5 * TWO_PI / BOX[2]
    w = phys(oracle.curl(spec([0 * one, 0 * one, np.sin(a * x) * np.cos(b * y) * one]), BOX))
    assert np.abs(w[0] - (-b * np.sin(a * x) * np.sin(b * y) * one)).max() < 1e-12
    assert np.abs(w[1] - (-a * np.cos(a * x) * np.cos(b * y) * one)).max() < 1e-12
    assert np.abs(w[2]).max() < 1e-12
    w = phys(oracle.curl(spec([np.sin(c * z) * one, 0 * one, 0 * one]), BOX))
    assert np.abs(w[1] - c * np.cos(c * z) * one).max() < 1e-12
    assert np.abs(w[0]).max() < 1e-12 and np.abs(w[2]).max() < 1e-12


def test_projection_annihilates_a_gradient_of_the_stretched_box():
    """grad phi, phi = sin(2 aX + bY) cos(3 cZ) with the box's own fundamental wavenumbers, written in closed form in
    physical space: P removes it, and leaves a field that is solenoidal in THIS box untouched."""
    x, y, z = synth.box_axes(SHAPE, BOX)
    a, b, c = TWO_PI / BOX[0], TWO_PI / BOX[1], TWO_PI / BOX[2]
    ph = 2 * a * x + b * y
    grad = spec([2 * a * np.cos(ph) * np.cos(3 * c * z), b * np.cos(ph) * np.cos(3 * c * z),
                 -3 * c * np.sin(ph) * np.sin(3 * c * z)])
    assert np.abs(oracle.project(grad, BOX)).max() / np.abs(grad).max() < 1e-13
    sol = synth.aniso_spectrum(SHAPE, BOX, seed=5)
    assert rel(oracle.project(sol + grad, BOX), sol) < 1e-13
    # the same gradient is NOT a gradient for the 2 pi box: the box really enters
    assert np.abs(oracle.project(grad)).max() / np.abs(grad).max() > 1e-2


# ---- O6: Taylor-Green with three different wavenumbers -------------------------------------------------------

def stretched_taylor_green(shape, box, A=1.3):
    """u = (A sin ax cos by cos cz, B cos ax sin by cos cz, 0), a A + b B = 0, and its closed-form right-hand side
    P[u x w] = ( -A^2 a c^2/(4(a^2+c^2)) sin 2ax cos 2cz,  -B^2 b c^2/(4(b^2+c^2)) sin 2by cos 2cz,
                 (c/4) [A^2 a^2/(a^2+c^2) cos 2ax + B^2 b^2/(b^2+c^2) cos 2by] sin 2cz )
    (u.grad u = ((A^2 a/2) sin 2ax, (B^2 b/2) sin 2by, 0) cos^2 cz; the z-independent half is a pure gradient)."""
    x, y, z = synth.box_axes(shape, box)
    a, b, c = TWO_PI / box[0], TWO_PI / box[1], TWO_PI / box[2]
    B = -a * A / b
    one = np.ones(shape[::-1])
    u = np.stack([A * np.sin(a * x) * np.cos(b * y) * np.cos(c * z) * one,
                  B * np.cos(a * x) * np.sin(b * y) * np.cos(c * z) * one, 0 * one])
    r = np.stack([-A * A * a * c * c / (4 * (a * a + c * c)) * np.sin(2 * a * x) * np.cos(2 * c * z) * one,
                  -B * B * b * c * c / (4 * (b * b + c * c)) * np.sin(2 * b * y) * np.cos(2 * c * z) * one,
                  (c / 4) * (A * A * a * a / (a * a + c * c) * np.cos(2 * a * x)
                             + B * B * b * b / (b * b + c * c) * np.cos(2 * b * y)) * np.sin(2 * c * z) * one])
    return u, r, a * a + b * b + c * c


@pytest.mark.parametrize("shape,box", [(SHAPE, BOX), ((24, 24, 8), (TWO_PI, TWO_PI, TWO_PI / 4)), ((16, 16, 16), (1.0, 2.0, 3.0))])
@pytest.mark.parametrize("nu", [0.0, 0.3])
def test_stretched_taylor_green_closed_form(shape, box, nu):
    u, want, k2 = stretched_taylor_green(shape, box)
    uh = spec(u)
    got = phys(oracle.hd_rhs(uh, nu, box=box))
    want = want - nu * k2 * u
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-13


def test_stretched_taylor_green_reduces_to_the_golden_cubic_one():
    """the closed form above at a = b = c = 1, A = 1 is the P7 closed form of tests/golden/taylor_green_rhs.txt"""
    u, want, _ = stretched_taylor_green((16, 16, 16), (TWO_PI,) * 3, A=1.0)
    assert np.abs(u - synth.taylor_green(16)).max() < 1e-15
    assert np.abs(phys(oracle.hd_rhs(spec(u))) - want).max() < 1e-14


# ---- exact symmetries ---------------------------------------------------------------------------------------

def test_isotropic_dilation_scaling_law():
    """Box s (2 pi) in every direction: k -> k/s, so the nonlinear term scales with 1/s and the viscous term with
    1/s^2: hd_rhs(u; s, nu) = hd_rhs(u; 1, 0)/s + [hd_rhs(u; 1, nu) - hd_rhs(u; 1, 0)]/s^2 (same coefficients)."""
    N, s, nu = 16, 2.5, 0.7
    uh = synth.broadband_spectrum(N, seed=3)
    r0, r1 = oracle.hd_rhs(uh, 0.0), oracle.hd_rhs(uh, nu)
    got = oracle.hd_rhs(uh, nu, box=(s * TWO_PI,) * 3)
    assert rel(got, r0 / s + (r1 - r0) / s**2) < 1e-13


def test_covariance_under_cyclic_relabelling_of_the_axes():
    """(x, y, z) -> (y, z, x) is a proper rotation: relabel grid, box, coordinates and components of a real field
    together and the right-hand side (compared in physical space) is relabelled the same way.  A slip that takes
    N_y for N_z, L_y for L_z, or one component's wavenumber for another's breaks it."""
    shape, box = (16, 12, 24), (TWO_PI, 3.0, 9.5)
    uh = synth.aniso_spectrum(shape, box, seed=11, fill=0.3)
    u = phys(uh)                                        # [c][z][y][x]
    r = phys(oracle.hd_rhs(uh, 0.2, box=box))
    # new axes (x', y', z') = (y, z, x): array [z'][y'][x'] = old [x... ] -> transpose (z,y,x) -> (x,z,y)
    perm = lambda f: np.ascontiguousarray(np.transpose(f, (2, 0, 1)))
    u2 = np.stack([perm(u[1]), perm(u[2]), perm(u[0])])     # u'_x' = u_y, u'_y' = u_z, u'_z' = u_x
    shape2, box2 = (shape[1], shape[2], shape[0]), (box[1], box[2], box[0])
    assert u2.shape[1:] == shape2[::-1]
    r2 = phys(oracle.hd_rhs(spec(u2), 0.2, box=box2))
    want = np.stack([perm(r[1]), perm(r[2]), perm(r[0])])
    # the input lies inside both masks (fill 0.3 < 1/3) and the mask is relabelling-invariant, so equality is exact
    assert rel(r2, want) < 1e-13


def test_embedding_into_the_cubic_grid():
    """P12 for anisotropic grids: the same band-limited coefficients on (16, 12, 24) and on 24^3 (box 2 pi) give the
    same right-hand side on every mode inside both masks."""
    shape, N = (16, 12, 24), 24
    small = synth.aniso_spectrum(shape, None, seed=2, fill=0.3)
    Nx, Ny, Nz = shape
    big = np.zeros((3, N, N, N // 2 + 1), dtype=complex)
    nx, ny, nz = (np.broadcast_to(a, small.shape[1:]) for a in indices(shape))
    big[:, nz % N, ny % N, nx] = small * (N**3 / (Nx * Ny * Nz))
    rs = oracle.hd_rhs(small, 0.1) / (Nx * Ny * Nz)
    rb = oracle.hd_rhs(big, 0.1) / N**3
    both = oracle.dealias_mask(Nx, Ny, Nz) & oracle.dealias_mask(N)[nz % N, ny % N, nx]
    assert both.sum() > 200
    assert rel(rs[:, both], rb[:, nz % N, ny % N, nx][:, both]) < 1e-13


def test_invariants_on_a_random_field_in_a_stretched_box():
    """P9 in the box: k . R = 0 with the physical k, energy and helicity conserved by the nonlinear term, exact zeros
    outside the ellipsoidal mask, Hermitian kx = 0 plane."""
    uh = synth.aniso_spectrum(SHAPE, BOX, seed=7)
    r = oracle.hd_rhs(uh, 0.0, box=BOX)
    kx, ky, kz = wavenumbers(SHAPE, BOX)
    m = oracle.dealias_mask(*SHAPE)
    um = uh * m
    assert np.abs(kx * r[0] + ky * r[1] + kz * r[2]).max() / np.abs(r).max() < 1e-13
    w = half_weights(SHAPE)
    scale = np.sum(w * np.abs(um) ** 2) * np.sqrt(np.sum(w * np.abs(r) ** 2) / np.sum(w * np.abs(um) ** 2))
    assert abs(np.sum(w * np.real(np.conj(um) * r))) / scale < 1e-13
    wh = oracle.curl(um, BOX)
    assert abs(np.sum(w * np.real(np.conj(wh) * r))) / (scale * np.sqrt(np.sum(np.abs(wh) ** 2) / np.sum(np.abs(um) ** 2))) < 1e-13
    assert np.all(r[:, ~m] == 0)
    Nz, Ny = SHAPE[2], SHAPE[1]
    p0 = r[:, :, :, 0]
    assert np.abs(p0 - np.conj(p0[:, (-np.arange(Nz)) % Nz][:, :, (-np.arange(Ny)) % Ny])).max() / np.abs(r).max() < 1e-13


# ---- O7, O8, O10, O9 in the box ---------------------------------------------------------------------------------

def test_mhd_uniform_field_closed_forms_in_the_box():
    """b = B0 z^ (the k = 0 mode): R_b = curl(u x B0) = B0 d_z u = i k_z B0 u^ with k_z = n_z 2 pi / L_z, and
    R_u = the hydrodynamic right-hand side (j = 0); b = 0 reduces to O6."""
    uh = synth.aniso_spectrum(SHAPE, BOX, seed=4, fill=0.3)
    B0 = 0.8
    bh = np.zeros_like(uh)
    bh[2, 0, 0, 0] = B0 * np.prod(SHAPE)
    ru, rb = oracle.mhd_rhs(uh, bh, 0.1, 0.0, box=BOX)
    _, _, kz = wavenumbers(SHAPE, BOX)
    m = oracle.dealias_mask(*SHAPE)
    assert rel(rb, 1j * kz * B0 * uh * m) < 1e-13
    assert rel(ru, oracle.hd_rhs(uh, 0.1, box=BOX)) < 1e-13
    ru0, rb0 = oracle.mhd_rhs(uh, 0 * uh, 0.1, 0.2, box=BOX)
    assert rel(ru0, oracle.hd_rhs(uh, 0.1, box=BOX)) < 1e-14 and np.abs(rb0).max() == 0


def test_boussinesq_closed_form_in_the_box():
    """Stretched Taylor-Green u with theta = sin(a x): u . grad theta = u_x a cos ax = (A a/2) sin 2ax cos by cos cz,
    so R_theta = -(A a/2) sin 2ax cos by cos cz - kappa a^2 theta (u_z = 0); and R_u = HD closed form + the projected
    buoyancy -N_bv P[theta z^] = -N_bv sin(ax) z^ (theta z^ is solenoidal: no z-dependence)."""
    shape, box = SHAPE, BOX
    u, want_u, k2 = stretched_taylor_green(shape, box)
    x, y, z = synth.box_axes(shape, box)
    a, b, c = TWO_PI / box[0], TWO_PI / box[1], TWO_PI / box[2]
    one = np.ones(shape[::-1])
    th = np.sin(a * x) * one
    nu, kappa, nbv, A = 0.2, 0.4, 1.7, 1.3
    ru, rt = oracle.boussinesq_rhs(spec(u), oracle.r2c3d(th), nu, kappa, nbv, box=box)
    want_t = -(A * a / 2) * np.sin(2 * a * x) * np.cos(b * y) * np.cos(c * z) * one - kappa * a * a * th
    assert np.abs(oracle.c2r3d(rt) - want_t).max() / np.abs(want_t).max() < 1e-13
    want_u = want_u - nu * k2 * u
    want_u[2] -= nbv * th
    assert np.abs(phys(ru) - want_u).max() / np.abs(want_u).max() < 1e-13
    # theta = 0 reduces to O6 in the same box
    ru0, rt0 = oracle.boussinesq_rhs(spec(u), 0 * oracle.r2c3d(th), nu, kappa, nbv, box=box)
    assert rel(ru0, oracle.hd_rhs(spec(u), nu, box=box)) < 1e-14


def test_boussinesq_energy_conservation_in_the_box():
    """Total energy 1/2 <|u|^2 + theta^2> is conserved by the inviscid system for any box: the buoyancy work
    -N_bv <w theta> cancels the source N_bv <theta w>."""
    uh = synth.aniso_spectrum(SHAPE, BOX, seed=8)
    th = synth.aniso_spectrum(SHAPE, BOX, seed=8, tag=7, ncomp=1)
    m = oracle.dealias_mask(*SHAPE)
    ru, rt = oracle.boussinesq_rhs(uh, th, 0.0, 0.0, 1.3, box=BOX)
    w = half_weights(SHAPE)
    dE = np.sum(w * np.real(np.conj(uh * m) * ru)) + np.sum(w * np.real(np.conj(th * m) * rt))
    norm = np.sqrt(np.sum(w * np.abs(uh * m) ** 2) * (np.sum(w * np.abs(ru) ** 2) + np.sum(w * np.abs(rt) ** 2)))
    assert abs(dE) / norm < 1e-13


def test_gpe_plane_wave_in_the_box():
    """psi = A exp(i k.x), k = (2 (2 pi/Lx), -1 (2 pi/Ly), 3 (2 pi/Lz)): d_t psi = -i (alpha |k|^2 + beta A^2) psi."""
    shape, box = (16, 12, 32), BOX
    x, y, z = synth.box_axes(shape, box)
    k = np.array([2 * TWO_PI / box[0], -1 * TWO_PI / box[1], 3 * TWO_PI / box[2]])
    A, alpha, beta = 0.7, 0.3, 1.9
    ph = k[0] * x + k[1] * y + k[2] * z + 0 * np.ones(shape[::-1])
    psi = A * np.exp(1j * ph)
    r = oracle.gpe_rhs(spec([psi.real, psi.imag]), alpha, beta, box=box)
    got = oracle.c2r3d(r[0]) + 1j * oracle.c2r3d(r[1])
    want = -1j * (alpha * k.dot(k) + beta * A * A) * psi
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-13


def test_rk_step_in_the_box_is_the_stage_loop_and_decays_a_beltrami_like_mode():
    """ord 1 = forward Euler with the box's right-hand side; and a single Fourier mode (nonlinear term zero) under
    viscosity follows the truncated exponential sum_{j<=ord} (-nu k^2 dt)^j / j! with the PHYSICAL k^2."""
    uh = synth.aniso_spectrum(SHAPE, BOX, seed=9, fill=0.3)
    dt, nu = 0.01, 0.3
    m = oracle.dealias_mask(*SHAPE)
    assert rel(oracle.rk_step(0, uh, 1, dt, nu, box=BOX), uh * m + dt * oracle.hd_rhs(uh, nu, box=BOX)) < 1e-14
    x, y, z = synth.box_axes(SHAPE, BOX)
    b, c = 2 * TWO_PI / BOX[1], 3 * TWO_PI / BOX[2]
    one = np.ones(SHAPE[::-1])
    u = spec([np.sin(b * y + c * z) * one, 0 * one, 0 * one])   # u_x(y, z): u . grad u = 0
    for ord_ in (2, 3, 4):
        got = oracle.rk_step(0, u, ord_, dt, nu, box=BOX)
        lam = -nu * (b * b + c * c) * dt
        poly = sum(lam**j / np.prod(np.arange(1, j + 1)) for j in range(ord_ + 1))
        assert rel(got, poly * u) < 1e-13
