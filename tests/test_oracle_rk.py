"""Pins for the oracle's Runge-Kutta step (O9; reading G21) -- CPU only.

The scheme y^(o-1) = M y_n + (dt/o) R(y^(o)), o = ord..1, is pinned by what the mathematics fixes:
the truncated exponential on linear problems (Beltrami flow under viscosity, internal gravity waves),
forward Euler at ord = 1, a numpy re-statement of the stage loop built from the already pinned right-hand
sides, second-order convergence on a nonlinear problem, and the dealiased output.  A wrong stage
coefficient (dt/(ord-o+1), dt/ord, ...), a wrong base state (previous stage instead of y_n), a missing mask
or a swapped parameter fails at least one of them.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1808_01309_b200 import synth


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


def spec3(fields):
    return np.stack([oracle.r2c3d(f) for f in fields])


def taylor_poly(x, n):
    return sum(x ** j / math.factorial(j) for j in range(n + 1))


@pytest.mark.parametrize("ord", [1, 2, 3, 4])
@pytest.mark.parametrize("k", [1, 2])
def test_beltrami_flow_decays_by_the_truncated_exponential(ord, k):
    """ABC flow: u x w = 0, every mode has |k|^2 = k^2, so R = -nu k^2 u and one step multiplies u^ by
    sum_{j<=ord} (-nu k^2 dt)^j / j!  (the degree-ord Taylor polynomial of exp)."""
    N, nu, dt = 16, 0.7, 0.05
    uh = spec3(synth.abc_flow(N, k=k))
    got = oracle.rk_step(0, uh, ord, dt, nu)
    assert rel(got, taylor_poly(-nu * k * k * dt, ord) * uh) < 1e-13


def test_order_one_is_forward_euler():
    N = 16
    uh = synth.solenoidal_spectrum(N, 2.0, 7, 3)          # kcut above N/3: the mask on y_n matters
    got = oracle.rk_step(0, uh, 1, 0.01, 0.2)
    assert rel(got, oracle.apply_mask(uh) + 0.01 * oracle.hd_rhs(uh, 0.2)) < 1e-15
    M = oracle.dealias_mask(N)
    assert np.all(got[:, ~M] == 0)


@pytest.mark.parametrize("sys", [0, 1, 2, 3])
@pytest.mark.parametrize("ord", [2, 3, 4])
def test_stage_loop_restated_in_numpy(sys, ord):
    """The stage loop written out with the (separately pinned) right-hand sides.  sys = 3 (Gross-Pitaevskii,
    PAPER.md:54-56 Eq. 7) runs with alpha and beta both non-zero and different, and with a third parameter that must
    be ignored, so rk_rhs cannot take beta from the wrong slot of `par` (the only other CPU pin of that
    branch has beta = 0)."""
    N, dt, nu, c2, nbv = 12, 0.02, 0.11, 0.07, 1.3
    u = synth.solenoidal_spectrum(N, 2.0, 5, 5, tag=0)
    if sys == 3:
        y = 0.5 * u[:2]                                      # (p^, q^) of psi = p + i q: any two real fields
        rhs = lambda y: oracle.gpe_rhs(y, nu, c2)            # alpha = 0.11, beta = 0.07
        assert rel(oracle.gpe_rhs(y, nu, c2), oracle.gpe_rhs(y, nu, nbv)) > 1e-3     # beta matters on this input
    elif sys == 0:
        y = u
        rhs = lambda y: oracle.hd_rhs(y, nu)
    elif sys == 1:
        y = np.concatenate([u, synth.solenoidal_spectrum(N, 2.0, 5, 5, tag=1)])
        rhs = lambda y: np.concatenate(oracle.mhd_rhs(y[:3], y[3:], nu, c2))
    else:
        y = np.concatenate([u, synth.scalar_spectrum(N, 2.0, 5, 5)[None]])
        def rhs(y):
            ru, rt = oracle.boussinesq_rhs(y[:3], y[3], nu, c2, nbv)
            return np.concatenate([ru, rt[None]])
    ym = np.stack([oracle.apply_mask(f[None])[0] for f in y])
    cur = y
    for o in range(ord, 0, -1):
        cur = ym + (dt / o) * rhs(cur)
    assert rel(oracle.rk_step(sys, y, ord, dt, nu, c2, nbv), cur) < 1e-14


def test_internal_gravity_wave_frequency():
    """Linear Boussinesq (tiny amplitude): a plane wave with wavevector (kx, 0, kz) oscillates with
    omega = N_bv kx / |k| (Eqs. 1-3 linearised): w(t) = w0 cos(omega t), theta(t) = (|k|/kx)... checked through
    the exact 2x2 propagator on (w^, theta^) after n RK4 steps."""
    N, nbv, dt, nsteps = 16, 2.0, 0.01, 20
    kx, kz = 2, 1
    k2 = kx * kx + kz * kz
    amp = 1e-9                                               # nonlinear terms are O(amp^2)
    x, y, z = synth.grid_axes(N)
    phase = kx * x + kz * z + 0 * y
    # solenoidal velocity in the (x, z) plane: u = (-kz, 0, kx) cos(phase) * amp
    u = np.stack([-kz * amp * np.cos(phase), np.zeros_like(phase), kx * amp * np.cos(phase)])
    th = 0.5 * amp * np.sin(phase)
    st = np.concatenate([spec3(u), oracle.r2c3d(th)[None]])
    y0 = st.copy()
    for _ in range(nsteps):
        st = oracle.rk_step(2, st, 4, dt, 0.0, 0.0, nbv)
    # linear system for the Fourier amplitudes at this k:  dw/dt = -N_bv (kx^2/k^2) theta,  dtheta/dt = N_bv w
    om = nbv * kx / math.sqrt(k2)
    t = nsteps * dt
    w0, t0 = y0[2, kz, 0, kx], y0[3, kz, 0, kx]
    c, s = math.cos(om * t), math.sin(om * t)
    w_exact = w0 * c - (kx / math.sqrt(k2)) * t0 * s
    t_exact = t0 * c + (math.sqrt(k2) / kx) * w0 * s
    scale = abs(w0) + abs(t0)
    assert abs(st[2, kz, 0, kx] - w_exact) / scale < 1e-9    # RK4: (om dt)^4 * nsteps ~ 1e-7 * small consts
    assert abs(st[3, kz, 0, kx] - t_exact) / scale < 1e-9
    # u_x follows from incompressibility: kx u_x + kz u_z = 0
    assert abs(kx * st[0, kz, 0, kx] + kz * st[2, kz, 0, kx]) / scale < 1e-12


def test_second_order_convergence_on_taylor_green():
    """Nonlinear problem: the global error at fixed T falls by ~4 when dt is halved (ord = 2), measured
    against a much finer RK4 integration."""
    N, nu, T = 16, 0.05, 0.4
    u0 = spec3(synth.taylor_green(N))

    def integrate(ord, n):
        y = u0
        for _ in range(n):
            y = oracle.rk_step(0, y, ord, T / n, nu)
        return y

    ref = integrate(4, 64)
    e1 = rel(integrate(2, 4), ref)
    e2 = rel(integrate(2, 8), ref)
    assert 3.0 < e1 / e2 < 5.5
    # ord = 4 is more accurate than ord = 2 at the same dt (fourth order on the linear part, second on the rest)
    assert rel(integrate(4, 8), ref) < 0.2 * e2


def test_state_stays_solenoidal_and_dealiased():
    N = 16
    y = oracle.rk_step(0, synth.solenoidal_spectrum(N, 2.0, 7, 11), 3, 0.05, 0.1)
    k = np.arange(N)
    k = np.where(k < N // 2, k, k - N)
    div = np.arange(N // 2 + 1)[None, None, :] * y[0] + k[None, :, None] * y[1] + k[:, None, None] * y[2]
    assert np.abs(div).max() / np.abs(y).max() < 1e-14
    assert np.all(y[:, ~oracle.dealias_mask(N)] == 0)
