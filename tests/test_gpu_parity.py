"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Run on the B200 box:  python -m pytest tests -m gpu

Tolerances (BASELINE.json north_star): relative L2 error <= 1e-12 (fp64), <= 2e-5 (fp32) over the whole
output; the dealias mask bit-exact (masked outputs exactly +0).
"""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_1808_01309_b200 import psfft, synth  # noqa: E402
from parity_util import assert_shells  # noqa: E402

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-12, torch.float32: 2e-5}
CDT = {torch.float64: np.complex128, torch.float32: np.complex64}
RDT = {torch.float64: np.float64, torch.float32: np.float32}
SMALL = [8, 12, 16, 24, 32, 48, 64, 96, 128]


def rel(a, b):
    a = np.asarray(a).astype(np.complex128 if np.iscomplexobj(a) else np.float64)
    b = np.asarray(b).astype(a.dtype)
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.fixture(autouse=True)
def _sync():
    yield
    torch.cuda.synchronize()


# ---- config 1 and friends: r2c / c2r -------------------------------------------------------------

@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", SMALL)
def test_r2c_matches_oracle(N, dtype):
    batch = 2 if N <= 48 else 1
    x = synth.uniform_field(N, batch, 1234, RDT[dtype])
    p = psfft.Plan(N, dtype, batch)
    X = p.r2c(dev(x)).cpu().numpy()
    assert X.shape == (batch, N, N, N // 2 + 1)
    for b in range(batch):
        assert rel(X[b], oracle.r2c3d(x[b].astype(np.float64))) < TOL[dtype]


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", SMALL)
def test_c2r_matches_oracle_on_non_hermitian_input(N, dtype):
    """Any half spectrum is a valid input; the imaginary parts at kx = 0, N/2 are ignored as the oracle defines."""
    rng = np.random.default_rng(N)
    X = (rng.standard_normal((1, N, N, N // 2 + 1)) + 1j * rng.standard_normal((1, N, N, N // 2 + 1))).astype(CDT[dtype])
    p = psfft.Plan(N, dtype, 1)
    Xd = dev(X)
    x = p.c2r(Xd).cpu().numpy()
    assert rel(x[0], oracle.c2r3d(X[0].astype(np.complex128), N)) < TOL[dtype]
    assert np.array_equal(Xd.cpu().numpy(), X)          # input not modified


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [192, 256, 384])
def test_r2c_c2r_at_the_remaining_sizes(N, dtype):
    x = synth.uniform_field(N, 1, 99, RDT[dtype])
    p = psfft.Plan(N, dtype, 1)
    X = p.r2c(dev(x))
    Xo = oracle.r2c3d(x[0].astype(np.float64))
    assert rel(X.cpu().numpy()[0], Xo) < TOL[dtype]
    assert rel(p.c2r(X).cpu().numpy(), x) < TOL[dtype]


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_config1_roundtrip_32(dtype):
    """BASELINE.json config 1: 32^3, uniform [-1,1) from seed, r2c then c2r; spectrum and round trip vs oracle."""
    N = 32
    x = synth.uniform_field(N, 1, 1234, RDT[dtype])
    p = psfft.Plan(N, dtype, 1)
    X = p.r2c(dev(x))
    back = p.c2r(X).cpu().numpy()
    Xo = oracle.r2c3d(x[0].astype(np.float64))
    assert rel(X.cpu().numpy()[0], Xo) < TOL[dtype]
    assert rel(back[0], oracle.c2r3d(Xo)) < TOL[dtype]
    assert rel(back, x) < TOL[dtype]


# ---- anisotropic grids (transforms) ---------------------------

@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(32, 16, 8), (8, 24, 48), (64, 64, 16), (48, 32, 32), (128, 96, 24), (16, 128, 64)])
def test_anisotropic_r2c_c2r_match_oracle(shape, dtype):
    """(Nx, Ny, Nz) all different, incl. radix-3 sizes and the paper's flat-box aspect ratio (4:4:1)."""
    Nx, Ny, Nz = shape
    x = synth.uniform01(77, np.arange(Nz * Ny * Nx, dtype=np.uint64)).reshape(1, Nz, Ny, Nx) * 2 - 1
    x = x.astype(RDT[dtype])
    p = psfft.Plan(shape, dtype, 1)
    assert (p.layout.N, p.layout.Ny, p.layout.Nz, p.layout.ldk) == (Nx, Ny, Nz, Nx // 2 + 1)
    X = p.r2c(dev(x))
    assert tuple(X.shape) == (1, Nz, Ny, Nx // 2 + 1)
    Xo = oracle.r2c3d(x[0].astype(np.float64))
    assert rel(X.cpu().numpy()[0], Xo) < TOL[dtype]
    back = p.c2r(X).cpu().numpy()
    assert rel(back, x) < TOL[dtype]
    rng = np.random.default_rng(5)
    Y = (rng.standard_normal(Xo.shape) + 1j * rng.standard_normal(Xo.shape)).astype(CDT[dtype])   # non-Hermitian input
    y = p.c2r(dev(Y[None])).cpu().numpy()[0]
    assert rel(y, oracle.c2r3d(Y.astype(np.complex128), Nx)) < TOL[dtype]


def test_unfused_cross_check_path_needs_a_cubic_plan():
    """Only the *_unfused variants are cubic-only; the fused right-hand sides take any plan (tests/test_gpu_aniso.py)."""
    p = psfft.Plan((32, 32, 16), torch.float64, 1, work="hd")
    assert p.layout.work_bytes_hd > 0 and psfft.rk_work_bytes(p.handle, psfft.SYS_HD) > 0
    u = torch.zeros((3, 16, 32, 17), dtype=torch.complex128, device="cuda")
    with pytest.raises(psfft.PsfftError):
        psfft.hd_rhs_unfused(p.handle, u, torch.empty_like(u), 0.0, p.ensure_work("hd"))


def test_unfused_cross_check_path_needs_the_default_box():
    """The *_unfused kernels use integer wavenumbers: after psfft_plan_set_box to another box they must refuse
    (PSFFT_E_SIZE) instead of returning the 2 pi-box answer; setting the box back to 2 pi re-enables them."""
    import math
    N = 16
    p = psfft.Plan(N, torch.float64, 1, work="mhd")
    u = dev(synth.solenoidal_spectrum(N, 3.0, 5, 21))
    b = dev(synth.solenoidal_spectrum(N, 3.0, 5, 22, tag=1))
    L = psfft.lib()
    st = torch.cuda.current_stream().cuda_stream
    ru, rb = torch.full_like(u, 7.0), torch.full_like(b, 7.0)
    want = torch.empty_like(u)
    psfft.hd_rhs_unfused(p.handle, u, want, 0.1, p._work)
    psfft.plan_set_box(p.handle, 2 * math.pi, 2 * math.pi, math.pi)
    assert L.psfft_hd_rhs_unfused(p.handle, u.data_ptr(), ru.data_ptr(), 0.1, p._work.data_ptr(), st) == -2
    assert L.psfft_mhd_rhs_unfused(p.handle, u.data_ptr(), b.data_ptr(), ru.data_ptr(), rb.data_ptr(), 0.1, 0.1,
                                   p._work.data_ptr(), st) == -2
    torch.cuda.synchronize()
    assert bool((ru == 7.0).all()) and bool((rb == 7.0).all())            # nothing was enqueued
    fused_box = p.hd_rhs(u, 0.1)                                            # the fused call does take the box
    assert not torch.equal(fused_box, want)
    psfft.plan_set_box(p.handle, 2 * math.pi, 2 * math.pi, 2 * math.pi)
    psfft.hd_rhs_unfused(p.handle, u, ru, 0.1, p._work)
    assert torch.equal(ru, want)


def test_degenerate_inputs():
    N = 16
    p = psfft.Plan(N, torch.float64, 1)
    z = torch.zeros((1, N, N, N), dtype=torch.float64, device="cuda")
    assert torch.count_nonzero(p.r2c(z)) == 0
    one = torch.ones_like(z)
    X = p.r2c(one).cpu().numpy()
    want = np.zeros_like(X)
    want[0, 0, 0, 0] = N**3
    assert np.abs(X - want).max() < 1e-9
    X = p.r2c(dev(synth.single_mode(N, 3, 2, -1)[None])).cpu().numpy()[0]
    want = np.zeros_like(X)
    want[N - 1, 2, 3] = N**3 / 2
    assert np.abs(X - want).max() < 1e-9


def test_streams_and_graph_capture():
    """Execute calls only enqueue on the given stream and are CUDA-graph capturable."""
    N = 32
    x = dev(synth.uniform_field(N, 1, 5))
    p = psfft.Plan(N, torch.float64, 1)
    ref = p.r2c(x).clone()
    out = torch.empty_like(ref)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        psfft.fft3d_r2c(p.handle, x, out, None)          # warm (func attributes) outside capture
        g = torch.cuda.CUDAGraph()
        out.zero_()
        with torch.cuda.graph(g, stream=s):
            psfft.fft3d_r2c(p.handle, x, out, None, stream=s)
        g.replay()
    s.synchronize()
    assert torch.equal(out, ref)
    assert psfft.last_launch_count(p.handle) == 3


def test_time_loop_as_one_cuda_graph():
    """A whole RK2 time step (two fused RHS evaluations, 10 launches) captured once and replayed: the replayed
    trajectory equals the eagerly stepped one bit for bit (same kernels, same order)."""
    N, steps = 32, 4
    y0 = dev(rk_state(psfft.SYS_BOUSSINESQ, N, 3.0, N // 2 - 1, torch.float64))
    p = psfft.Plan(N, torch.float64, 1)
    a, b = y0.clone(), torch.empty_like(y0)
    for _ in range(steps):                                   # eager reference, ping-pong a -> b -> a
        p.rk_step(psfft.SYS_BOUSSINESQ, a, 2, 0.01, 0.01, 0.02, 1.5, out=b)
        a, b = b, a
    want = a.clone()
    a, b = y0.clone(), torch.empty_like(y0)
    work = p.ensure_work("rk_boussinesq")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):                  # two steps per replay: a -> b -> a
            psfft.rk_step(p.handle, psfft.SYS_BOUSSINESQ, a, b, 2, 0.01, (0.01, 0.02, 1.5), work, stream=s)
            psfft.rk_step(p.handle, psfft.SYS_BOUSSINESQ, b, a, 2, 0.01, (0.01, 0.02, 1.5), work, stream=s)
        for _ in range(steps // 2):
            g.replay()
    s.synchronize()
    assert torch.equal(a, want)
    assert psfft.last_launch_count(p.handle) == 10


# ---- config 2 and friends: HD right-hand side ------------------------------------------------------

def hd_case(N, k0, kcut, dtype, nu=0.0, seed=1234):
    uh = synth.solenoidal_spectrum(N, k0, kcut, seed).astype(CDT[dtype])
    p = psfft.Plan(N, dtype, 1, work="hd")
    got = p.hd_rhs(dev(uh), nu).cpu().numpy()
    want = oracle.hd_rhs(uh.astype(np.complex128), nu)
    return got, want


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N,k0,kcut", [(16, 2.0, 7), (24, 2.0, 11), (32, 4.0, 15), (48, 4.0, 23), (64, 4.0, 31), (96, 4.0, 32)])
def test_hd_rhs_matches_oracle(N, k0, kcut, dtype):
    """kcut above N/3 on purpose: the input mask of step 1 has to act."""
    got, want = hd_case(N, k0, kcut, dtype)
    assert rel(got, want) < TOL[dtype]
    M = oracle.dealias_mask(N)
    assert np.all(got[:, ~M] == 0) and not np.any(np.signbit(got[:, ~M].real)) and not np.any(np.signbit(got[:, ~M].imag))


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_config2_hd_rhs_128(dtype):
    """BASELINE.json config 2: 128^3 HD RHS, E(k) ~ k^4 exp(-2 (k/4)^2), unit energy, seed 1234."""
    got, want = hd_case(128, 4.0, 32, dtype)
    assert rel(got, want) < TOL[dtype]
    M = oracle.dealias_mask(128)
    assert np.all(got[:, ~M] == 0)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [192, 256, 384])
def test_rhs_at_the_remaining_sizes(N, dtype):
    """Every supported size runs its own radix schedules (mid_x: 8 3 8, 8 4 8, 8 2 3 8): HD and Boussinesq against
    the oracle on the grid itself."""
    got, want = hd_case(N, 4.0, 32, dtype, nu=0.01)
    assert rel(got, want) < TOL[dtype]
    assert np.all(got[:, ~oracle.dealias_mask(N)] == 0)
    if N != 384:
        ru, rt, wu, wt = boussinesq_case(N, 4.0, 32, dtype, 0.01, 0.02, 1.5)
        assert rel(ru, wu) < TOL[dtype] and rel(rt, wt) < TOL[dtype]


def test_hd_rhs_viscous_term():
    got, want = hd_case(32, 4.0, 12, torch.float64, nu=0.37)
    assert rel(got, want) < 1e-12


def test_hd_rhs_taylor_green_closed_form():
    """P7 directly on the GPU result: 12 entries +-i N^3/32."""
    N = 32
    uh = np.stack([oracle.r2c3d(f) for f in synth.taylor_green(N)])
    p = psfft.Plan(N, torch.float64, 1, work="hd")
    got = p.hd_rhs(dev(uh)).cpu().numpy() / N**3
    assert abs(got[0, 2, 0, 2] - 0.03125j) < 1e-15 and abs(got[0, N - 2, 0, 2] - 0.03125j) < 1e-15
    assert abs(got[2, 2, 0, 2] + 0.03125j) < 1e-15 and abs(got[2, N - 2, 2, 0] - 0.03125j) < 1e-15
    assert np.count_nonzero(np.abs(got) > 1e-13) == 12


def test_hd_rhs_abc_is_steady_and_input_untouched():
    N = 16
    uh = np.stack([oracle.r2c3d(f) for f in synth.abc_flow(N)])
    d = dev(uh)
    p = psfft.Plan(N, torch.float64, 1, work="hd")
    got = p.hd_rhs(d).cpu().numpy()
    assert np.abs(got).max() / N**3 < 1e-14
    assert np.array_equal(d.cpu().numpy(), uh)


# ---- MHD ----------------------------------------------------------------------------------------------

@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [16, 32, 48, 64])
def test_mhd_rhs_matches_oracle(N, dtype):
    kcut = N // 2 - 1
    uh = synth.solenoidal_spectrum(N, 3.0, kcut, 1234, tag=0).astype(CDT[dtype])
    bh = synth.solenoidal_spectrum(N, 3.0, kcut, 1234, tag=1).astype(CDT[dtype])
    p = psfft.Plan(N, dtype, 1, work="mhd")
    ru, rb = p.mhd_rhs(dev(uh), dev(bh), 0.01, 0.02)
    wu, wb = oracle.mhd_rhs(uh.astype(np.complex128), bh.astype(np.complex128), 0.01, 0.02)
    assert rel(ru.cpu().numpy(), wu) < TOL[dtype]
    assert rel(rb.cpu().numpy(), wb) < TOL[dtype]
    M = oracle.dealias_mask(N)
    assert np.all(ru.cpu().numpy()[:, ~M] == 0) and np.all(rb.cpu().numpy()[:, ~M] == 0)


# ---- Boussinesq (Eqs. 1-3) ------------------------------------------

def boussinesq_case(N, k0, kcut, dtype, nu, kappa, nbv):
    uh = synth.solenoidal_spectrum(N, k0, kcut, 1234).astype(CDT[dtype])
    th = synth.scalar_spectrum(N, k0, kcut, 1234).astype(CDT[dtype])
    p = psfft.Plan(N, dtype, 1, work="boussinesq")
    ud, td = dev(uh), dev(th)
    ru, rt = p.boussinesq_rhs(ud, td, nu, kappa, nbv)
    assert np.array_equal(ud.cpu().numpy(), uh) and np.array_equal(td.cpu().numpy(), th)     # inputs untouched
    wu, wt = oracle.boussinesq_rhs(uh.astype(np.complex128), th.astype(np.complex128), nu, kappa, nbv)
    return ru.cpu().numpy(), rt.cpu().numpy(), wu, wt


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N,k0,kcut", [(16, 2.0, 7), (24, 2.0, 11), (32, 4.0, 15), (48, 4.0, 23), (64, 4.0, 31), (96, 4.0, 32),
                                       (128, 4.0, 32)])
def test_boussinesq_rhs_matches_oracle(N, k0, kcut, dtype):
    """All terms on: nu, kappa, N_bv != 0; kcut above N/3 so that the input mask has to act.  N = 64 runs the
    radix-8 two-for-one mid_x kernel, the others the generic one."""
    ru, rt, wu, wt = boussinesq_case(N, k0, kcut, dtype, 0.013, 0.021, 2.5)
    assert rel(ru, wu) < TOL[dtype]
    assert rel(rt, wt) < TOL[dtype]
    M = oracle.dealias_mask(N)
    assert np.all(ru[:, ~M] == 0) and np.all(rt[~M] == 0)


@pytest.mark.parametrize("nu,kappa,nbv", [(0.0, 0.0, 0.0), (0.0, 0.0, 1.7), (0.02, 0.0, 0.0), (0.0, 0.03, 0.0)])
def test_boussinesq_rhs_term_by_term(nu, kappa, nbv):
    """Each optional term alone (the epilogue skips the reads of a term whose coefficient is zero)."""
    ru, rt, wu, wt = boussinesq_case(32, 4.0, 12, torch.float64, nu, kappa, nbv)
    assert rel(ru, wu) < 1e-12 and rel(rt, wt) < 1e-12


def test_boussinesq_reduces_to_hd_when_theta_vanishes():
    N = 32
    uh = synth.solenoidal_spectrum(N, 4.0, 12, 1234)
    p = psfft.Plan(N, torch.float64, 1, work="boussinesq")
    ru, rt = p.boussinesq_rhs(dev(uh), dev(np.zeros((N, N, N // 2 + 1), np.complex128)), 0.01, 0.02, 0.0)
    hd = p.hd_rhs(dev(uh), 0.01)
    assert float((ru - hd).norm() / hd.norm()) < 1e-14 and float(rt.abs().max()) == 0.0


# ---- Runge-Kutta step -------------------------------------------------

def rk_state(system, N, k0, kcut, dtype):
    u = synth.solenoidal_spectrum(N, k0, kcut, 1234, tag=0)
    if system == psfft.SYS_HD:
        y = u
    elif system == psfft.SYS_MHD:
        y = np.concatenate([u, synth.solenoidal_spectrum(N, k0, kcut, 1234, tag=1)])
    else:
        y = np.concatenate([u, synth.scalar_spectrum(N, k0, kcut, 1234)[None]])
    return np.ascontiguousarray(y.astype(CDT[dtype]))


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("system", [0, 1, 2])
@pytest.mark.parametrize("N,ord", [(16, 1), (24, 2), (32, 3), (48, 4), (64, 2), (96, 4)])
def test_rk_step_matches_oracle(N, ord, system, dtype):
    """dt chosen so that dt * |R| is comparable to |y| (CFL-like): the stages feed on each other."""
    y = rk_state(system, N, 3.0, N // 2 - 1, dtype)
    dt, nu, c2, nbv = 0.02, 0.013, 0.021, 2.5
    p = psfft.Plan(N, dtype, 1)
    yd = dev(y)
    got = p.rk_step(system, yd, ord, dt, nu, c2, nbv).cpu().numpy()
    assert np.array_equal(yd.cpu().numpy(), y)                      # y_n untouched
    want = oracle.rk_step(system, y.astype(np.complex128), ord, dt, nu, c2, nbv)
    assert rel(got, want) < TOL[dtype]
    assert np.all(got[:, ~oracle.dealias_mask(N)] == 0)
    assert rel(got, y) > 1e-3                                        # the step did something


@pytest.mark.parametrize("system", [0, 3])
def test_rk_intermediate_stages_never_read_outside_the_sphere(system):
    """Intermediate stages skip the zero fill outside the truncation sphere (the next stage masks on load): poison
    the workspace and the output with NaN bit patterns first; the result must still match the oracle and be fully
    defined."""
    N, ord = 32, 4
    y = rk_state(system, N, 3.0, N // 2 - 1, torch.float64) if system == 0 else gpe_state(N, N // 2 - 1, torch.float64)
    p = psfft.Plan(N, torch.float64, 1)
    p.ensure_work("rk_hd" if system == 0 else "rk_gpe").fill_(0xFF)
    out = torch.full(y.shape, float("nan"), dtype=torch.complex128, device="cuda")
    got = p.rk_step(system, dev(y), ord, 0.02, 0.013, 0.5, out=out).cpu().numpy()
    want = oracle.rk_step(system, y, ord, 0.02, 0.013, 0.5)
    assert np.isfinite(got).all() and rel(got, want) < 1e-12
    assert np.all(got[:, ~oracle.dealias_mask(N)] == 0)


def test_rk_step_beltrami_closed_form_and_argument_checks():
    """ABC flow under viscosity: one RK4 step multiplies u^ by 1 + x + x^2/2 + x^3/6 + x^4/24, x = -nu dt."""
    N, nu, dt = 32, 0.7, 0.05
    uh = np.stack([oracle.r2c3d(f) for f in synth.abc_flow(N)])
    p = psfft.Plan(N, torch.float64, 1)
    got = p.rk_step(psfft.SYS_HD, dev(uh), 4, dt, nu).cpu().numpy()
    x = -nu * dt
    assert rel(got, (1 + x + x * x / 2 + x ** 3 / 6 + x ** 4 / 24) * uh) < 1e-13
    yd = dev(uh)
    work = p.ensure_work("rk_hd")
    with pytest.raises(psfft.PsfftError):
        psfft.rk_step(p.handle, psfft.SYS_HD, yd, yd, 2, dt, (nu, 0, 0), work)          # in == out
    with pytest.raises(psfft.PsfftError):
        psfft.rk_step(p.handle, psfft.SYS_HD, yd, torch.empty_like(yd), 5, dt, (nu, 0, 0), work)   # ord > 4


# ---- Gross-Pitaevskii (Eq. 7; the paper's fourth solver) ----------------------------------------

def gpe_state(N, kcut, dtype):
    y = np.stack([synth.scalar_spectrum(N, 3.0, kcut, 1234, tag=11), synth.scalar_spectrum(N, 3.0, kcut, 1234, tag=12)])
    y[0, 0, 0, 0] = float(N) ** 3                                   # condensate: psi = 1 + fluctuations
    return np.ascontiguousarray(y.astype(CDT[dtype]))


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [16, 24, 32, 48, 64, 96, 128])
def test_gpe_rhs_matches_oracle(N, dtype):
    y = gpe_state(N, N // 2 - 1, dtype)                             # kcut above N/3: the input mask acts
    p = psfft.Plan(N, dtype, 1, work="gpe")
    yd = dev(y)
    got = p.gpe_rhs(yd, 0.37, 1.3).cpu().numpy()
    assert np.array_equal(yd.cpu().numpy(), y)
    want = oracle.gpe_rhs(y.astype(np.complex128), 0.37, 1.3)
    assert rel(got, want) < TOL[dtype]
    assert np.all(got[:, ~oracle.dealias_mask(N)] == 0)


def test_gpe_plane_wave_closed_form():
    """psi = A exp(i k.x) is an exact solution: rhs = -i (alpha |k|^2 + beta A^2) psi."""
    N, A, alpha, beta = 32, 0.7, 0.3, 1.1
    x, y, z = synth.grid_axes(N)
    psi = A * np.exp(1j * (2 * x + y - 3 * z + 0 * x * y * z))
    pk = lambda f: np.stack([oracle.r2c3d(np.ascontiguousarray(f.real)), oracle.r2c3d(np.ascontiguousarray(f.imag))])
    p = psfft.Plan(N, torch.float64, 1, work="gpe")
    got = p.gpe_rhs(dev(pk(psi)), alpha, beta).cpu().numpy()
    assert rel(got, pk(-1j * (alpha * 14 + beta * A * A) * psi)) < 1e-13


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N,ord", [(16, 1), (32, 2), (48, 3), (64, 4)])
def test_gpe_rk_step_matches_oracle(N, ord, dtype):
    y = gpe_state(N, N // 2 - 1, dtype)
    p = psfft.Plan(N, dtype, 1)
    got = p.rk_step(psfft.SYS_GPE, dev(y), ord, 0.01, 0.37, 1.3).cpu().numpy()
    want = oracle.rk_step(3, y.astype(np.complex128), ord, 0.01, 0.37, 1.3)
    assert rel(got, want) < TOL[dtype]


# ---- broadband (full-sphere) inputs: every retained mode populated, per-shell error bounds ----------------------
# The band-limited config fields (k0 = 4, kcut = 32) leave the outer shells of the 2/3 sphere empty from N = 96 on
# (ADVICE r1): the pruned column ranges, the kx_count / pitch edge and the mirrored loads of mid_x would then only
# ever move zeros there.  synth.broadband_* fills E(k) ~ k^-5/3 up to the Nyquist planes.

def broadband_state(system, N, dtype):
    u = synth.broadband_spectrum(N, seed=77, tag=0)
    if system == psfft.SYS_HD:
        y = u
    elif system == psfft.SYS_MHD:
        y = np.concatenate([u, synth.broadband_spectrum(N, seed=77, tag=1)])
    elif system == psfft.SYS_BOUSSINESQ:
        y = np.concatenate([u, synth.broadband_scalar(N, seed=77)[None]])
    else:
        y = np.stack([synth.broadband_scalar(N, seed=77, tag=11), synth.broadband_scalar(N, seed=77, tag=12)])
        y[0, 0, 0, 0] = float(N) ** 3
    return np.ascontiguousarray(y.astype(CDT[dtype]))


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [128, 192, 256])
@pytest.mark.parametrize("system", [0, 1, 2, 3])
def test_rhs_broadband_per_shell(system, N, dtype):
    y = broadband_state(system, N, dtype)
    yw = y.astype(np.complex128)
    M = oracle.dealias_mask(N)
    assert np.count_nonzero(y[0][M]) > 0.99 * M.sum() and np.count_nonzero(y[0][~M]) > 0.2 * (~M).sum()
    yd = dev(y)
    p = psfft.Plan(N, dtype, 1, work="mhd")
    if system == psfft.SYS_HD:
        got = p.hd_rhs(yd, 0.003).cpu().numpy()
        want = oracle.hd_rhs(yw, 0.003)
    elif system == psfft.SYS_MHD:
        ru, rb = p.mhd_rhs(yd[:3].contiguous(), yd[3:].contiguous(), 0.003, 0.002)
        got = np.concatenate([ru.cpu().numpy(), rb.cpu().numpy()])
        want = np.concatenate(oracle.mhd_rhs(yw[:3], yw[3:], 0.003, 0.002))
    elif system == psfft.SYS_BOUSSINESQ:
        ru, rt = p.boussinesq_rhs(yd[:3].contiguous(), yd[3].contiguous(), 0.003, 0.002, 1.5)
        got = np.concatenate([ru.cpu().numpy(), rt.cpu().numpy()[None]])
        wu, wt = oracle.boussinesq_rhs(yw[:3], yw[3], 0.003, 0.002, 1.5)
        want = np.concatenate([wu, wt[None]])
    else:
        got = p.gpe_rhs(yd, 0.37, 1.3).cpu().numpy()
        want = oracle.gpe_rhs(yw, 0.37, 1.3)
    assert rel(got, want) < TOL[dtype]
    for f in range(0, got.shape[0], 3):              # vector fields (and the scalar) separately, shell by shell
        assert_shells(got[f:f + 3], want[f:f + 3], N, TOL[dtype])
    assert np.all(got[:, ~M] == 0)
    assert np.count_nonzero(got[0][M]) > 0.99 * M.sum()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("system", [0, 1, 2, 3])
def test_rk2_broadband_per_shell(system, dtype):
    N = 128
    y = broadband_state(system, N, dtype)
    p = psfft.Plan(N, dtype, 1)
    par = (0.37, 1.3, 0.0) if system == psfft.SYS_GPE else (0.003, 0.002, 1.5)
    got = p.rk_step(system, dev(y), 2, 0.01, *par).cpu().numpy()
    want = oracle.rk_step(system, y.astype(np.complex128), 2, 0.01, *par)
    assert rel(got, want) < TOL[dtype]
    assert_shells(got, want, N, TOL[dtype])
    assert np.all(got[:, ~oracle.dealias_mask(N)] == 0)


# ---- host-buffer (end-to-end) entry points -----------------------------------------------------------

def test_host_entry_points():
    N = 32
    x = synth.uniform_field(N, 1, 77)
    p = psfft.Plan(N, torch.float64, 1, work="hd")
    hx = torch.from_numpy(x).pin_memory()
    hX = torch.empty((1, N, N, N // 2 + 1), dtype=torch.complex128).pin_memory()
    d_in = torch.empty(p.layout.spec_bytes * 3, dtype=torch.uint8, device="cuda")
    d_out = torch.empty(p.layout.spec_bytes * 3, dtype=torch.uint8, device="cuda")
    psfft.fft3d_r2c_host(p.handle, hx, hX, d_in, d_out, p._work)
    assert rel(hX.numpy()[0], oracle.r2c3d(x[0])) < 1e-12
    hb = torch.empty_like(hx)
    psfft.fft3d_c2r_host(p.handle, hX, hb, d_in, d_out, p._work)
    assert rel(hb.numpy(), x) < 1e-12
    uh = synth.solenoidal_spectrum(N, 4.0, 12, 3)
    hu = torch.from_numpy(uh).pin_memory()
    hr = torch.empty_like(hu)
    psfft.hd_rhs_host(p.handle, hu, hr, 0.0, d_in, d_out, p._work)
    assert rel(hr.numpy(), oracle.hd_rhs(uh, 0.0)) < 1e-12


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(32, 32, 32), (48, 48, 48), (48, 24, 32), (12, 8, 16)])
def test_host_box_entry_point_moves_only_the_retained_box(shape, dtype):
    """psfft_hd_rhs_host_box: the FULL host array equals the oracle's (the array was zeroed once; the call writes the box),
    nothing outside the box is touched, the staging buffers need no initialisation, and the byte count is the box's."""
    Nx, Ny, Nz = shape
    p = psfft.Plan(shape if len(set(shape)) > 1 else Nx, dtype, 1, work="hd")
    uh = synth.aniso_spectrum(shape, seed=11).astype(CDT[dtype])              # broadband: fills the retained ellipsoid
    want = oracle.hd_rhs(uh.astype(np.complex128), 0.05)
    hu = torch.from_numpy(uh).pin_memory()
    d_in = torch.full((3 * p.layout.spec_elems,), complex(float("nan"), float("nan")), dtype=p.cdtype, device="cuda")
    d_out = torch.full_like(d_in, complex(float("nan"), float("nan")))
    hr = torch.zeros_like(hu).pin_memory()
    psfft.hd_rhs_host_box(p.handle, hu, hr, 0.05, d_in, d_out, p._work)
    got = hr.numpy()
    assert rel(got, want) < TOL[dtype]
    # the box: kx < ceil(Nx / 3), |ky| < Ny / 3, |kz| < Nz / 3 (index ranges [0, b] and [N - b, N))
    bx, by, bz = (Nx - 1) // 3 + 1, (Ny - 1) // 3, (Nz - 1) // 3
    inside = np.zeros((Nz, Ny, Nx // 2 + 1), dtype=bool)
    zi = np.r_[0:bz + 1, Nz - bz:Nz]
    yi = np.r_[0:by + 1, Ny - by:Ny]
    inside[np.ix_(zi, yi, np.arange(bx))] = True
    assert psfft.host_box_bytes(p.handle) == int(inside.sum()) * uh.itemsize
    assert np.all(want[:, ~inside] == 0)                                       # the oracle agrees that nothing lives outside
    hr2 = torch.full_like(hu, 7.0).pin_memory()                                 # second call into a marked array
    psfft.hd_rhs_host_box(p.handle, hu, hr2, 0.05, d_in, d_out, p._work)
    got2 = hr2.numpy()
    assert np.all(got2[:, ~inside] == 7.0) and np.array_equal(got2[:, inside], got[:, inside])
    # and it agrees bit for bit with the dense host entry point
    hr3 = torch.empty_like(hu).pin_memory()
    psfft.hd_rhs_host(p.handle, hu, hr3, 0.05, d_in, d_out, p._work)
    assert np.array_equal(hr3.numpy(), got)


# ---- the unfused composition (second CUDA path) ------------------------------------------------------

@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [16, 48, 64])
def test_unfused_rhs_matches_oracle(N, dtype):
    kcut = N // 2 - 1
    uh = synth.solenoidal_spectrum(N, 3.0, kcut, 7, tag=0).astype(CDT[dtype])
    bh = synth.solenoidal_spectrum(N, 3.0, kcut, 7, tag=1).astype(CDT[dtype])
    p = psfft.Plan(N, dtype, 1, work="mhd")
    du, db = dev(uh), dev(bh)
    out = torch.empty_like(du)
    psfft.hd_rhs_unfused(p.handle, du, out, 0.05, p._work)
    assert rel(out.cpu().numpy(), oracle.hd_rhs(uh.astype(np.complex128), 0.05)) < TOL[dtype]
    ru, rb = torch.empty_like(du), torch.empty_like(du)
    psfft.mhd_rhs_unfused(p.handle, du, db, ru, rb, 0.01, 0.02, p._work)
    wu, wb = oracle.mhd_rhs(uh.astype(np.complex128), bh.astype(np.complex128), 0.01, 0.02)
    assert rel(ru.cpu().numpy(), wu) < TOL[dtype] and rel(rb.cpu().numpy(), wb) < TOL[dtype]


# ---- argument checks that need a live plan ---------------------------------------------------------------------

def test_overlapping_buffers_and_dead_handles_are_rejected():
    """psfft.h: "input and output of one call must not overlap; the workspace must overlap neither" -- every
    execute call checks the byte ranges it will touch and returns PSFFT_E_OVERLAP (-8) before enqueuing."""
    N = 32
    p = psfft.Plan(N, torch.float64, 1, work="mhd")
    C = p.layout.spec_bytes
    buf = torch.zeros(16 * C, dtype=torch.uint8, device="cuda")
    work = p.ensure_work("rk_mhd")
    u, b, ru, rb = buf[:3 * C], buf[3 * C:6 * C], buf[6 * C:9 * C], buf[9 * C:12 * C]
    L = psfft.lib()
    st = torch.cuda.current_stream().cuda_stream
    h = p.handle
    ptr = lambda t: ctypes.c_void_p(t.data_ptr())
    assert L.psfft_hd_rhs(h, ptr(u), ptr(u), 0.0, ptr(work), st) == -8                      # in place
    assert L.psfft_hd_rhs(h, ptr(u), ptr(buf[C:4 * C]), 0.0, ptr(work), st) == -8           # partial overlap
    assert L.psfft_hd_rhs(h, ptr(u), ptr(ru), 0.0, ptr(buf[8 * C:]), st) == -8              # workspace over the output
    assert L.psfft_hd_rhs(h, ptr(u), ptr(ru), 0.0, ptr(u), st) == -8                        # workspace over the input
    assert L.psfft_mhd_rhs(h, ptr(u), ptr(b), ptr(ru), ptr(ru), 0.0, 0.0, ptr(work), st) == -8
    assert L.psfft_mhd_rhs(h, ptr(u), ptr(u), ptr(ru), ptr(rb), 0.0, 0.0, ptr(work), st) == 0   # inputs may alias
    assert psfft.last_launch_count(h) == 5
    assert L.psfft_boussinesq_rhs(h, ptr(u), ptr(b), ptr(ru), ptr(buf[8 * C:9 * C]), 0.0, 0.0, 0.0, ptr(work), st) == -8
    assert L.psfft_gpe_rhs(h, ptr(u), ptr(buf[C:3 * C]), 0.1, 1.0, ptr(work), st) == -8
    par = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    assert L.psfft_rk_step(h, 0, ptr(u), ptr(u), 2, 0.01, par, ptr(work), st) == -8
    assert L.psfft_rk_step(h, 0, ptr(u), ptr(buf[2 * C:5 * C]), 2, 0.01, par, ptr(work), st) == -8
    assert L.psfft_rk_step(h, 0, ptr(u), ptr(ru), 2, 0.01, par, ptr(ru), st) == -8
    assert L.psfft_fft3d_c2r(h, ptr(u), ptr(u), ptr(work), st) == -8
    assert L.psfft_fft3d_r2c(h, ptr(u), ptr(u), None, st) == -8
    torch.cuda.synchronize()
    assert psfft.last_launch_count(h) == 5               # still the accepted MHD call: the rejected ones enqueued nothing
    # a destroyed plan is gone from the registry: every later use of the handle is PSFFT_E_PLAN
    p.close()
    assert L.psfft_hd_rhs(h, ptr(u), ptr(ru), 0.0, ptr(work), st) == -6
    assert L.psfft_plan_destroy(h) == -6


# ---- guard bands: no call writes outside the buffers it was given ------------------------------------------

class Arena:
    """One device allocation carved into 256-byte aligned blocks separated by guard bands of a known pattern."""
    GUARD = 4096

    def __init__(self, nbytes):
        self.buf = torch.full((nbytes,), 0xA5, dtype=torch.uint8, device="cuda")
        self.off = self.GUARD
        self.blocks = []

    def take(self, nbytes):
        start = (self.off + 255) // 256 * 256
        self.off = start + nbytes + self.GUARD
        assert self.off <= self.buf.numel()
        self.blocks.append((start, nbytes))
        return self.buf[start:start + nbytes]

    def guards_intact(self):
        mask = torch.ones(self.buf.numel(), dtype=torch.bool, device="cuda")
        for start, n in self.blocks:
            mask[start:start + n] = False
        return bool((self.buf[mask] == 0xA5).all())


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("N", [12, 32, 48, 64])
def test_no_call_writes_outside_its_buffers(N, dtype):
    code = psfft.F64 if dtype == torch.float64 else psfft.F32
    lay = psfft.plan_query(N, code, 2)
    C = lay.spec_bytes
    work_bytes = max(lay.work_bytes_fft, 6 * C + lay.work_bytes_mhd, 4 * C + lay.work_bytes_boussinesq,
                     2 * C + lay.work_bytes_gpe)
    ar = Arena(lay.table_bytes + 2 * lay.real_bytes * 2 + 14 * C + work_bytes + 64 * Arena.GUARD)
    tables = ar.take(lay.table_bytes)
    h = psfft.plan_create(N, code, 2, tables, lay.table_bytes)
    real, real2 = ar.take(2 * lay.real_bytes), ar.take(2 * lay.real_bytes)
    yin, yout, work = ar.take(6 * C), ar.take(6 * C), ar.take(work_bytes)
    real.view(dtype).uniform_(-1, 1)
    kc = N // 2 - 1
    y = np.concatenate([synth.solenoidal_spectrum(N, 2.0, kc, 3, tag=0), synth.solenoidal_spectrum(N, 2.0, kc, 3, tag=1)])
    yin.view(torch.complex128 if dtype == torch.float64 else torch.complex64).copy_(
        torch.from_numpy(y.astype(CDT[dtype])).reshape(-1))
    u, b = yin[:3 * C], yin[3 * C:]
    try:
        psfft.fft3d_r2c(h, real, yout[:2 * C], work)
        psfft.fft3d_c2r(h, yout[:2 * C], real2, work)
        psfft.hd_rhs(h, u, yout[:3 * C], 0.1, work)
        psfft.mhd_rhs(h, u, b, yout[:3 * C], yout[3 * C:], 0.1, 0.1, work)
        psfft.boussinesq_rhs(h, u, b[:C], yout[:3 * C], yout[3 * C:4 * C], 0.1, 0.1, 1.0, work)
        psfft.gpe_rhs(h, u[:2 * C], yout[:2 * C], 0.1, 1.0, work)
        for system, nf in ((0, 3), (1, 6), (2, 4), (3, 2)):
            psfft.rk_step(h, system, yin[:nf * C], yout[:nf * C], 3, 0.01, (0.1, 0.1, 1.0), work)
        torch.cuda.synchronize()
        assert ar.guards_intact()
        assert np.array_equal(yin.view(torch.complex128 if dtype == torch.float64 else torch.complex64).cpu().numpy(),
                              y.astype(CDT[dtype]).reshape(-1))                      # inputs untouched by every call
    finally:
        psfft.plan_destroy(h)
