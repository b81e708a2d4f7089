"""GPU parity of the right-hand sides on anisotropic grids (Nx, Ny, Nz) and boxes (Lx, Ly, Lz) against the oracle
(readings G24, G25).  Run with -m gpu on the B200 box.

Inputs: synth.aniso_spectrum -- broadband, filled up to the Nyquist planes (so the input mask has to act and the
outermost retained shell of the ellipsoid carries data), solenoidal in the box's own wavenumbers.
Tolerances as everywhere: relative L2 <= 1e-12 (fp64), <= 2e-5 (fp32); the ellipsoidal mask bit-exact.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_1808_01309_b200 import psfft, synth  # noqa: E402

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-12, torch.float32: 2e-5}
CDT = {torch.float64: np.complex128, torch.float32: np.complex64}
TWO_PI = 2.0 * np.pi
# (Nx, Ny, Nz), (Lx, Ly, Lz): every axis in every role, radix-3 sizes, the paper's 4:4:1 flat box, tiles of different
# widths for the y and z passes (small N widen the tile), a stretched box on a cubic grid
CASES = [((16, 12, 24), (TWO_PI, 3.0, 9.5)),
         ((32, 64, 16), (TWO_PI, TWO_PI, TWO_PI)),
         ((64, 32, 128), (1.0, 2.0, 3.0)),
         ((128, 128, 32), (TWO_PI, TWO_PI, TWO_PI / 4)),
         ((48, 96, 24), (4.0, TWO_PI, 2.5)),
         ((24, 8, 64), (TWO_PI, 1.5, 7.0)),
         ((32, 32, 32), (5.0, 3.0, 11.0))]


def rel(a, b):
    a = np.asarray(a).astype(np.complex128)
    b = np.asarray(b).astype(np.complex128)
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_mask(got, shape):
    M = oracle.dealias_mask(*shape)
    out = got[..., ~M]
    assert np.all(out == 0) and not np.any(np.signbit(out.real)) and not np.any(np.signbit(out.imag))


@pytest.fixture(autouse=True)
def _sync():
    yield
    torch.cuda.synchronize()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape,box", CASES)
def test_hd_rhs_anisotropic(shape, box, dtype):
    uh = synth.aniso_spectrum(shape, box, seed=21).astype(CDT[dtype])
    p = psfft.Plan(shape, dtype, 1, work="hd", box=box)
    d = dev(uh)
    got = p.hd_rhs(d, 0.07).cpu().numpy()
    assert np.array_equal(d.cpu().numpy(), uh)
    want = oracle.hd_rhs(uh.astype(np.complex128), 0.07, box=box)
    assert rel(got, want) < TOL[dtype]
    check_mask(got, shape)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape,box", CASES[:5])
def test_boussinesq_rhs_anisotropic(shape, box, dtype):
    """The paper's reference equations on its flat-box geometry (1024 x 1024 x 256), all terms on."""
    uh = synth.aniso_spectrum(shape, box, seed=22).astype(CDT[dtype])
    th = synth.aniso_spectrum(shape, box, seed=22, tag=7, ncomp=1).astype(CDT[dtype])
    p = psfft.Plan(shape, dtype, 1, work="boussinesq", box=box)
    ru, rt = p.boussinesq_rhs(dev(uh), dev(th), 0.013, 0.021, 2.5)
    wu, wt = oracle.boussinesq_rhs(uh.astype(np.complex128), th.astype(np.complex128), 0.013, 0.021, 2.5, box=box)
    assert rel(ru.cpu().numpy(), wu) < TOL[dtype] and rel(rt.cpu().numpy(), wt) < TOL[dtype]
    check_mask(ru.cpu().numpy(), shape)
    check_mask(rt.cpu().numpy(), shape)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape,box", CASES[:4])
def test_mhd_rhs_anisotropic(shape, box, dtype):
    uh = synth.aniso_spectrum(shape, box, seed=23, tag=0).astype(CDT[dtype])
    bh = synth.aniso_spectrum(shape, box, seed=23, tag=1).astype(CDT[dtype])
    p = psfft.Plan(shape, dtype, 1, work="mhd", box=box)
    ru, rb = p.mhd_rhs(dev(uh), dev(bh), 0.01, 0.02)
    wu, wb = oracle.mhd_rhs(uh.astype(np.complex128), bh.astype(np.complex128), 0.01, 0.02, box=box)
    assert rel(ru.cpu().numpy(), wu) < TOL[dtype] and rel(rb.cpu().numpy(), wb) < TOL[dtype]
    check_mask(ru.cpu().numpy(), shape)
    check_mask(rb.cpu().numpy(), shape)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape,box", CASES[:4])
def test_gpe_rhs_anisotropic(shape, box, dtype):
    psi = np.stack([synth.aniso_spectrum(shape, box, seed=24, tag=t, ncomp=1) for t in (3, 4)]).astype(CDT[dtype])
    p = psfft.Plan(shape, dtype, 1, work="gpe", box=box)
    got = p.gpe_rhs(dev(psi), 0.3, 1.1).cpu().numpy()
    want = oracle.gpe_rhs(psi.astype(np.complex128), 0.3, 1.1, box=box)
    assert rel(got, want) < TOL[dtype]
    check_mask(got, shape)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("system,ord", [(0, 2), (2, 2), (2, 4), (1, 3), (3, 2)])
def test_rk_step_anisotropic(system, ord, dtype):
    shape, box = CASES[3]
    u = synth.aniso_spectrum(shape, box, seed=25, tag=0)
    if system == psfft.SYS_HD:
        y = u
    elif system == psfft.SYS_MHD:
        y = np.concatenate([u, synth.aniso_spectrum(shape, box, seed=25, tag=1)])
    elif system == psfft.SYS_BOUSSINESQ:
        y = np.concatenate([u, synth.aniso_spectrum(shape, box, seed=25, tag=7, ncomp=1)[None]])
    else:
        y = np.stack([synth.aniso_spectrum(shape, box, seed=25, tag=t, ncomp=1) for t in (3, 4)])
    y = np.ascontiguousarray(y.astype(CDT[dtype]))
    p = psfft.Plan(shape, dtype, 1, work="fft", box=box)
    dt, nu, c2, nbv = 2e-3, 0.05, 0.03, 1.5
    if system == psfft.SYS_GPE:
        nu, c2, nbv = 0.3, 1.1, 0.0
    got = p.rk_step(system, dev(y), ord, dt, nu, c2, nbv).cpu().numpy()
    want = oracle.rk_step(system, y.astype(np.complex128), ord, dt, nu, c2, nbv, box=box)
    assert rel(got, want) < TOL[dtype]
    check_mask(got, shape)


def test_stretched_taylor_green_closed_form_on_the_gpu():
    """The closed form of tests/test_oracle_aniso.py::stretched_taylor_green directly against the CUDA path: twelve
    modes with three different wavenumbers 2 pi / L_i."""
    shape, box, A = (32, 16, 64), (TWO_PI, 3.0, 9.5), 1.3
    x, y, z = synth.box_axes(shape, box)
    a, b, c = TWO_PI / box[0], TWO_PI / box[1], TWO_PI / box[2]
    B = -a * A / b
    one = np.ones(shape[::-1])
    u = np.stack([A * np.sin(a * x) * np.cos(b * y) * np.cos(c * z) * one,
                  B * np.cos(a * x) * np.sin(b * y) * np.cos(c * z) * one, 0 * one])
    want = np.stack([-A * A * a * c * c / (4 * (a * a + c * c)) * np.sin(2 * a * x) * np.cos(2 * c * z) * one,
                     -B * B * b * c * c / (4 * (b * b + c * c)) * np.sin(2 * b * y) * np.cos(2 * c * z) * one,
                     (c / 4) * (A * A * a * a / (a * a + c * c) * np.cos(2 * a * x)
                                + B * B * b * b / (b * b + c * c) * np.cos(2 * b * y)) * np.sin(2 * c * z) * one])
    p = psfft.Plan(shape, torch.float64, 3, work="hd", box=box)
    uh = p.r2c(dev(u))
    got = p.c2r(p.hd_rhs(uh)).cpu().numpy()
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-13


def test_box_on_a_cubic_plan_and_bad_boxes():
    """set_box on a cubic plan: the dilation law rhs(s) = rhs(1)/s for nu = 0; non-positive lengths are refused."""
    N, s = 32, 2.5
    uh = synth.broadband_spectrum(N, seed=3)
    p = psfft.Plan(N, torch.float64, 1, work="hd")
    r1 = p.hd_rhs(dev(uh)).cpu().numpy()
    psfft.plan_set_box(p.handle, s * TWO_PI, s * TWO_PI, s * TWO_PI)
    rs = p.hd_rhs(dev(uh)).cpu().numpy()
    assert rel(rs, r1 / s) < 1e-13
    assert rel(rs, oracle.hd_rhs(uh, 0.0, box=(s * TWO_PI,) * 3)) < 1e-12
    for bad in [(0.0, 1.0, 1.0), (1.0, -2.0, 1.0), (1.0, 1.0, float("inf")), (float("nan"), 1.0, 1.0)]:
        with pytest.raises(psfft.PsfftError):
            psfft.plan_set_box(p.handle, *bad)


def test_anisotropic_rk_step_is_graph_capturable_and_replays_bit_for_bit():
    """A Boussinesq RK2 step on the flat-box aspect ratio captured as one CUDA graph (the execute calls only enqueue)."""
    shape, box = (128, 128, 32), (TWO_PI, TWO_PI, TWO_PI / 4)
    y = np.concatenate([synth.aniso_spectrum(shape, box, seed=5), synth.aniso_spectrum(shape, box, seed=5, tag=7, ncomp=1)[None]])
    p = psfft.Plan(shape, torch.float64, 1, work="rk_boussinesq", box=box)
    yd = dev(y)
    out = torch.empty_like(yd)
    work = p.ensure_work("rk_boussinesq")
    eager = p.rk_step(psfft.SYS_BOUSSINESQ, yd, 2, 1e-3, 0.01, 0.02, 1.5).clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        psfft.rk_step(p.handle, psfft.SYS_BOUSSINESQ, yd, out, 2, 1e-3, (0.01, 0.02, 1.5), work, stream=s)   # warm-up
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            psfft.rk_step(p.handle, psfft.SYS_BOUSSINESQ, yd, out, 2, 1e-3, (0.01, 0.02, 1.5), work, stream=s)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager)


# ---- N = 2048 (the paper's largest grid is 2048 x 2048 x 512) on every axis ------------------------------

@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(2048, 16, 8), (16, 2048, 8), (8, 16, 2048)])
def test_length_2048_transforms_and_rhs_on_each_axis(shape, dtype):
    """The 8 8 8 4 column schedule / 8 8 4 8 row schedule of length 2048 in the x-, y- and z-pass: plain transforms
    and the Boussinesq right-hand side against the oracle."""
    Nx, Ny, Nz = shape
    box = (TWO_PI, 3.0, 5.0)
    x = synth.uniform01(3, np.arange(Nz * Ny * Nx, dtype=np.uint64)).reshape(1, Nz, Ny, Nx) * 2 - 1
    x = x.astype(np.float64 if dtype == torch.float64 else np.float32)
    p = psfft.Plan(shape, dtype, 1, work="boussinesq", box=box)
    X = p.r2c(dev(x))
    assert rel(X.cpu().numpy()[0], oracle.r2c3d(x[0].astype(np.float64))) < TOL[dtype]
    assert rel(p.c2r(X).cpu().numpy(), x) < TOL[dtype]
    uh = synth.aniso_spectrum(shape, box, seed=31).astype(CDT[dtype])
    th = synth.aniso_spectrum(shape, box, seed=31, tag=7, ncomp=1).astype(CDT[dtype])
    ru, rt = p.boussinesq_rhs(dev(uh), dev(th), 0.01, 0.02, 1.5)
    wu, wt = oracle.boussinesq_rhs(uh.astype(np.complex128), th.astype(np.complex128), 0.01, 0.02, 1.5, box=box)
    assert rel(ru.cpu().numpy(), wu) < TOL[dtype] and rel(rt.cpu().numpy(), wt) < TOL[dtype]
    check_mask(ru.cpu().numpy(), shape)
