"""Pins for the oracle's transforms (O1-O5) -- CPU only.

Each test pins the oracle to something other than itself: the O(N^6) definition, closed forms,
identities, and numpy's pocketfft as an independent library.
"""
import numpy as np
import pytest

import oracle
from paper_1808_01309_b200 import synth

RNG = np.random.default_rng(7)


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


# ---- O1 / O2: one axis -------------------------------------------------------------------------

def test_dft1d_direct_closed_forms():
    """Delta -> all ones; shifted delta -> pure phase with the forward sign '-' (Eq. 8)."""
    n = 12
    d = np.zeros(n, complex)
    d[0] = 1
    assert np.allclose(oracle.dft1d_direct(d, -1), np.ones(n), atol=1e-15)
    d = np.zeros(n, complex)
    d[1] = 1
    p = np.arange(n)
    assert np.allclose(oracle.dft1d_direct(d, -1), np.exp(-2j * np.pi * p / n), atol=1e-15)
    assert np.allclose(oracle.dft1d_direct(d, +1), np.exp(+2j * np.pi * p / n), atol=1e-15)
    # constant -> n at p = 0 only
    X = oracle.dft1d_direct(np.ones(n), -1)
    assert abs(X[0] - n) < 1e-13 and np.all(np.abs(X[1:]) < 1e-13)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 8, 9, 12, 16, 24, 30, 32, 48, 49, 64, 96, 128, 384, 768])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft1d_equals_definition(n, sign):
    """O2 (recursive mixed radix) equals O1 (the definition) for radix 2, 3, mixed and prime lengths."""
    x = RNG.standard_normal(n) + 1j * RNG.standard_normal(n)
    assert rel(oracle.fft1d(x, sign), oracle.dft1d_direct(x, sign)) < 1e-13


@pytest.mark.parametrize("n", [8, 12, 96, 512, 768, 1024])
def test_fft1d_vs_numpy(n):
    """P6, one axis: numpy.fft.fft uses the same sign convention as Eq. 8 (exp(-2 pi i p j/n))."""
    x = RNG.standard_normal(n) + 1j * RNG.standard_normal(n)
    assert rel(oracle.fft1d(x, -1), np.fft.fft(x)) < 1e-14
    assert rel(oracle.fft1d(x, +1), np.fft.ifft(x) * n) < 1e-14


# ---- O3 / O4 / O5: three axes ------------------------------------------------------------------

@pytest.mark.parametrize("shape", [(8, 8, 8), (16, 16, 16), (4, 6, 8), (6, 4, 10), (3, 5, 4)])
def test_r2c3d_equals_bruteforce(shape):
    """P1: O3 equals the O(N^6) triple sum (O5).  Non-cubic shapes catch swapped axes / strides."""
    x = RNG.uniform(-1, 1, shape)
    full = oracle.dft3d_bruteforce(x)
    H = shape[2] // 2 + 1
    X = oracle.r2c3d(x)
    assert X.shape == (shape[0], shape[1], H)
    assert rel(X, full[:, :, :H]) < 1e-13


def test_bruteforce_itself_single_point():
    """O5 pinned by hand: N = 2 in each direction is a sum/difference table."""
    x = np.arange(8, dtype=float).reshape(2, 2, 2)
    X = oracle.dft3d_bruteforce(x)
    assert np.isclose(X[0, 0, 0], x.sum())
    assert np.isclose(X[0, 0, 1], (x[:, :, 0] - x[:, :, 1]).sum())
    assert np.isclose(X[0, 1, 0], (x[:, 0, :] - x[:, 1, :]).sum())
    assert np.isclose(X[1, 0, 0], (x[0] - x[1]).sum())
    assert np.isclose(X[1, 1, 1], sum(x[k, j, i] * (-1) ** (i + j + k) for k in range(2) for j in range(2) for i in range(2)))


@pytest.mark.parametrize("shape", [(8, 8, 8), (4, 6, 8), (6, 4, 10)])
def test_c2r3d_equals_bruteforce_inverse(shape):
    """P1 for O4: Hermitian-extend the half spectrum and evaluate the inverse triple sum point by point."""
    Nz, Ny, Nx = shape
    x = RNG.uniform(-1, 1, shape)
    full = oracle.dft3d_bruteforce(x)
    H = Nx // 2 + 1
    back = oracle.c2r3d(full[:, :, :H], Nx)
    for (k, j, i) in [(0, 0, 0), (1, 2, 3), (Nz - 1, Ny - 1, Nx - 1), (2, 0, 5)]:
        v = oracle.idft3d_point(full, k, j, i)
        assert abs(v.imag) < 1e-13
        assert abs(back[k, j, i] - v.real) < 1e-13
        assert abs(back[k, j, i] - x[k, j, i]) < 1e-13


def test_c2r3d_row_formula_non_hermitian():
    """O4's definition for ANY half spectrum: x_i = (1/N^3)[Re Y0 + (-1)^i Re Y_{N/2} + 2 sum Re(Y_p e^{+2 pi i p i/N})]
    after complex inverse transforms along z and y."""
    N = 8
    H = N // 2 + 1
    X = RNG.standard_normal((N, N, H)) + 1j * RNG.standard_normal((N, N, H))   # not Hermitian-consistent
    Y = np.fft.ifft(np.fft.ifft(X, axis=0), axis=1) * N * N                      # unnormalised inverse z, y
    i = np.arange(N)
    want = np.empty((N, N, N))
    for k in range(N):
        for j in range(N):
            row = Y[k, j]
            acc = row[0].real + (-1.0) ** i * row[N // 2].real
            for p in range(1, N // 2):
                acc = acc + 2.0 * (row[p] * np.exp(2j * np.pi * p * i / N)).real
            want[k, j] = acc / N**3
    got = oracle.c2r3d(X, N)
    assert rel(got, want) < 1e-14
    assert rel(got, np.fft.irfftn(X, s=(N, N, N), axes=(0, 1, 2))) < 1e-14


def test_single_mode_lands_in_exact_bin():
    """P2: cos(2 pi (3 i + 2 j - k)/N), N = 8 -> one non-zero half-spectrum bin [kz=7][ky=2][kx=3] = N^3/2."""
    N = 8
    X = oracle.r2c3d(synth.single_mode(N, 3, 2, -1))
    want = np.zeros_like(X)
    want[7, 2, 3] = N**3 / 2
    assert np.abs(X - want).max() < 1e-12
    # a mode with kx = 0 gives two conjugate bins in the kx = 0 plane
    X = oracle.r2c3d(synth.single_mode(N, 0, 2, -1))
    want = np.zeros_like(X)
    want[7, 2, 0] = N**3 / 2
    want[1, 6, 0] = N**3 / 2
    assert np.abs(X - want).max() < 1e-12
    # sine phase: sin(2 pi i/N) -> -i N^3/2 at kx = 1 (sign of the exponent)
    t = 2 * np.pi * np.arange(N) / N
    X = oracle.r2c3d(np.broadcast_to(np.sin(t)[None, None, :], (N, N, N)))
    assert abs(X[0, 0, 1] - (-0.5j * N**3)) < 1e-12


@pytest.mark.parametrize("N", [8, 12, 32])
def test_parseval(N):
    """P3: sum x^2 = (1/N^3) sum_half w_p |X|^2, w_p = 1 for p in {0, N/2}, else 2."""
    x = synth.uniform_field(N, seed=3)[0]
    X = oracle.r2c3d(x)
    w = np.full(N // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    lhs = np.sum(x * x)
    rhs = np.sum(w[None, None, :] * np.abs(X) ** 2) / N**3
    assert abs(lhs - rhs) / lhs < 1e-14


@pytest.mark.parametrize("N", [8, 24, 32, 48])
def test_round_trip(N):
    """P4: c2r(r2c(x)) = x (forward unnormalised, inverse x 1/N^3; BASELINE.json config 1)."""
    x = synth.uniform_field(N, seed=1234)[0]
    assert rel(oracle.c2r3d(oracle.r2c3d(x)), x) < 1e-14


@pytest.mark.parametrize("shape", [(8, 8, 8), (12, 12, 12), (32, 32, 32), (48, 48, 48), (96, 96, 96), (6, 10, 12)])
def test_vs_numpy_rfftn(shape):
    """P6: library special case -- numpy.fft.rfftn / irfftn over axes (0,1,2) is the same definition."""
    x = RNG.uniform(-1, 1, shape)
    X = oracle.r2c3d(x)
    assert rel(X, np.fft.rfftn(x, axes=(0, 1, 2))) < 1e-14
    assert rel(oracle.c2r3d(X, shape[2]), np.fft.irfftn(X, s=shape, axes=(0, 1, 2))) < 1e-14


def test_r2c3d_mode_matches_full_transform():
    """The sampled single-mode evaluator is the same triple sum (used for 512^3 parity)."""
    x = RNG.uniform(-1, 1, (12, 12, 12))
    X = np.fft.rfftn(x)
    for (r, q, p) in [(0, 0, 0), (5, 7, 3), (11, 1, 6), (6, 6, 6)]:
        assert abs(oracle.r2c3d_mode(x, r, q, p) - X[r, q, p]) < 1e-11


def test_hermitian_symmetry_of_real_input():
    """G2: real input => X(-k) = conj X(k) (the paper prints this relation with a wrong sign)."""
    N = 8
    x = RNG.uniform(-1, 1, (N, N, N))
    X = oracle.r2c3d(x)
    for (r, q) in [(1, 2), (3, 0), (0, 5)]:
        assert abs(X[(-r) % N, (-q) % N, 0] - np.conj(X[r, q, 0])) < 1e-13
        assert abs(X[(-r) % N, (-q) % N, N // 2] - np.conj(X[r, q, N // 2])) < 1e-13
