"""Seeded input generators: properties the recipe promises -- CPU only."""
import os

import numpy as np

from paper_1808_01309_b200 import synth


def test_golden_values(golden_dir):
    for l in open(os.path.join(golden_dir, "synth_values.txt")):
        t = l.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] in ("uniform64", "uniform32"):
            dt = np.float64 if t[0] == "uniform64" else np.float32
            x = synth.uniform_field(int(t[1]), 1, int(t[2]), dt)[0]
            assert float(x[int(t[3]), int(t[4]), int(t[5])]) == float(t[6])
        elif t[0] == "solenoidal":
            u = synth.solenoidal_spectrum(int(t[1]), float(t[2]), int(t[3]), int(t[4]), int(t[5]))
            v = u[int(t[6]), int(t[7]), int(t[8]), int(t[9])]
            assert v.real == float(t[10]) and v.imag == float(t[11])
        elif t[0] == "broadband":        # (the global energy sum may round differently across numpy builds)
            v = synth.broadband_spectrum(int(t[1]), seed=int(t[2]), tag=int(t[3]))[int(t[4]), int(t[5]), int(t[6]), int(t[7])]
            assert abs(v - complex(float(t[8]), float(t[9]))) <= 1e-13 * abs(v)
        elif t[0] == "broadband_scalar":
            v = synth.broadband_scalar(int(t[1]), seed=int(t[2]), tag=int(t[3]))[int(t[4]), int(t[5]), int(t[6])]
            assert abs(v - complex(float(t[7]), float(t[8]))) <= 1e-13 * abs(v)


def test_uniform_field_range_and_batch_indexing():
    x = synth.uniform_field(16, 3, 99)
    assert x.shape == (3, 16, 16, 16) and x.min() >= -1.0 and x.max() < 1.0
    assert abs(x.mean()) < 0.05 and abs(x.var() - 1.0 / 3.0) < 0.02
    # counter-based: element idx does not depend on the batch size
    assert np.array_equal(synth.uniform_field(16, 1, 99)[0], x[0])
    x32 = synth.uniform_field(16, 1, 99, np.float32)
    assert x32.dtype == np.float32 and x32.min() >= -1.0 and x32.max() < 1.0
    assert np.array_equal(x32.astype(np.float64) * 2**23, np.round(x32.astype(np.float64) * 2**23))  # 24-bit exact


def test_solenoidal_spectrum_properties():
    N = 32
    u = synth.solenoidal_spectrum(N, 4.0, 12, 1234)
    k = np.arange(N)
    k = np.where(k < N // 2, k, k - N)
    kx, ky, kz = np.arange(N // 2 + 1)[None, None, :], k[None, :, None], k[:, None, None]
    w = np.full(N // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    a = u / N**3
    assert abs(0.5 * np.sum(w * np.abs(a) ** 2) - 1.0) < 1e-14            # unit energy (G18)
    assert np.abs(kx * a[0] + ky * a[1] + kz * a[2]).max() < 1e-16          # solenoidal
    assert np.abs(a[:, (-k[:, None]) % N, (-k[None, :]) % N, 0] - np.conj(a[:, k[:, None] % N, k[None, :] % N, 0])).max() == 0  # Hermitian plane
    k2 = kx**2 + ky**2 + kz**2
    assert np.all(a[:, (k2 > 144) | (k2 == 0)] == 0)                        # support 1 <= |k| <= kcut


def test_solenoidal_field_is_grid_independent():
    a = synth.solenoidal_spectrum(24, 2.0, 6, 5) / 24**3
    b = synth.solenoidal_spectrum(40, 2.0, 6, 5) / 40**3
    for kz in range(-6, 7):
        for ky in range(-6, 7):
            x, y = a[:, kz % 24, ky % 24, :7], b[:, kz % 40, ky % 40, :7]
            assert np.abs(x - y).max() <= 1e-15 * max(np.abs(y).max(), 1e-300)
    # different tags give different fields
    c = synth.solenoidal_spectrum(24, 2.0, 6, 5, tag=1) / 24**3
    assert np.abs(a - c).max() > 1e-3


def test_broadband_fields_fill_the_spectrum_below_nyquist():
    """Unit energy, solenoidal, Hermitian kx = 0 plane, E(k) ~ k^-5/3 shell by shell, every mode with
    1 <= |k| <= N/2 - 1 populated (inside AND outside the 2/3 sphere), grid independent up to the normalisation."""
    N = 48
    u = synth.broadband_spectrum(N, seed=3)
    th = synth.broadband_scalar(N, seed=3)
    k = np.arange(N)
    k = np.where(k < N // 2, k, k - N)
    kx, ky, kz = np.arange(N // 2 + 1)[None, None, :], k[None, :, None], k[:, None, None]
    w = np.full(N // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    a = u / N**3
    assert abs(0.5 * np.sum(w * np.abs(a) ** 2) - 1.0) < 1e-13
    assert abs(0.5 * np.sum(w * np.abs(th / N**3) ** 2) - 1.0) < 1e-13
    assert np.abs(kx * a[0] + ky * a[1] + kz * a[2]).max() < 1e-15
    for f in (a[0], a[1], a[2], th):
        assert np.abs(f[(-k[:, None]) % N, (-k[None, :]) % N, 0] - np.conj(f[k[:, None] % N, k[None, :] % N, 0])).max() == 0
    k2 = kx**2 + ky**2 + kz**2 + 0 * a[0].real
    inside = (k2 >= 1) & (k2 <= (N // 2 - 1) ** 2)
    assert np.all(np.abs(th[inside]) > 0) and np.all(th[~inside] == 0)
    assert np.all(np.sum(np.abs(a), axis=0)[inside] > 0) and np.all(a[:, ~inside] == 0)
    shell = np.rint(np.sqrt(k2)).astype(int)
    E = np.bincount(shell.ravel(), weights=(0.5 * w * np.sum(np.abs(a) ** 2, axis=0)).ravel())
    comp = E[4:N // 2 - 1] * np.arange(4, N // 2 - 1) ** (5.0 / 3.0)
    assert comp.max() / comp.min() < 1.35                               # flat compensated spectrum (lattice noise)
    b = synth.broadband_spectrum(64, kcut=N // 2 - 1, seed=3) / 64**3   # same kcut => same normalisation
    assert abs(b[1, 64 - 3, 5, 7] - a[1, N - 3, 5, 7]) < 1e-15 * abs(b[1, 64 - 3, 5, 7])


def test_taylor_green_spectrum_is_the_transform_of_the_field():
    N, m = 16, 3
    x, y, z = synth.grid_axes(N)
    u = np.stack([np.sin(m * x) * np.cos(m * y) * np.cos(m * z), -np.cos(m * x) * np.sin(m * y) * np.cos(m * z),
                  np.zeros((N, N, N))])
    want = np.fft.rfftn(u, axes=(1, 2, 3))
    assert np.abs(synth.taylor_green_spectrum(N, m) - want).max() < 1e-10
    assert np.count_nonzero(synth.taylor_green_spectrum(N, m)) == 8
