"""Helpers shared by the parity tests (comparison arithmetic only: no transform, no right-hand side)."""
import numpy as np


def rel(a, b):
    """Relative L2 error of a against b, accumulated in fp64."""
    a = np.asarray(a)
    b = np.asarray(b)
    wide = np.complex128 if (np.iscomplexobj(a) or np.iscomplexobj(b)) else np.float64
    num = 0.0
    den = 0.0
    a = a.reshape(a.shape[0], -1) if a.ndim > 1 else a.reshape(1, -1)
    b = b.reshape(a.shape)
    for x, y in zip(a, b):                       # slab by slab: no full-size fp64 temporaries at 1024^3
        y = y.astype(wide)
        d = x.astype(wide) - y
        num += float(np.vdot(d, d).real)
        den += float(np.vdot(y, y).real)
    return np.sqrt(num / max(den, 1e-300))


def shell_index(N, width):
    """Integer shell number floor(|k| / width) of every half-spectrum mode [kz][ky][kx] (uint8/16 array)."""
    k = np.fft.fftfreq(N, 1.0 / N)
    kx = np.arange(N // 2 + 1, dtype=np.float64)
    k2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + kx[None, None, :] ** 2
    return (np.sqrt(k2) / width).astype(np.int32)


def shell_rel_errors(got, want, N, width=None, mask=None):
    """Per-shell relative L2 error of a spectral result [fields][kz][ky][kx]: shells of width `width` in |k|
    (default N/24, i.e. eight shells inside the 2/3 sphere), optionally restricted to `mask`.  A defect confined
    to the outermost retained shell cannot hide behind the energy of the low shells, as it could in one global
    norm.  Returns (shell numbers with non-zero reference, their relative errors)."""
    if width is None:
        width = N / 24.0
    sh = shell_index(N, width)
    nb = int(sh.max()) + 1
    num = np.zeros(nb)
    den = np.zeros(nb)
    for g, w in zip(got, want):
        w = w.astype(np.complex128)
        d = np.abs(g.astype(np.complex128) - w) ** 2
        r = np.abs(w) ** 2
        if mask is not None:
            d = d * mask
            r = r * mask
        num += np.bincount(sh.ravel(), weights=d.ravel(), minlength=nb)
        den += np.bincount(sh.ravel(), weights=r.ravel(), minlength=nb)
    live = den > 0
    return np.nonzero(live)[0], np.sqrt(num[live] / den[live])


def assert_shells(got, want, N, tol, min_shells=8):
    """Every populated shell of the reference within tol, and the populated shells reach the sphere's edge."""
    shells, err = shell_rel_errors(got, want, N)
    assert len(shells) >= min_shells, f"reference populates only {len(shells)} shells"
    assert shells.max() >= 7, "reference does not reach the outermost retained shell"
    bad = {int(s): float(e) for s, e in zip(shells, err) if not e < tol}
    assert not bad, f"per-shell relative error above {tol}: {bad}"
    return float(err.max())


def shell_rel_errors_device(got, want, N, width=None):
    """shell_rel_errors for torch tensors that live on the GPU (the 1024^3 comparisons: 3 x 537 M modes per field
    set would take minutes in numpy).  Accumulates in fp64.  Returns (shells, errors) as numpy arrays."""
    import torch
    if width is None:
        width = N / 24.0
    dev = got.device
    k = torch.fft.fftfreq(N, 1.0 / N, device=dev, dtype=torch.float64)
    kx = torch.arange(N // 2 + 1, device=dev, dtype=torch.float64)
    nb = int(np.sqrt(3.0) * (N // 2) / width) + 2
    num = torch.zeros(nb, dtype=torch.float64, device=dev)
    den = torch.zeros(nb, dtype=torch.float64, device=dev)
    kyx2 = k[:, None] ** 2 + kx[None, :] ** 2
    for f in range(got.shape[0]):
        for z in range(N):                               # plane by plane: small temporaries
            sh = (torch.sqrt(kyx2 + k[z] ** 2) / width).to(torch.int64).reshape(-1)
            w = want[f, z].reshape(-1).to(torch.complex128)
            d = got[f, z].reshape(-1).to(torch.complex128) - w
            num.index_add_(0, sh, d.real ** 2 + d.imag ** 2)
            den.index_add_(0, sh, w.real ** 2 + w.imag ** 2)
    num, den = num.cpu().numpy(), den.cpu().numpy()
    live = den > 0
    return np.nonzero(live)[0], np.sqrt(num[live] / den[live])


def assert_shells_device(got, want, N, tol, min_shells=8):
    shells, err = shell_rel_errors_device(got, want, N)
    assert len(shells) >= min_shells and shells.max() >= 7
    bad = {int(s): float(e) for s, e in zip(shells, err) if not e < tol}
    assert not bad, f"per-shell relative error above {tol}: {bad}"
    return float(err.max())


def ellipsoid_shell_index(shape, nshell=8):
    """Shell number floor(nshell * 3 * sqrt(sum (n_i / N_i)^2)) of every half-spectrum mode of an (Nx, Ny, Nz) grid:
    shells 0 .. nshell-1 tile the 2/3-rule ellipsoid sum (n_i / N_i)^2 < 1/9 (reading G25)."""
    Nx, Ny, Nz = shape
    fy = np.fft.fftfreq(Ny)          # n / N
    fz = np.fft.fftfreq(Nz)
    fx = np.arange(Nx // 2 + 1) / Nx
    rho = np.sqrt(fz[:, None, None] ** 2 + fy[None, :, None] ** 2 + fx[None, None, :] ** 2)
    return (rho * (3 * nshell)).astype(np.int32)


def assert_ellipsoid_shells(got, want, shape, tol, nshell=8):
    """Per-shell relative L2 error on an anisotropic grid: every populated shell within tol and the reference reaches
    the outermost retained shell."""
    sh = ellipsoid_shell_index(shape, nshell)
    nb = int(sh.max()) + 1
    num = np.zeros(nb)
    den = np.zeros(nb)
    for g, w in zip(got, want):
        w = w.astype(np.complex128)
        num += np.bincount(sh.ravel(), weights=(np.abs(g.astype(np.complex128) - w) ** 2).ravel(), minlength=nb)
        den += np.bincount(sh.ravel(), weights=(np.abs(w) ** 2).ravel(), minlength=nb)
    live = den > 0
    shells, err = np.nonzero(live)[0], np.sqrt(num[live] / den[live])
    assert len(shells) >= nshell and shells.max() >= nshell - 1, f"reference populates shells {shells}"
    bad = {int(s): float(e) for s, e in zip(shells, err) if not e < tol}
    assert not bad, f"per-shell relative error above {tol}: {bad}"
    return float(err.max())
