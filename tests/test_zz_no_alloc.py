"""psfft_fft3d_c2r_static -- the inverse transform for callers that cannot allocate device memory.

Who that is: code that was handed a fixed set of device buffers and may not ask the driver for more -- a solver
plugged into an application whose own arena already holds all of HBM (a cudaMalloc there simply fails), a time
loop that must never stall on the device-wide synchronisation cudaMalloc / cudaFree imply, a plug-in living in a
process whose allocator it does not own.  Such a caller has nowhere to take the workspace of psfft_fft3d_c2r
from, so this entry point brings its own: a 32 MiB `static __device__` array inside libpsfft.so (include/psfft.h).

What is checked here, always against the existing path (Plan.c2r = psfft_fft3d_c2r with a torch-allocated
workspace), which the rest of the suite checks against the oracle:
  * two calls in a row on the same plan, different inputs: each result equals the existing path's bit for bit (same
    kernels, same order -- so the comparison is `torch.equal`, tighter than the 1e-12 / 2e-5 of the parity tests);
  * a third call on a smaller plan of the other dtype right after a larger one: what the larger call left in the
    shared array does not leak into the result (nothing is, or needs to be, cleared);
  * the second call takes no device memory (free memory reported by the driver does not drop) and the input
    spectrum is left untouched;
  * a plan whose workspace exceeds the limit is refused with PSFFT_E_SCRATCH (-9), a readable message, and an
    untouched output buffer.

This file sorts last on purpose (`pytest --collect-only`): `pytest -x` stops at the first failure, and a failure of
this add-on must not hide the parity tests.  It passes alone in a fresh process (the first call then does the
per-device symbol lookup) and after the rest of the suite.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1808_01309_b200 import psfft  # noqa: E402

pytestmark = pytest.mark.gpu

CDT = {torch.float64: np.complex128, torch.float32: np.complex64}


def spectrum(plan, seed):
    """Any half spectrum is a valid input of the inverse transform (non-Hermitian ones included)."""
    rng = np.random.default_rng(seed)
    shape = plan.spec_shape(plan.batch)
    z = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    return torch.from_numpy(z.astype(CDT[plan.rdtype])).cuda()


def test_static_scratch_c2r_equals_the_workspace_path_on_consecutive_calls():
    # 96 = 2^5 * 3: several tiles and a ragged tail (ldk = 49) in every pass; 2 fields = 14.5 MB of the 32 MiB
    p = psfft.Plan(96, torch.float64, batch=2)
    assert p.layout.work_bytes_fft <= psfft.STATIC_SCRATCH_BYTES
    s1, s2 = spectrum(p, 1), spectrum(p, 2)
    keep1, keep2 = s1.clone(), s2.clone()
    want1, want2 = p.c2r(s1), p.c2r(s2)                    # existing path, workspace from torch
    out1 = torch.full_like(want1, float("nan"))
    out2 = torch.full_like(want2, float("nan"))
    torch.cuda.synchronize()

    p.c2r_static(s1, out1)                                 # first call: per-device set-up happens in here
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    p.c2r_static(s2, out2)                                 # second call, straight after, other input
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]

    assert psfft.last_launch_count(p.handle) == 3          # z-pass, y-pass, c2r x-pass: our kernels ran
    assert torch.equal(out1, want1) and torch.equal(out2, want2)
    assert not torch.equal(out1, out2)                     # the two calls really computed different things
    assert torch.equal(s1, keep1) and torch.equal(s2, keep2)          # inputs are never modified
    assert free_after >= free_before, "the call took device memory"

    # a smaller plan of the other dtype right after: the array still holds the fp64 data of the call above
    q = psfft.Plan(48, torch.float32, batch=3)
    s3 = spectrum(q, 3)
    want3 = q.c2r(s3)
    out3 = torch.full_like(want3, float("nan"))
    q.c2r_static(s3, out3)
    torch.cuda.synchronize()
    assert torch.equal(out3, want3)
    # and back to the first plan once more
    out1.fill_(float("nan"))
    p.c2r_static(s1, out1)
    torch.cuda.synchronize()
    assert torch.equal(out1, want1)


def test_static_scratch_rejects_plans_beyond_its_limit():
    p = psfft.Plan(256, torch.float64, batch=1)            # 129 * 256 * 256 * 16 B = 135 MB > 32 MiB
    assert p.layout.work_bytes_fft > psfft.STATIC_SCRATCH_BYTES
    s = torch.zeros(p.spec_shape(1), dtype=torch.complex128, device="cuda")
    out = torch.full((1, 256, 256, 256), 7.0, dtype=torch.float64, device="cuda")
    rc = psfft.lib().psfft_fft3d_c2r_static(p.handle, s.data_ptr(), out.data_ptr(), None)
    assert rc == psfft.E_SCRATCH
    assert "32 MiB" in psfft.strerror(rc) and "psfft_fft3d_c2r" in psfft.strerror(rc)
    with pytest.raises(psfft.PsfftError, match="built-in workspace"):
        p.c2r_static(s, out)
    torch.cuda.synchronize()
    assert psfft.last_launch_count(p.handle) == 0          # nothing was enqueued
    assert bool((out == 7.0).all())
    # the other argument checks of psfft_fft3d_c2r still come first
    assert psfft.lib().psfft_fft3d_c2r_static(None, s.data_ptr(), out.data_ptr(), None) == -6
    assert psfft.lib().psfft_fft3d_c2r_static(p.handle, None, out.data_ptr(), None) == -1
    assert psfft.lib().psfft_fft3d_c2r_static(p.handle, s.data_ptr() + 8, out.data_ptr(), None) == -4
