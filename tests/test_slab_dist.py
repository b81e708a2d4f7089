"""The exchange schedule of the slab-decomposed transform with world_size-2 gloo on CPU tensors.

The product's kernels need a GPU; what runs here is the product's COMMUNICATION code (slab.exchange_forward /
exchange_inverse with slab.forward_splits) around local passes done with numpy in this test only -- laid out exactly
as psfft_slab_r2c_xy / psfft_slab_z / psfft_slab_c2r_yx lay them out (include/psfft.h) -- and checked against numpy's
rfftn of the global field.  A wrong split size, slice order or block layout breaks it.
"""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_1808_01309_b200 import slab  # noqa: E402


def test_ranges_and_splits():
    assert slab.x_ranges(257, 8) == [0, 32, 64, 96, 128, 160, 192, 224, 257]
    assert slab.x_ranges(17, 2) == [0, 8, 17]
    for ldk, P in [(257, 8), (513, 16), (17, 3), (9, 9)]:
        x0 = slab.x_ranges(ldk, P)
        w = np.diff(x0)
        assert x0[0] == 0 and x0[-1] == ldk and w.min() >= 1 and w.max() - w.min() <= 1
    send, recv = slab.forward_splits(64, 32, 17, 2, 1)
    assert send == [32 * 32 * 8, 32 * 32 * 9] and recv == [32 * 32 * 9] * 2
    # every element is sent exactly once and received exactly once
    P, Nz, Ny, ldk = 4, 16, 12, 13
    tot_send = sum(sum(slab.forward_splits(Nz, Ny, ldk, P, r)[0]) for r in range(P))
    tot_recv = sum(sum(slab.forward_splits(Nz, Ny, ldk, P, r)[1]) for r in range(P))
    assert tot_send == tot_recv == Nz * Ny * ldk


def _worker(rank, world, port, shape, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        Nx, Ny, Nz = shape
        ldk, Mz = Nx // 2 + 1, Nz // world
        x0 = slab.x_ranges(ldk, world)
        w = x0[rank + 1] - x0[rank]
        rng = np.random.default_rng(7)
        full = rng.standard_normal((Nz, Ny, Nx))                       # every rank draws the same global field
        mine = full[rank * Mz:(rank + 1) * Mz]
        # phase 1 as psfft_slab_r2c_xy lays it out (packed mode): x, y passes, slices [q][Mz][Ny][w_q]
        zs = np.fft.fft(np.fft.rfft(mine, axis=2), axis=1)
        send = np.concatenate([zs[:, :, x0[q]:x0[q + 1]].ravel() for q in range(world)])
        sendbuf = torch.from_numpy(send)
        xslab = torch.empty(Nz * Ny * w, dtype=torch.complex128)
        slab.exchange_forward(sendbuf, xslab, Nz, Ny, ldk)
        X = np.fft.fft(xslab.numpy().reshape(Nz, Ny, w), axis=0)         # phase 2: z-pass of the x-slab
        want = np.fft.rfftn(full)[:, :, x0[rank]:x0[rank + 1]]
        err_f = np.abs(X - want).max() / np.abs(want).max()
        # inverse: z-pass, exchange of contiguous z-ranges, gather-load y-pass, c2r x-pass
        Y = np.ascontiguousarray(np.fft.ifft(X, axis=0) * Nz)               # unnormalised, as psfft_slab_z(+1)
        recvbuf = torch.empty(Mz * Ny * ldk, dtype=torch.complex128)
        slab.exchange_inverse(torch.from_numpy(Y.ravel()), recvbuf, Nz, Ny, ldk)
        send_counts, _ = slab.forward_splits(Nz, Ny, ldk, world, rank)
        zs2 = np.empty((Mz, Ny, ldk), dtype=np.complex128)
        off = 0
        for q in range(world):
            zs2[:, :, x0[q]:x0[q + 1]] = recvbuf.numpy()[off:off + send_counts[q]].reshape(Mz, Ny, x0[q + 1] - x0[q])
            off += send_counts[q]
        back = np.fft.irfft(np.fft.ifft(zs2, axis=1), n=Nx, axis=2) / Nz
        err_b = np.abs(back - mine).max()
        out[rank] = (float(err_f), float(err_b))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("shape", [(16, 12, 8), (32, 8, 16)])
def test_exchange_schedule_world_size_2_gloo(shape):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, shape, out), nprocs=world, join=True)
        assert len(out) == world
        for r in range(world):
            assert out[r][0] < 1e-13 and out[r][1] < 1e-13, out[r]
