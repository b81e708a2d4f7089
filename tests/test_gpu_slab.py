"""Slab-decomposed transform on ONE GPU: P virtual ranks in direct
mode -- each rank's y-pass stores straight into the x-slabs of all ranks -- must reproduce the single-GPU transform
BIT FOR BIT (same kernels, same butterfly order per column), and the oracle within tolerance.  -m gpu."""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_1808_01309_b200 import psfft, slab, synth  # noqa: E402

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

TOL = {torch.float64: 1e-12, torch.float32: 2e-5}
RDT = {torch.float64: np.float64, torch.float32: np.float32}


def field(shape, dtype, seed=31):
    Nx, Ny, Nz = shape
    x = synth.uniform01(seed, np.arange(Nz * Ny * Nx, dtype=np.uint64)).reshape(Nz, Ny, Nx) * 2 - 1
    return x.astype(RDT[dtype])


def rel(a, b):
    a = np.asarray(a).astype(np.complex128)
    b = np.asarray(b).astype(np.complex128)
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape,P", [((32, 32, 32), 2), ((32, 32, 32), 8), ((64, 48, 16), 4), ((128, 128, 128), 8),
                                     ((24, 16, 48), 3), ((64, 8, 16), 16), ((256, 64, 32), 2), ((32, 32, 32), 1), ((16, 2048, 16), 4)])
def test_virtual_ranks_equal_the_single_gpu_transform_bit_for_bit(shape, P, dtype):
    Nx, Ny, Nz = shape
    x = field(shape, dtype)
    plan = psfft.Plan(shape, dtype, 1)
    xd = torch.from_numpy(x).cuda()
    single = plan.r2c(xd[None])[0]
    vs = slab.VirtualSlabs(plan, P)
    got = vs.r2c(xd)
    assert torch.equal(got, single)                              # bit for bit
    assert rel(got.cpu().numpy(), oracle.r2c3d(x.astype(np.float64))) < TOL[dtype]
    # the kx ranges partition [0, ldk) as evenly as possible
    x0 = list(vs.lays[0].x0[:P + 1])
    assert x0[0] == 0 and x0[-1] == Nx // 2 + 1 and max(np.diff(x0)) - min(np.diff(x0)) <= 1
    # inverse through the virtual ranks: bit for bit the single-GPU c2r, and the round trip
    back = vs.c2r(single)
    assert torch.equal(back, plan.c2r(single[None])[0])
    assert rel(back.cpu().numpy(), x) < TOL[dtype]


def test_packed_mode_blocks_and_argument_checks():
    """Packed mode on one rank-0-of-2 call: the send buffer holds the slices [q][Mz][Ny][w_q] of the y-transformed
    slab; bad (P, rank) are refused."""
    shape, P = (32, 16, 8), 2
    Nx, Ny, Nz = shape
    plan = psfft.Plan(shape, torch.float64, 1)
    lay = psfft.slab_query(plan.handle, P, 0)
    assert (lay.Mz, lay.z0, lay.w) == (4, 0, 8) and list(lay.x0[:3]) == [0, 8, 17]
    x = field(shape, torch.float64)
    xd = torch.from_numpy(x).cuda()
    send = torch.zeros(lay.zspec_elems, dtype=torch.complex128, device="cuda")
    zs = torch.empty_like(send)
    counts, _ = slab.forward_splits(Nz, Ny, Nx // 2 + 1, P, 0)
    psfft.slab_r2c_xy(plan.handle, P, 0, xd[:4], zs, slab._slice_ptrs(send, counts), 0)
    want = np.fft.fft(np.fft.rfft(x[:4].astype(np.float64), axis=2), axis=1)       # x then y of the slab (check only)
    s = send.cpu().numpy()
    b0 = s[:counts[0]].reshape(4, Ny, 8)
    b1 = s[counts[0]:].reshape(4, Ny, 9)
    assert rel(b0, want[:, :, :8]) < 1e-13 and rel(b1, want[:, :, 8:]) < 1e-13
    for bad in [(3, 0), (2, 2), (0, 0), (17, 0)]:
        with pytest.raises(psfft.PsfftError):
            psfft.slab_query(plan.handle, *bad)


def test_slab_argument_checks_and_guard_bands():
    """Bad pointers are refused before anything is enqueued; a phase-1 call writes its work buffer and the blocks it was
    given and nothing around them (buffers carved from one arena with NaN guard bands)."""
    import ctypes
    shape, P = (32, 16, 16), 4
    Nx, Ny, Nz = shape
    plan = psfft.Plan(shape, torch.float64, 1)
    lay = psfft.slab_query(plan.handle, P, 1)
    L = psfft.lib()
    real = torch.rand((lay.Mz, Ny, Nx), dtype=torch.float64, device="cuda")
    zs = torch.empty(lay.zspec_elems, dtype=torch.complex128, device="cuda")
    blocks = [torch.empty(psfft.slab_query(plan.handle, P, q).xslab_elems, dtype=torch.complex128, device="cuda") for q in range(P)]
    st = torch.cuda.current_stream().cuda_stream
    arr = (ctypes.c_void_p * P)(*[b.data_ptr() for b in blocks])
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), None, 0, st) == -1          # NULL
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr() + 8, zs.data_ptr(), arr, 0, st) == -4       # alignment
    bad = (ctypes.c_void_p * P)(blocks[0].data_ptr(), None, blocks[2].data_ptr(), blocks[3].data_ptr())
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), bad, 0, st) == -1
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), arr, -1, st) == -2          # zoff < 0
    # planes past the end of a block (here zoff + Mz = 13 + 4 > Nz = 16) would be stores into a peer's memory: refused
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), arr, Nz - lay.Mz + 1, st) == -2
    assert L.psfft_slab_c2r_yx(plan.handle, P, 1, arr, Nz - lay.Mz + 1, zs.data_ptr(), real.data_ptr(), st) == -2
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), arr, Nz - lay.Mz, st) == 0  # last planes: fine
    assert L.psfft_slab_z(plan.handle, P, 1, 0, blocks[1].data_ptr(), st) == -2                               # dir
    # the blocks are part of the overlap check: a block on the work buffer, on the input, or two blocks on one another
    for alias in (zs.data_ptr(), real.data_ptr(), blocks[0].data_ptr()):
        arr2 = (ctypes.c_void_p * P)(blocks[0].data_ptr(), blocks[1].data_ptr(), alias, blocks[3].data_ptr())
        assert L.psfft_slab_r2c_xy(plan.handle, P, 1, real.data_ptr(), zs.data_ptr(), arr2, 0, st) == -8
    arr2 = (ctypes.c_void_p * P)(blocks[0].data_ptr(), blocks[1].data_ptr(), zs.data_ptr(), blocks[3].data_ptr())
    assert L.psfft_slab_c2r_yx(plan.handle, P, 1, arr2, 0, zs.data_ptr(), real.data_ptr(), st) == -8          # reads what it writes
    arr2 = (ctypes.c_void_p * P)(blocks[0].data_ptr(), blocks[0].data_ptr(), blocks[2].data_ptr(), blocks[3].data_ptr())
    assert L.psfft_slab_c2r_yx(plan.handle, P, 1, arr2, 0, zs.data_ptr(), real.data_ptr(), st) == 0           # read-only blocks may alias
    assert L.psfft_slab_r2c_xy(plan.handle, P, 1, zs.data_ptr(), zs.data_ptr(), arr, 0, st) == -8             # overlap
    # guard bands: arena = [guard | zspec | guard | block 0 | guard | ... ]
    G = 512
    sizes = [lay.zspec_elems] + [psfft.slab_query(plan.handle, P, q).xslab_elems for q in range(P)]
    arena = torch.full((sum(sizes) + G * (len(sizes) + 1),), complex(float("nan"), float("nan")), dtype=torch.complex128,
                       device="cuda")
    offs, o = [], G
    for n in sizes:
        offs.append(o)
        o += n + G
    views = [arena[a:a + n] for a, n in zip(offs, sizes)]
    for v in views[1:]:
        v.zero_()
    psfft.slab_r2c_xy(plan.handle, P, 1, real, views[0], views[1:], lay.z0)
    torch.cuda.synchronize()
    mask = torch.ones_like(arena, dtype=torch.bool)
    for a, n in zip(offs, sizes):
        mask[a:a + n] = False
    assert bool(torch.isnan(arena[mask].real).all())                     # every guard element untouched
    assert not bool(torch.isnan(views[0].real).any())                   # the work buffer was written
    for q, v in enumerate(views[1:]):                                    # each block got exactly this rank's planes
        w = psfft.slab_query(plan.handle, P, q).w
        blk = v.view(Nz, Ny, w)
        assert bool((blk[lay.z0:lay.z0 + lay.Mz] != 0).any()) and bool((blk[:lay.z0] == 0).all()) and bool((blk[lay.z0 + lay.Mz:] == 0).all())


def test_packed_mode_class_under_torch_distributed_world_size_1():
    """slab.SlabFFT (the torch.distributed / NCCL path: send buffer of contiguous slices, one all_to_all_single, x-slab
    z-pass) on the one GPU this box has: a world of one rank must reproduce the single-GPU transform bit for bit.  (The
    exchange schedule for P > 1 is covered on CPU tensors by tests/test_slab_dist.py.)"""
    import os
    import socket
    import torch.distributed as dist
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        shape = (64, 48, 32)
        x = field(shape, torch.float64)
        plan = psfft.Plan(shape, torch.float64, 1)
        xd = torch.from_numpy(x).cuda()
        single = plan.r2c(xd[None])[0]
        sf = slab.SlabFFT(plan)
        X = sf.r2c(xd)
        assert torch.equal(X, single)
        back = sf.c2r(X.clone())
        assert torch.equal(back, plan.c2r(single[None])[0])
        # caller-owned result buffers (what a time loop passes every step): same bits, and it is those buffers that come back
        xbuf = torch.full((sf.lay.xslab_elems,), complex(float("nan"), 0.0), dtype=torch.complex128, device="cuda")
        rbuf = torch.full_like(xd, float("nan"))
        X2 = sf.r2c(xd, out=xbuf)
        assert X2.data_ptr() == xbuf.data_ptr() and torch.equal(X2, single)
        back2 = sf.c2r(X2, out=rbuf)
        assert back2.data_ptr() == rbuf.data_ptr() and torch.equal(back2, back)
    finally:
        dist.destroy_process_group()


def test_bench_multi_gpu_slab_row_in_a_world_of_one():
    """bench.py's slab_multi (what `--gpus N` adds to the line for N > 1) runs end to end under NCCL with one rank."""
    import os
    import socket
    import sys
    import torch.distributed as dist
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        res = bench.slab_multi(torch, psfft, torch.device("cuda", 0), torch.cuda.current_stream(), 3, N=128)
        assert "failed" not in res, res
        assert res["roundtrip_max_abs_err"] < 1e-13 and res["ms_r2c"] > 0 and res["ms_c2r"] > 0
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("shape,P", [((64, 32, 32), 4), ((32, 48, 24), 3), ((128, 64, 64), 8)])
def test_packed_mode_for_P_ranks_emulated_on_one_gpu(shape, P):
    """The packed (NCCL) mode for P > 1 without a process group: every rank's phase 1 fills its send buffer, the
    all_to_all_single is replayed as tensor copies with slab.forward_splits' counts (slice q of rank p's send buffer
    becomes slice p of rank q's receive buffer -- the semantics of the collective), phase 2 runs on the receive
    buffers, and the assembled x-slabs equal the single-GPU transform bit for bit; then the inverse the same way."""
    Nx, Ny, Nz = shape
    ldk = Nx // 2 + 1
    x = field(shape, torch.float64)
    plan = psfft.Plan(shape, torch.float64, 1)
    xd = torch.from_numpy(x).cuda()
    single = plan.r2c(xd[None])[0]
    lays = [psfft.slab_query(plan.handle, P, r) for r in range(P)]
    Mz = lays[0].Mz
    cd = torch.complex128
    sends = [torch.empty(l.zspec_elems, dtype=cd, device="cuda") for l in lays]
    zs = torch.empty(lays[0].zspec_elems, dtype=cd, device="cuda")
    splits = [slab.forward_splits(Nz, Ny, ldk, P, r) for r in range(P)]
    for r in range(P):
        psfft.slab_r2c_xy(plan.handle, P, r, xd[r * Mz:(r + 1) * Mz], zs, slab._slice_ptrs(sends[r], splits[r][0]), 0)
    recvs = []
    for q in range(P):                                   # all_to_all_single, replayed
        parts = []
        for p_ in range(P):
            off = sum(splits[p_][0][:q])
            parts.append(sends[p_][off:off + splits[p_][0][q]])
            assert splits[p_][0][q] == splits[q][1][p_]  # what p sends to q is what q expects from p
        recvs.append(torch.cat(parts))
        assert recvs[q].numel() == lays[q].xslab_elems
    for q in range(P):
        psfft.slab_z(plan.handle, P, q, -1, recvs[q])
    got = torch.cat([recvs[q].view(Nz, Ny, lays[q].w) for q in range(P)], dim=2)
    assert torch.equal(got, single)
    # inverse: z-pass on the x-slabs, exchange of contiguous z-ranges, gather-load y-pass + c2r
    for q in range(P):
        psfft.slab_z(plan.handle, P, q, +1, recvs[q])
    back = torch.empty((Nz, Ny, Nx), dtype=torch.float64, device="cuda")
    for r in range(P):
        parts = [recvs[q].view(Nz, Ny, lays[q].w)[r * Mz:(r + 1) * Mz].reshape(-1) for q in range(P)]   # what q sends to r
        rbuf = torch.cat(parts)
        psfft.slab_c2r_yx(plan.handle, P, r, slab._slice_ptrs(rbuf, splits[r][0]), 0, zs, back[r * Mz:(r + 1) * Mz])
    assert torch.equal(back, plan.c2r(single[None])[0])


DIRECT_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_1808_01309_b200 import psfft, slab
rank, P = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(0)                                   # both ranks on the one GPU of the box
dist.init_process_group("gloo", rank=rank, world_size=P)   # handles and barriers only: direct mode needs no NCCL
out = {}
for shape, dtype in (((32, 24, 16), torch.float64), ((48, 16, 32), torch.float32), ((64, 64, 64), torch.float64)):
    Nx, Ny, Nz = shape
    plan = psfft.Plan(shape if len(set(shape)) > 1 else Nx, dtype, 1)
    g = torch.Generator(device="cuda").manual_seed(99)     # the same global field in both processes
    x = torch.rand((1, Nz, Ny, Nx), dtype=dtype, device="cuda", generator=g) * 2 - 1
    want = plan.r2c(x)[0]                                  # single-GPU transform of the whole field
    sf = slab.DirectSlabFFT(plan)
    Mz, x0 = sf.lay.Mz, sf.lay.x0
    for rep in range(2):                                   # twice: the barriers make the buffers reusable
        X = sf.r2c(x[0, rank * Mz:(rank + 1) * Mz].contiguous())
        fwd = bool(torch.equal(X, want[:, :, x0[rank]:x0[rank + 1]]))
        back = sf.c2r()
        inv = bool(torch.equal(back, plan.c2r(want[None].contiguous())[0, rank * Mz:(rank + 1) * Mz]))
        out[f"{shape}-{dtype}-{rep}"] = [fwd, inv, float((back - x[0, rank * Mz:(rank + 1) * Mz]).abs().max())]
    del sf
    dist.barrier()
print(json.dumps({"rank": rank, "results": out}))
dist.destroy_process_group()
""" % ROOT


def test_direct_mode_with_two_real_processes_sharing_the_gpu(tmp_path):
    """slab.DirectSlabFFT: two PROCESSES (gloo group for handles and barriers), both on cuda:0, each exporting its x-slab
    to the other through CUDA IPC; rank p's y-pass stores straight into the peer's x-slab.  Each rank's x-slab equals the
    matching kx range of psfft_fft3d_r2c of the whole field BIT FOR BIT, and the inverse equals psfft_fft3d_c2r's
    planes bit for bit."""
    import json
    import subprocess
    import sys
    script = tmp_path / "direct_worker.py"
    script.write_text(DIRECT_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29541", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=600) for p in procs]
    assert all(p.returncode == 0 for p in procs), [o[1][-1500:] for o in outs]
    for r, (out, _) in enumerate(outs):
        got = json.loads(out.strip().splitlines()[-1])
        assert got["rank"] == r and len(got["results"]) == 6
        for key, (fwd, inv, err) in got["results"].items():
            assert fwd and inv, (r, key)
            assert err < (1e-5 if "float32" in key else 1e-13), (r, key, err)
