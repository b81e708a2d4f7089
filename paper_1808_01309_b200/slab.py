"""Slab-decomposed 3D transform over P ranks (Sec. 2, Fig. 1): orchestration only.

Every transform step runs in libpsfft's kernels (``psfft.slab_r2c_xy / slab_z / slab_c2r_yx``); this module decides
where the x-distributed blocks live and moves them:

* ``VirtualSlabs``   P virtual ranks in ONE process on one GPU, *direct* mode: rank p's y-pass stores straight into the
                     x-slab buffers of all ranks (on a multi-GPU node those would be peer-mapped buffers; here they
                     are ordinary device buffers), so the all-to-all is the store pattern of the kernel itself.  The
                     result equals ``psfft_fft3d_r2c`` bit for bit -- the single-GPU check of the multi-GPU path.
* ``SlabFFT``        one rank of a ``torch.distributed`` job, *packed* mode: the y-pass stores into a send buffer laid
                     out as P contiguous slices, ONE ``all_to_all_single`` (NCCL over NVLink on GPUs) delivers the
                     x-slab -- the receive buffer [sender][Mz][Ny][w] is the x-slab [Nz][Ny][w], no unpack.
* ``DirectSlabFFT``  one rank of a ``torch.distributed`` job on one node, *direct* mode with REAL processes: every rank's
                     x-slab is mapped into every other rank through CUDA IPC, the y-pass stores / loads go straight
                     to the owners, a barrier separates the phases; no NCCL needed.
* ``exchange_forward / exchange_inverse``  the two all-to-alls with their split sizes; pure communication on torch
                     tensors of any device (the world_size-2 gloo test drives them on CPU tensors).

Unmeasured on multi-GPU hardware: this round's GPU box has one GPU.
"""
from __future__ import annotations

import torch

from . import psfft


def x_ranges(ldk: int, P: int):
    """kx range [x0[q], x0[q+1]) of every rank: x0[q] = floor(q ldk / P) (as psfft_slab_query)."""
    return [q * ldk // P for q in range(P + 1)]


def forward_splits(Nz: int, Ny: int, ldk: int, P: int, rank: int):
    """(send counts, receive counts) in complex elements of the forward all-to-all of rank `rank`: it sends rank q the
    slice [Mz][Ny][w_q] and receives [Mz][Ny][w_rank] from everyone.  The inverse exchange swaps the two lists."""
    x0 = x_ranges(ldk, P)
    Mz = Nz // P
    send = [Mz * Ny * (x0[q + 1] - x0[q]) for q in range(P)]
    recv = [Mz * Ny * (x0[rank + 1] - x0[rank])] * P
    return send, recv


def exchange_forward(sendbuf: torch.Tensor, xslab: torch.Tensor, Nz: int, Ny: int, ldk: int, group=None) -> None:
    """The global transpose of PAPER.md:76 (step 2) as one all-to-all of contiguous slices.  sendbuf: flat complex,
    slices [q][Mz][Ny][w_q]; xslab: flat complex [Nz][Ny][w_rank] (= [p][Mz][Ny][w_rank])."""
    import torch.distributed as dist
    P, rank = dist.get_world_size(group), dist.get_rank(group)
    send, recv = forward_splits(Nz, Ny, ldk, P, rank)
    dist.all_to_all_single(xslab, sendbuf, output_split_sizes=recv, input_split_sizes=send, group=group)


def exchange_inverse(xslab: torch.Tensor, recvbuf: torch.Tensor, Nz: int, Ny: int, ldk: int, group=None) -> None:
    """Inverse direction: rank q sends rank p the contiguous z-range [p Mz, (p+1) Mz) of its x-slab; recvbuf gets the
    slices [q][Mz][Ny][w_q] that the inverse y-pass loads from."""
    import torch.distributed as dist
    P, rank = dist.get_world_size(group), dist.get_rank(group)
    send, recv = forward_splits(Nz, Ny, ldk, P, rank)
    dist.all_to_all_single(recvbuf, xslab, output_split_sizes=send, input_split_sizes=recv, group=group)


def _slice_ptrs(buf: torch.Tensor, counts):
    """Device pointers of consecutive slices of `counts` elements of a flat tensor."""
    out, off = [], 0
    for c in counts:
        out.append(buf.data_ptr() + off * buf.element_size())
        off += c
    return out


class SlabFFT:
    """One rank of the distributed transform (packed mode).  `plan` is a psfft.Plan of the GLOBAL grid."""

    def __init__(self, plan: "psfft.Plan", group=None):
        import torch.distributed as dist
        self.plan, self.group = plan, group
        self.P, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.lay = psfft.slab_query(plan.handle, self.P, self.rank)
        dev, cd = plan.device, plan.cdtype
        self.zspec = torch.empty(self.lay.zspec_elems, dtype=cd, device=dev)
        self.sendbuf = torch.empty(self.lay.zspec_elems, dtype=cd, device=dev)   # sum of the slices = Mz Ny ldk
        self.send, self.recv = forward_splits(plan.Nz, plan.Ny, plan.ldk, self.P, self.rank)

    def r2c(self, real_slab: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        """real_slab [Mz][Ny][Nx] -> this rank's x-slab [Nz][Ny][w].  `out`: a flat complex buffer of xslab_elems to
        receive it (a time loop passes the same one every step); allocated here when omitted."""
        p, h = self.plan, self.plan.handle
        xslab = out if out is not None else torch.empty(self.lay.xslab_elems, dtype=p.cdtype, device=p.device)
        assert xslab.numel() == self.lay.xslab_elems and xslab.dtype == p.cdtype and xslab.is_contiguous()
        xslab = xslab.view(-1)
        psfft.slab_r2c_xy(h, self.P, self.rank, real_slab, self.zspec, _slice_ptrs(self.sendbuf, self.send), 0)
        exchange_forward(self.sendbuf, xslab, p.Nz, p.Ny, p.ldk, self.group)
        psfft.slab_z(h, self.P, self.rank, -1, xslab)
        return xslab.view(p.Nz, p.Ny, self.lay.w)

    def c2r(self, xslab: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        """x-slab [Nz][Ny][w] (overwritten) -> real z-slab [Mz][Ny][Nx] (into `out` when given)."""
        p, h = self.plan, self.plan.handle
        psfft.slab_z(h, self.P, self.rank, +1, xslab)
        exchange_inverse(xslab.reshape(-1), self.sendbuf, p.Nz, p.Ny, p.ldk, self.group)
        real = out if out is not None else torch.empty((self.lay.Mz, p.Ny, p.N), dtype=p.rdtype, device=p.device)
        assert real.numel() == self.lay.real_elems and real.dtype == p.rdtype and real.is_contiguous()
        psfft.slab_c2r_yx(h, self.P, self.rank, _slice_ptrs(self.sendbuf, self.send), 0, self.zspec, real)
        return real


class DirectSlabFFT:
    """One rank of a ``torch.distributed`` job on ONE node, *direct* mode (psfft.h): the fused compute + exchange path.

    Every rank owns its x-slab [Nz][Ny][w] and exports it to the other ranks through CUDA IPC (the handles travel as
    pickled objects over the process group -- ``all_gather_object`` -- so the group may be gloo: this mode needs no NCCL
    at all).  The forward y-pass of a rank then stores each finished column straight into the x-slab of the rank that
    owns its kx -- over NVLink when that rank sits on another GPU -- so the all-to-all of PAPER.md:76 IS the store
    pattern of the kernel and overlaps the y-pass tile by tile; the inverse y-pass loads its columns from the peers'
    x-slabs the same way.  The only synchronisation is a barrier between the two phases (all stores have landed before
    anyone starts the z-pass; all loads are done before anyone overwrites its x-slab again).

    Buffers (x-slab, phase-1 work buffer, the real output slab) are allocated once, here.  ``plan`` is a psfft.Plan of
    the GLOBAL grid on this rank's device.  Verified with two processes sharing the one GPU of the test box
    (tests/test_gpu_slab.py); between different GPUs it relies on CUDA IPC peer mappings and is unmeasured."""

    def __init__(self, plan: "psfft.Plan", group=None):
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        self.plan, self.group = plan, group
        self.P, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.lay = psfft.slab_query(plan.handle, self.P, self.rank)
        dev, cd = plan.device, plan.cdtype
        with torch.cuda.device(dev):
            self.xslab = torch.empty(self.lay.xslab_elems, dtype=cd, device=dev)
            self.zspec = torch.empty(self.lay.zspec_elems, dtype=cd, device=dev)
            self.real = torch.empty((self.lay.Mz, plan.Ny, plan.N), dtype=plan.rdtype, device=dev)
            exported = reduce_tensor(self.xslab)                # (rebuild function, IPC handle + geometry): picklable
            gathered = [None] * self.P
            dist.all_gather_object(gathered, exported, group=group)
            # d_blocks[q]: rank q's x-slab as THIS process addresses it (own buffer; IPC mapping of a peer's)
            self.blocks = [self.xslab if q == self.rank else fn(*args) for q, (fn, args) in enumerate(gathered)]
        for q, b in enumerate(self.blocks):
            assert b.numel() == psfft.slab_query(plan.handle, self.P, q).xslab_elems and b.dtype == cd
        self._barrier()

    def _barrier(self):
        import torch.distributed as dist
        torch.cuda.synchronize(self.plan.device)
        dist.barrier(group=self.group)

    def r2c(self, real_slab: torch.Tensor) -> torch.Tensor:
        """real_slab [Mz][Ny][Nx] -> this rank's x-slab [Nz][Ny][w] (the object's own buffer, valid until the next call)."""
        p, h = self.plan, self.plan.handle
        with torch.cuda.device(p.device):
            psfft.slab_r2c_xy(h, self.P, self.rank, real_slab, self.zspec, self.blocks, self.rank * self.lay.Mz)
            self._barrier()                                     # every rank's stores have landed in every x-slab
            psfft.slab_z(h, self.P, self.rank, -1, self.xslab)
        return self.xslab.view(p.Nz, p.Ny, self.lay.w)

    def c2r(self) -> torch.Tensor:
        """The x-slab held by this object (as r2c left it, or as the caller filled ``self.xslab``; overwritten) ->
        real z-slab [Mz][Ny][Nx] (the object's own buffer)."""
        p, h = self.plan, self.plan.handle
        with torch.cuda.device(p.device):
            psfft.slab_z(h, self.P, self.rank, +1, self.xslab)
            self._barrier()                                     # every x-slab holds its inverse z-pass
            psfft.slab_c2r_yx(h, self.P, self.rank, self.blocks, self.rank * self.lay.Mz, self.zspec, self.real)
            self._barrier()                                     # all peer loads done: x-slabs may be overwritten again
        return self.real


class VirtualSlabs:
    """P virtual ranks on one device, direct mode: every rank's x-slab is a buffer all ranks can address."""

    def __init__(self, plan: "psfft.Plan", P: int):
        self.plan, self.P = plan, P
        self.lays = [psfft.slab_query(plan.handle, P, r) for r in range(P)]
        cd, dev = plan.cdtype, plan.device
        self.xslabs = [torch.empty(l.xslab_elems, dtype=cd, device=dev) for l in self.lays]
        self.zspec = torch.empty(self.lays[0].zspec_elems, dtype=cd, device=dev)

    def r2c(self, real: torch.Tensor) -> torch.Tensor:
        """real [Nz][Ny][Nx] (the ranks' z-slabs are its consecutive plane ranges) -> assembled half spectrum
        [Nz][Ny][ldk] gathered from the P x-slabs."""
        p, h, P = self.plan, self.plan.handle, self.P
        Mz = self.lays[0].Mz
        for r in range(P):      # phase 1 of every rank: x, y passes + the all-to-all as peer stores
            psfft.slab_r2c_xy(h, P, r, real[r * Mz:(r + 1) * Mz], self.zspec, self.xslabs, r * Mz)
        for r in range(P):      # (barrier here on real hardware)  phase 2: z-pass of every x-slab
            psfft.slab_z(h, P, r, -1, self.xslabs[r])
        return self.gather()

    def gather(self) -> torch.Tensor:
        p = self.plan
        return torch.cat([x.view(p.Nz, p.Ny, l.w) for x, l in zip(self.xslabs, self.lays)], dim=2)

    def c2r(self, spec: torch.Tensor) -> torch.Tensor:
        """half spectrum [Nz][Ny][ldk] -> real [Nz][Ny][Nx] through the P virtual ranks."""
        p, h, P = self.plan, self.plan.handle, self.P
        for r, l in enumerate(self.lays):
            self.xslabs[r].view(p.Nz, p.Ny, l.w).copy_(spec[:, :, l.x0[r]:l.x0[r + 1]])
            psfft.slab_z(h, P, r, +1, self.xslabs[r])
        real = torch.empty((p.Nz, p.Ny, p.N), dtype=p.rdtype, device=p.device)
        Mz = self.lays[0].Mz
        for r in range(P):
            psfft.slab_c2r_yx(h, P, r, self.xslabs, r * Mz, self.zspec, real[r * Mz:(r + 1) * Mz])
        return real
