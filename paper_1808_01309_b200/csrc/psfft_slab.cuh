// psfft_slab.cuh -- the slab-decomposed (multi-GPU) transform of the paper, B200 form.
//
// PAPER.md:68-81 (Sec. 2, Fig. 1): P tasks, task p owns the z-slab of M = Nz / P planes.  Forward transform:
//   1. local 2D transform (x, then y) in every plane of the slab  -> z-incomplete
//   2. global transpose (all-to-all, "the only communication")    -> z- and y-complete, x-incomplete
//   3. local 1D transform along z
// and the paper adds a local transpose on either side of the exchange (cost (3)).
//
// Here steps 1-2 are ONE kernel: the y-pass of the slab stores each finished column straight into the x-slab of the
// task that owns its kx ("x-distributed" addressing below), so there is no pack buffer, no local transpose and no
// unpack: after the exchange every task holds its x-slab [Nz][Ny][w] in the natural layout and the plain strided
// z-pass (psfft_kernels.cuh k_cpass) finishes the transform.  Where the blocks live is the caller's choice:
//   direct   base[q] = peer-mapped x-slab of rank q (NVLink P2P / symmetric memory), zoff = rank * M: the stores ARE the
//            all-to-all; a barrier between the two phases is the only synchronisation
//   packed   base[q] = slice q of a local send buffer, zoff = 0: one all_to_all_single (NCCL) of contiguous slices then
//            delivers the x-slab, again with no pack / unpack kernel (the receive buffer is the x-slab)
// The inverse mirrors it: plain inverse z-pass on the x-slab, then the inverse y-pass of each z-slab LOADS its columns
// from the x-distributed blocks (direct: peer loads; packed: the slices an all_to_all_single of contiguous z-ranges of
// the x-slabs delivered), then the c2r x-pass.
#pragma once
#include "psfft_kernels.cuh"

namespace psfft {

constexpr int kMaxRanks = 16;

// An array [z][ky][kx] distributed over P ranks by kx: rank q holds kx in [x0[q], x0[q + 1]) as [rows][Ny][w_q]
template <typename C> struct XDist {
    C *base[kMaxRanks];      // block of rank q
    int x0[kMaxRanks + 1];
    int P;
    long zoff;               // row (z plane) of this slab's first plane inside each block
};

// y-pass of one z-slab [Mz][N = Ny][ldk] with one side x-distributed.
//   SCATTER = true  (forward, DIR = -1): load the slab, store into the blocks
//   SCATTER = false (inverse, DIR = +1): load from the blocks, store the slab
// grid (ceil(ldk / (TC EW)), Mz); same tile shape, butterflies and twiddles as k_cpass, so every column is transformed
// bit for bit as by the single-GPU y-pass.
template <typename T, int N, int DIR, int TC, int TPF, int MINB, bool SCATTER>
__global__ void __launch_bounds__(TC *TPF, MINB)
    k_cpass_xdist(const Cx<T> *slab_in, Cx<T> *slab_out, XDist<Cx<T>> xd, const Cx<T> *__restrict__ tw, int ldk)
{
    using C = Cx<T>;
    using E = Ex<T>;
    constexpr int EW = ElemWidth<E>::value;
    constexpr bool PAD = (TC * sizeof(E) < 128);
    using Map = ColMap<N, TC, PAD>;
    extern __shared__ __align__(16) unsigned char smraw[];
    E *sm = reinterpret_cast<E *>(smraw);

    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    const int col = ((int)blockIdx.x * TC + c) * EW;
    const long pbase = (long)blockIdx.y * N * ldk;
    bool valid[EW];
    C *dptr[EW];
    long dw[EW];
#pragma unroll
    for (int j = 0; j < EW; ++j) {
        const int kx = col + j;
        valid[j] = kx < ldk;
        int q = 0;
        while (q + 1 < xd.P && kx >= xd.x0[q + 1]) ++q;
        dw[j] = xd.x0[q + 1] - xd.x0[q];
        dptr[j] = xd.base[q] + (xd.zoff + blockIdx.y) * (long)N * dw[j] + (kx - xd.x0[q]);
    }
    auto ld = [&](int i) -> E {
        E x = ezero<E>();
#pragma unroll
        for (int j = 0; j < EW; ++j)
            if (valid[j]) ecol_set(x, j, SCATTER ? ld_stream(slab_in + pbase + (long)i * ldk + col + j) : ld_stream(dptr[j] + i * dw[j]));
        return x;
    };
    auto st = [&](int i, E v) {
#pragma unroll
        for (int j = 0; j < EW; ++j) {
            if (!valid[j]) continue;
            if (SCATTER) st_stream(dptr[j] + i * dw[j], ecol(v, j));
            else st_stream(slab_out + pbase + (long)i * ldk + col + j, ecol(v, j));
        }
    };
    fft_stages<T, N, 1, DIR, TPF, false, false, false, Map>(sm, tw, c, t, ld, st);
}

}  // namespace psfft
