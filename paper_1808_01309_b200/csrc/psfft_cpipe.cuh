// psfft_cpipe.cuh -- software-pipelined strided column pass (y or z axis) of the plain 3D transforms.
//
// Same transform as k_cpass (psfft_kernels.cuh; a2 / a4 / a5 of SURVEY.md §8(a)) with a
// different schedule: persistent CTAs walk over the tiles [N rows] x [TC contiguous columns]; the
// NEXT tile of a CTA is fetched with cp.async (global -> shared memory, no registers) into a second
// shared-memory buffer while the butterflies of the current tile run, so that HBM latency is hidden
// behind the compute phases instead of being exposed once per tile (profiles/r1b_summary.md: the
// unpipelined column passes sit at 50 % warps active and 55-65 % DRAM utilisation).
#pragma once
#include "psfft_core.cuh"

namespace psfft {

// 16-byte (fp64 complex) / 8-byte (fp32 complex) asynchronous copy; `ok == false` zero-fills
__device__ __forceinline__ void cp_async_c(double2 *smem_dst, const double2 *gsrc, bool ok)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_c(float2 *smem_dst, const float2 *gsrc, bool ok)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = ok ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int PENDING> __device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(PENDING) : "memory");
}

// tiles are numbered w = by * ntx + bx:  bx = tile along the contiguous axis, by = outer slice
template <typename T, int N, int DIR, int TC, int TPF, int NBUF>
__global__ void __launch_bounds__(TC *TPF, 1)
    k_cpass_pipe(const Cx<T> *in, Cx<T> *out, const Cx<T> *__restrict__ tw, long axis_stride, long inner,
                 long outer_stride, int ntx, long ntiles)
{
    using C = Cx<T>;
    constexpr bool PAD = (TC * sizeof(C) < 128);
    using Map = ColMap<N, TC, PAD>;
    constexpr int ROWS_PER_THREAD = N / TPF;
    extern __shared__ __align__(16) unsigned char smraw[];
    C *sm = reinterpret_cast<C *>(smraw);

    const int c = threadIdx.x % TC, t = threadIdx.x / TC;

    auto issue = [&](long w, int buf) {
        const long bx = w % ntx, by = w / ntx;
        const long col = bx * TC + c;
        const bool valid = col < inner;
        const C *src = in + by * outer_stride + (valid ? col : 0);
        C *dstb = sm + buf * Map::size;
#pragma unroll
        for (int r = 0; r < ROWS_PER_THREAD; ++r) {
            const int i = t + r * TPF;
            cp_async_c(dstb + Map::at(i, c), src + i * axis_stride, valid);
        }
        cp_async_commit();
    };

    long w = blockIdx.x;
    if (w >= ntiles) return;
    int buf = 0;
    // prologue: NBUF - 1 tiles in flight
    {
        long wp = w;
#pragma unroll
        for (int k = 0; k < NBUF - 1; ++k) {
            if (wp < ntiles) issue(wp, k);
            else cp_async_commit();
            wp += gridDim.x;
        }
    }
    for (; w < ntiles; w += gridDim.x) {
        // the buffer freed at the end of the previous iteration receives the tile NBUF - 1 ahead
        const long wn = w + (long)(NBUF - 1) * gridDim.x;
        const int bufn = (buf + NBUF - 1) % NBUF;
        if (wn < ntiles) issue(wn, bufn);
        else cp_async_commit();
        cp_async_wait<NBUF - 1>();
        __syncthreads();

        const long bx = w % ntx, by = w / ntx;
        const long col = bx * TC + c;
        const bool valid = col < inner;
        C *dst = out + by * outer_stride + (valid ? col : 0);
        auto ld = [&](int) -> C { return mk<T>(0, 0); };
        auto st = [&](int i, C v) {
            if (valid) st_stream(dst + i * axis_stride, v);
        };
        fft_stages<T, N, 1, DIR, TPF, true, false, false, Map>(sm + buf * Map::size, tw, c, t, ld, st);
        __syncthreads();   // every read of this buffer is done before it is refilled
        buf = (buf + 1) % NBUF;
    }
}

}  // namespace psfft
