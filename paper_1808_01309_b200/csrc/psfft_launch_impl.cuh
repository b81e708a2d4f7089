// psfft_launch_impl.cuh -- definitions of the launchers; included by psfft_f32.cu / psfft_f64.cu,
// which instantiate them for one dtype each (two translation units compile in parallel).
#pragma once
#include "psfft_kernels.cuh"
#include "psfft_launch.cuh"

namespace psfft {

// tile shapes ------------------------------------------------------------------------------
// x-pass: transforms per CTA so that a CTA has about 256 threads
__host__ __device__ constexpr int xpass_rows(int N)
{
    int tpf = threads_per_fft(N / 2);
    return tpf >= 256 ? 1 : 256 / tpf;
}
// column passes: TC contiguous columns per CTA; at least 64 B per tile row
__host__ __device__ constexpr int cpass_cols(int N, int csize)
{
    int tpf = threads_per_fft(N);
    int tc = tpf >= 256 ? 1 : 256 / tpf;
    int mn = 64 / csize;
    return tc < mn ? mn : tc;
}

template <typename K> static cudaError_t set_smem(K kernel, size_t bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <typename T, int N>
static cudaError_t xpass_r2c_n(const PassArgs &a, const void *in, void *out, long nrows)
{
    constexpr int ROWS = xpass_rows(N);
    constexpr int TPF = threads_per_fft(N / 2);
    constexpr size_t smem = (size_t)ROWS * RowMap<N / 2>::ld * sizeof(Cx<T>);
    auto kern = k_xpass_r2c<T, N, ROWS>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((nrows + ROWS - 1) / ROWS);
    kern<<<grid, ROWS * TPF, smem, a.stream>>>((const T *)in, (Cx<T> *)out, (const Cx<T> *)a.tab, nrows, a.ldk);
    return cudaGetLastError();
}

template <typename T, int N>
static cudaError_t xpass_c2r_n(const PassArgs &a, const void *in, void *out, long nrows, double scale)
{
    constexpr int ROWS = xpass_rows(N);
    constexpr int TPF = threads_per_fft(N / 2);
    constexpr size_t smem = (size_t)ROWS * RowMap<N / 2>::ld * sizeof(Cx<T>);
    auto kern = k_xpass_c2r<T, N, ROWS>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((nrows + ROWS - 1) / ROWS);
    kern<<<grid, ROWS * TPF, smem, a.stream>>>((const Cx<T> *)in, (T *)out, (const Cx<T> *)a.tab, nrows, a.ldk,
                                                (T)scale);
    return cudaGetLastError();
}

template <typename T, int N, int DIR>
static cudaError_t cpass_n(const PassArgs &a, int axis, const void *in, void *out, int fields)
{
    using C = Cx<T>;
    constexpr int TC = cpass_cols(N, (int)sizeof(C));
    constexpr int TPF = threads_per_fft(N);
    constexpr bool PAD = (TC * sizeof(C) < 128);
    constexpr size_t smem = (size_t)ColMap<N, TC, PAD>::size * sizeof(C);
    auto kern = k_cpass<T, N, DIR, TC>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    const long plane = (long)a.ldk * N;
    long axis_stride, inner, outer_stride, outer;
    if (axis == 1) { axis_stride = a.ldk; inner = a.ldk; outer_stride = plane; outer = (long)N * fields; }
    else { axis_stride = plane; inner = plane; outer_stride = plane * N; outer = fields; }
    dim3 grid((unsigned)((inner + TC - 1) / TC), (unsigned)outer);
    kern<<<grid, TC * TPF, smem, a.stream>>>((const C *)in, (C *)out, (const C *)a.tab, axis_stride, inner,
                                              outer_stride);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_xpass_r2c(const PassArgs &a, const void *in, void *out, long nrows, int *launches)
{
    ++*launches;
    switch (a.N) {
#define X(n) case n: return xpass_r2c_n<T, n>(a, in, out, nrows);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t launch_xpass_c2r(const PassArgs &a, const void *in, void *out, long nrows, double scale, int *launches)
{
    ++*launches;
    switch (a.N) {
#define X(n) case n: return xpass_c2r_n<T, n>(a, in, out, nrows, scale);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t launch_cpass(const PassArgs &a, int dir, int axis, const void *in, void *out, int fields, int *launches)
{
    ++*launches;
    switch (a.N) {
#define X(n) case n: return dir < 0 ? cpass_n<T, n, -1>(a, axis, in, out, fields) : cpass_n<T, n, +1>(a, axis, in, out, fields);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

template <typename T> cudaError_t launch_mask_curl(const PassArgs &a, const void *u, void *out6, int *launches)
{
    ++*launches;
    const long nf = (long)a.ldk * a.N * a.N;
    k_mask_curl<T><<<(unsigned)((nf + 255) / 256), 256, 0, a.stream>>>((const Cx<T> *)u, (Cx<T> *)out6, a.N, a.ldk, nf);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_cross(const PassArgs &a, const void *pa, const void *pb, void *pc, int *launches)
{
    ++*launches;
    const long n = (long)a.N * a.N * a.N;
    k_cross<T><<<(unsigned)((n + 255) / 256), 256, 0, a.stream>>>((const T *)pa, (const T *)pb, (T *)pc, n);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_cross_mhd(const PassArgs &a, const void *u, const void *b, const void *w, const void *j, void *om,
                             void *oe, int *launches)
{
    ++*launches;
    const long n = (long)a.N * a.N * a.N;
    k_cross_mhd<T><<<(unsigned)((n + 255) / 256), 256, 0, a.stream>>>((const T *)u, (const T *)b, (const T *)w,
                                                                      (const T *)j, (T *)om, (T *)oe, n);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_finish(const PassArgs &a, int mode, const void *f, const void *u, void *out, double nu, int *launches)
{
    ++*launches;
    const long nf = (long)a.ldk * a.N * a.N;
    const unsigned grid = (unsigned)((nf + 255) / 256);
    if (mode == 0)
        k_finish<T, 0><<<grid, 256, 0, a.stream>>>((const Cx<T> *)f, (const Cx<T> *)u, (Cx<T> *)out, a.N, a.ldk, nf, (T)nu);
    else
        k_finish<T, 1><<<grid, 256, 0, a.stream>>>((const Cx<T> *)f, (const Cx<T> *)u, (Cx<T> *)out, a.N, a.ldk, nf, (T)nu);
    return cudaGetLastError();
}

#define PSFFT_INSTANTIATE(T)                                                                                          \
    template cudaError_t launch_xpass_r2c<T>(const PassArgs &, const void *, void *, long, int *);                    \
    template cudaError_t launch_xpass_c2r<T>(const PassArgs &, const void *, void *, long, double, int *);            \
    template cudaError_t launch_cpass<T>(const PassArgs &, int, int, const void *, void *, int, int *);               \
    template cudaError_t launch_mask_curl<T>(const PassArgs &, const void *, void *, int *);                          \
    template cudaError_t launch_cross<T>(const PassArgs &, const void *, const void *, void *, int *);                \
    template cudaError_t launch_cross_mhd<T>(const PassArgs &, const void *, const void *, const void *, const void *, \
                                             void *, void *, int *);                                                  \
    template cudaError_t launch_finish<T>(const PassArgs &, int, const void *, const void *, void *, double, int *);

}  // namespace psfft
