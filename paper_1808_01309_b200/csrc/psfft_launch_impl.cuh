// psfft_launch_impl.cuh -- definitions of the launchers; included by psfft_f{32,64}_{fft,col,midx}.cu,
// which instantiate one group of them for one dtype each (six translation units compile in parallel).
#pragma once
#include "psfft_kernels.cuh"
#include "psfft_rhs.cuh"
#include "psfft_midxg.cuh"
#include "psfft_xpass2.cuh"
#include "psfft_slab.cuh"
#include "psfft_launch.cuh"

namespace psfft {

// tile shapes ------------------------------------------------------------------------------
template <typename K> static cudaError_t set_smem(K kernel, size_t bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// x-passes: two adjacent rows per complex length-N transform (psfft_xpass2.cuh); nrows is even for every
// supported size
template <typename T, int N> constexpr int xpass2_minb()
{
    constexpr int threads = xg_rows<N>() * XSched<N>::TPR;
    constexpr int m = 512 / threads;
    return m < 1 ? 1 : m;
}

template <typename T, int N>
static cudaError_t xpass_r2c_n(const PassArgs &a, const void *in, void *out, long nrows)
{
    using C = Cx<T>;
    constexpr int ROWS = xg_rows<N>(), THREADS = ROWS * XSched<N>::TPR;
    constexpr size_t smem = (size_t)ROWS * 2 * XPad<N, (int)sizeof(C)>::BUF * sizeof(C);
    auto kern = k_xpass2_r2c<T, N, xpass2_minb<T, N>()>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    const long npairs = nrows / 2;
    kern<<<(unsigned)((npairs + ROWS - 1) / ROWS), THREADS, smem, a.stream>>>((const T *)in, (C *)out, (const C *)a.twX,
                                                                              npairs, a.ldk);
    return cudaGetLastError();
}

template <typename T, int N>
static cudaError_t xpass_c2r_n(const PassArgs &a, const void *in, void *out, long nrows, double scale)
{
    using C = Cx<T>;
    constexpr int ROWS = xg_rows<N>(), THREADS = ROWS * XSched<N>::TPR;
    constexpr size_t smem = (size_t)ROWS * XPad<N, (int)sizeof(C)>::BUF * sizeof(C);
    auto kern = k_xpass2_c2r<T, N, xpass2_minb<T, N>()>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    const long npairs = nrows / 2;
    kern<<<(unsigned)((npairs + ROWS - 1) / ROWS), THREADS, smem, a.stream>>>((const C *)in, (T *)out, (const C *)a.twX,
                                                                              npairs, a.ldk, (T)scale);
    return cudaGetLastError();
}

template <typename T, int N, int DIR, int TC, int TPF, int MINB>
static cudaError_t cpass_strided(const PassArgs &a, const void *tw, const void *in, void *out, long axis_stride, long inner,
                                 long outer_stride, long outer)
{
    using C = Cx<T>;
    using E = Ex<T>;
    constexpr int EW = ElemWidth<E>::value;
    constexpr bool PAD = (TC * sizeof(E) < 128);
    constexpr size_t smem = (size_t)ColMap<N, TC, PAD>::size * sizeof(E);
    auto kern = k_cpass<T, N, DIR, TC, TPF, MINB>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((inner + TC * EW - 1) / (TC * EW)), (unsigned)outer);
    // fp32 pairs: 16-byte access when every pair of columns is aligned (even strides; the bases are 16-byte aligned)
    const bool vec = axis_stride % 2 == 0 && outer_stride % 2 == 0 && inner % 2 == 0 &&
                     (reinterpret_cast<uintptr_t>(in) & 15u) == 0 && (reinterpret_cast<uintptr_t>(out) & 15u) == 0;
    kern<<<grid, TC * TPF, smem, a.stream>>>((const C *)in, (C *)out, (const C *)tw, axis_stride, inner, outer_stride, vec);
    return cudaGetLastError();
}

template <typename T, int N, int DIR, int TC, int TPF, int MINB>
static cudaError_t cpass_v(const PassArgs &a, int axis, const void *in, void *out, int fields)
{
    // N is the length of the transformed axis: Ny for the y-pass, Nz for the z-pass
    const long plane = (long)a.ldk * a.Ny;
    if (axis == 1)
        return cpass_strided<T, N, DIR, TC, TPF, MINB>(a, a.twY, in, out, a.ldk, a.ldk, plane, (long)a.Nz * fields);
    return cpass_strided<T, N, DIR, TC, TPF, MINB>(a, a.twZ, in, out, plane, plane, plane * a.Nz, fields);
}

// Column passes: 8 elements per thread (one radix-8 butterfly per stage) while the CTA stays within
// 512 threads -- twice the warps of the 16-element shape for the same two tiles per SM (measured, 512^3
// fp64: inv_y 1.67 -> 1.50 ms, fwd_y 0.85 -> 0.60 ms; profiles/r1b_summary.md)
// (A tile above 64 KB is alone on its SM and may take 1024 threads.)
__host__ __device__ constexpr int job_tpf(int N, int TC, int esize)
{
    const int cap = (long)N * TC * esize > 65536 ? 1024 : 512;
    return (N >= 64 && N % 8 == 0 && max_radix(N) == 8 && TC * (N / 8) <= cap) ? N / 8 : cpass_tpf(N);
}

// plain passes: 64 KB tiles; at N = 2048 a 64 KB tile would have 32-byte rows, so one 128 KB tile with 64-byte rows
__host__ __device__ constexpr long plain_tile_cap(int N) { return N >= 2048 ? 131072 : 65536; }

template <typename T, int N, int DIR>
static cudaError_t cpass_n(const PassArgs &a, int axis, const void *in, void *out, int fields)
{
    // 16-byte elements in both precisions; the plain passes keep 64 KB tiles at every N (measured: 1024 x 1024 x 256
    // r2c + c2r 5.77 ms with 64 KB tiles, 5.96 ms with 128 KB ones)
    constexpr int TC = cpass_cols_cap(N, (int)sizeof(Ex<T>), plain_tile_cap(N));
    constexpr int TPF = job_tpf(N, TC, 16);
    constexpr int MINB = ((long)N * TC * 16 * 2 <= 220 * 1024 && 2 * TC * TPF <= 1024) ? 2 : 1;
    return cpass_v<T, N, DIR, TC, TPF, MINB>(a, axis, in, out, fields);
}

// plain strided pass with caller-given strides (the z-pass of an x-slab: psfft_slab.cuh)
template <typename T, int N, int DIR>
static cudaError_t cpass_raw_n(const PassArgs &a, const void *tw, const void *in, void *out, long axis_stride, long inner,
                               long outer_stride, long outer)
{
    constexpr int TC = cpass_cols_cap(N, (int)sizeof(Ex<T>), plain_tile_cap(N));
    constexpr int TPF = job_tpf(N, TC, 16);
    constexpr int MINB = ((long)N * TC * 16 * 2 <= 220 * 1024 && 2 * TC * TPF <= 1024) ? 2 : 1;
    return cpass_strided<T, N, DIR, TC, TPF, MINB>(a, tw, in, out, axis_stride, inner, outer_stride, outer);
}

template <typename T>
cudaError_t launch_cpass_raw(const PassArgs &a, int dir, int len, const void *tw, const void *in, void *out, long axis_stride,
                             long inner, long outer_stride, long outer, int *launches)
{
    ++*launches;
    switch (len) {
#define X(n) case n: return dir < 0 ? cpass_raw_n<T, n, -1>(a, tw, in, out, axis_stride, inner, outer_stride, outer) \
                                    : cpass_raw_n<T, n, +1>(a, tw, in, out, axis_stride, inner, outer_stride, outer);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

// y-pass of a z-slab with the all-to-all fused into its store (forward) or load (inverse): psfft_slab.cuh
template <typename T, int N, bool SCATTER>
static cudaError_t cpass_xdist_n(const PassArgs &a, const void *slab_in, void *slab_out, const XDistArgs &xa, int mz)
{
    using C = Cx<T>;
    using E = Ex<T>;
    constexpr int EW = ElemWidth<E>::value;
    constexpr int TC = cpass_cols_cap(N, (int)sizeof(E), plain_tile_cap(N));
    constexpr int TPF = job_tpf(N, TC, 16);
    constexpr int MINB = ((long)N * TC * 16 * 2 <= 220 * 1024 && 2 * TC * TPF <= 1024) ? 2 : 1;
    constexpr bool PAD = (TC * sizeof(E) < 128);
    constexpr size_t smem = (size_t)ColMap<N, TC, PAD>::size * sizeof(E);
    auto kern = k_cpass_xdist<T, N, SCATTER ? -1 : +1, TC, TPF, MINB, SCATTER>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    XDist<C> xd;
    for (int q = 0; q < kMaxRanks; ++q) xd.base[q] = (C *)xa.base[q];
    for (int q = 0; q <= kMaxRanks; ++q) xd.x0[q] = xa.x0[q];
    xd.P = xa.P;
    xd.zoff = xa.zoff;
    dim3 grid((unsigned)((a.ldk + TC * EW - 1) / (TC * EW)), (unsigned)mz);
    kern<<<grid, TC * TPF, smem, a.stream>>>((const C *)slab_in, (C *)slab_out, xd, (const C *)a.twY, a.ldk);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_cpass_xdist(const PassArgs &a, bool scatter, const void *slab_in, void *slab_out, const XDistArgs &xd,
                               int mz, int *launches)
{
    ++*launches;
    switch (a.Ny) {
#define X(n) case n: return scatter ? cpass_xdist_n<T, n, true>(a, slab_in, slab_out, xd, mz) \
                                    : cpass_xdist_n<T, n, false>(a, slab_in, slab_out, xd, mz);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

// ---- fused right-hand side -------------------------------------------------------------------
// N below is always the length of the axis the pass transforms (Nz for the z passes, Ny for the y passes, Nx for
// mid_x); everything about the other axes and the box comes from PassArgs (psfft_rhs.cuh Geom).
// geometry policy of a pass whose own axis has length N: compile-time for the N^3 grid in the 2 pi box (CUBE),
// run-time values of the plan otherwise
template <typename T, int N, bool CUBE> struct GeomSel {
    using type = GeomAny<T>;
    static type make(const PassArgs &a)
    {
        type g;
        g.ny = a.Ny; g.nz = a.Nz; g.kxc = a.kxc;
        g.rx2 = a.rx2; g.ry2 = a.ry2; g.rz2 = a.rz2; g.lim = a.lim;
        g.kfx = (T)a.kf[0]; g.kfy = (T)a.kf[1]; g.kfz = (T)a.kf[2];
        return g;
    }
};
template <typename T, int N> struct GeomSel<T, N, true> {
    using type = GeomCube<T, N>;
    static type make(const PassArgs &) { return type(); }
};

template <typename T, int N, int DIR, int TPF, int MINB, class Job>
static cudaError_t run_job_v(const PassArgs &a, const Job &job, dim3 grid, const void *tw)
{
    using C = Cx<T>;
    using E = typename Job::Elem;
    constexpr int TC = Job::is_fwdz ? fwdz_cols(N, (int)sizeof(E)) : cpass_cols(N, (int)sizeof(E));   // elements per tile row
    constexpr bool PAD = (TC * sizeof(E) < 128);
    constexpr size_t smem = (size_t)ColMap<N, TC, PAD>::size * sizeof(E);
    auto kern = k_cpass_job<T, N, DIR, TC, TPF, MINB, Job>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    // small grids (N <= 256): one CTA per (tile position, round) instead of looping over the rounds, so that
    // the pass fills the machine
    if (Job::split_rounds && (long)grid.x * grid.y < 2048) grid.z = (unsigned)job.rounds();
    kern<<<grid, TC * TPF, smem, a.stream>>>(job, (const C *)tw);
    return cudaGetLastError();
}

template <typename T, int N, int DIR, class Job>
static cudaError_t run_job(const PassArgs &a, const Job &job, dim3 grid, const void *tw)
{
    using E = typename Job::Elem;
    constexpr int TC = Job::is_fwdz ? fwdz_cols(N, (int)sizeof(E)) : cpass_cols(N, (int)sizeof(E));
    // two CTAs per SM when two tiles fit in shared memory and two CTAs' threads in the register file at 64 each
    constexpr int TPF = job_tpf(N, TC, (int)sizeof(E));
    constexpr int MINB = ((long)N * TC * sizeof(E) * 2 <= 220 * 1024 && 2 * TC * TPF <= 1024) ? 2 : 1;
    return run_job_v<T, N, DIR, TPF, MINB>(a, job, grid, tw);
}

// z passes: N = Nz
template <typename T, int N, int NV, int NS, bool CUBE> static cudaError_t rhs_inv_z_n(const PassArgs &a, const RhsArgs &r)
{
    using C = Cx<T>;
    using GS = GeomSel<T, N, CUBE>;
    constexpr int TC = job_cols(N), EW = 16 / (int)sizeof(C);   // element columns per tile, columns per element
    JobInvZ<T, N, TC, NV, NS, typename GS::type> job;
    for (int v = 0; v < NV; ++v) job.src[v] = (const C *)r.src[v];
    job.ssrc = (const C *)r.ssrc;
    job.dst = (C *)r.zbuf;
    job.plane = (long)a.ldk * a.Ny;
    job.nf = job.plane * N;
    job.wplane = (long)a.kxp * a.Ny;
    job.wnf = job.wplane * N;
    job.ldk = a.ldk;
    job.kxp = a.kxp;
    job.geo = GS::make(a);
    return run_job<T, N, +1>(a, job, dim3((unsigned)(a.kxp / (TC * EW)), (unsigned)a.Ny), a.twZ);
}

// y passes: N = Ny
template <typename T, int N, int NV, int NS, bool CUBE> static cudaError_t rhs_inv_y_n(const PassArgs &a, const RhsArgs &r)
{
    using C = Cx<T>;
    using GS = GeomSel<T, N, CUBE>;
    constexpr int TC = job_cols(N), EW = 16 / (int)sizeof(C);   // element columns per tile, columns per element
    JobInvY<T, N, TC, NV, NS, typename GS::type> job;
    job.src = (const C *)r.zbuf;
    job.dst = (C *)r.ybuf;
    job.wplane = (long)a.kxp * N;
    job.wnf = job.wplane * a.Nz;
    job.kxp = a.kxp;
    job.geo = GS::make(a);
    return run_job<T, N, +1>(a, job, dim3((unsigned)(a.kxp / (TC * EW)), (unsigned)a.Nz), a.twY);
}

// mid_x: N = Nx
template <typename T, int N, int NV, int NS, int MINB>
static cudaError_t mid_xg_launch(const PassArgs &a, const RhsArgs &r, long wnf, int kxp)
{
    using C = Cx<T>;
    using PX = XPad<N, (int)sizeof(C)>;
    constexpr int ROWS = xg_rows<N>();
    constexpr size_t smem = (size_t)ROWS * (3 * NV + 2 * NS) * PX::BUF * sizeof(C);
    auto kern = k_mid_xg<T, N, NV, NS, MINB>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    const double npts = (double)N * a.Ny * a.Nz;
    const T scale2 = (T)(1.0 / (npts * npts));   // both c2r factors, applied to the product
    const long nrows = (long)a.Ny * a.Nz;        // a multiple of ROWS (<= 8): Ny, Nz are multiples of 4, Ny Nz of 16
    kern<<<(unsigned)(nrows / ROWS), ROWS * XSched<N>::TPR, smem, a.stream>>>((const C *)r.ybuf, (C *)r.zbuf,
                                                                               (const C *)a.twX, wnf, kxp, scale2, (T)a.kf[0]);
    return cudaGetLastError();
}

template <typename T, int N, int NV, int NS> static cudaError_t rhs_mid_x_n(const PassArgs &a, const RhsArgs &r)
{
    const long wnf = (long)a.kxp * a.Ny * a.Nz;
    // register budget: about 8 (fp64) / 16 (fp32) warps per SM for HD, half of that for MHD / Boussinesq
    constexpr int THREADS = xg_rows<N>() * XSched<N>::TPR;
    constexpr int M0 = (sizeof(T) == 8 ? 256 : 512) / (THREADS * (NV + NS));
    constexpr int MINB = M0 < 1 ? 1 : M0;
    return mid_xg_launch<T, N, NV, NS, MINB>(a, r, wnf, a.kxp);
}

template <typename T, int N, int NV, int NS, bool CUBE> static cudaError_t rhs_fwd_y_n(const PassArgs &a, const RhsArgs &r)
{
    using C = Cx<T>;
    using GS = GeomSel<T, N, CUBE>;
    constexpr int TC = job_cols(N), EW = 16 / (int)sizeof(C);   // element columns per tile, columns per element
    JobFwdY<T, N, TC, typename GS::type> job;
    job.buf = (C *)r.zbuf;
    job.wplane = (long)a.kxp * N;
    job.wnf = job.wplane * a.Nz;
    job.kxp = a.kxp;
    job.nfields = 3 * NV + NS;
    job.geo = GS::make(a);
    return run_job<T, N, -1>(a, job, dim3((unsigned)(a.kxp / (TC * EW)), (unsigned)a.Nz), a.twY);
}

template <typename T, int N, int NV, int NS, bool CUBE> static cudaError_t rhs_fwd_z_n(const PassArgs &a, const RhsArgs &r)
{
    using C = Cx<T>;
    using GS = GeomSel<T, N, CUBE>;
    constexpr int TC = fwdz_cols(N, (int)sizeof(C)), EW = 1;   // single columns in both precisions
    JobFwdZ<T, N, TC, NV, NS, typename GS::type> job;
    job.sdst = (C *)r.sdst;
    job.saux = (const C *)r.ssrc;
    job.sdiff = (T)r.sdiff;
    job.nbv = (T)r.nbv;
    for (int v = 0; v < NV; ++v) job.base[v] = (const C *)r.base[v];
    job.sbase = (const C *)r.sbase;
    job.cstep = (T)r.cstep;
    job.sparse = r.sparse_out;
    job.src = (const C *)r.zbuf;
    for (int v = 0; v < NV; ++v) {
        job.dst[v] = (C *)r.dst[v];
        job.aux[v] = (const C *)r.src[v];
        job.diff[v] = (T)r.diff[v];
    }
    job.plane = (long)a.ldk * a.Ny;
    job.nf = job.plane * N;
    job.wplane = (long)a.kxp * a.Ny;
    job.wnf = job.wplane * N;
    job.ldk = a.ldk;
    job.kxp = a.kxp;
    job.geo = GS::make(a);
    return run_job<T, N, -1>(a, job, dim3((unsigned)((job.plane + TC * EW - 1) / (TC * EW))), a.twZ);
}

// ---- Gross-Pitaevskii right-hand side ------------------------------------------------------------
// N = the length of the pass's own axis: Nz for pass 0 / 4, Ny for 1 / 3, Nx for 2 (see launch_gpe_pass)
template <typename T, int N, bool CUBE> static cudaError_t gpe_pass_n(const PassArgs &a, const GpeArgs &g, int pass)
{
    using C = Cx<T>;
    using GS = GeomSel<T, N, CUBE>;
    using G = typename GS::type;
    constexpr int TC = job_cols(N), EW = 16 / (int)sizeof(C);
    const int KXP = a.kxp;
    const long plane = (long)a.ldk * a.Ny, wplane = (long)KXP * a.Ny, wnf = wplane * a.Nz;
    const G geo = GS::make(a);
    if (pass == 0) {
        JobPlainInvZ<T, N, TC, 2, G> job;
        job.src = (const C *)g.psi; job.dst = (C *)g.zbuf;
        job.plane = plane; job.nf = plane * N; job.wplane = wplane; job.wnf = wnf; job.ldk = a.ldk; job.kxp = KXP;
        job.geo = geo;
        return run_job<T, N, +1>(a, job, dim3((unsigned)(KXP / (TC * EW)), (unsigned)a.Ny), a.twZ);
    }
    if (pass == 1 || pass == 3) {
        const dim3 ygrid((unsigned)(KXP / (TC * EW)), (unsigned)a.Nz);
        if (pass == 1) {
            JobPlainInvY<T, N, TC, G> job;
            job.buf = (C *)g.zbuf; job.wplane = wplane; job.wnf = wnf; job.kxp = KXP; job.nfields = 2; job.geo = geo;
            return run_job<T, N, +1>(a, job, ygrid, a.twY);
        }
        JobFwdY<T, N, TC, G> job;
        job.buf = (C *)g.obuf; job.wplane = wplane; job.wnf = wnf; job.kxp = KXP; job.nfields = 2; job.geo = geo;
        return run_job<T, N, -1>(a, job, ygrid, a.twY);
    }
    if (pass == 2) {
        using PX = XPad<N, (int)sizeof(C)>;
        constexpr int ROWS = xg_rows<N>(), THREADS = ROWS * XSched<N>::TPR;
        constexpr int M0 = (sizeof(T) == 8 ? 512 : 1024) / THREADS;
        constexpr int MINB = M0 < 1 ? 1 : M0;
        constexpr size_t smem = (size_t)ROWS * 2 * PX::BUF * sizeof(C);
        auto kern = k_mid_x_gpe<T, N, MINB>;
        cudaError_t e = set_smem(kern, smem);
        if (e != cudaSuccess) return e;
        kern<<<(unsigned)((long)a.Ny * a.Nz / ROWS), THREADS, smem, a.stream>>>(
            (const C *)g.zbuf, (C *)g.obuf, (const C *)a.twX, wnf, KXP, (T)(1.0 / ((double)N * a.Ny * a.Nz)));
        return cudaGetLastError();
    }
    constexpr int TCZ = fwdz_cols(N, (int)sizeof(C));
    JobGpeFwdZ<T, N, TCZ, G> job;
    job.src = (const C *)g.obuf; job.dst = (C *)g.dst; job.psi = (const C *)g.psi; job.base = (const C *)g.base;
    job.alpha = (T)g.alpha; job.beta = (T)g.beta; job.cstep = (T)g.cstep; job.sparse = g.sparse_out;
    job.plane = plane; job.nf = plane * N; job.wplane = wplane; job.wnf = wnf; job.ldk = a.ldk; job.kxp = KXP;
    job.geo = geo;
    return run_job<T, N, -1>(a, job, dim3((unsigned)((plane + TCZ - 1) / TCZ)), a.twZ);
}

template <typename T, bool CUBE> cudaError_t launch_gpe_pass_g(const PassArgs &a, const GpeArgs &g, int pass, int *launches)
{
    ++*launches;
    switch (pass == 2 ? a.N : (pass == 1 || pass == 3) ? a.Ny : a.Nz) {
#define X(n) case n: return gpe_pass_n<T, n, CUBE>(a, g, pass);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

#define PSFFT_RHS_LAUNCHER(name, axislen)                                                              \
    template <typename T, bool CUBE> cudaError_t launch_rhs_##name##_g(const PassArgs &a, const RhsArgs &r, int *launches) \
    {                                                                                                  \
        ++*launches;                                                                                   \
        switch (axislen) {                                                                             \
            PSFFT_FOR_EACH_N(PSFFT_RHS_CASE_##name)                                                    \
        }                                                                                              \
        return cudaErrorInvalidValue;                                                                  \
    }
#define PSFFT_RHS_CASE_inv_z(n) case n: return r.ns == 1 ? rhs_inv_z_n<T, n, 1, 1, CUBE>(a, r) : r.nv == 1 ? rhs_inv_z_n<T, n, 1, 0, CUBE>(a, r) : rhs_inv_z_n<T, n, 2, 0, CUBE>(a, r);
#define PSFFT_RHS_CASE_inv_y(n) case n: return r.ns == 1 ? rhs_inv_y_n<T, n, 1, 1, CUBE>(a, r) : r.nv == 1 ? rhs_inv_y_n<T, n, 1, 0, CUBE>(a, r) : rhs_inv_y_n<T, n, 2, 0, CUBE>(a, r);
#define PSFFT_RHS_CASE_fwd_y(n) case n: return r.ns == 1 ? rhs_fwd_y_n<T, n, 1, 1, CUBE>(a, r) : r.nv == 1 ? rhs_fwd_y_n<T, n, 1, 0, CUBE>(a, r) : rhs_fwd_y_n<T, n, 2, 0, CUBE>(a, r);
#define PSFFT_RHS_CASE_fwd_z(n) case n: return r.ns == 1 ? rhs_fwd_z_n<T, n, 1, 1, CUBE>(a, r) : r.nv == 1 ? rhs_fwd_z_n<T, n, 1, 0, CUBE>(a, r) : rhs_fwd_z_n<T, n, 2, 0, CUBE>(a, r);
PSFFT_RHS_LAUNCHER(inv_z, a.Nz)
PSFFT_RHS_LAUNCHER(inv_y, a.Ny)
PSFFT_RHS_LAUNCHER(fwd_y, a.Ny)
PSFFT_RHS_LAUNCHER(fwd_z, a.Nz)

template <typename T> cudaError_t launch_rhs_mid_x(const PassArgs &a, const RhsArgs &r, int *launches)
{
    ++*launches;
    switch (a.N) {
#define X(n) case n: return r.ns == 1 ? rhs_mid_x_n<T, n, 1, 1>(a, r) : r.nv == 1 ? rhs_mid_x_n<T, n, 1, 0>(a, r) : rhs_mid_x_n<T, n, 2, 0>(a, r);
        PSFFT_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
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
    switch (axis == 1 ? a.Ny : a.Nz) {
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

// Explicit instantiations, in three groups per dtype so that six translation units compile in parallel
// (psfft_f{32,64}_{fft,col,midx}.cu).
#define PSFFT_INSTANTIATE_FFT(T)                                                                                      \
    template cudaError_t launch_xpass_r2c<T>(const PassArgs &, const void *, void *, long, int *);                    \
    template cudaError_t launch_xpass_c2r<T>(const PassArgs &, const void *, void *, long, double, int *);            \
    template cudaError_t launch_cpass<T>(const PassArgs &, int, int, const void *, void *, int, int *);               \
    template cudaError_t launch_cpass_raw<T>(const PassArgs &, int, int, const void *, const void *, void *, long, long, \
                                             long, long, int *);                                                      \
    template cudaError_t launch_cpass_xdist<T>(const PassArgs &, bool, const void *, void *, const XDistArgs &, int,  \
                                               int *);                                                                \
    template cudaError_t launch_mask_curl<T>(const PassArgs &, const void *, void *, int *);                          \
    template cudaError_t launch_cross<T>(const PassArgs &, const void *, const void *, void *, int *);                \
    template cudaError_t launch_cross_mhd<T>(const PassArgs &, const void *, const void *, const void *, const void *, \
                                             void *, void *, int *);                                                  \
    template cudaError_t launch_finish<T>(const PassArgs &, int, const void *, const void *, void *, double, int *);
// column passes of the right-hand sides: CUBE = true (N^3 grid, 2 pi box: compile-time geometry) and false
// (any grid and box) in separate translation units
#define PSFFT_INSTANTIATE_COL(T, CUBE)                                                                                \
    template cudaError_t launch_rhs_inv_z_g<T, CUBE>(const PassArgs &, const RhsArgs &, int *);                       \
    template cudaError_t launch_rhs_inv_y_g<T, CUBE>(const PassArgs &, const RhsArgs &, int *);                       \
    template cudaError_t launch_rhs_fwd_y_g<T, CUBE>(const PassArgs &, const RhsArgs &, int *);                       \
    template cudaError_t launch_gpe_pass_g<T, CUBE>(const PassArgs &, const GpeArgs &, int, int *);
#define PSFFT_INSTANTIATE_FWDZ(T)                                                                                     \
    template cudaError_t launch_rhs_fwd_z_g<T, false>(const PassArgs &, const RhsArgs &, int *);
#define PSFFT_INSTANTIATE_MIDX(T)                                                                                     \
    template cudaError_t launch_rhs_mid_x<T>(const PassArgs &, const RhsArgs &, int *);

}  // namespace psfft
