// psfft_kernels.cuh -- the axis passes and pointwise kernels of libpsfft (sm_100a).
//
// Pass structure: a 3D transform is three passes, each reading and
// writing the field exactly once (the minimal-pass count for an out-of-cache 3D FFT):
//   x-pass  contiguous rows; real <-> half-complex, two rows per complex transform (psfft_xpass2.cuh;
//           PAPER.md:70 step 1, first half)
//   y-pass  columns with element stride ldk (PAPER.md:70 step 1, second half)
//   z-pass  columns with element stride ldk*N (PAPER.md:77 step 3)
// The paper's transpose (PAPER.md:76 step 2) is not a pass: the y/z kernels read tiles of
// [all rows of the axis] x [TC contiguous elements] and transform them in shared memory.
#pragma once
#include "psfft_core.cuh"

namespace psfft {

// ------------------------------------------------------------------------------------------
// strided column pass (y or z): complex FFT of length N along an axis with element stride
// `axis_stride`, for `inner` contiguous columns, repeated for blockIdx.y outer slices.
//   element (i, col, o) at  base[o * outer_stride + i * axis_stride + col]
// y-pass: axis_stride = ldk,   inner = ldk,   outer = N * fields, outer_stride = ldk*N
// z-pass: axis_stride = ldk*N, inner = ldk*N, outer = fields,     outer_stride = ldk*N*N
// In place (in == out) is allowed: a CTA reads all of its columns before it writes any.
// ------------------------------------------------------------------------------------------
// The tile is [N rows] x [TC elements Ex<T>]: one fp64 column or two adjacent fp32 columns per element
// (packed fp32x2 butterflies, psfft_core.cuh).  vec: every pair of columns is 16-byte aligned (z-pass: the
// strides are even) so that an fp32 element moves with one 16-byte access; otherwise (y-pass: odd pitch ldk)
// with two 8-byte ones.
template <typename T, int N, int DIR, int TC, int TPF, int MINB>
__global__ void __launch_bounds__(TC *TPF, MINB)
    k_cpass(const Cx<T> *in, Cx<T> *out, const Cx<T> *__restrict__ tw, long axis_stride, long inner,
            long outer_stride, bool vec)
{
    using C = Cx<T>;
    using E = Ex<T>;
    constexpr int EW = ElemWidth<E>::value;
    constexpr bool PAD = (TC * sizeof(E) < 128);
    using Map = ColMap<N, TC, PAD>;
    extern __shared__ __align__(16) unsigned char smraw[];
    E *sm = reinterpret_cast<E *>(smraw);

    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    const long col = ((long)blockIdx.x * TC + c) * EW;
    const bool valid = col < inner, valid1 = col + 1 < inner;   // valid1: second column of an fp32 pair
    const long base = (long)blockIdx.y * outer_stride + (valid ? col : 0);
    const C *src = in + base;
    C *dst = out + base;

    auto ld = [&](int i) -> E {
        if constexpr (EW == 1) {
            return valid ? ld_stream(src + i * axis_stride) : mk<T>(0, 0);
        } else {
            E x = ezero<E>();
            if (vec && valid1) {
                const float4 q = __ldcs(reinterpret_cast<const float4 *>(src + i * axis_stride));
                x.re = make_float2(q.x, q.z);
                x.im = make_float2(q.y, q.w);
            } else {
                if (valid) ecol_set(x, 0, ld_stream(src + i * axis_stride));
                if (valid1) ecol_set(x, 1, ld_stream(src + i * axis_stride + 1));
            }
            return x;
        }
    };
    auto st = [&](int i, E v) {
        if constexpr (EW == 1) {
            if (valid) st_stream(dst + i * axis_stride, v);
        } else {
            if (vec && valid1) {
                __stcs(reinterpret_cast<float4 *>(dst + i * axis_stride), make_float4(v.re.x, v.im.x, v.re.y, v.im.y));
            } else {
                if (valid) st_stream(dst + i * axis_stride, ecol(v, 0));
                if (valid1) st_stream(dst + i * axis_stride + 1, ecol(v, 1));
            }
        }
    };
    fft_stages<T, N, 1, DIR, TPF, false, false, false, Map>(sm, tw, c, t, ld, st);
}

// ------------------------------------------------------------------------------------------
// pointwise spectral / physical kernels (first, unfused RHS path)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int wavenumber(int idx, int N) { return idx < N / 2 ? idx : idx - N; }
// a9: 2/3-rule spherical truncation in integers
__device__ __forceinline__ bool keep_mode(int N, int kx, int ky, int kz)
{
    return 9ll * ((long long)kx * kx + (long long)ky * ky + (long long)kz * kz) < (long long)N * N;
}

// a7 (+ a9 on load): um = M u^, w^ = i k x um.  u: [3][nf]; out: [6][nf] = (um, w^)
template <typename T>
__global__ void k_mask_curl(const Cx<T> *__restrict__ u, Cx<T> *__restrict__ out, int N, int ldk, long nf)
{
    using C = Cx<T>;
    const long o = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nf) return;
    const int p = (int)(o % ldk);
    const long zy = o / ldk;
    const int ky = wavenumber((int)(zy % N), N), kz = wavenumber((int)(zy / N), N);
    C ux = mk<T>(0, 0), uy = ux, uz = ux;
    if (p <= N / 2 && keep_mode(N, p, ky, kz)) { ux = u[o]; uy = u[nf + o]; uz = u[2 * nf + o]; }
    const T kx = (T)p, fy = (T)ky, fz = (T)kz;
    out[o] = ux;
    out[nf + o] = uy;
    out[2 * nf + o] = uz;
    // i * (a + i b) = -b + i a
    C w;
    w = mk<T>(-(fy * uz.y - fz * uy.y), fy * uz.x - fz * uy.x); out[3 * nf + o] = w;
    w = mk<T>(-(fz * ux.y - kx * uz.y), fz * ux.x - kx * uz.x); out[4 * nf + o] = w;
    w = mk<T>(-(kx * uy.y - fy * ux.y), kx * uy.x - fy * ux.x); out[5 * nf + o] = w;
}

// a8: c = a x b (+ c2 = a2 x b2) pointwise; fields [3][n]
template <typename T>
__global__ void k_cross(const T *__restrict__ a, const T *__restrict__ b, T *__restrict__ c, long n)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const T ax = a[i], ay = a[n + i], az = a[2 * n + i];
    const T bx = b[i], by = b[n + i], bz = b[2 * n + i];
    c[i] = ay * bz - az * by;
    c[n + i] = az * bx - ax * bz;
    c[2 * n + i] = ax * by - ay * bx;
}

// MHD: m = u x w + j x b, e = u x b; inputs (u, b, w, j) each [3][n]; outputs m -> om, e -> oe
template <typename T>
__global__ void k_cross_mhd(const T *__restrict__ u, const T *__restrict__ b, const T *__restrict__ w,
                            const T *__restrict__ j, T *__restrict__ om, T *__restrict__ oe, long n)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const T ux = u[i], uy = u[n + i], uz = u[2 * n + i];
    const T bx = b[i], by = b[n + i], bz = b[2 * n + i];
    const T wx = w[i], wy = w[n + i], wz = w[2 * n + i];
    const T jx = j[i], jy = j[n + i], jz = j[2 * n + i];
    om[i] = (uy * wz - uz * wy) + (jy * bz - jz * by);
    om[n + i] = (uz * wx - ux * wz) + (jz * bx - jx * bz);
    om[2 * n + i] = (ux * wy - uy * wx) + (jx * by - jy * bx);
    oe[i] = uy * bz - uz * by;
    oe[n + i] = uz * bx - ux * bz;
    oe[2 * n + i] = ux * by - uy * bx;
}

// a9 + a10 (+ a11): out = M P f - nu |k|^2 M u^   (MODE 0), or
//                   out = M i k x f - nu |k|^2 M u^ (MODE 1, induction equation)
template <typename T, int MODE>
__global__ void k_finish(const Cx<T> *__restrict__ f, const Cx<T> *__restrict__ u, Cx<T> *__restrict__ out,
                         int N, int ldk, long nf, T nu)
{
    using C = Cx<T>;
    const long o = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nf) return;
    const int p = (int)(o % ldk);
    const long zy = o / ldk;
    const int ky = wavenumber((int)(zy % N), N), kz = wavenumber((int)(zy / N), N);
    const C zero = mk<T>(0, 0);
    if (p > N / 2 || !keep_mode(N, p, ky, kz)) {
        out[o] = zero; out[nf + o] = zero; out[2 * nf + o] = zero;
        return;
    }
    const T kx = (T)p, fy = (T)ky, fz = (T)kz;
    const T k2 = kx * kx + fy * fy + fz * fz;
    C fx = f[o], fyv = f[nf + o], fzv = f[2 * nf + o];
    C rx, ry, rz;
    if (MODE == 0) {
        rx = fx; ry = fyv; rz = fzv;
        if (k2 != (T)0) {
            const T inv = (T)1 / k2;
            const T dr = (kx * fx.x + fy * fyv.x + fz * fzv.x) * inv;
            const T di = (kx * fx.y + fy * fyv.y + fz * fzv.y) * inv;
            rx.x -= kx * dr; rx.y -= kx * di;
            ry.x -= fy * dr; ry.y -= fy * di;
            rz.x -= fz * dr; rz.y -= fz * di;
        }
    } else {
        rx = mk<T>(-(fy * fzv.y - fz * fyv.y), fy * fzv.x - fz * fyv.x);
        ry = mk<T>(-(fz * fx.y - kx * fzv.y), fz * fx.x - kx * fzv.x);
        rz = mk<T>(-(kx * fyv.y - fy * fx.y), kx * fyv.x - fy * fx.x);
    }
    if (nu != (T)0) {
        const T s = nu * k2;
        const C ux = u[o], uy = u[nf + o], uz = u[2 * nf + o];
        rx.x -= s * ux.x; rx.y -= s * ux.y;
        ry.x -= s * uy.x; ry.y -= s * uy.y;
        rz.x -= s * uz.x; rz.y -= s * uz.y;
    }
    out[o] = rx; out[nf + o] = ry; out[2 * nf + o] = rz;
}

}  // namespace psfft
