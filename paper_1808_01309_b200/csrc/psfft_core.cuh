// psfft_core.cuh -- device-side building blocks of libpsfft (sm_100a).
//
// Batched 1D FFTs as register-resident radix-2/3/4/8 butterflies with a shared-memory
// exchange between stages (Stockham autosort, decimation in time).  One "FFT group" of
// TPF = L / max_radix threads owns one transform of length L; the first stage reads its
// inputs straight from a caller-supplied loader (global memory), the last stage hands its
// outputs to a caller-supplied storer, so a transform costs (stages - 1) shared-memory round
// trips and exactly one global read and one global write per element.
//
// What is computed: Eq. 8 of arxiv 1808.01309 along one axis,
//   X[p] = sum_j x[j] exp(DIR * 2 pi i p j / L),   DIR = -1 forward, +1 backward,
// unnormalised in both directions.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace psfft {

// ------------------------------------------------------------------------------------------
// complex arithmetic on float2 / double2
// ------------------------------------------------------------------------------------------
template <typename T> struct CxOf;
template <> struct CxOf<float> { using type = float2; };
template <> struct CxOf<double> { using type = double2; };
template <typename T> using Cx = typename CxOf<T>::type;

template <typename T> __device__ __forceinline__ Cx<T> mk(T re, T im) { Cx<T> r; r.x = re; r.y = im; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b)
{
    C r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
template <typename C> __device__ __forceinline__ C cconj(C a) { a.y = -a.y; return a; }
// multiply by DIR * i  (DIR = -1: times -i, DIR = +1: times +i)
template <int DIR, typename C> __device__ __forceinline__ C mul_diri(C a)
{
    C r;
    if (DIR < 0) { r.x = a.y; r.y = -a.x; }
    else { r.x = -a.y; r.y = a.x; }
    return r;
}
template <typename C, typename T> __device__ __forceinline__ C cscale(C a, T s) { a.x *= s; a.y *= s; return a; }

// ------------------------------------------------------------------------------------------
// fp32 column passes: one thread carries TWO adjacent columns as a float2x2 -- two complex numbers
// (a, b) held component-wise, re = (re_a, re_b), im = (im_a, im_b) -- so that every complex add /
// multiply of a butterfly is issued once for both columns with Blackwell's packed fp32 instructions
// (FADD2 / FMUL2 / FFMA2, add/mul/fma.f32x2: sm_100+), twiddles entering as scalar broadcast operands.
// Ex<T> is the element a column pass works on: double2 (one column) or float2x2 (two columns), 16 bytes
// either way, so tile shapes, shared-memory maps and thread counts are the same for both precisions.
// ------------------------------------------------------------------------------------------
struct __align__(16) float2x2 { float2 re, im; };
template <typename T> struct ExOf;
template <> struct ExOf<float> { using type = float2x2; };
template <> struct ExOf<double> { using type = double2; };
template <typename T> using Ex = typename ExOf<T>::type;
template <typename E> struct ElemWidth { static constexpr int value = 1; };
template <> struct ElemWidth<float2x2> { static constexpr int value = 2; };

__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }
__device__ __forceinline__ float2 bc2(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2x2 cadd(float2x2 a, float2x2 b)
{
    float2x2 r;
    r.re = __fadd2_rn(a.re, b.re);
    r.im = __fadd2_rn(a.im, b.im);
    return r;
}
__device__ __forceinline__ float2x2 csub(float2x2 a, float2x2 b)
{
    float2x2 r;
    r.re = __fadd2_rn(a.re, neg2(b.re));
    r.im = __fadd2_rn(a.im, neg2(b.im));
    return r;
}
// both columns times the same complex scalar w
__device__ __forceinline__ float2x2 cmul(float2x2 a, float2 w)
{
    float2x2 r;
    r.re = __ffma2_rn(a.re, bc2(w.x), neg2(__fmul2_rn(a.im, bc2(w.y))));
    r.im = __ffma2_rn(a.re, bc2(w.y), __fmul2_rn(a.im, bc2(w.x)));
    return r;
}
template <int DIR> __device__ __forceinline__ float2x2 mul_diri(float2x2 a)
{
    float2x2 r;
    if (DIR < 0) { r.re = a.im; r.im = neg2(a.re); }
    else { r.re = neg2(a.im); r.im = a.re; }
    return r;
}
__device__ __forceinline__ float2x2 cscale(float2x2 a, float s)
{
    a.re = __fmul2_rn(a.re, bc2(s));
    a.im = __fmul2_rn(a.im, bc2(s));
    return a;
}
template <typename E> __device__ __forceinline__ E ezero();
template <> __device__ __forceinline__ double2 ezero<double2>() { return make_double2(0.0, 0.0); }
template <> __device__ __forceinline__ float2 ezero<float2>() { return make_float2(0.f, 0.f); }
template <> __device__ __forceinline__ float2x2 ezero<float2x2>()
{
    float2x2 r;
    r.re = make_float2(0.f, 0.f);
    r.im = r.re;
    return r;
}
// column j of an element / set column j
__device__ __forceinline__ double2 ecol(double2 e, int) { return e; }
__device__ __forceinline__ float2 ecol(float2 e, int) { return e; }
__device__ __forceinline__ float2 ecol(float2x2 e, int j) { return j == 0 ? make_float2(e.re.x, e.im.x) : make_float2(e.re.y, e.im.y); }
__device__ __forceinline__ void ecol_set(double2 &e, int, double2 v) { e = v; }
__device__ __forceinline__ void ecol_set(float2 &e, int, float2 v) { e = v; }
__device__ __forceinline__ void ecol_set(float2x2 &e, int j, float2 v)
{
    if (j == 0) { e.re.x = v.x; e.im.x = v.y; }
    else { e.re.y = v.x; e.im.y = v.y; }
}
// v (1 + DIR i)/sqrt 2  and  v (-1 + DIR i)/sqrt 2  (the odd eighth roots of a radix-8 butterfly)
template <int DIR, typename T, typename C> __device__ __forceinline__ C mul_w8_1(C v)
{
    const T h = (T)0.70710678118654752440084436210485;
    return DIR < 0 ? mk<T>((v.x + v.y) * h, (v.y - v.x) * h) : mk<T>((v.x - v.y) * h, (v.x + v.y) * h);
}
template <int DIR, typename T, typename C> __device__ __forceinline__ C mul_w8_3(C v)
{
    const T h = (T)0.70710678118654752440084436210485;
    return DIR < 0 ? mk<T>((v.y - v.x) * h, -(v.x + v.y) * h) : mk<T>(-(v.x + v.y) * h, (v.x - v.y) * h);
}
template <int DIR, typename T> __device__ __forceinline__ float2x2 mul_w8_1(float2x2 v)
{
    const float h = 0.70710678118654752440f;
    float2x2 r;
    if (DIR < 0) { r.re = __fmul2_rn(__fadd2_rn(v.re, v.im), bc2(h)); r.im = __fmul2_rn(__fadd2_rn(v.im, neg2(v.re)), bc2(h)); }
    else { r.re = __fmul2_rn(__fadd2_rn(v.re, neg2(v.im)), bc2(h)); r.im = __fmul2_rn(__fadd2_rn(v.re, v.im), bc2(h)); }
    return r;
}
template <int DIR, typename T> __device__ __forceinline__ float2x2 mul_w8_3(float2x2 v)
{
    const float h = 0.70710678118654752440f;
    float2x2 r;
    if (DIR < 0) { r.re = __fmul2_rn(__fadd2_rn(v.im, neg2(v.re)), bc2(h)); r.im = __fmul2_rn(__fadd2_rn(v.re, v.im), bc2(-h)); }
    else { r.re = __fmul2_rn(__fadd2_rn(v.re, v.im), bc2(-h)); r.im = __fmul2_rn(__fadd2_rn(v.re, neg2(v.im)), bc2(h)); }
    return r;
}

// ------------------------------------------------------------------------------------------
// compile-time radix schedule
// ------------------------------------------------------------------------------------------
__host__ __device__ constexpr int pow2_part(int n) { int p = 1; while (n % 2 == 0) { n /= 2; p *= 2; } return p; }
// radix of the stage that starts with `rem` = L / Ns still to be factored
__host__ __device__ constexpr int pick_radix(int rem)
{
    int p2 = pow2_part(rem);
    return p2 == 16 ? 4 : p2 >= 8 ? 8 : p2 == 4 ? 4 : p2 == 2 ? 2 : 3;
}
__host__ __device__ constexpr int max_radix(int L)
{
    int m = 1, rem = L;
    while (rem > 1) { int r = pick_radix(rem); m = r > m ? r : m; rem /= r; }
    return m;
}
__host__ __device__ constexpr int num_stages(int L)
{
    int n = 0, rem = L;
    while (rem > 1) { rem /= pick_radix(rem); ++n; }
    return n;
}
// threads per transform
__host__ __device__ constexpr int threads_per_fft(int L) { return L / max_radix(L); }
__host__ __device__ constexpr bool supported_len(int L)
{
    int rem = L / pow2_part(L);
    return L >= 4 && (rem == 1 || rem == 3);
}

// column passes: 16 elements per thread for N >= 128 (two radix-8 butterflies in flight), and TC
// contiguous columns per CTA: 128-byte tile rows, capped so a tile stays within 64 KB, widened for
// small N until a CTA has at least 128 threads.  (Measured on B200, 512^3 fp64: 64-byte rows run
// the z-pass at 3.5 TB/s, 128-byte rows at 5.4 TB/s; profiles/r1a_summary.md.)
__host__ __device__ constexpr int cpass_tpf(int N) { return N >= 128 ? N / 16 : threads_per_fft(N); }
// `cap`: largest tile in bytes.  64 KB (two tiles per SM) is the rule; at N = 1024 a 64 KB tile would have
// 64-byte rows, and one 128 KB tile per SM with 128-byte rows is faster (measured, 1024^3 fp32 MHD: fwd_z
// 15.1 -> 10.8 ms, fwd_y 7.7 -> 7.0 ms, inv_y unchanged); at N = 768 only the z-pass with the epilogue gains.
__host__ __device__ constexpr int cpass_cols_cap(int N, int csize, long cap)
{
    int tc = 128 / csize;
    while (tc > 1 && (long)N * tc * csize > cap) tc /= 2;
    while (tc * cpass_tpf(N) < 128 && (long)N * tc * 2 * csize <= 65536) tc *= 2;
    return tc;
}
__host__ __device__ constexpr int cpass_cols(int N, int csize) { return cpass_cols_cap(N, csize, N >= 1024 ? 131072 : 65536); }
// fwd_z (the pass that also writes the dense output) takes the big tile from N = 768 on
__host__ __device__ constexpr int fwdz_cols(int N, int csize) { return cpass_cols_cap(N, csize, N >= 768 ? 131072 : 65536); }

// number of kx with 9 kx^2 < N^2 (2/3-rule), and the compact row pitch of the RHS workspace fields:
// kx_count rounded up to whole tiles of TC columns
__host__ __device__ constexpr int kx_count(int N) { return (N - 1) / 3 + 1; }
__host__ __device__ constexpr int kx_pitch(int N, int TC) { return (kx_count(N) + TC - 1) / TC * TC; }

// RHS column passes work on 16-byte elements Ex<T> (one fp64 column or two packed fp32 columns, below):
// tile = [N rows] x [job_cols(N) elements]; the workspace row pitch is a whole number of tiles.
__host__ __device__ constexpr int job_cols(int N) { return cpass_cols(N, 16); }
__host__ __device__ constexpr int rhs_pitch(int N, int csize) { return kx_pitch(N, job_cols(N) * (16 / csize)); }

// Per-stage twiddle tables.  Stage with earlier radix product Ns (> 1) and radix R needs
// w_{Ns R}^{r k}, k in [0, Ns), r in [1, R).  They are stored as [r-1][k] (k contiguous, so the
// lanes of a warp -- consecutive k -- read consecutive 16-byte entries), stage after stage.
__host__ __device__ constexpr int tw_offset(int L, int Ns_target)
{
    int off = 0, Ns = 1;
    while (Ns < Ns_target) {
        int r = pick_radix(L / Ns);
        if (Ns > 1) off += (r - 1) * Ns;
        Ns *= r;
    }
    return off;
}
__host__ __device__ constexpr int tw_size(int L) { return tw_offset(L, L); }

// ------------------------------------------------------------------------------------------
// in-register butterflies: v[0..R) <- DFT_R(v), natural order out
// ------------------------------------------------------------------------------------------
template <int DIR, typename C> __device__ __forceinline__ void bfly2(C &a, C &b)
{
    C t = csub(a, b);
    a = cadd(a, b);
    b = t;
}

template <int DIR, typename C> __device__ __forceinline__ void bfly4(C &v0, C &v1, C &v2, C &v3)
{
    C t0 = cadd(v0, v2), t1 = csub(v0, v2), t2 = cadd(v1, v3), t3 = mul_diri<DIR>(csub(v1, v3));
    v0 = cadd(t0, t2);
    v2 = csub(t0, t2);
    v1 = cadd(t1, t3);
    v3 = csub(t1, t3);
}

template <int DIR, typename T, typename C> __device__ __forceinline__ void bfly3(C &v0, C &v1, C &v2)
{
    const T s = (T)0.86602540378443864676372317075294;  // sqrt(3)/2
    C t = cadd(v1, v2);
    C m = csub(v0, cscale(t, (T)0.5));
    C d = mul_diri<DIR>(cscale(csub(v1, v2), s));
    v0 = cadd(v0, t);
    v1 = cadd(m, d);
    v2 = csub(m, d);
}

template <int DIR, typename T, typename C> __device__ __forceinline__ void bfly8(C *v)
{
    bfly4<DIR>(v[0], v[2], v[4], v[6]);
    bfly4<DIR>(v[1], v[3], v[5], v[7]);
    // w8^1 = (1 + DIR i)/sqrt2, w8^2 = DIR i, w8^3 = (-1 + DIR i)/sqrt2
    const C o1 = mul_w8_1<DIR, T>(v[3]), o3 = mul_w8_3<DIR, T>(v[7]);
    C o2 = mul_diri<DIR>(v[5]);
    C e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
    v[0] = cadd(e0, o0);
    v[4] = csub(e0, o0);
    v[1] = cadd(e1, o1);
    v[5] = csub(e1, o1);
    v[2] = cadd(e2, o2);
    v[6] = csub(e2, o2);
    v[3] = cadd(e3, o3);
    v[7] = csub(e3, o3);
}

template <int R, int DIR, typename T, typename C> __device__ __forceinline__ void bfly(C *v)
{
    if (R == 2) bfly2<DIR>(v[0], v[1]);
    else if (R == 3) bfly3<DIR, T>(v[0], v[1], v[2]);
    else if (R == 4) bfly4<DIR>(v[0], v[1], v[2], v[3]);
    else bfly8<DIR, T>(v);
}

// ------------------------------------------------------------------------------------------
// read-only table load (roots of unity): w_N^m = exp(-2 pi i m / N), m in [0, N)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 ldg_c(const double2 *p) { return __ldg(p); }
__device__ __forceinline__ float2 ldg_c(const float2 *p) { return __ldg(p); }

// streaming (touch-once) global access for field data: keeps the twiddle tables resident in L1
__device__ __forceinline__ double2 ld_stream(const double2 *p) { return __ldcs(p); }
__device__ __forceinline__ float2 ld_stream(const float2 *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(double2 *p, double2 v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream(float2 *p, float2 v) { __stcs(p, v); }

template <int DIR, typename C> __device__ __forceinline__ C root_of(const C *__restrict__ tab, int m)
{
    C w = ldg_c(tab + m);
    if (DIR > 0) w.y = -w.y;
    return w;
}

// ------------------------------------------------------------------------------------------
// shared-memory index maps.  Elements are whole complex numbers.
//   ColMap : tile [row][TC columns]; thread column c, rows along the FFT axis.
//            One padding row of TC elements after every 8 rows when a row is 64 B, so that
//            the two rows of a 128 B wavefront never share banks in the stride-8 writes.
// ------------------------------------------------------------------------------------------
template <int L, int TC, bool PAD> struct ColMap {
    static constexpr int rows = PAD ? L + (L >> 3) : L;
    static constexpr int size = rows * TC;
    __device__ __forceinline__ static int at(int i, int c) { return (PAD ? i + (i >> 3) : i) * TC + c; }
};

// ------------------------------------------------------------------------------------------
// group-level synchronisation between stages
// ------------------------------------------------------------------------------------------
template <bool WARP> __device__ __forceinline__ void group_sync()
{
    if (WARP) __syncwarp();
    else __syncthreads();
}

// ------------------------------------------------------------------------------------------
// One Stockham stage of radix R on a length-L transform whose earlier stages have radix
// product Ns.  Butterfly b in [0, L/R): k = b mod Ns,
//     v[r] = src[b + r L/R] * w_{Ns R}^{r k},  V = DFT_R(v),  dst[(b/Ns) Ns R + k + r Ns] = V[r].
// src is the loader (SRC_SMEM = false) or shared memory; dst likewise.
// tw = per-stage twiddle tables of length L (layout: tw_offset above), forward sign.
// ------------------------------------------------------------------------------------------
// ld(i) must be a bare (possibly predicated) load so that all loads of a stage issue back to
// back; px(i, x) is applied to the loaded values afterwards (masking factors, i k multipliers).
struct NoPost {
    template <typename C> __device__ __forceinline__ C operator()(int, C x) const { return x; }
};

// E is the element the transform works on: Cx<T> (one column per thread) or float2x2 (two fp32 columns per
// thread, packed arithmetic); the twiddles are always scalar complex numbers Cx<T>.
template <typename T, int L, int Ns, int DIR, int TPF, bool SRC_SMEM, bool DST_SMEM, bool WARP, class Map,
          class LD, class ST, class PX, typename E>
__device__ __forceinline__ void fft_stages(E *sm, const Cx<T> *__restrict__ tw, int c, int t, LD &ld, ST &st,
                                           PX &px)
{
    using C = Cx<T>;
    constexpr int R = pick_radix(L / Ns);
    constexpr bool first = (Ns == 1), last = (Ns * R == L);
    constexpr int NB = L / R;
    constexpr int ITER = (NB + TPF - 1) / TPF;
    constexpr bool ragged = (NB % TPF) != 0;
    constexpr bool from_smem = !first || SRC_SMEM;
    constexpr bool to_smem = !last || DST_SMEM;

    E v[ITER][R];
#pragma unroll
    for (int it = 0; it < ITER; ++it) {
        const int b = t + it * TPF;
        if (!ragged || b < NB) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (from_smem) v[it][r] = sm[Map::at(b + r * NB, c)];
                else v[it][r] = ld(b + r * NB);
            }
        }
    }
#pragma unroll
    for (int it = 0; it < ITER; ++it) {
        const int b = t + it * TPF;
        if (!ragged || b < NB) {
            if (!from_smem) {
#pragma unroll
                for (int r = 0; r < R; ++r) v[it][r] = px(b + r * NB, v[it][r]);
            }
            if (Ns > 1) {
                const C *__restrict__ ts = tw + tw_offset(L, Ns) + (b % Ns);
                if (R == 8) {  // three loads, the other four by one or two multiplications
                    const C w1 = root_of<DIR>(ts, 0), w2 = root_of<DIR>(ts, Ns), w4 = root_of<DIR>(ts, 3 * Ns);
                    const C w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4);
                    const C w7 = cmul(w3, w4);
                    v[it][1] = cmul(v[it][1], w1); v[it][2] = cmul(v[it][2], w2); v[it][3] = cmul(v[it][3], w3);
                    v[it][4] = cmul(v[it][4], w4); v[it][5] = cmul(v[it][5], w5); v[it][6] = cmul(v[it][6], w6);
                    v[it][7] = cmul(v[it][7], w7);
                } else {
#pragma unroll
                    for (int r = 1; r < R; ++r) v[it][r] = cmul(v[it][r], root_of<DIR>(ts, (r - 1) * Ns));
                }
            }
            bfly<R, DIR, T>(v[it]);
        }
    }
    if (from_smem && to_smem) group_sync<WARP>();  // in place: every read done before any write
#pragma unroll
    for (int it = 0; it < ITER; ++it) {
        const int b = t + it * TPF;
        if (!ragged || b < NB) {
            const int j0 = (b / Ns) * Ns * R + (b % Ns);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (to_smem) sm[Map::at(j0 + r * Ns, c)] = v[it][r];
                else st(j0 + r * Ns, v[it][r]);
            }
        }
    }
    if (to_smem) group_sync<WARP>();
    if constexpr (!last)
        fft_stages<T, L, Ns * R, DIR, TPF, SRC_SMEM, DST_SMEM, WARP, Map, LD, ST, PX, E>(sm, tw, c, t, ld, st, px);
}

template <typename T, int L, int Ns, int DIR, int TPF, bool SRC_SMEM, bool DST_SMEM, bool WARP, class Map,
          class LD, class ST, typename E>
__device__ __forceinline__ void fft_stages(E *sm, const Cx<T> *__restrict__ tw, int c, int t, LD &ld, ST &st)
{
    NoPost px;
    fft_stages<T, L, Ns, DIR, TPF, SRC_SMEM, DST_SMEM, WARP, Map, LD, ST, NoPost, E>(sm, tw, c, t, ld, st, px);
}

}  // namespace psfft
