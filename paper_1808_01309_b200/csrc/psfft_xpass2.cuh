// psfft_xpass2.cuh -- the x-passes of the plain 3D transforms as "two for one" complex transforms.
//
// a1 / a6 of SURVEY.md §8(a) (PAPER.md:70 step 1, first half): N reals <-> N/2 + 1 complex per
// row.  Two adjacent rows a, b are packed into one complex row z = a + i b, transformed with ONE complex
// length-N transform in the symmetric radix schedule of psfft_midxg.cuh (XSched / XPad / twX), and
// separated with the Hermitian split
//     A[k] = (Z[k] + conj Z[N-k]) / 2,      B[k] = -i (Z[k] - conj Z[N-k]) / 2,      k = 0 .. N/2
// (inverse: Z[k] = A[k] + i B[k], Z[N-k] = conj A[k] + i conj B[k], imaginary parts of the k = 0 and k = N/2
// entries ignored as the c2r definition O4 says).  Against the half-length formulation (k_xpass_r2c /
// k_xpass_c2r: a length-N/2 transform per row plus a split / merge step staged through shared memory) this
// moves a third less through shared memory per row and the exchanges are conflict-free (XPad), so the pass
// is bound by HBM instead of the L1 data pipe (profiles/r1c_summary.md: 96 % L1 pipe for the half-length
// kernel).  N / RM threads per row PAIR.
#pragma once
#include "psfft_midxg.cuh"

namespace psfft {

template <typename T, int N, int MINB>
__global__ void __launch_bounds__(xg_rows<N>() * XSched<N>::TPR, MINB)
    k_xpass2_r2c(const T *__restrict__ in, Cx<T> *__restrict__ out, const Cx<T> *__restrict__ twx, long npairs, int ldk)
{
    using C = Cx<T>;
    using X = XSched<N>;
    using P = XPad<N, (int)sizeof(C)>;
    constexpr int RM = X::RM, TPR = X::TPR, S = X::S, BUF = P::BUF, H = RM / 2;
    extern __shared__ __align__(16) unsigned char smraw[];

    const int g = threadIdx.x / TPR, b = threadIdx.x % TPR;
    C *sm = reinterpret_cast<C *>(smraw) + g * (2 * BUF);   // buffer 0: the transform, buffer 1: split exchange
    long pair = (long)blockIdx.x * xg_rows<N>() + g;
    const bool valid = pair < npairs;
    if (!valid) pair = npairs - 1;   // keep the CTA in lock step; results discarded
    const T *xa = in + 2 * pair * N, *xb = xa + N;

    // ---- first stage from global memory: z = a + i b at x = b + TPR r; outputs into the slots "just read" ----
    C F[RM];
#pragma unroll
    for (int r = 0; r < RM; ++r) F[r] = mk<T>(__ldcs(xa + b + TPR * r), __ldcs(xb + b + TPR * r));
    bfly<RM, -1, T>(F);
#pragma unroll
    for (int r = 0; r < RM; ++r) sm[P::pad(b + TPR * r)] = F[r];
    __syncthreads();
    xg_middle_stages<T, N, 1, -1, 1>(sm, twx, b);
    {
        const C *ts = twx + X::tw_off(S - 1) + b;
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            const int e = b + TPR * r;
            F[r] = sm[P::pad(S == 2 ? e / RM + TPR * (e % RM) : e)];
        }
        twiddle_r<RM, -1, T>(F, ts, TPR);
        bfly<RM, -1, T>(F);   // F[r] = Z[b + TPR r]
    }
    // ---- split: thread TPR - b holds Z[N - k] at r' = RM - 1 - r (thread 0 pairs with itself at r' = RM - r) ----
    C *ex = sm + BUF;
#pragma unroll
    for (int e = 0; e < H; ++e) ex[e * TPR + b] = F[H + e];
    __syncthreads();
    if (!valid) return;
    const int bp = (TPR - b) % TPR;
    C *oa = out + 2 * pair * ldk, *ob = oa + ldk;
#pragma unroll
    for (int r = 0; r < H; ++r) {
        const int k = b + TPR * r;
        const int e = (b == 0) ? (r == 0 ? 0 : H - r) : H - 1 - r;
        C c = ex[e * TPR + bp];
        if (b == 0 && r == 0) c = F[0];
        const C a = F[r];
        const C s = mk<T>((T)0.5 * (a.x + c.x), (T)0.5 * (a.y - c.y));   // (a + conj c)/2
        const C d = mk<T>((T)0.5 * (a.x - c.x), (T)0.5 * (a.y + c.y));   // (a - conj c)/2
        st_stream(oa + k, s);
        st_stream(ob + k, mk<T>(d.y, -d.x));                             // -i d
    }
    if (b == 0) {   // k = N/2 pairs with itself: A = Re Z, B = Im Z
        st_stream(oa + N / 2, mk<T>(F[H].x, (T)0));
        st_stream(ob + N / 2, mk<T>(F[H].y, (T)0));
    }
}

template <typename T, int N, int MINB>
__global__ void __launch_bounds__(xg_rows<N>() * XSched<N>::TPR, MINB)
    k_xpass2_c2r(const Cx<T> *__restrict__ in, T *__restrict__ out, const Cx<T> *__restrict__ twx, long npairs, int ldk,
                 T scale)
{
    using C = Cx<T>;
    using X = XSched<N>;
    using P = XPad<N, (int)sizeof(C)>;
    constexpr int RM = X::RM, TPR = X::TPR, S = X::S, BUF = P::BUF, H = RM / 2;
    extern __shared__ __align__(16) unsigned char smraw[];

    const int g = threadIdx.x / TPR, b = threadIdx.x % TPR;
    C *sm = reinterpret_cast<C *>(smraw) + g * BUF;
    long pair = (long)blockIdx.x * xg_rows<N>() + g;
    const bool valid = pair < npairs;
    if (!valid) pair = npairs - 1;
    const C *ya = in + 2 * pair * ldk, *yb = ya + ldk;

    // ---- first stage: Z[b + TPR r] from the two half spectra ----
    C v[RM];
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        const int e = b + TPR * r;
        const bool mirror = r > H || (r == H && b > 0);        // e > N/2
        const int k = mirror ? N - e : e;
        const C pa = ld_stream(ya + k), pb = ld_stream(yb + k);
        if (mirror) v[r] = mk<T>(pa.x + pb.y, pb.x - pa.y);    // conj A + i conj B
        else if ((r == 0 || r == H) && b == 0) v[r] = mk<T>(pa.x, pb.x);   // k = 0, N/2: imaginary parts ignored
        else v[r] = mk<T>(pa.x - pb.y, pa.y + pb.x);           // A + i B
    }
    bfly<RM, +1, T>(v);
#pragma unroll
    for (int r = 0; r < RM; ++r) sm[P::pad(RM * b + r)] = v[r];
    __syncthreads();
    xg_middle_stages<T, N, 1, +1, 1>(sm, twx, b);
    {
        const C *ts = twx + X::tw_off(S - 1) + b;
#pragma unroll
        for (int r = 0; r < RM; ++r) v[r] = sm[P::pad(b + TPR * r)];
        twiddle_r<RM, +1, T>(v, ts, TPR);
        bfly<RM, +1, T>(v);   // v[r] = a + i b at x = b + TPR r
    }
    if (!valid) return;
    T *xa = out + 2 * pair * N, *xb = xa + N;
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        __stcs(xa + b + TPR * r, v[r].x * scale);
        __stcs(xb + b + TPR * r, v[r].y * scale);
    }
}

}  // namespace psfft
