// psfft_midxg.cuh -- RHS pass 3 ("mid_x") for every supported N: the inverse x-transforms, the pointwise
// products (a8) and the forward x-transforms of one (z, y) row as complex length-N transforms of PAIRS of
// real fields ("two for one"), with the products formed in registers between the last inverse and the
// first forward stage.
//
// What is computed per row:
//   u_c = c2r U_c, w_x = c2r W_x, w_y = c2r (P - i kx U_z), w_z = c2r (i kx U_y - D)   (six per vector field)
//   n = u x w                                     (MHD: m = u x w + j x b, e = u x b)
//   n^_c = r2c n_c, kept for kx < N/3
//
// Packing.  For Hermitian rows A, B (real a, b) the complex row Z[k] = A[k] + i B[k] (0 <= k < N/2),
// Z[N-k] = conj A[k] + i conj B[k] has the inverse transform z = a + i b: three complex transforms
// give (u_x, w_x), (u_y, w_y), (u_z, w_z) with no merge step, and a thread that finishes a
// last-stage butterfly of all three holds u and w at its RM grid points x = b + (N/RM) r.  The
// products are formed in registers and go straight into the first stage of the forward
// transforms F1 = n_x + i n_y, F2 = n_z (MHD: m_x + i m_y, m_z + i e_x, e_y + i e_z), whose output
// is split as n^_x[k] = (F1[k] + conj F1[N-k])/2, n^_y[k] = -i (F1[k] - conj F1[N-k])/2.
// Boussinesq (NS = 1): two more inverse transforms (g_x + i g_y, g_z) for grad theta and F2 = n_z + i s,
// s = u . grad theta (Eq. 2).
//
// Shared memory: one buffer of N complex per inverse transform, padded so that the exchanges are (nearly)
// conflict-free (XPad).  The first forward stage writes into the slots its thread has just read, so the
// inverse -> product -> forward hand-over needs no barrier and no extra buffer.  At N = 512 (8 8 8): two
// exchanges per transform, 20 N complex shared-memory accesses per HD row.
//
// Schedule.  The hand-over in registers needs the LAST inverse stage and the FIRST forward stage to have
// the same radix RM and the same butterfly -> thread map: a last-stage Stockham butterfly b of radix RM
// produces the points x = b + (N/RM) r, which are exactly the inputs of first-stage butterfly b.  So the
// length-N transforms here use the SYMMETRIC radix schedule  RM, (factors of N / RM^2), RM  with
// RM = 8 if 64 | N, 4 if 16 | N, else 2:
//     8: 2 2 2    12: 2 3 2    16: 4 4      24: 2 2 3 2   32: 4 2 4     48: 4 3 4     64: 8 8
//    96: 4 2 3 4 128: 8 2 8   192: 8 3 8   256: 8 4 8    384: 8 2 3 8  512: 8 8 8    768: 8 4 3 8
//  1024: 8 4 4 8   2048: 8 8 4 8
// N / RM threads own one row; a thread does one radix-RM butterfly in the outer stages and RM / R (rounded
// up, predicated) radix-R butterflies in a middle stage.  The twiddle tables of this schedule are a third
// table of the plan (PassArgs::twX), laid out per stage as [r - 1][k] like the others.
#pragma once
#include "psfft_rhs.cuh"

namespace psfft {

template <int N> struct XSched {
    static constexpr int RM = (N % 64 == 0) ? 8 : (N % 16 == 0) ? 4 : 2;
    static constexpr int TPR = N / RM;   // threads per row = butterflies of an outer stage
    __host__ __device__ static constexpr int mid_radix(int m)
    {
        return (m % 8 == 0 && m != 16) ? 8 : (m % 4 == 0) ? 4 : (m % 2 == 0) ? 2 : 3;
    }
    __host__ __device__ static constexpr int stages()
    {
        int n = 2, m = N / (RM * RM);
        while (m > 1) { m /= mid_radix(m); ++n; }
        return n;
    }
    static constexpr int S = stages();
    __host__ __device__ static constexpr int radix(int s)
    {
        if (s == 0 || s == S - 1) return RM;
        int m = N / (RM * RM), r = 1;
        for (int i = 1; i <= s; ++i) { r = mid_radix(m); m /= r; }
        return r;
    }
    // product of the radices of the stages before s
    __host__ __device__ static constexpr int ns(int s)
    {
        int p = 1;
        for (int i = 0; i < s; ++i) p *= radix(i);
        return p;
    }
    // entries of the stage tables before stage s (stage 0 has none)
    __host__ __device__ static constexpr int tw_off(int s)
    {
        int off = 0;
        for (int i = 1; i < s; ++i) off += (radix(i) - 1) * ns(i);
        return off;
    }
    static constexpr int tw_size = tw_off(S);
};

// Shared-memory slot of element i of one transform buffer: i + X (i >> A) + Y (i >> B) + Z (i >> C), found by
// exhaustive search over this family for the fewest bank conflicts summed over every exchange of the
// inverse and forward transforms (16-byte elements: per quarter warp; 8-byte elements: per half warp).
// To regenerate a row of the table: for every (a, x, b, y, c, z) with a < b < c <= 9 and x, y, z in 0..4, walk the
// exchanges of XSched<N> (first-stage writes RM b + r; middle-stage reads bb + r NBF / writes j0 + r Ns, through the
// slot map e / RM + TPR (e % RM) where SLOT applies; last-stage reads b + TPR r) for the lanes of each quarter (half)
// warp, count the lanes beyond the first that fall into an occupied 16-byte (8-byte) bank group, and keep the
// minimum, ties to the smaller buffer pad(N - 1) + 1.  The search takes seconds in plain Python.
template <int N, int CSIZE> struct XPad {
    struct P { int a, x, b, y, c, z; };
    __host__ __device__ static constexpr P params()
    {
        if (CSIZE == 16) {
            switch (N) {
                case 2048: return {3, 1, 8, 1, 11, 0};
                case 1024: return {3, 1, 7, 1, 9, 0};
                case 768: return {3, 1, 6, 1, 8, 4};
                case 384: return {3, 1, 6, 3, 7, 2};
                case 192: return {3, 1, 6, 0, 9, 0};
                default: return {3, 1, 6, 1, 9, 0};   // 512, 256, 128 (and the small sizes)
            }
        } else {
            switch (N) {
                case 1024: return {4, 2, 5, 4, 6, 1};
                case 192: return {2, 4, 3, 4, 6, 1};
                default: return {4, 1, 6, 4, 7, 2};   // the small sizes
            }
        }
    }
    // 8-byte elements (fp32), 128 <= N <= 768: no additive padding of the family above removes the conflicts of the
    // stride-8 first-stage writes (17 % of mid_x's shared-memory wavefronts, profiles/r2_summary.md).  An XOR map does:
    //     slot(i) = i ^ ((i >> s1) & m1) ^ ((i >> s2) & m2),
    // each term feeding index bits >= 4 into the low four bits (so the map is a bijection of every aligned block of 16
    // slots, the buffer needs no padding, BUF = N), found by the same exhaustive walk of the exchanges, per half warp:
    // zero conflicts at every size listed.  Measured on B200, fp32 mid_x: 512^3 1.129 -> 1.098 ms, 768^3 5.09 -> 4.87 ms.
    // N = 1024 needs three terms ({5, 15}, {2, 12}, {6, 14}) for zero conflicts; the MHD kernel then takes 173 instead
    // of 167 registers, loses its third CTA per SM and runs 23.3 -> 27.3 ms, so 1024 keeps its additive padding (8 %
    // conflict wavefronts).
    struct X3 { int s1, m1, s2, m2, s3, m3; };
    __host__ __device__ static constexpr bool use_xor()
    {
        return CSIZE == 8 && (N == 128 || N == 256 || N == 384 || N == 512 || N == 768);
    }
    __host__ __device__ static constexpr X3 xor_params()
    {
        switch (N) {
            case 768: case 256: return {4, 15, 2, 8, 0, 0};
            case 512: return {3, 14, 6, 7, 0, 0};
            default: return {4, 7, 1, 8, 0, 0};       // 384, 128
        }
    }
    __host__ __device__ static constexpr int pad(int i)
    {
        if constexpr (use_xor()) {
            constexpr X3 q = xor_params();
            return i ^ ((i >> q.s1) & q.m1) ^ ((i >> q.s2) & q.m2) ^ ((i >> q.s3) & q.m3);
        } else {
            constexpr P p = params();
            return i + p.x * (i >> p.a) + p.y * (i >> p.b) + p.z * (i >> p.c);
        }
    }
    static constexpr int BUF = use_xor() ? N : pad(N - 1) + 1;
};

// radix-8 inter-stage twiddles w_{8 Ns}^{r k}: three table loads, the rest by multiplication
template <int DIR, typename T, typename C>
__device__ __forceinline__ void twiddle8(C *v, const C *__restrict__ ts, int Ns)
{
    const C w1 = root_of<DIR>(ts, 0), w2 = root_of<DIR>(ts, Ns), w4 = root_of<DIR>(ts, 3 * Ns);
    const C w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4);
    const C w7 = cmul(w3, w4);
    v[1] = cmul(v[1], w1); v[2] = cmul(v[2], w2); v[3] = cmul(v[3], w3); v[4] = cmul(v[4], w4);
    v[5] = cmul(v[5], w5); v[6] = cmul(v[6], w6); v[7] = cmul(v[7], w7);
}

// twiddles of one butterfly of radix R whose k-th entries start at ts: v[r] *= w^{r k}, rows [r - 1][k] of length Ns
template <int R, int DIR, typename T, typename C>
__device__ __forceinline__ void twiddle_r(C *v, const C *__restrict__ ts, int Ns)
{
    if constexpr (R == 8) {
        twiddle8<DIR, T>(v, ts, Ns);
    } else {
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul(v[r], root_of<DIR>(ts, (r - 1) * Ns));
    }
}

// One middle stage (0 < s < S - 1) of NT transforms held in consecutive shared-memory buffers, in place.
// SLOT: the elements sit where the first forward stage left them (slot of element j = j / RM + TPR (j % RM)).
template <typename T, int N, int s, int DIR, bool SLOT, int NT>
__device__ __forceinline__ void xg_middle_stage(Cx<T> *sm, const Cx<T> *__restrict__ twx, int b)
{
    using C = Cx<T>;
    using X = XSched<N>;
    using P = XPad<N, (int)sizeof(C)>;
    constexpr int R = X::radix(s), Ns = X::ns(s), NBF = N / R, TPR = X::TPR, RM = X::RM;
    constexpr int ITER = (NBF + TPR - 1) / TPR;
    constexpr bool ragged = (NBF % TPR) != 0;
    C v[ITER][R];
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        C *buf = sm + t * P::BUF;
#pragma unroll
        for (int it = 0; it < ITER; ++it) {
            const int bb = b + it * TPR;
            if (!ragged || bb < NBF) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int e = bb + r * NBF;
                    v[it][r] = buf[P::pad(SLOT ? e / RM + TPR * (e % RM) : e)];
                }
                twiddle_r<R, DIR, T>(v[it], twx + X::tw_off(s) + (bb % Ns), Ns);
                bfly<R, DIR, T>(v[it]);
            }
        }
        __syncthreads();   // every thread has read buffer t
#pragma unroll
        for (int it = 0; it < ITER; ++it) {
            const int bb = b + it * TPR;
            if (!ragged || bb < NBF) {
                const int j0 = (bb / Ns) * Ns * R + (bb % Ns);
#pragma unroll
                for (int r = 0; r < R; ++r) buf[P::pad(j0 + r * Ns)] = v[it][r];
            }
        }
    }
    __syncthreads();
}

template <typename T, int N, int s, int DIR, int NT>
__device__ __forceinline__ void xg_middle_stages(Cx<T> *sm, const Cx<T> *__restrict__ twx, int b)
{
    if constexpr (s < XSched<N>::S - 1) {
        xg_middle_stage<T, N, s, DIR, (DIR < 0 && s == 1), NT>(sm, twx, b);
        xg_middle_stages<T, N, s + 1, DIR, NT>(sm, twx, b);
    }
}

// rows per CTA: a CTA has at least 64 threads when N / RM is smaller (power of two, divides N^2)
template <int N> __host__ __device__ constexpr int xg_rows()
{
    int rows = 1;
    while (rows * 2 * XSched<N>::TPR <= 64) rows *= 2;
    return rows;
}

template <typename T, int N, int NV, int NS, int MINB>
__global__ void __launch_bounds__(xg_rows<N>() * XSched<N>::TPR, MINB)
    k_mid_xg(const Cx<T> *__restrict__ in, Cx<T> *__restrict__ out, const Cx<T> *__restrict__ twx, long nfw, int kxp,
             T scale2, T kfx)
{
    using C = Cx<T>;
    using X = XSched<N>;
    using P = XPad<N, (int)sizeof(C)>;
    constexpr int RM = X::RM, TPR = X::TPR, S = X::S, BUF = P::BUF, KX = kx_count(N);
    constexpr int NI = 3 * NV + 2 * NS;        // inverse complex transforms: (u_c, w_c) pairs, (g_x, g_y), (g_z, -)
    constexpr int NF = (3 * NV + NS + 1) / 2;  // forward complex transforms
    constexpr int NSPLIT = (3 * NV + NS) / 2;  // forward transforms that carry two real fields
    constexpr int ND = (KX + TPR - 1) / TPR;   // outer-stage outputs r = 0..ND-1 can lie below the cutoff
    extern __shared__ __align__(16) unsigned char smraw[];

    const int g = threadIdx.x / TPR, b = threadIdx.x % TPR;
    C *sm = reinterpret_cast<C *>(smraw) + g * (NI * BUF);
    const long rowoff = ((long)blockIdx.x * xg_rows<N>() + g) * kxp;
    const C zero = mk<T>(0, 0);

    // ---- inverse, first stage: Z_t[b + TPR r] from global memory ----
    // class of r (compile time): direct  k = b + TPR r      possible iff TPR r < KX
    //                            mirror  k = N - b - TPR r  possible iff TPR r + TPR - 1 > N - KX
    int kq[RM];
    bool pq[RM];
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        const int e = b + TPR * r;
        const bool dc = TPR * r < KX, mc = TPR * r + TPR - 1 > N - KX;
        kq[r] = dc ? e : N - e;
        pq[r] = (dc || mc) && kq[r] < KX;
    }
    auto first_stage = [&](const C *a, const C *bb, int t) {
        C v[RM];
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            const bool dc = TPR * r < KX, mc = TPR * r + TPR - 1 > N - KX;
            if (dc) {
                C x = a[r], y = bb[r];
                if (r == 0 && b == 0) { x.y = (T)0; y.y = (T)0; }   // k = 0: imaginary parts ignored (c2r, O4)
                v[r] = mk<T>(x.x - y.y, x.y + y.x);                  // A + i B
            } else if (mc) {
                v[r] = mk<T>(a[r].x + bb[r].y, bb[r].x - a[r].y);    // conj A + i conj B
            } else {
                v[r] = zero;
            }
        }
        bfly<RM, +1, T>(v);
        C *buf = sm + t * BUF;
#pragma unroll
        for (int r = 0; r < RM; ++r) buf[P::pad(RM * b + r)] = v[r];
    };
#pragma unroll
    for (int vv = 0; vv < NV; ++vv) {
        const C *f = in + (long)(vv * 6) * nfw + rowoff;
        C ux[RM], uy[RM], uz[RM], wx[RM], wy[RM], wz[RM];
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            ux[r] = uy[r] = uz[r] = wx[r] = wy[r] = wz[r] = zero;
            if (pq[r]) {
                ux[r] = ld_stream(f + kq[r]);
                wx[r] = ld_stream(f + 3 * nfw + kq[r]);
                uy[r] = ld_stream(f + nfw + kq[r]);
                uz[r] = ld_stream(f + 2 * nfw + kq[r]);
                wy[r] = ld_stream(f + 4 * nfw + kq[r]);   // P
                wz[r] = ld_stream(f + 5 * nfw + kq[r]);   // D
            }
        }
#pragma unroll
        for (int r = 0; r < RM; ++r) {   // w^_y = P - i kx U_z,  w^_z = i kx U_y - D
            const T kk = (T)kq[r] * kfx;   // k_x = n_x 2 pi / L_x
            const C p = wy[r], d = wz[r];
            wy[r] = csub(p, mul_ik(uz[r], kk));
            wz[r] = csub(mul_ik(uy[r], kk), d);
        }
        first_stage(ux, wx, vv * 3 + 0);
        first_stage(uy, wy, vv * 3 + 1);
        first_stage(uz, wz, vv * 3 + 2);
    }
    if constexpr (NS > 0) {   // gradient of the scalar: g_x = c2r (i kx Th), g_y = c2r Dt, g_z = c2r Gz
        const C *f = in + (long)(6 * NV) * nfw + rowoff;
        C gx[RM], gy[RM], gz[RM], zz[RM];
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            gx[r] = gy[r] = gz[r] = zz[r] = zero;
            if (pq[r]) {
                gx[r] = mul_ik(ld_stream(f + kq[r]), (T)kq[r] * kfx);
                gy[r] = ld_stream(f + nfw + kq[r]);
                gz[r] = ld_stream(f + 2 * nfw + kq[r]);
            }
        }
        first_stage(gx, gy, 3 * NV);
        first_stage(gz, zz, 3 * NV + 1);
    }
    __syncthreads();

    // ---- inverse, middle stages ----
    xg_middle_stages<T, N, 1, +1, NI>(sm, twx, b);

    // ---- inverse, last stage (Ns = TPR, k = b): results stay in registers ----
    C z[NI][RM];
    {
        const C *ts = twx + X::tw_off(S - 1) + b;
#pragma unroll
        for (int t = 0; t < NI; ++t) {
            const C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < RM; ++r) z[t][r] = buf[P::pad(b + TPR * r)];
            twiddle_r<RM, +1, T>(z[t], ts, TPR);
            bfly<RM, +1, T>(z[t]);
        }
    }

    // ---- a8: products at x = b + TPR r; first forward stage in registers ----
    // z[c] = u_c + i w_c (c = 0..2);  MHD: z[3 + c] = b_c + i j_c;  Boussinesq: z[3] = g_x + i g_y, z[4] = g_z
    C F[NF][RM];
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        const T ux = z[0][r].x, uy = z[1][r].x, uz = z[2][r].x;
        const T wx = z[0][r].y, wy = z[1][r].y, wz = z[2][r].y;
        T m0 = uy * wz - uz * wy, m1 = uz * wx - ux * wz, m2 = ux * wy - uy * wx;
        if constexpr (NV == 2) {
            const T bx = z[3][r].x, by = z[4][r].x, bz = z[5][r].x;
            const T jx = z[3][r].y, jy = z[4][r].y, jz = z[5][r].y;
            m0 += jy * bz - jz * by; m1 += jz * bx - jx * bz; m2 += jx * by - jy * bx;
            const T e0 = uy * bz - uz * by, e1 = uz * bx - ux * bz, e2 = ux * by - uy * bx;
            F[1][r] = mk<T>(m2 * scale2, e0 * scale2);
            F[2][r] = mk<T>(e1 * scale2, e2 * scale2);
        } else if constexpr (NS > 0) {
            const T s = ux * z[3][r].x + uy * z[3][r].y + uz * z[4][r].x;
            F[1][r] = mk<T>(m2 * scale2, s * scale2);
        } else {
            F[1][r] = mk<T>(m2 * scale2, (T)0);
        }
        F[0][r] = mk<T>(m0 * scale2, m1 * scale2);
    }
#pragma unroll
    for (int t = 0; t < NF; ++t) {
        bfly<RM, -1, T>(F[t]);
        C *buf = sm + t * BUF;
        // element RM b + r of the forward transform goes to the slot this thread read above
#pragma unroll
        for (int r = 0; r < RM; ++r) buf[P::pad(b + TPR * r)] = F[t][r];
    }
    __syncthreads();

    // ---- forward, middle stages (the first one reads through the slot map) ----
    xg_middle_stages<T, N, 1, -1, NF>(sm, twx, b);

    // ---- forward, last stage: X_t[b + TPR r] in registers ----
    {
        const C *ts = twx + X::tw_off(S - 1) + b;
#pragma unroll
        for (int t = 0; t < NF; ++t) {
            const C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < RM; ++r) {
                const int e = b + TPR * r;
                F[t][r] = buf[P::pad(S == 2 ? e / RM + TPR * (e % RM) : e)];
            }
            twiddle_r<RM, -1, T>(F[t], ts, TPR);
            bfly<RM, -1, T>(F[t]);
        }
    }

    // ---- split of the packed transforms: thread TPR - b holds X[N - k] at r' = RM - 1 - r ----
    C *ex = sm + NF * BUF;   // buffers NF.. are free since the last inverse stage
#pragma unroll
    for (int t = 0; t < NSPLIT; ++t)
#pragma unroll
        for (int e = 0; e < ND; ++e) ex[(t * ND + e) * TPR + b] = F[t][RM - ND + e];
    __syncthreads();
    const int bp = (TPR - b) % TPR;
    C *o = out + rowoff;
#pragma unroll
    for (int r = 0; r < ND; ++r) {
        const int k = b + TPR * r;
        if (k < KX) {
#pragma unroll
            for (int t = 0; t < NF; ++t) {
                if (t < NSPLIT) {
                    // thread 0 is its own partner: X[N - TPR r] sits at r' = RM - r (r > 0), X[0] pairs with itself
                    const int e = (b == 0) ? (r == 0 ? 0 : ND - r) : ND - 1 - r;
                    C c = ex[(t * ND + e) * TPR + bp];
                    if (b == 0 && r == 0) c = F[t][0];
                    const C a = F[t][r];
                    const C s = mk<T>((T)0.5 * (a.x + c.x), (T)0.5 * (a.y - c.y));   // (a + conj c)/2
                    const C d = mk<T>((T)0.5 * (a.x - c.x), (T)0.5 * (a.y + c.y));   // (a - conj c)/2
                    st_stream(o + (long)(2 * t) * nfw + k, s);
                    st_stream(o + (long)(2 * t + 1) * nfw + k, mk<T>(d.y, -d.x));    // -i d
                } else {
                    st_stream(o + (long)(2 * t) * nfw + k, F[t][r]);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// mid_x of the Gross-Pitaevskii equation (Eq. 7): psi = p + i q.  The packed row
// Z = P^ + i Q^ inverse-transforms to psi itself (ONE complex length-N transform per row), the cubic term
// rho = |psi|^2, F = rho q + i rho p is formed in registers, and one forward transform + split gives
// a^ = F[rho q], b^ = F[rho p] for kx < N/3.   in: 2 compact fields (P, Q rows);  out: 2 compact fields.
// ------------------------------------------------------------------------------------------
template <typename T, int N, int MINB>
__global__ void __launch_bounds__(xg_rows<N>() * XSched<N>::TPR, MINB)
    k_mid_x_gpe(const Cx<T> *__restrict__ in, Cx<T> *__restrict__ out, const Cx<T> *__restrict__ twx, long nfw, int kxp,
                T scale1)
{
    using C = Cx<T>;
    using X = XSched<N>;
    using P = XPad<N, (int)sizeof(C)>;
    constexpr int RM = X::RM, TPR = X::TPR, S = X::S, BUF = P::BUF, KX = kx_count(N);
    constexpr int ND = (KX + TPR - 1) / TPR;
    extern __shared__ __align__(16) unsigned char smraw[];

    const int g = threadIdx.x / TPR, b = threadIdx.x % TPR;
    C *sm = reinterpret_cast<C *>(smraw) + g * (2 * BUF);   // buffer 0: the transform, buffer 1: split exchange
    const long rowoff = ((long)blockIdx.x * xg_rows<N>() + g) * kxp;
    const C zero = mk<T>(0, 0);

    // ---- inverse, first stage (same classes of r as k_mid_xg) ----
    C z[RM];
    {
        const C *f = in + rowoff;
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            const int e = b + TPR * r;
            const bool dc = TPR * r < KX, mc = TPR * r + TPR - 1 > N - KX;
            const int k = dc ? e : N - e;
            C pa = zero, qa = zero;
            if ((dc || mc) && k < KX) { pa = ld_stream(f + k); qa = ld_stream(f + nfw + k); }
            if (dc) {
                if (r == 0 && b == 0) { pa.y = (T)0; qa.y = (T)0; }
                z[r] = mk<T>(pa.x - qa.y, pa.y + qa.x);        // P + i Q
            } else if (mc) {
                z[r] = mk<T>(pa.x + qa.y, qa.x - pa.y);        // conj P + i conj Q
            } else {
                z[r] = zero;
            }
        }
        bfly<RM, +1, T>(z);
#pragma unroll
        for (int r = 0; r < RM; ++r) sm[P::pad(RM * b + r)] = z[r];
    }
    __syncthreads();
    xg_middle_stages<T, N, 1, +1, 1>(sm, twx, b);
    {
        const C *ts = twx + X::tw_off(S - 1) + b;
#pragma unroll
        for (int r = 0; r < RM; ++r) z[r] = sm[P::pad(b + TPR * r)];
        twiddle_r<RM, +1, T>(z, ts, TPR);
        bfly<RM, +1, T>(z);
    }
    // ---- cubic term at x = b + TPR r: psi = scale1 z;  F = |psi|^2 (q + i p) ----
    C F[RM];
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        const T pr = z[r].x * scale1, qr = z[r].y * scale1;
        const T rho = pr * pr + qr * qr;
        F[r] = mk<T>(rho * qr, rho * pr);
    }
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
        bfly<RM, -1, T>(F);
    }
    // ---- split: a^[k] = (F[k] + conj F[N-k])/2, b^[k] = -i (F[k] - conj F[N-k])/2 ----
    C *ex = sm + BUF;
#pragma unroll
    for (int e = 0; e < ND; ++e) ex[e * TPR + b] = F[RM - ND + e];
    __syncthreads();
    const int bp = (TPR - b) % TPR;
    C *o = out + rowoff;
#pragma unroll
    for (int r = 0; r < ND; ++r) {
        const int k = b + TPR * r;
        if (k < KX) {
            const int e = (b == 0) ? (r == 0 ? 0 : ND - r) : ND - 1 - r;
            C c = ex[e * TPR + bp];
            if (b == 0 && r == 0) c = F[0];
            const C a = F[r];
            const C sa = mk<T>((T)0.5 * (a.x + c.x), (T)0.5 * (a.y - c.y));
            const C d = mk<T>((T)0.5 * (a.x - c.x), (T)0.5 * (a.y + c.y));
            st_stream(o + k, sa);
            st_stream(o + nfw + k, mk<T>(d.y, -d.x));
        }
    }
}

}  // namespace psfft
