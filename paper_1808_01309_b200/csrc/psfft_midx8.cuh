// psfft_midx8.cuh -- RHS pass 3 ("mid_x") for N = 8^S (64, 512): the inverse x-transforms, the pointwise
// products (a8) and the forward x-transforms of one (z, y) row, as complex length-N transforms of
// PAIRS of real fields ("two for one"), radix 8 throughout, one butterfly per thread and stage.
//
// What is computed per row:
//   u_c = c2r U_c, w_x = c2r W_x, w_y = c2r (P - i kx U_z), w_z = c2r (i kx U_y - D)   (six per vector field)
//   n = u x w                                     (MHD: m = u x w + j x b, e = u x b)
//   n^_c = r2c n_c, kept for kx < N/3
//
// Packing.  For Hermitian rows A, B (real a, b) the complex row Z[k] = A[k] + i B[k] (0 <= k < N/2),
// Z[N-k] = conj A[k] + i conj B[k] has the inverse transform z = a + i b: three complex transforms
// give (u_x, w_x), (u_y, w_y), (u_z, w_z) with no merge step, and a thread that finishes a
// last-stage butterfly of all three holds u and w at its eight grid points x = b + (N/8) r.  The
// products are formed in registers and go straight into the first stage of the forward
// transforms F1 = n_x + i n_y, F2 = n_z (MHD: m_x + i m_y, m_z + i e_x, e_y + i e_z), whose output
// is split as n^_x[k] = (F1[k] + conj F1[N-k])/2, n^_y[k] = -i (F1[k] - conj F1[N-k])/2.
// Boussinesq (NS = 1): two more inverse transforms (g_x + i g_y, g_z) for grad theta and F2 = n_z + i s,
// s = u . grad theta (Eq. 2).
//
// Shared memory: one buffer of N complex per inverse transform; every exchange is conflict-free
// (Mid8::pad).  The first forward stage writes into the slots its thread has just read, so the
// inverse -> product -> forward hand-over needs no barrier and no extra buffer.  Per row and
// transform: two exchanges (write + read) instead of the three stages + merge + product staging of
// k_mid_x, i.e. 20 N complex accesses per HD row instead of 36 N.
#pragma once
#include "psfft_rhs.cuh"

namespace psfft {

template <int N, int CSIZE> struct Mid8 {
    static_assert(N == 64 || N == 512, "k_mid_x8: N must be 8^2 or 8^3");
    static constexpr int NB = N / 8;           // butterflies per stage = threads per row
    static constexpr int S = (N == 64) ? 2 : 3;
    // element index -> padded slot.  Conflict-free (fp64) for: stride-8 over b (first-stage writes), unit
    // stride over b (reads b + NB r), 64 (b>>3) + (b&7) + 8 r (middle-stage writes) and
    // (b>>3) + 8 r + 64 (b&7) (middle-stage reads of the forward transform); _work-free derivation in DESIGN.md.
    __host__ __device__ static constexpr int pad(int i)
    {
        return CSIZE == 16 ? i + (i >> 3) + (i >> 6) : i + (i >> 4) + 4 * (i >> 6) + 2 * (i >> 7);
    }
    static constexpr int BUF = pad(N - 1) + 1;
    // slot of forward-transform element j after its first stage: thread b = j >> 3 wrote output r = j & 7 into
    // the slot it had read as inverse element b + NB r
    __host__ __device__ static constexpr int fwd_slot(int j) { return (j >> 3) + NB * (j & 7); }
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

template <typename T, int N, int NV, int NS, int MINB>
__global__ void __launch_bounds__(N / 8, MINB)
    k_mid_x8(const Cx<T> *__restrict__ in, Cx<T> *__restrict__ out, const Cx<T> *__restrict__ tw, long nfw, int kxp,
             T scale2)
{
    using C = Cx<T>;
    using L = Mid8<N, (int)sizeof(C)>;
    constexpr int NB = L::NB, BUF = L::BUF, KX = kx_count(N);
    constexpr int NI = 3 * NV + 2 * NS;        // inverse complex transforms: (u_c, w_c) pairs, (g_x, g_y), (g_z, -)
    constexpr int NF = (3 * NV + NS + 1) / 2;  // forward complex transforms
    constexpr int NSPLIT = (3 * NV + NS) / 2;  // forward transforms that carry two real fields
    extern __shared__ __align__(16) unsigned char smraw[];
    C *sm = reinterpret_cast<C *>(smraw);

    const int b = threadIdx.x;
    const long rowoff = (long)blockIdx.x * kxp;
    const C zero = mk<T>(0, 0);

    // ---- inverse, first stage: Z_t[b + NB r] from global memory (r = 3, 4 lie in the truncated band) ----
    // positions: q = 0..2 direct k = b + NB q;  q = 3..5 mirrored k = N - b - NB (q + 2)  (r = q + 2)
    int kq[6];
    bool pq[6];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        kq[q] = b + NB * q;
        pq[q] = kq[q] < KX;
        kq[q + 3] = N - b - NB * (q + 5);
        pq[q + 3] = kq[q + 3] < KX;
    }
#pragma unroll
    for (int vv = 0; vv < NV; ++vv) {
        const C *f = in + (long)(vv * 6) * nfw + rowoff;
        C ux[6], uy[6], uz[6], wx[6], pp[6], dd[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            ux[q] = uy[q] = uz[q] = wx[q] = pp[q] = dd[q] = zero;
            if (pq[q]) {
                ux[q] = ld_stream(f + kq[q]);
                wx[q] = ld_stream(f + 3 * nfw + kq[q]);
                uy[q] = ld_stream(f + nfw + kq[q]);
                uz[q] = ld_stream(f + 2 * nfw + kq[q]);
                pp[q] = ld_stream(f + 4 * nfw + kq[q]);
                dd[q] = ld_stream(f + 5 * nfw + kq[q]);
            }
        }
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            C v[8];
            v[3] = zero; v[4] = zero;
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                const T kk = (T)kq[q];
                C a, bb;   // A = U_comp, B = w^_comp row
                if (comp == 0) { a = ux[q]; bb = wx[q]; }
                else if (comp == 1) { a = uy[q]; bb = csub(pp[q], mul_ik(uz[q], kk)); }
                else { a = uz[q]; bb = csub(mul_ik(uy[q], kk), dd[q]); }
                C z;
                if (q < 3) {
                    if (q == 0 && b == 0) { a.y = (T)0; bb.y = (T)0; }   // k = 0: imaginary parts ignored (c2r, O4)
                    z = mk<T>(a.x - bb.y, a.y + bb.x);                     // A + i B
                    v[q] = z;
                } else {
                    z = mk<T>(a.x + bb.y, bb.x - a.y);                     // conj A + i conj B
                    v[q + 2] = z;
                }
            }
            bfly8<+1, T>(v);
            C *buf = sm + (vv * 3 + comp) * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r) buf[L::pad(8 * b + r)] = v[r];
        }
    }
    if constexpr (NS > 0) {   // gradient of the scalar: g_x = c2r (i kx Th), g_y = c2r Dt, g_z = c2r Gz
        const C *f = in + (long)(6 * NV) * nfw + rowoff;
        C th[6], dt[6], gz[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            th[q] = dt[q] = gz[q] = zero;
            if (pq[q]) {
                th[q] = ld_stream(f + kq[q]);
                dt[q] = ld_stream(f + nfw + kq[q]);
                gz[q] = ld_stream(f + 2 * nfw + kq[q]);
            }
        }
#pragma unroll
        for (int tt = 0; tt < 2; ++tt) {
            C v[8];
            v[3] = zero; v[4] = zero;
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                C a, bb;
                if (tt == 0) { a = mul_ik(th[q], (T)kq[q]); bb = dt[q]; }
                else { a = gz[q]; bb = zero; }
                if (q < 3) {
                    if (q == 0 && b == 0) { a.y = (T)0; bb.y = (T)0; }
                    v[q] = mk<T>(a.x - bb.y, a.y + bb.x);
                } else {
                    v[q + 2] = mk<T>(a.x + bb.y, bb.x - a.y);
                }
            }
            bfly8<+1, T>(v);
            C *buf = sm + (3 * NV + tt) * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r) buf[L::pad(8 * b + r)] = v[r];
        }
    }
    __syncthreads();

    // ---- inverse, middle stage (N = 512): Ns = 8, in place, software-pipelined over the transforms ----
    if constexpr (L::S == 3) {
        const C *ts = tw + tw_offset(N, 8) + (b & 7);
        const int j0 = (b >> 3) * 64 + (b & 7);
        C v[8];
#pragma unroll
        for (int t = 0; t < NI; ++t) {
            C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r) v[r] = buf[L::pad(b + NB * r)];
            twiddle8<+1, T>(v, ts, 8);
            bfly8<+1, T>(v);
            __syncthreads();   // every thread has read buffer t
#pragma unroll
            for (int r = 0; r < 8; ++r) buf[L::pad(j0 + 8 * r)] = v[r];
        }
        __syncthreads();
    }

    // ---- inverse, last stage (Ns = NB, k = b): results stay in registers ----
    C z[NI][8];
    {
        const C *ts = tw + tw_offset(N, NB) + b;
#pragma unroll
        for (int t = 0; t < NI; ++t) {
            const C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r) z[t][r] = buf[L::pad(b + NB * r)];
            twiddle8<+1, T>(z[t], ts, NB);
            bfly8<+1, T>(z[t]);
        }
    }

    // ---- a8: products at x = b + NB r; first forward stage in registers ----
    // z[c] = u_c + i w_c (c = 0..2), z[3 + c] = b_c + i j_c
    C F[NF][8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
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
        } else if constexpr (NS > 0) {   // z[3] = g_x + i g_y, z[4] = g_z:  s = u . grad theta
            const T s = ux * z[3][r].x + uy * z[3][r].y + uz * z[4][r].x;
            F[1][r] = mk<T>(m2 * scale2, s * scale2);
        } else {
            F[1][r] = mk<T>(m2 * scale2, (T)0);
        }
        F[0][r] = mk<T>(m0 * scale2, m1 * scale2);
    }
#pragma unroll
    for (int t = 0; t < NF; ++t) {
        bfly8<-1, T>(F[t]);
        C *buf = sm + t * BUF;
        // element 8 b + r of the forward transform goes to the slot this thread read above
#pragma unroll
        for (int r = 0; r < 8; ++r) buf[L::pad(b + NB * r)] = F[t][r];
    }
    __syncthreads();

    // ---- forward, middle stage (N = 512) ----
    if constexpr (L::S == 3) {
        const C *ts = tw + tw_offset(N, 8) + (b & 7);
        const int j0 = (b >> 3) * 64 + (b & 7);
        C v[8];
#pragma unroll
        for (int t = 0; t < NF; ++t) {
            C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r) v[r] = buf[L::pad(L::fwd_slot(b + NB * r))];
            twiddle8<-1, T>(v, ts, 8);
            bfly8<-1, T>(v);
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 8; ++r) buf[L::pad(j0 + 8 * r)] = v[r];
        }
        __syncthreads();
    }

    // ---- forward, last stage: X_t[b + NB r] in registers ----
    {
        const C *ts = tw + tw_offset(N, NB) + b;
#pragma unroll
        for (int t = 0; t < NF; ++t) {
            const C *buf = sm + t * BUF;
#pragma unroll
            for (int r = 0; r < 8; ++r)
                F[t][r] = buf[L::pad(L::S == 3 ? b + NB * r : L::fwd_slot(b + NB * r))];
            twiddle8<-1, T>(F[t], ts, NB);
            bfly8<-1, T>(F[t]);
        }
    }

    // ---- split of the packed transforms: partner class NB - b holds X[N - k] at r' = 7 - r ----
    C *ex = sm + NF * BUF;   // buffers NF.. are free since the last inverse stage
#pragma unroll
    for (int t = 0; t < NSPLIT; ++t)
#pragma unroll
        for (int r = 5; r < 8; ++r) ex[(t * 3 + (r - 5)) * NB + b] = F[t][r];
    __syncthreads();
    const int bp = (NB - b) % NB;
    C *o = out + rowoff;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int k = b + NB * r;
        if (k < KX) {
#pragma unroll
            for (int t = 0; t < NF; ++t) {
                if (t < NSPLIT) {
                    // class 0 is its own partner: X[N - NB r] sits at r' = 8 - r (r > 0), X[0] pairs with itself
                    const int e = (b == 0) ? (r == 0 ? 0 : 3 - r) : 2 - r;
                    C c = ex[(t * 3 + e) * NB + bp];
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

}  // namespace psfft
