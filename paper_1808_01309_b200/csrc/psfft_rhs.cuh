// psfft_rhs.cuh -- the fused right-hand-side passes (HD: NV = 1; MHD: NV = 2; Boussinesq: NV = 1 plus
// NS = 1 scalar field theta, Eqs. 1-3).
//
// One evaluation is five kernels; physical-space data never reaches HBM and the spectral
// pointwise work rides on the loads / stores of the transform passes:
//
//   inv_z   u^ (masked on load) -> A_c = F_z^-1 u^_c (c = x,y,z),  B_x = F_z^-1 (i kz u^_x),
//           G_x = F_z^-1 (i (ky u^_z - kz u^_y))  [= w^_x, complete]
//   inv_y   -> U_c = F_y^-1 A_c,  W_x = F_y^-1 G_x,  P = F_y^-1 B_x,  D = F_y^-1 (i ky A_x)
//   mid_x   (psfft_midxg.cuh) per (z,y) row: u_c = c2r U_c, w_x = c2r W_x, w_y = c2r (P - i kx U_z), w_z = c2r (i kx U_y - D);
//           n = u x w (MHD: m = u x w + j x b, e = u x b);  r2c of n -> kx < N/3 only
//   fwd_y   in place, kx < N/3
//   fwd_z   + epilogue on the store: 2/3 mask, projection (or i k x for the induction equation),
//           diffusion term
//
// The curl i k x u^ (a7) is distributed over the three inverse passes: each wavenumber factor is
// applied in the pass whose FFT runs along that axis (the multiplier is then per-element of the
// loaded column), everything else commutes with the remaining transforms by linearity.  This
// needs 5 z-transforms and 6 y-transforms per vector field instead of 6 + 6.
//
// Boussinesq (NS = 1): the gradient g = i k theta^ is split over the passes in the same way,
//   inv_z   T_A = F_z^-1 theta^,  T_B = F_z^-1 (i kz theta^)
//   inv_y   Th = F_y^-1 T_A,  Dt = F_y^-1 (i ky T_A),  Gz = F_y^-1 T_B
//   mid_x   g_x = c2r (i kx Th), g_y = c2r Dt, g_z = c2r Gz;  s = u . g;  r2c of s
//   fwd_z   epilogue: n^_z -= N_bv M theta^ before the projection (Eq. 1: buoyancy is inside the
//           pressure projection);  R_theta = -s^ + N_bv M u^_z - kappa |k|^2 M theta^ (Eq. 2)
// i.e. 2 + 3 + 3 inverse and 1 forward axis transforms on top of HD (theta itself is never needed in
// physical space).
//
// Pruning: after the mask of step 1 (and before the mask of step 6) every mode with
// 9 |k|^2 >= N^2 is zero (does not matter), so columns / rows that are entirely outside the
// truncation sphere are neither read, transformed nor written, and loads inside a column are
// predicated on the mode being retained.
//
// Intermediate layout: every workspace field is [z][y][kxp] with the COMPACT row pitch
// kxp = kx_pitch(N, TC) >= kx_count(N), a multiple of the tile width TC, so every 128-byte tile
// row of the y passes, of mid_x and of the z passes' workspace side starts on a 128-byte line
// (the caller's layout has the odd pitch ldk = N/2+1, whose tile rows straddle two lines).
// Skipped entries of the workspace are simply never touched.
#pragma once
#include "psfft_kernels.cuh"

namespace psfft {


template <typename C, typename T> __device__ __forceinline__ C mul_ik(C v, T k) { return mk<T>(-k * v.y, k * v.x); }
__device__ __forceinline__ float2x2 mul_ik(float2x2 v, float k)
{
    float2x2 r;
    r.re = __fmul2_rn(v.im, bc2(-k));
    r.im = __fmul2_rn(v.re, bc2(k));
    return r;
}

// Geometry of a right-hand side on an (Nx, Ny, Nz) grid in an (Lx, Ly, Lz) box (box size and grid points
// independent per direction; readings G24, G25).  Index n_i (integer, the wavenumber of the 2 pi box):
//   mask         keep iff sum_i (n_i / N_i)^2 < 1/9, in integers  rx2 nx^2 + ry2 ny^2 + rz2 nz^2 < lim  with
//                r_i = lcm(Nx, Ny, Nz) / N_i,  lim = ceil(lcm^2 / 9)   (cubic: r_i = 1, i.e. 9 |n|^2 < N^2)
//   wavenumbers  k_i = n_i kf_i,  kf_i = 2 pi / L_i  (exactly 1 in the 2 pi box)
// A job template's N is the length of ITS transform axis only; everything about the other two axes comes from its
// geometry policy G: GeomCube (the N^3 grid in the 2 pi box of every BASELINE.json config: all compile-time, the
// multiplications by 1 fold away) or GeomAny (run-time values from the plan).  Measured on B200, 512^3 fp64: with
// run-time geometry alone inv_y ran 1.56 -> 2.03 ms (spills at the 64-register budget), hence the two policies.
template <typename T, int N> struct GeomCube {
    static constexpr int ny = N, nz = N, kxc = kx_count(N);
    static constexpr int rx2 = 1, ry2 = 1, rz2 = 1, lim = (N * N + 8) / 9;
    static constexpr T kfx = (T)1, kfy = (T)1, kfz = (T)1;
    __device__ __forceinline__ static int w2(int kx, int ky) { return kx * kx + ky * ky; }
    __device__ __forceinline__ static bool keep2(int kxy2) { return 9 * kxy2 < N * N; }
    __device__ __forceinline__ static bool keep3(int kxy2, int kz) { return 9 * (kxy2 + kz * kz) < N * N; }
};
template <typename T> struct GeomAny {
    int ny, nz;           // grid points along y, z
    int kxc;              // retained kx: kx < kxc = kx_count(Nx)
    int rx2, ry2, rz2, lim;
    T kfx, kfy, kfz;
    __device__ __forceinline__ int w2(int kx, int ky) const { return rx2 * kx * kx + ry2 * ky * ky; }
    __device__ __forceinline__ bool keep2(int kxy2) const { return kxy2 < lim; }
    __device__ __forceinline__ bool keep3(int kxy2, int kz) const { return kxy2 + rz2 * kz * kz < lim; }
};

// 16-byte access to two adjacent fp32 columns (re0, im0, re1, im1) <-> float2x2; p must be 16-byte aligned
__device__ __forceinline__ float2x2 pack2(float4 q)
{
    float2x2 e;
    e.re = make_float2(q.x, q.z);
    e.im = make_float2(q.y, q.w);
    return e;
}
__device__ __forceinline__ float4 unpack2(float2x2 e) { return make_float4(e.re.x, e.im.x, e.re.y, e.im.y); }
// zero the columns whose flag is false
__device__ __forceinline__ float2x2 mask2(float2x2 e, bool m0, bool m1)
{
    if (!m0) { e.re.x = 0.f; e.im.x = 0.f; }
    if (!m1) { e.re.y = 0.f; e.im.y = 0.f; }
    return e;
}
// store the flagged columns of e at p (16-byte aligned), one 16-byte store when both are flagged
__device__ __forceinline__ void st_stream2(float2 *p, float2x2 e, bool m0, bool m1)
{
    if (m0 && m1) __stcs(reinterpret_cast<float4 *>(p), unpack2(e));
    else if (m0) __stcs(p, make_float2(e.re.x, e.im.x));
    else if (m1) __stcs(p + 1, make_float2(e.re.y, e.im.y));
}

// Element-level entry points of a job, by default assembled column by column from the job's per-column
// load / post / store (s[j] = state of column j of the element).  Jobs whose tiles are 16-byte aligned
// override them with one vector access per element.
template <class Derived, typename C, typename E> struct JobElems {
    static constexpr int EW = ElemWidth<E>::value;
    using Elem = E;
    static constexpr bool prefetch_next = false;
    static constexpr bool split_rounds = true;   // rounds are independent: may run in different CTAs
    static constexpr bool is_fwdz = false;       // tile width rule: cpass_cols (fwdz_cols for the last pass)
    template <class State> __device__ __forceinline__ const void *next_addr(const State &, int, int) const { return nullptr; }
    template <class State> __device__ __forceinline__ E load_e(const State *s, int r, int i) const
    {
        E x;
#pragma unroll
        for (int j = 0; j < EW; ++j) ecol_set(x, j, static_cast<const Derived *>(this)->load(s[j], r, i));
        return x;
    }
    template <class State> __device__ __forceinline__ E post_e(const State *s, int r, int i, E x) const
    {
#pragma unroll
        for (int j = 0; j < EW; ++j) ecol_set(x, j, static_cast<const Derived *>(this)->post(s[j], r, i, ecol(x, j)));
        return x;
    }
    template <class State> __device__ __forceinline__ void store_e(const State *s, int r, int i, E v) const
    {
#pragma unroll
        for (int j = 0; j < EW; ++j) static_cast<const Derived *>(this)->store(s[j], r, i, ecol(v, j));
    }
};

// ------------------------------------------------------------------------------------------
// generic multi-round column pass: Job supplies begin(c) / load(r,i) / store(r,i,v)
// ------------------------------------------------------------------------------------------
// The tile is [N rows] x [TC elements]; an element (Job::Elem) is one column (Cx<T>) or TWO adjacent fp32
// columns (float2x2) whose butterflies run on packed fp32x2 arithmetic (psfft_core.cuh).  Column j of
// element c is column (blockIdx.x TC + c) EW + j of the job's column grid.
template <typename T, int N, int DIR, int TC, int TPF, int MINB, class Job>
__global__ void __launch_bounds__(TC *TPF, MINB) k_cpass_job(Job job, const Cx<T> *__restrict__ tw)
{
    using E = typename Job::Elem;
    constexpr int EW = ElemWidth<E>::value;
    constexpr bool PAD = (TC * sizeof(E) < 128);
    using Map = ColMap<N, TC, PAD>;
    extern __shared__ __align__(16) unsigned char smraw[];
    E *sm = reinterpret_cast<E *>(smraw);
    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    typename Job::State s[EW];
    bool any = false;
#pragma unroll
    for (int j = 0; j < EW; ++j) any |= job.begin(s[j], ((long)blockIdx.x * TC + c) * EW + j);
    if (!__syncthreads_or(any)) {   // nothing of this tile is retained (CTA-uniform)
#pragma unroll
        for (int j = 0; j < EW; ++j) job.idle(s[j], t, blockDim.x / TC);
        return;
    }
    // gridDim.z > 1 (small grids, see run_job_v): the rounds of a tile position are spread over blockIdx.z
#pragma unroll 1
    for (int r = blockIdx.z; r < job.rounds(); r += gridDim.z) {
        // Jobs that ask for it: pull the next round's tile into L2 while this round computes -- one prefetch
        // per 128-byte tile row, issued by the threads of the tile's first column (whose retained range is the
        // widest).  Measured at 512^3: fp32 inv_y 1.05 -> 0.94 ms, fwd_y 0.41 -> 0.35 ms; no gain in fp64 and
        // for the z passes, which leave it off.
        if constexpr (Job::prefetch_next) {
            if (c == 0 && r + (int)gridDim.z < job.rounds()) {
                for (int i = t; i < N; i += TPF) {
                    const void *p = job.next_addr(s[0], r + (int)gridDim.z, i);
                    if (p) asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
                }
            }
        }
        auto ld = [&](int i) -> E { return job.load_e(s, r, i); };
        auto px = [&](int i, E x) -> E { return job.post_e(s, r, i, x); };
        auto st = [&](int i, E v) { job.store_e(s, r, i, v); };
        fft_stages<T, N, 1, DIR, TPF, false, false, false, Map>(sm, tw, c, t, ld, st, px);
        __syncthreads();  // the next round's first stage overwrites the tile
    }
}

// ---- inv_z -------------------------------------------------------------------------------------
// grid (kxp / TC, N): tile = TC consecutive kx at one ky.  Reads the caller's layout (pitch ldk),
// writes the compact workspace layout (pitch kxp).
template <typename T, int N, int TC, int NV, int NS, class G> struct JobInvZ : JobElems<JobInvZ<T, N, TC, NV, NS, G>, Cx<T>, Ex<T>> {
    using C = Cx<T>;
    const C *src[NV];   // NV x 3 spectral fields (u^, b^), caller layout
    const C *ssrc;      // NS = 1: theta^, caller layout
    C *dst;             // NV x 5 fields: A_x, A_y, A_z, B_x = F_z^-1(i kz u_x), G_x = F_z^-1(w^_x); then NS x 2: T_A, T_B
    long plane, nf;     // caller layout: ldk Ny, ldk Ny Nz
    long wplane, wnf;   // workspace layout: kxp Ny, kxp Ny Nz
    int ldk, kxp;
    G geo;
    struct State { long col, wcol; int kxy2, ky; bool active; };

    __host__ __device__ __forceinline__ int rounds() const { return 5 * NV + 2 * NS; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        const int kx = (int)colidx, ky = wavenumber((int)blockIdx.y, geo.ny);
        s.kxy2 = geo.w2(kx, ky);
        s.ky = ky;
        s.active = geo.keep2(s.kxy2);
        s.col = (long)blockIdx.y * ldk + kx;
        s.wcol = (long)blockIdx.y * kxp + kx;
        return s.active;
    }
    __device__ __forceinline__ void idle(const State &, int, int) const {}
    __device__ __forceinline__ bool keep(const State &s, int i) const
    {
        return s.active && geo.keep3(s.kxy2, wavenumber(i, N));
    }
    __device__ __forceinline__ const C *field(int r) const { return (NV == 2 && r >= 5) ? src[NV - 1] : src[0]; }
    // rr: 0..2 A_c <- u_c | 3 B_x <- i kz u_x | 4 G_x <- i (ky u_z - kz u_y);  scalar: T_A <- th | T_B <- i kz th
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (NS > 0 && r >= 5 * NV) {
            if (keep(s, i)) x = ldg_c(ssrc + i * plane + s.col);
            return x;
        }
        const int rr = r % 5;
        const int comp = rr < 3 ? rr : rr == 3 ? 0 : 2;
        if (keep(s, i)) x = ldg_c(field(r) + comp * nf + i * plane + s.col);
        return x;
    }
    __device__ __forceinline__ C post(const State &s, int r, int i, C x) const
    {
        if (NS > 0 && r >= 5 * NV) return r == 5 * NV ? x : mul_ik(x, (T)wavenumber(i, N) * geo.kfz);
        const int rr = r % 5;
        if (rr < 3) return x;
        const T kz = (T)wavenumber(i, N) * geo.kfz;
        if (rr == 3) return mul_ik(x, kz);
        C y = mk<T>(0, 0);
        if (keep(s, i)) y = ldg_c(field(r) + nf + i * plane + s.col);   // u_y (sparse, L1/L2 resident)
        const T ky = (T)s.ky * geo.kfy;
        return mk<T>(-(ky * x.y - kz * y.y), ky * x.x - kz * y.x);
    }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (s.active) st_stream(dst + r * wnf + i * wplane + s.wcol, v);
    }
    // fp32 pairs: the workspace side is 16-byte aligned (kx even, pitch a multiple of the tile)
    __device__ __forceinline__ void store_e(const State *s, int r, int i, float2x2 v) const
    {
        st_stream2(dst + r * wnf + i * wplane + s[0].wcol, v, s[0].active, s[1].active);
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, double2 v) const { store(s[0], r, i, v); }
};

// ---- inv_y -------------------------------------------------------------------------------------
// grid (kxp / TC, N): tile = TC consecutive kx of one z plane, all in the compact layout.
template <typename T, int N, int TC, int NV, int NS, class G> struct JobInvY : JobElems<JobInvY<T, N, TC, NV, NS, G>, Cx<T>, Ex<T>> {
    using C = Cx<T>;
    const C *src;  // NV x 5 (+ NS x 2) fields from inv_z
    C *dst;        // NV x 6 fields: U_x, U_y, U_z, W_x, P, D;  then NS x 3: Th, Dt, Gz
    long wplane, wnf;
    int kxp;
    G geo;
    struct State { long base; int kx; bool active; };
    static constexpr bool prefetch_next = sizeof(T) == 4;

    __host__ __device__ __forceinline__ int rounds() const { return 6 * NV + 3 * NS; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        s.kx = (int)colidx;
        s.active = s.kx < geo.kxc;
        s.base = (long)blockIdx.y * wplane + s.kx;
        return true;
    }
    __device__ __forceinline__ bool keepy(const State &s, int ky) const { return s.active && geo.keep2(geo.w2(s.kx, ky)); }
    __device__ __forceinline__ void idle(const State &, int, int) const {}
    // scalar rounds (r >= 6 NV): Th <- T_A | Dt <- i ky T_A | Gz <- T_B
    // round order: U_x <- A_x | D <- i ky A_x | U_y | U_z | W_x <- G_x | P <- B_x.  A_x is read in two
    // consecutive rounds: the first read leaves it in L2 (default policy), the second streams.
    __device__ __forceinline__ static int src_field(int rr) { return rr == 0 ? 0 : rr == 1 ? 0 : rr == 2 ? 1 : rr == 3 ? 2 : rr == 4 ? 4 : 3; }
    __device__ __forceinline__ static int dst_field(int rr) { return rr == 0 ? 0 : rr == 1 ? 5 : rr == 2 ? 1 : rr == 3 ? 2 : rr == 4 ? 3 : 4; }
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        const int ky = wavenumber(i, N);
        const bool sc = NS > 0 && r >= 6 * NV;
        const int v = r / 6, rr = sc ? r - 6 * NV : r % 6;
        C x = mk<T>(0, 0);
        if (keepy(s, ky)) {
            const int f = sc ? 5 * NV + (rr >> 1) : v * 5 + src_field(rr);
            const C *p = src + (long)f * wnf + s.base + (long)i * kxp;
            x = rr == 0 ? *p : ld_stream(p);
        }
        return x;
    }
    __device__ __forceinline__ const void *next_addr(const State &s, int r, int i) const
    {
        const int ky = wavenumber(i, N);
        const bool sc = NS > 0 && r >= 6 * NV;
        const int v = r / 6, rr = sc ? r - 6 * NV : r % 6;
        if (rr == 1 || !keepy(s, ky)) return nullptr;   // rr 1 re-reads rr 0's field
        const int f = sc ? 5 * NV + (rr >> 1) : v * 5 + src_field(rr);
        return src + (long)f * wnf + s.base + (long)i * kxp;
    }
    __device__ __forceinline__ C post(const State &, int r, int i, C x) const
    {
        const int rr = (NS > 0 && r >= 6 * NV) ? r - 6 * NV : r % 6;
        return rr == 1 ? mul_ik(x, (T)wavenumber(i, N) * geo.kfy) : x;
    }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        const int f = (NS > 0 && r >= 6 * NV) ? r : (r / 6) * 6 + dst_field(r % 6);
        if (s.active) st_stream(dst + (long)f * wnf + s.base + (long)i * kxp, v);
    }
    // fp32 pairs: one 16-byte access per element (both sides are the aligned compact layout)
    __device__ __forceinline__ Ex<T> load_e(const State *s, int r, int i) const
    {
        if constexpr (sizeof(T) == 8) return load(s[0], r, i);
        else return load_pair(s, r, i);
    }
    __device__ __forceinline__ float2x2 load_pair(const State *s, int r, int i) const
    {
        const int ky = wavenumber(i, N);
        const bool sc = NS > 0 && r >= 6 * NV;
        const int v = r / 6, rr = sc ? r - 6 * NV : r % 6;
        const bool m0 = keepy(s[0], ky), m1 = keepy(s[1], ky);
        float2x2 x = ezero<float2x2>();
        if (m0 || m1) {
            const int f = sc ? 5 * NV + (rr >> 1) : v * 5 + src_field(rr);
            const float4 *p = reinterpret_cast<const float4 *>(src + (long)f * wnf + s[0].base + (long)i * kxp);
            x = mask2(pack2(rr == 0 ? *p : __ldcs(p)), m0, m1);
        }
        return x;
    }
    __device__ __forceinline__ float2x2 post_e(const State *, int r, int i, float2x2 x) const
    {
        const int rr = (NS > 0 && r >= 6 * NV) ? r - 6 * NV : r % 6;
        return rr == 1 ? mul_ik(x, (float)wavenumber(i, N) * geo.kfy) : x;
    }
    __device__ __forceinline__ double2 post_e(const State *s, int r, int i, double2 x) const { return post(s[0], r, i, x); }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, float2x2 v) const
    {
        const int f = (NS > 0 && r >= 6 * NV) ? r : (r / 6) * 6 + dst_field(r % 6);
        st_stream2(dst + (long)f * wnf + s[0].base + (long)i * kxp, v, s[0].active, s[1].active);
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, double2 v) const { store(s[0], r, i, v); }
};

// ---- fwd_y -------------------------------------------------------------------------------------
template <typename T, int N, int TC, class G> struct JobFwdY : JobElems<JobFwdY<T, N, TC, G>, Cx<T>, Ex<T>> {
    using C = Cx<T>;
    C *buf;  // NF fields, in place, compact layout
    long wplane, wnf;
    int kxp, nfields;
    G geo;
    struct State { long base; int kx; bool active; };
    static constexpr bool prefetch_next = sizeof(T) == 4;

    __host__ __device__ __forceinline__ int rounds() const { return nfields; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        s.kx = (int)colidx;
        s.active = s.kx < geo.kxc;
        s.base = (long)blockIdx.y * wplane + s.kx;
        return true;
    }
    __device__ __forceinline__ bool keepy(const State &s, int ky) const { return s.active && geo.keep2(geo.w2(s.kx, ky)); }
    __device__ __forceinline__ void idle(const State &, int, int) const {}
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (s.active) x = ld_stream(buf + r * wnf + s.base + (long)i * kxp);
        return x;
    }
    __device__ __forceinline__ const void *next_addr(const State &s, int r, int i) const
    {
        return s.active ? buf + r * wnf + s.base + (long)i * kxp : nullptr;
    }
    __device__ __forceinline__ C post(const State &, int, int, C x) const { return x; }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (keepy(s, wavenumber(i, N))) st_stream(buf + r * wnf + s.base + (long)i * kxp, v);
    }
    // fp32 pairs: one 16-byte access per element
    __device__ __forceinline__ Ex<T> load_e(const State *s, int r, int i) const
    {
        if constexpr (sizeof(T) == 8) return load(s[0], r, i);
        else return load_pair(s, r, i);
    }
    __device__ __forceinline__ float2x2 load_pair(const State *s, int r, int i) const
    {
        float2x2 x = ezero<float2x2>();
        if (s[0].active || s[1].active)
            x = mask2(pack2(__ldcs(reinterpret_cast<const float4 *>(buf + r * wnf + s[0].base + (long)i * kxp))),
                      s[0].active, s[1].active);
        return x;
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, float2x2 v) const
    {
        const int ky = wavenumber(i, N);
        st_stream2(buf + r * wnf + s[0].base + (long)i * kxp, v, keepy(s[0], ky), keepy(s[1], ky));
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, double2 v) const { store(s[0], r, i, v); }
};

// ---- fwd_z + epilogue ----------------------------------------------------------------------------
// groups of 3 rounds (components x, y, z of one vector field).  Group g: mode[g] = 0 -> P f - d |k|^2 a
// (momentum), 1 -> i k x f - d |k|^2 a (induction); a = aux[g] (u^ or b^), d = diff[g].
// Boussinesq (NS = 1): one more round for s^ = F[u . grad theta]; its store forms
// R_theta = -s^ + N_bv u^_z - kappa |k|^2 theta^, and the z component of group 0 gets -N_bv theta^
// before the projection (Eqs. 1-2).
// Works on single columns in both precisions (the two columns of an fp32 pair would sit in different rows
// of the caller's odd-pitch layout, and the epilogue is per mode anyway).
template <typename T, int N, int TC, int NV, int NS, class G> struct JobFwdZ : JobElems<JobFwdZ<T, N, TC, NV, NS, G>, Cx<T>, Cx<T>> {
    using C = Cx<T>;
    const C *src;        // NV x 3 (+ NS) fields (after fwd_y), compact layout
    C *dst[NV];          // NV outputs of 3 fields, caller layout
    const C *aux[NV];    // u^, b^ for the diffusion term
    T diff[NV];
    C *sdst;             // NS = 1: R_theta, caller layout
    const C *saux;       // NS = 1: theta^
    T sdiff, nbv;        // kappa, N_bv
    const C *base[NV];   // Runge-Kutta stage: y_n (NULL: plain right-hand side); out = base + cstep * rhs
    const C *sbase;
    T cstep;
    bool sparse;         // intermediate Runge-Kutta stage: the zeros outside the truncation sphere are not written
                         // (the next stage masks on load and never reads them)
    static constexpr bool split_rounds = false;   // the third component's epilogue reads the first two back
    static constexpr bool is_fwdz = true;
    long plane, nf;      // caller layout
    long wplane, wnf;    // workspace layout
    int ldk, kxp;
    G geo;
    struct State { long col, wcol; int kx, ky, kxy2; bool active, valid; };   // kxy2: weighted (mask) form

    __host__ __device__ __forceinline__ int rounds() const { return 3 * NV + NS; }
    // grid (ceil(ldk N / TC)): tile = TC consecutive columns of the caller's (ky, kx) plane, whose
    // 128-byte rows are line-aligned (the plane size ldk N is a multiple of TC); the workspace side
    // is read at the compact address of the same (ky, kx)
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        s.col = colidx;
        s.valid = s.col < plane;
        s.active = false;
        s.kx = s.ky = s.kxy2 = 0;
        s.wcol = 0;
        if (s.valid) {
            s.kx = (int)(s.col % ldk);
            const int q = (int)(s.col / ldk);
            s.ky = wavenumber(q, geo.ny);
            s.kxy2 = geo.w2(s.kx, s.ky);
            s.active = geo.keep2(s.kxy2);
            s.wcol = (long)q * kxp + s.kx;
        }
        return s.active;
    }
    // nothing retained in this tile: the output is all zeros (thread t of nt writes rows t, t + nt, ...)
    __device__ __forceinline__ void idle(const State &s, int t, int nt) const
    {
        if (!s.valid || sparse) return;
        const C z = mk<T>(0, 0);
        for (int g = 0; g < NV; ++g)
            for (int comp = 0; comp < 3; ++comp)
                for (int i = t; i < N; i += nt)
                    st_stream((g == 0 ? dst[0] : dst[NV - 1]) + comp * nf + i * plane + s.col, z);
        if (NS > 0)
            for (int i = t; i < N; i += nt) st_stream(sdst + i * plane + s.col, z);
    }
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (s.active) x = ld_stream(src + r * wnf + i * wplane + s.wcol);
        return x;
    }
    __device__ __forceinline__ C post(const State &, int, int, C x) const { return x; }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (!s.valid) return;
        const int g = r / 3, comp = r % 3;
        const int kz = wavenumber(i, N);
        const bool keep = s.active && geo.keep3(s.kxy2, kz);
        if (NS > 0 && r == 3 * NV) {   // Eq. 2: R_theta = -s^ + N_bv u^_z - kappa |k|^2 theta^
            C *os = sdst + i * plane + s.col;
            if (!keep) { if (!sparse) *os = mk<T>(0, 0); return; }
            C rt = mk<T>(-v.x, -v.y);
            if (nbv != (T)0) {
                const C uz = ldg_c(aux[0] + 2 * nf + i * plane + s.col);
                rt.x += nbv * uz.x; rt.y += nbv * uz.y;
            }
            if (sdiff != (T)0) {
                const T qx = (T)s.kx * geo.kfx, qy = (T)s.ky * geo.kfy, qz = (T)kz * geo.kfz;
                const T sc = sdiff * (qx * qx + qy * qy + qz * qz);
                const C th = ldg_c(saux + i * plane + s.col);
                rt.x -= sc * th.x; rt.y -= sc * th.y;
            }
            if (sbase != nullptr) {   // Runge-Kutta stage
                const C y0 = ldg_c(sbase + i * plane + s.col);
                rt.x = y0.x + cstep * rt.x; rt.y = y0.y + cstep * rt.y;
            }
            *os = rt;
            return;
        }
        C *o = (g == 0 ? dst[0] : dst[NV - 1]) + i * plane + s.col;
        if (!keep) { if (!sparse) o[comp * nf] = mk<T>(0, 0); return; }
        if (comp < 2) { o[comp * nf] = v; return; }   // raw; read back here by this same thread (same address: ordered)
        finish(s, g, i, o, __ldcg(o), __ldcg(o + nf), v);
    }
    // epilogue of one retained mode: (fx, fy, fz) = raw transform of the three components
    __device__ __forceinline__ void finish(const State &s, int g, int i, C *o, C fx, C fy, C fz) const
    {
        const int kz = wavenumber(i, N);
        const T qx = (T)s.kx * geo.kfx, qy = (T)s.ky * geo.kfy, qz = (T)kz * geo.kfz;
        const T k2 = qx * qx + qy * qy + qz * qz;
        if (g == 0) {            // a10: projection, identity at k = 0
            if (NS > 0 && nbv != (T)0) {   // Eq. 1: buoyancy -N_bv theta z^, inside the projection
                const C th = ldg_c(saux + i * plane + s.col);
                fz.x -= nbv * th.x; fz.y -= nbv * th.y;
            }
            if (k2 != (T)0) {
                const T inv = (T)1 / k2;
                const T dr = (qx * fx.x + qy * fy.x + qz * fz.x) * inv;
                const T di = (qx * fx.y + qy * fy.y + qz * fz.y) * inv;
                fx.x -= qx * dr; fx.y -= qx * di;
                fy.x -= qy * dr; fy.y -= qy * di;
                fz.x -= qz * dr; fz.y -= qz * di;
            }
        } else {                 // induction: i k x e
            const C rx = mk<T>(-(qy * fz.y - qz * fy.y), qy * fz.x - qz * fy.x);
            const C ry = mk<T>(-(qz * fx.y - qx * fz.y), qz * fx.x - qx * fz.x);
            const C rz = mk<T>(-(qx * fy.y - qy * fx.y), qx * fy.x - qy * fx.x);
            fx = rx; fy = ry; fz = rz;
        }
        const T dg = g == 0 ? diff[0] : diff[NV - 1];
        if (dg != (T)0) {   // a11
            const T sc = dg * k2;
            const C *a = (g == 0 ? aux[0] : aux[NV - 1]) + i * plane + s.col;
            const C ax = ldg_c(a), ay = ldg_c(a + nf), az = ldg_c(a + 2 * nf);
            fx.x -= sc * ax.x; fx.y -= sc * ax.y;
            fy.x -= sc * ay.x; fy.y -= sc * ay.y;
            fz.x -= sc * az.x; fz.y -= sc * az.y;
        }
        const C *yb = g == 0 ? base[0] : base[NV - 1];
        if (yb != nullptr) {   // Runge-Kutta stage: y_n + (dt / o) R
            yb += i * plane + s.col;
            const C bx = ldg_c(yb), by = ldg_c(yb + nf), bz = ldg_c(yb + 2 * nf);
            fx.x = bx.x + cstep * fx.x; fx.y = bx.y + cstep * fx.y;
            fy.x = by.x + cstep * fy.x; fy.y = by.y + cstep * fy.y;
            fz.x = bz.x + cstep * fz.x; fz.y = bz.y + cstep * fz.y;
        }
        o[0] = fx; o[nf] = fy; o[2 * nf] = fz;
    }
};

// ------------------------------------------------------------------------------------------
// Gross-Pitaevskii equation (Eq. 7), psi = p + i q as two real fields: plain masked
// inverse z / y passes of NF fields, and the fwd_z epilogue R_p = beta a^ + alpha |k|^2 q^,
// R_q = -beta b^ - alpha |k|^2 p^ (a = |psi|^2 q, b = |psi|^2 p from mid_x).
// ------------------------------------------------------------------------------------------
template <typename T, int N, int TC, int NF, class G> struct JobPlainInvZ : JobElems<JobPlainInvZ<T, N, TC, NF, G>, Cx<T>, Ex<T>> {
    using C = Cx<T>;
    const C *src;       // NF spectral fields, caller layout
    C *dst;             // NF compact fields
    long plane, nf, wplane, wnf;
    int ldk, kxp;
    G geo;
    struct State { long col, wcol; int kxy2; bool active; };
    __host__ __device__ __forceinline__ int rounds() const { return NF; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        const int kx = (int)colidx, ky = wavenumber((int)blockIdx.y, geo.ny);
        s.kxy2 = geo.w2(kx, ky);
        s.active = geo.keep2(s.kxy2);
        s.col = (long)blockIdx.y * ldk + kx;
        s.wcol = (long)blockIdx.y * kxp + kx;
        return s.active;
    }
    __device__ __forceinline__ void idle(const State &, int, int) const {}
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (s.active && geo.keep3(s.kxy2, wavenumber(i, N))) x = ldg_c(src + r * nf + i * plane + s.col);
        return x;
    }
    __device__ __forceinline__ C post(const State &, int, int, C x) const { return x; }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (s.active) st_stream(dst + r * wnf + i * wplane + s.wcol, v);
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, float2x2 v) const
    {
        st_stream2(dst + r * wnf + i * wplane + s[0].wcol, v, s[0].active, s[1].active);
    }
    __device__ __forceinline__ void store_e(const State *s, int r, int i, double2 v) const { store(s[0], r, i, v); }
};

// in place on NF compact fields; reads only the retained (ky, kx), writes every ky of the retained kx
template <typename T, int N, int TC, class G> struct JobPlainInvY : JobElems<JobPlainInvY<T, N, TC, G>, Cx<T>, Ex<T>> {
    using C = Cx<T>;
    C *buf;
    long wplane, wnf;
    int kxp, nfields;
    G geo;
    struct State { long base; int kx; bool active; };
    __host__ __device__ __forceinline__ int rounds() const { return nfields; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        s.kx = (int)colidx;
        s.active = s.kx < geo.kxc;
        s.base = (long)blockIdx.y * wplane + s.kx;
        return true;
    }
    __device__ __forceinline__ void idle(const State &, int, int) const {}
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (s.active && geo.keep2(geo.w2(s.kx, wavenumber(i, N)))) x = ld_stream(buf + r * wnf + s.base + (long)i * kxp);
        return x;
    }
    __device__ __forceinline__ C post(const State &, int, int, C x) const { return x; }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (s.active) st_stream(buf + r * wnf + s.base + (long)i * kxp, v);
    }
};

template <typename T, int N, int TC, class G> struct JobGpeFwdZ : JobElems<JobGpeFwdZ<T, N, TC, G>, Cx<T>, Cx<T>> {
    using C = Cx<T>;
    const C *src;        // 2 compact fields (after fwd_y): a^, b^
    C *dst;              // 2 fields, caller layout: R_p, R_q
    const C *psi;        // p^, q^ (caller layout) for the dispersion term
    const C *base;       // Runge-Kutta stage: y_n (NULL: plain right-hand side)
    T alpha, beta, cstep;
    bool sparse;         // as in JobFwdZ
    static constexpr bool split_rounds = false;   // the idle path fills both fields
    static constexpr bool is_fwdz = true;
    long plane, nf, wplane, wnf;
    int ldk, kxp;
    G geo;
    struct State { long col, wcol; int kxy2; T kr2; bool active, valid; };   // kr2 = kx^2 + ky^2 (physical)
    __host__ __device__ __forceinline__ int rounds() const { return 2; }
    __device__ __forceinline__ bool begin(State &s, long colidx) const
    {
        s.col = colidx;
        s.valid = s.col < plane;
        s.active = false;
        s.kxy2 = 0;
        s.kr2 = (T)0;
        s.wcol = 0;
        if (s.valid) {
            const int kx = (int)(s.col % ldk), q = (int)(s.col / ldk), ky = wavenumber(q, geo.ny);
            s.kxy2 = geo.w2(kx, ky);
            const T qx = (T)kx * geo.kfx, qy = (T)ky * geo.kfy;
            s.kr2 = qx * qx + qy * qy;
            s.active = geo.keep2(s.kxy2);
            s.wcol = (long)q * kxp + kx;
        }
        return s.active;
    }
    __device__ __forceinline__ void idle(const State &s, int t, int nt) const
    {
        if (!s.valid || sparse) return;
        for (int r = 0; r < 2; ++r)
            for (int i = t; i < N; i += nt) st_stream(dst + r * nf + i * plane + s.col, mk<T>(0, 0));
    }
    __device__ __forceinline__ C load(const State &s, int r, int i) const
    {
        C x = mk<T>(0, 0);
        if (s.active) x = ld_stream(src + r * wnf + i * wplane + s.wcol);
        return x;
    }
    __device__ __forceinline__ C post(const State &, int, int, C x) const { return x; }
    __device__ __forceinline__ void store(const State &s, int r, int i, C v) const
    {
        if (!s.valid) return;
        const int kz = wavenumber(i, N);
        C *o = dst + r * nf + i * plane + s.col;
        if (!(s.active && geo.keep3(s.kxy2, kz))) { if (!sparse) *o = mk<T>(0, 0); return; }
        // r = 0: R_p = beta a^ + alpha |k|^2 q^;   r = 1: R_q = -beta b^ - alpha |k|^2 p^
        const T sg = r == 0 ? (T)1 : (T)-1;
        const C other = ldg_c(psi + (1 - r) * nf + i * plane + s.col);
        const T qz = (T)kz * geo.kfz;
        const T d = sg * alpha * (s.kr2 + qz * qz), b = sg * beta;
        C res = mk<T>(b * v.x + d * other.x, b * v.y + d * other.y);
        if (base != nullptr) {
            const C y0 = ldg_c(base + r * nf + i * plane + s.col);
            res.x = y0.x + cstep * res.x; res.y = y0.y + cstep * res.y;
        }
        *o = res;
    }
};

}  // namespace psfft
