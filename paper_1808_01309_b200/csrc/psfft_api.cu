// psfft_api.cu -- plan object and the extern "C" boundary declared in include/psfft.h.
// Host logic only; every step of the path runs in the kernels of psfft_kernels.cuh.
#include <math.h>
#include <cmath>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <initializer_list>
#include <mutex>
#include <new>
#include <unordered_set>
#include <vector>

#include "../../include/psfft.h"
#include "psfft_core.cuh"
#include "psfft_launch.cuh"

using namespace psfft;

namespace psfft {
// entries are padded to multiples of 16 so that each table starts 256-byte aligned
// the symmetric schedule RM, (factors of N / RM^2), RM of psfft_midxg.cuh (XSched) for a runtime N
int xsched_stages(int N, int *radix)
{
    const int RM = (N % 64 == 0) ? 8 : (N % 16 == 0) ? 4 : 2;
    int n = 0, m = N / (RM * RM);
    radix[n++] = RM;
    while (m > 1) {
        const int r = (m % 8 == 0 && m != 16) ? 8 : (m % 4 == 0) ? 4 : (m % 2 == 0) ? 2 : 3;
        radix[n++] = r;
        m /= r;
    }
    radix[n++] = RM;
    return n;
}

TableOffsets table_entries(int Nx, int Ny, int Nz)
{
    auto up = [](size_t n) { return (n + 15) / 16 * 16; };
    TableOffsets o;
    o.y = up((size_t)Nx);
    o.x = o.y + up((size_t)tw_size(Ny));
    int radix[8];
    const int S = xsched_stages(Nx, radix);
    size_t x = 0, Ns = radix[0];
    for (int s = 1; s < S; ++s) { x += (size_t)(radix[s] - 1) * Ns; Ns *= radix[s]; }
    const size_t end_x = o.x + up(x);
    o.z = Nz == Ny ? o.y : end_x;
    o.total = Nz == Ny ? end_x : end_x + up((size_t)tw_size(Nz));
    return o;
}

// Row pitch (complex elements) of the compact RHS workspace fields [Nz][Ny][kxp]: the retained kx count of Nx
// rounded up to whole tiles of BOTH column passes (tile widths are powers of two, so the wider one decides).
int rhs_pitch3(int Nx, int Ny, int Nz, int csize)
{
    const int ew = 16 / csize;
    const int ty = job_cols(Ny) * ew, tz = job_cols(Nz) * ew;
    return kx_pitch(Nx, ty > tz ? ty : tz);
}
}  // namespace psfft

namespace {

const uint32_t PLAN_MAGIC = 0x50534654u;  // "PSFT"

struct ProfRec {
    int kind;
    double bytes;
    cudaEvent_t start, stop;
};

struct Plan {
    uint32_t magic;
    psfft_layout lay;
    void *d_tab;
    int launches;
    bool prof;
    double kf[3];                   // 2 pi / L_i of the box (psfft_plan_set_box; 1 for the default 2 pi box)
    int rx2, ry2, rz2, lim;         // integer form of the 2/3-rule ellipsoid (psfft_rhs.cuh Geom)
    double n_disc, n_sphere;        // retained (ky,kx) columns / retained modes of the half spectrum
    std::vector<ProfRec> recs;      // records since the last reset
    std::vector<cudaEvent_t> pool;  // events available for reuse
};

const char *const KERNEL_NAMES[] = {"xpass_r2c", "xpass_c2r", "cpass_y", "cpass_z", "mask_curl", "cross", "finish",
                                    "rhs_inv_z", "rhs_inv_y", "rhs_mid_x", "rhs_fwd_y", "rhs_fwd_z"};
enum { K_XR2C = 0, K_XC2R, K_CPY, K_CPZ, K_MASKCURL, K_CROSS, K_FINISH, K_INVZ, K_INVY, K_MIDX, K_FWDY, K_FWDZ, K_COUNT };

cudaEvent_t take_event(Plan *pl)
{
    cudaEvent_t e = nullptr;
    if (!pl->pool.empty()) { e = pl->pool.back(); pl->pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}

// per-launch CUDA events on the launching stream (only when profiling is on)
struct ProfScope {
    Plan *pl;
    cudaStream_t st;
    ProfScope(Plan *p, cudaStream_t s, int kind, double bytes) : pl(p), st(s)
    {
        if (!pl->prof) return;
        ProfRec r;
        r.kind = kind;
        r.bytes = bytes;
        r.start = take_event(pl);
        r.stop = take_event(pl);
        cudaEventRecord(r.start, st);
        pl->recs.push_back(r);
    }
    ~ProfScope()
    {
        if (pl->prof) cudaEventRecord(pl->recs.back().stop, st);
    }
};

bool supported_n(int N)
{
    switch (N) {
#define X(n) case n:
        PSFFT_FOR_EACH_N(X)
#undef X
        return true;
    }
    return false;
}

int fill_layout(int N, int Ny, int Nz, int dtype, int batch, psfft_layout *o)
{
    if (!o) return PSFFT_E_NULL;
    if (dtype != PSFFT_F32 && dtype != PSFFT_F64) return PSFFT_E_DTYPE;
    if (!supported_n(N) || !supported_n(Ny) || !supported_n(Nz) || batch < 1) return PSFFT_E_SIZE;
    // the y-pass puts (z plane, field) on gridDim.y (<= 65535)
    if ((long)batch * Nz > 65535) return PSFFT_E_BATCH;
    const size_t s = dtype == PSFFT_F64 ? 8 : 4;
    memset(o, 0, sizeof(*o));
    o->N = N;
    o->Ny = Ny;
    o->Nz = Nz;
    o->dtype = dtype;
    o->batch = batch;
    o->ldk = N / 2 + 1;
    o->real_elems = (size_t)N * Ny * Nz;
    o->spec_elems = (size_t)o->ldk * Ny * Nz;
    o->real_bytes = o->real_elems * s;
    o->spec_bytes = o->spec_elems * 2 * s;
    o->table_bytes = table_entries(N, Ny, Nz).total * 2 * s;
    o->work_bytes_fft = (size_t)batch * o->spec_bytes;
    // fused path: 5 + 6 compact fields [Nz][Ny][kx pitch] per vector field; unfused path (cubic plans only): 12 C
    // per vector field
    const size_t wfield = (size_t)Nz * Ny * rhs_pitch3(N, Ny, Nz, (int)(2 * s)) * 2 * s;
    const bool cube = Ny == N && Nz == N;
    o->work_bytes_hd = (cube && 12 * o->spec_bytes > 11 * wfield) ? 12 * o->spec_bytes : 11 * wfield;
    o->work_bytes_mhd = 2 * o->work_bytes_hd;
    o->work_bytes_boussinesq = 16 * wfield;   // 5 + 2 z-fields, 6 + 3 y-fields
    o->work_bytes_gpe = 4 * wfield;           // 2 z/y-fields, 2 x-out fields
    return PSFFT_OK;
}

inline bool cubic(const psfft_layout &l) { return l.Ny == l.N && l.Nz == l.N; }
// cubic grid in the default 2 pi box (every 2 pi / L_i exactly 1): what the *_unfused kernels assume
inline bool unit_cube(const Plan *pl) { return cubic(pl->lay) && pl->kf[0] == 1.0 && pl->kf[1] == 1.0 && pl->kf[2] == 1.0; }
inline bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

// Live plans.  A handle is looked up here before it is dereferenced, so a destroyed or made-up handle is
// answered with PSFFT_E_PLAN instead of a read through a dangling pointer.
std::mutex g_plans_mu;
std::unordered_set<const Plan *> g_plans;

Plan *get(psfft_plan p)
{
    Plan *pl = reinterpret_cast<Plan *>(p);
    if (!pl) return nullptr;
    std::lock_guard<std::mutex> lock(g_plans_mu);
    return g_plans.count(pl) ? pl : nullptr;
}

// "Input and output of one call must not overlap; the workspace must overlap neither" (psfft.h): byte ranges
// of the call, checked on the host before anything is enqueued.  Inputs may alias one another (they are only
// read); every written range (outputs, workspace) must be disjoint from every other range.
struct Span {
    const void *p;
    size_t n;
    bool written;
};
bool spans_overlap(const Span *first, const Span *last)
{
    for (const Span *a = first; a != last; ++a) {
        if (!a->p || !a->n) continue;
        const uintptr_t a0 = reinterpret_cast<uintptr_t>(a->p), a1 = a0 + a->n;
        for (const Span *b = a + 1; b != last; ++b) {
            if (!b->p || !b->n || !(a->written || b->written)) continue;
            const uintptr_t b0 = reinterpret_cast<uintptr_t>(b->p), b1 = b0 + b->n;
            if (a0 < b1 && b0 < a1) return true;
        }
    }
    return false;
}
bool spans_overlap(std::initializer_list<Span> spans) { return spans_overlap(spans.begin(), spans.end()); }

PassArgs args_of(const Plan *pl, void *stream)
{
    PassArgs a;
    const size_t cs = pl->lay.dtype == PSFFT_F64 ? 16 : 8;
    const TableOffsets o = table_entries(pl->lay.N, pl->lay.Ny, pl->lay.Nz);
    a.tab = pl->d_tab;
    a.twN = a.twY = static_cast<const char *>(pl->d_tab) + o.y * cs;
    a.twX = static_cast<const char *>(pl->d_tab) + o.x * cs;
    a.twZ = static_cast<const char *>(pl->d_tab) + o.z * cs;
    a.N = pl->lay.N;
    a.Ny = pl->lay.Ny;
    a.Nz = pl->lay.Nz;
    a.ldk = pl->lay.ldk;
    a.stream = reinterpret_cast<cudaStream_t>(stream);
    a.kxp = rhs_pitch3(a.N, a.Ny, a.Nz, (int)cs);
    a.kxc = kx_count(a.N);
    a.rx2 = pl->rx2; a.ry2 = pl->ry2; a.rz2 = pl->rz2; a.lim = pl->lim;
    for (int i = 0; i < 3; ++i) a.kf[i] = pl->kf[i];
    a.unit_cube = unit_cube(pl);
    return a;
}

#define CU(call)                                   \
    do {                                           \
        cudaError_t e__ = (call);                  \
        if (e__ != cudaSuccess) return (int)e__;   \
    } while (0)

inline char *off(void *p, size_t bytes) { return static_cast<char *>(p) + bytes; }
inline const char *off(const void *p, size_t bytes) { return static_cast<const char *>(p) + bytes; }

// ---- transforms ----------------------------------------------------------------------------
template <typename T> int r2c_fields(Plan *pl, const PassArgs &a, const void *d_real, void *d_spec, int fields)
{
    const long nrows = (long)fields * a.Ny * a.Nz;
    const double C = (double)pl->lay.spec_bytes * fields, R = (double)pl->lay.real_bytes * fields;
    { ProfScope ps(pl, a.stream, K_XR2C, R + C); CU(launch_xpass_r2c<T>(a, d_real, d_spec, nrows, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass<T>(a, -1, 1, d_spec, d_spec, fields, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_CPZ, 2 * C); CU(launch_cpass<T>(a, -1, 2, d_spec, d_spec, fields, &pl->launches)); }
    return PSFFT_OK;
}

// d_spec_work holds the spectra and is overwritten
template <typename T> int c2r_fields_inplace(Plan *pl, const PassArgs &a, const void *d_spec_in, void *d_spec_work,
                                             void *d_real, int fields)
{
    const long nrows = (long)fields * a.Ny * a.Nz;
    const double scale = 1.0 / ((double)a.N * a.Ny * a.Nz);
    const double C = (double)pl->lay.spec_bytes * fields, R = (double)pl->lay.real_bytes * fields;
    { ProfScope ps(pl, a.stream, K_CPZ, 2 * C); CU(launch_cpass<T>(a, +1, 2, d_spec_in, d_spec_work, fields, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass<T>(a, +1, 1, d_spec_work, d_spec_work, fields, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_XC2R, R + C); CU(launch_xpass_c2r<T>(a, d_spec_work, d_real, nrows, scale, &pl->launches)); }
    return PSFFT_OK;
}

// ---- right-hand sides, fused five-pass path (psfft_rhs.cuh) ------------
// Algorithmic bytes per launch = what the pass must read and write given the known-zero structure
// of the dealiased spectra: n_disc retained (ky,kx) columns,
// n_sphere retained modes, KX = kx_count(N) retained kx.
// System: nv vector fields (1 = HD, 2 = MHD) and ns scalars (Boussinesq: nv = 1, ns = 1).
struct RhsSys {
    int nv, ns;
    const void *uhat, *bhat, *thhat;
    void *ru, *rb, *rt;
    double nu, eta, kappa, nbv;
    // Runge-Kutta stage: outputs are base + cstep * rhs (base_u == NULL: plain right-hand side)
    const void *base_u, *base_b, *base_t;
    double cstep;
    bool sparse_out;   // intermediate Runge-Kutta stage: zeros outside the sphere are not written
};

template <typename T> int rhs_fused_t(Plan *pl, const PassArgs &a, const RhsSys &y, void *work)
{
    const size_t C = pl->lay.spec_bytes;
    const double cs = (double)(2 * sizeof(T)), KX = a.kxc;
    const int nv = y.nv, ns = y.ns;
    RhsArgs r;
    r.nv = nv; r.ns = ns;
    r.src[0] = y.uhat; r.src[1] = y.bhat;
    r.dst[0] = y.ru; r.dst[1] = y.rb;
    r.diff[0] = y.nu; r.diff[1] = y.eta;
    r.ssrc = y.thhat; r.sdst = y.rt;
    r.sdiff = y.kappa; r.nbv = y.nbv;
    r.base[0] = y.base_u; r.base[1] = y.base_b; r.sbase = y.base_t; r.cstep = y.cstep;
    r.sparse_out = y.sparse_out;
    const size_t W = (size_t)a.Nz * a.Ny * a.kxp * 2 * sizeof(T);
    r.zbuf = work;                                         // 5 nv + 2 ns compact fields (later 3 nv + ns: mid_x out, fwd_y in place)
    r.ybuf = off(work, (size_t)(5 * nv + 2 * ns) * W);     // 6 nv + 3 ns compact fields
    const double disc = pl->n_disc * a.Nz * cs, rows = KX * a.Ny * a.Nz * cs, sph = pl->n_sphere * cs;
    // sparse re-reads of the inputs in the fwd_z epilogue: diffusion (3 per vector, 1 per scalar), buoyancy
    // (theta^ for R_u, u^_z for R_theta)
    const double nepi = (y.nu != 0.0 ? 3.0 : 0.0) + (nv == 2 && y.eta != 0.0 ? 3.0 : 0.0) +
                        (ns ? (y.kappa != 0.0 || y.nbv != 0.0 ? 1.0 : 0.0) + (y.nbv != 0.0 && y.nu == 0.0 ? 1.0 : 0.0) : 0.0);
    const int zin = 3 * nv + ns, zf = 5 * nv + 2 * ns, yf = 6 * nv + 3 * ns, ff = 3 * nv + ns;
    const double nbase = y.base_u ? (double)ff : 0.0;   // sparse reads of y_n in a Runge-Kutta stage
    { ProfScope ps(pl, a.stream, K_INVZ, zin * sph + zf * disc); CU(launch_rhs_inv_z<T>(a, r, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_INVY, zf * disc + yf * rows); CU(launch_rhs_inv_y<T>(a, r, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_MIDX, yf * rows + ff * rows); CU(launch_rhs_mid_x<T>(a, r, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_FWDY, ff * rows + ff * disc); CU(launch_rhs_fwd_y<T>(a, r, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_FWDZ, ff * disc + ff * (y.sparse_out ? sph : (double)C) + (nepi + nbase) * sph); CU(launch_rhs_fwd_z<T>(a, r, &pl->launches)); }
    return PSFFT_OK;
}

// ---- Gross-Pitaevskii right-hand side (five passes, psfft_rhs.cuh / psfft_midxg.cuh) -----------------
template <typename T>
int gpe_t(Plan *pl, const PassArgs &a, const void *psi, void *rhs, double alpha, double beta, const void *base,
          double cstep, bool sparse_out, void *work)
{
    const size_t C = pl->lay.spec_bytes;
    const double cs = (double)(2 * sizeof(T)), KX = a.kxc;
    const size_t W = (size_t)a.Nz * a.Ny * a.kxp * 2 * sizeof(T);
    GpeArgs g;
    g.psi = psi; g.dst = rhs; g.base = base;
    g.alpha = alpha; g.beta = beta; g.cstep = cstep; g.sparse_out = sparse_out;
    g.zbuf = work;
    g.obuf = off(work, 2 * W);
    const double disc = pl->n_disc * a.Nz * cs, rows = KX * a.Ny * a.Nz * cs, sph = pl->n_sphere * cs;
    const double nepi = (alpha != 0.0 ? 2.0 : 0.0) + (base ? 2.0 : 0.0);
    { ProfScope ps(pl, a.stream, K_INVZ, 2 * sph + 2 * disc); CU(launch_gpe_pass<T>(a, g, 0, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_INVY, 2 * disc + 2 * rows); CU(launch_gpe_pass<T>(a, g, 1, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_MIDX, 2 * rows + 2 * rows); CU(launch_gpe_pass<T>(a, g, 2, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_FWDY, 2 * rows + 2 * disc); CU(launch_gpe_pass<T>(a, g, 3, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_FWDZ, 2 * disc + 2 * (sparse_out ? sph : (double)C) + nepi * sph); CU(launch_gpe_pass<T>(a, g, 4, &pl->launches)); }
    return PSFFT_OK;
}

// ---- right-hand sides, unfused composition of the public passes (cross-check path) -------------
template <typename T> int hd_rhs_t(Plan *pl, const PassArgs &a, const void *uhat, void *rhs, double nu, void *work)
{
    const size_t C = pl->lay.spec_bytes, R = pl->lay.real_bytes;
    void *W0 = work;               // 6 C: (M u^, w^), later 3 R: u x w
    void *W1 = off(work, 6 * C);   // 6 R: (u, w), later 3 C: F[u x w]
    { ProfScope ps(pl, a.stream, K_MASKCURL, 9.0 * C); CU(launch_mask_curl<T>(a, uhat, W0, &pl->launches)); }
    int rc = c2r_fields_inplace<T>(pl, a, W0, W0, W1, 6);
    if (rc) return rc;
    { ProfScope ps(pl, a.stream, K_CROSS, 9.0 * R); CU(launch_cross<T>(a, W1, off(W1, 3 * R), W0, &pl->launches)); }
    rc = r2c_fields<T>(pl, a, W0, W1, 3);
    if (rc) return rc;
    { ProfScope ps(pl, a.stream, K_FINISH, (nu != 0.0 ? 9.0 : 6.0) * C); CU(launch_finish<T>(a, 0, W1, uhat, rhs, nu, &pl->launches)); }
    return PSFFT_OK;
}

template <typename T>
int mhd_rhs_t(Plan *pl, const PassArgs &a, const void *uhat, const void *bhat, void *ru, void *rb, double nu,
              double eta, void *work)
{
    const size_t C = pl->lay.spec_bytes, R = pl->lay.real_bytes;
    void *W0 = work;                // 12 C: (M u^, w^, M b^, j^), later 6 R: (m, e)
    void *W1 = off(work, 12 * C);   // 12 R: (u, w, b, j), later 6 C: (F[m], F[e])
    { ProfScope ps(pl, a.stream, K_MASKCURL, 9.0 * C); CU(launch_mask_curl<T>(a, uhat, W0, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_MASKCURL, 9.0 * C); CU(launch_mask_curl<T>(a, bhat, off(W0, 6 * C), &pl->launches)); }
    int rc = c2r_fields_inplace<T>(pl, a, W0, W0, W1, 12);
    if (rc) return rc;
    { ProfScope ps(pl, a.stream, K_CROSS, 18.0 * R);
      CU(launch_cross_mhd<T>(a, W1, off(W1, 6 * R), off(W1, 3 * R), off(W1, 9 * R), W0, off(W0, 3 * R), &pl->launches)); }
    rc = r2c_fields<T>(pl, a, W0, W1, 6);
    if (rc) return rc;
    { ProfScope ps(pl, a.stream, K_FINISH, (nu != 0.0 ? 9.0 : 6.0) * C); CU(launch_finish<T>(a, 0, W1, uhat, ru, nu, &pl->launches)); }
    { ProfScope ps(pl, a.stream, K_FINISH, (eta != 0.0 ? 9.0 : 6.0) * C); CU(launch_finish<T>(a, 1, off(W1, 3 * C), bhat, rb, eta, &pl->launches)); }
    return PSFFT_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

int psfft_plan_query(int N, int dtype, int batch, psfft_layout *out) { return fill_layout(N, N, N, dtype, batch, out); }

int psfft_plan_query3(int Nx, int Ny, int Nz, int dtype, int batch, psfft_layout *out)
{
    return fill_layout(Nx, Ny, Nz, dtype, batch, out);
}

int psfft_plan_create(psfft_plan *plan, int N, int dtype, int batch, void *d_tables, size_t table_bytes, void *stream)
{
    return psfft_plan_create3(plan, N, N, N, dtype, batch, d_tables, table_bytes, stream);
}

int psfft_plan_create3(psfft_plan *plan, int N, int Ny, int Nz, int dtype, int batch, void *d_tables, size_t table_bytes,
                       void *stream)
{
    if (!plan) return PSFFT_E_NULL;
    *plan = nullptr;
    psfft_layout lay;
    int rc = fill_layout(N, Ny, Nz, dtype, batch, &lay);
    if (rc) return rc;
    if (!d_tables) return PSFFT_E_NULL;
    if (misaligned(d_tables)) return PSFFT_E_ALIGN;
    if (table_bytes < lay.table_bytes) return PSFFT_E_TABLE;

    // Every entry is exp(-2 pi i m / n) from the reduced integer m, evaluated in long double and
    // rounded once to the plan dtype.  Layout: table_entries() above.
    std::vector<unsigned char> host(lay.table_bytes);
    const TableOffsets toff = table_entries(N, Ny, Nz);
    const size_t off_twN = toff.y, off_twX = toff.x;
    auto put = [&](size_t idx, long m, long n) {
        m %= n;
        const long double two_pi = 6.283185307179586476925286766559005768L;
        const long double ang = two_pi * (long double)m / (long double)n;
        long double c = cosl(ang), s = -sinl(ang);
        if (m == 0) { c = 1; s = 0; }
        else if (4 * m == n) { c = 0; s = -1; }
        else if (2 * m == n) { c = -1; s = 0; }
        else if (4 * m == 3 * n) { c = 0; s = 1; }
        if (dtype == PSFFT_F64) {
            double *t = reinterpret_cast<double *>(host.data());
            t[2 * idx] = (double)c;
            t[2 * idx + 1] = (double)s;
        } else {
            float *t = reinterpret_cast<float *>(host.data());
            t[2 * idx] = (float)c;
            t[2 * idx + 1] = (float)s;
        }
    };
    for (int m = 0; m < N; ++m) put(m, m, N);
    auto stage_tables = [&](size_t base, int L) {   // layout: psfft_core.cuh tw_offset()
        for (int Ns = 1; Ns < L;) {
            const int R = pick_radix(L / Ns);
            if (Ns > 1)
                for (int r = 1; r < R; ++r)
                    for (int k = 0; k < Ns; ++k) put(base + tw_offset(L, Ns) + (size_t)(r - 1) * Ns + k, (long)r * k, (long)Ns * R);
            Ns *= R;
        }
    };
    stage_tables(off_twN, Ny);
    if (Nz != Ny) stage_tables(toff.z, Nz);
    {   // symmetric schedule of the mid_x transforms: stage s >= 1 with earlier radix product Ns, [r-1][k]
        int radix[8];
        const int S = xsched_stages(N, radix);
        size_t o = off_twX;
        long Ns = radix[0];
        for (int s = 1; s < S; ++s) {
            const int R = radix[s];
            for (int r = 1; r < R; ++r)
                for (long k = 0; k < Ns; ++k) put(o + (size_t)(r - 1) * Ns + k, (long)r * k, Ns * R);
            o += (size_t)(R - 1) * Ns;
            Ns *= R;
        }
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    CU(cudaMemcpyAsync(d_tables, host.data(), lay.table_bytes, cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));

    Plan *pl = new (std::nothrow) Plan;
    if (!pl) return (int)cudaErrorMemoryAllocation;
    pl->magic = PLAN_MAGIC;
    pl->lay = lay;
    pl->d_tab = d_tables;
    pl->launches = 0;
    pl->prof = false;
    {   // 2/3 rule on a general grid (reading G25): keep iff sum (n_i / N_i)^2 < 1/9, in integers
        // 9 sum (r_i n_i)^2 < L^2 with L = lcm(Nx, Ny, Nz), r_i = L / N_i  (cubic: 9 |n|^2 < N^2)
        auto gcd = [](long x, long y) { while (y) { const long t = x % y; x = y; y = t; } return x; };
        long L = (long)N / gcd(N, Ny) * Ny;
        L = L / gcd(L, Nz) * Nz;
        // int32 headroom of GeomAny::w2 / keep3 (psfft_rhs.cuh): sum_i (r_i n_i)^2 <= 3 (L/2)^2 with |n_i| <= N_i / 2.
        // The supported sizes give L <= lcm(2048, 768) = 6144, i.e. 2.8e7; a future size list must not break this.
        if (3 * (L / 2) * (L / 2) > 0x7fffffffL) { delete pl; return PSFFT_E_SIZE; }
        const long rx = L / N, ry = L / Ny, rz = L / Nz;
        pl->rx2 = (int)(rx * rx); pl->ry2 = (int)(ry * ry); pl->rz2 = (int)(rz * rz);
        pl->lim = (int)((L * L + 8) / 9);
        pl->kf[0] = pl->kf[1] = pl->kf[2] = 1.0;   // 2 pi box
        // retained columns / modes, by integer enumeration
        double nd = 0, ns = 0;
        for (int q = 0; q < Ny; ++q) {
            const long ky = q < Ny / 2 ? q : q - Ny;
            for (long kx = 0; kx <= N / 2; ++kx) {
                const long kxy2 = pl->rx2 * kx * kx + pl->ry2 * ky * ky;
                if (kxy2 >= pl->lim) continue;
                nd += 1;
                long cnt = 0;   // kz = 0, 1, ... retained; each kz > 0 also stands for -kz
                while (kxy2 + pl->rz2 * cnt * cnt < pl->lim) ++cnt;
                ns += (double)(2 * cnt - 1);
            }
        }
        pl->n_disc = nd;
        pl->n_sphere = ns;
    }
    {
        std::lock_guard<std::mutex> lock(g_plans_mu);
        g_plans.insert(pl);
    }
    *plan = reinterpret_cast<psfft_plan>(pl);
    return PSFFT_OK;
}

int psfft_plan_destroy(psfft_plan plan)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    {
        std::lock_guard<std::mutex> lock(g_plans_mu);
        g_plans.erase(pl);
    }
    pl->magic = 0;
    for (ProfRec &r : pl->recs) { cudaEventDestroy(r.start); cudaEventDestroy(r.stop); }
    for (cudaEvent_t e : pl->pool) cudaEventDestroy(e);
    delete pl;
    return PSFFT_OK;
}

int psfft_plan_layout(psfft_plan plan, psfft_layout *out)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!out) return PSFFT_E_NULL;
    *out = pl->lay;
    return PSFFT_OK;
}

int psfft_plan_set_box(psfft_plan plan, double Lx, double Ly, double Lz)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    const double L[3] = {Lx, Ly, Lz};
    for (double v : L)
        if (!(v > 0.0) || !std::isfinite(v)) return PSFFT_E_SIZE;
    const double two_pi = 6.283185307179586476925286766559;
    for (int i = 0; i < 3; ++i) pl->kf[i] = two_pi / L[i];   // exactly 1 for L_i = 2 pi
    return PSFFT_OK;
}

int psfft_fft3d_r2c(psfft_plan plan, const void *d_real, void *d_spec, void *d_work, void *stream)
{
    (void)d_work;
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_real || !d_spec) return PSFFT_E_NULL;
    if (misaligned(d_real) || misaligned(d_spec)) return PSFFT_E_ALIGN;
    if (spans_overlap({{d_real, pl->lay.batch * pl->lay.real_bytes, false}, {d_spec, pl->lay.batch * pl->lay.spec_bytes, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    return pl->lay.dtype == PSFFT_F64 ? r2c_fields<double>(pl, a, d_real, d_spec, pl->lay.batch)
                                      : r2c_fields<float>(pl, a, d_real, d_spec, pl->lay.batch);
}

int psfft_fft3d_c2r(psfft_plan plan, const void *d_spec, void *d_real, void *d_work, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_real || !d_spec || !d_work) return PSFFT_E_NULL;
    if (misaligned(d_real) || misaligned(d_spec) || misaligned(d_work)) return PSFFT_E_ALIGN;
    if (spans_overlap({{d_spec, pl->lay.batch * pl->lay.spec_bytes, false}, {d_real, pl->lay.batch * pl->lay.real_bytes, true},
                       {d_work, pl->lay.work_bytes_fft, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    return pl->lay.dtype == PSFFT_F64 ? c2r_fields_inplace<double>(pl, a, d_spec, d_work, d_real, pl->lay.batch)
                                      : c2r_fields_inplace<float>(pl, a, d_spec, d_work, d_real, pl->lay.batch);
}

static int hd_entry(psfft_plan plan, const void *d_uhat, void *d_rhs, double nu, void *d_work, void *stream, bool fused)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    // the unfused cross-check path works in integer wavenumbers on a cube: Nx = Ny = Nz and the default 2 pi box
    if (!fused && !unit_cube(pl)) return PSFFT_E_SIZE;
    if (!d_uhat || !d_rhs || !d_work) return PSFFT_E_NULL;
    if (misaligned(d_uhat) || misaligned(d_rhs) || misaligned(d_work)) return PSFFT_E_ALIGN;
    {
        const size_t C = pl->lay.spec_bytes;
        if (spans_overlap({{d_uhat, 3 * C, false}, {d_rhs, 3 * C, true}, {d_work, pl->lay.work_bytes_hd, true}}))
            return PSFFT_E_OVERLAP;
    }
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    if (fused) {
        const RhsSys y = {1, 0, d_uhat, nullptr, nullptr, d_rhs, nullptr, nullptr, nu, 0.0, 0.0, 0.0,
                          nullptr, nullptr, nullptr, 0.0, false};
        return pl->lay.dtype == PSFFT_F64 ? rhs_fused_t<double>(pl, a, y, d_work) : rhs_fused_t<float>(pl, a, y, d_work);
    }
    return pl->lay.dtype == PSFFT_F64 ? hd_rhs_t<double>(pl, a, d_uhat, d_rhs, nu, d_work)
                                      : hd_rhs_t<float>(pl, a, d_uhat, d_rhs, nu, d_work);
}

static int mhd_entry(psfft_plan plan, const void *d_uhat, const void *d_bhat, void *d_rhs_u, void *d_rhs_b, double nu,
                     double eta, void *d_work, void *stream, bool fused)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    // the unfused cross-check path works in integer wavenumbers on a cube: Nx = Ny = Nz and the default 2 pi box
    if (!fused && !unit_cube(pl)) return PSFFT_E_SIZE;
    if (!d_uhat || !d_bhat || !d_rhs_u || !d_rhs_b || !d_work) return PSFFT_E_NULL;
    if (misaligned(d_uhat) || misaligned(d_bhat) || misaligned(d_rhs_u) || misaligned(d_rhs_b) || misaligned(d_work))
        return PSFFT_E_ALIGN;
    {
        const size_t C = pl->lay.spec_bytes;
        if (spans_overlap({{d_uhat, 3 * C, false}, {d_bhat, 3 * C, false}, {d_rhs_u, 3 * C, true}, {d_rhs_b, 3 * C, true},
                           {d_work, pl->lay.work_bytes_mhd, true}}))
            return PSFFT_E_OVERLAP;
    }
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    if (fused) {
        const RhsSys y = {2, 0, d_uhat, d_bhat, nullptr, d_rhs_u, d_rhs_b, nullptr, nu, eta, 0.0, 0.0,
                          nullptr, nullptr, nullptr, 0.0, false};
        return pl->lay.dtype == PSFFT_F64 ? rhs_fused_t<double>(pl, a, y, d_work) : rhs_fused_t<float>(pl, a, y, d_work);
    }
    return pl->lay.dtype == PSFFT_F64 ? mhd_rhs_t<double>(pl, a, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu, eta, d_work)
                                      : mhd_rhs_t<float>(pl, a, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu, eta, d_work);
}

int psfft_hd_rhs(psfft_plan plan, const void *d_uhat, void *d_rhs, double nu, void *d_work, void *stream)
{
    return hd_entry(plan, d_uhat, d_rhs, nu, d_work, stream, true);
}

int psfft_hd_rhs_unfused(psfft_plan plan, const void *d_uhat, void *d_rhs, double nu, void *d_work, void *stream)
{
    return hd_entry(plan, d_uhat, d_rhs, nu, d_work, stream, false);
}

int psfft_mhd_rhs(psfft_plan plan, const void *d_uhat, const void *d_bhat, void *d_rhs_u, void *d_rhs_b, double nu,
                  double eta, void *d_work, void *stream)
{
    return mhd_entry(plan, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu, eta, d_work, stream, true);
}

int psfft_mhd_rhs_unfused(psfft_plan plan, const void *d_uhat, const void *d_bhat, void *d_rhs_u, void *d_rhs_b,
                          double nu, double eta, void *d_work, void *stream)
{
    return mhd_entry(plan, d_uhat, d_bhat, d_rhs_u, d_rhs_b, nu, eta, d_work, stream, false);
}

int psfft_boussinesq_rhs(psfft_plan plan, const void *d_uhat, const void *d_thhat, void *d_rhs_u, void *d_rhs_th,
                         double nu, double kappa, double nbv, void *d_work, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_uhat || !d_thhat || !d_rhs_u || !d_rhs_th || !d_work) return PSFFT_E_NULL;
    if (misaligned(d_uhat) || misaligned(d_thhat) || misaligned(d_rhs_u) || misaligned(d_rhs_th) || misaligned(d_work))
        return PSFFT_E_ALIGN;
    {
        const size_t C = pl->lay.spec_bytes;
        if (spans_overlap({{d_uhat, 3 * C, false}, {d_thhat, C, false}, {d_rhs_u, 3 * C, true}, {d_rhs_th, C, true},
                           {d_work, pl->lay.work_bytes_boussinesq, true}}))
            return PSFFT_E_OVERLAP;
    }
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    const RhsSys y = {1, 1, d_uhat, nullptr, d_thhat, d_rhs_u, nullptr, d_rhs_th, nu, 0.0, kappa, nbv,
                      nullptr, nullptr, nullptr, 0.0, false};
    return pl->lay.dtype == PSFFT_F64 ? rhs_fused_t<double>(pl, a, y, d_work) : rhs_fused_t<float>(pl, a, y, d_work);
}

int psfft_gpe_rhs(psfft_plan plan, const void *d_psihat, void *d_rhs, double alpha, double beta, void *d_work,
                  void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_psihat || !d_rhs || !d_work) return PSFFT_E_NULL;
    if (misaligned(d_psihat) || misaligned(d_rhs) || misaligned(d_work)) return PSFFT_E_ALIGN;
    if (spans_overlap({{d_psihat, 2 * pl->lay.spec_bytes, false}, {d_rhs, 2 * pl->lay.spec_bytes, true},
                       {d_work, pl->lay.work_bytes_gpe, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    return pl->lay.dtype == PSFFT_F64 ? gpe_t<double>(pl, a, d_psihat, d_rhs, alpha, beta, nullptr, 0.0, false, d_work)
                                      : gpe_t<float>(pl, a, d_psihat, d_rhs, alpha, beta, nullptr, 0.0, false, d_work);
}

static int sys_fields(int system) { return system == PSFFT_SYS_HD ? 3 : system == PSFFT_SYS_MHD ? 6 : system == PSFFT_SYS_GPE ? 2 : 4; }

size_t psfft_rk_work_bytes(psfft_plan plan, int system)
{
    Plan *pl = get(plan);
    if (!pl || system < 0 || system > 3) return 0;
    const size_t rhs = system == PSFFT_SYS_HD ? pl->lay.work_bytes_hd
                     : system == PSFFT_SYS_MHD ? pl->lay.work_bytes_mhd
                     : system == PSFFT_SYS_GPE ? pl->lay.work_bytes_gpe : pl->lay.work_bytes_boussinesq;
    return (size_t)sys_fields(system) * pl->lay.spec_bytes + rhs;
}

int psfft_rk_step(psfft_plan plan, int system, const void *d_y_in, void *d_y_out, int ord, double dt,
                  const double *params, void *d_work, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_y_in || !d_y_out || !d_work || !params) return PSFFT_E_NULL;
    if (system < 0 || system > 3 || ord < 1 || ord > 4) return PSFFT_E_SIZE;
    if (misaligned(d_y_in) || misaligned(d_y_out) || misaligned(d_work)) return PSFFT_E_ALIGN;
    const size_t C = pl->lay.spec_bytes;
    const int nfields = sys_fields(system);
    if (spans_overlap({{d_y_in, nfields * C, false}, {d_y_out, nfields * C, true},
                       {d_work, psfft_rk_work_bytes(plan, system), true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    void *stage = d_work;                                  // one state-sized stage buffer
    void *rhswork = off(d_work, (size_t)nfields * C);
    const void *cur = d_y_in;
    for (int j = 1; j <= ord; ++j) {
        // stage outputs alternate between the stage buffer and d_y_out so that the last one lands in d_y_out
        void *out = ((ord - j) % 2 == 0) ? d_y_out : stage;
        if (system == PSFFT_SYS_GPE) {   // params = { alpha, beta }
            const double cstep = dt / (double)(ord - j + 1);
            const int rc = pl->lay.dtype == PSFFT_F64
                               ? gpe_t<double>(pl, a, cur, out, params[0], params[1], d_y_in, cstep, j < ord, rhswork)
                               : gpe_t<float>(pl, a, cur, out, params[0], params[1], d_y_in, cstep, j < ord, rhswork);
            if (rc) return rc;
            cur = out;
            continue;
        }
        RhsSys y;
        y.nv = system == PSFFT_SYS_MHD ? 2 : 1;
        y.ns = system == PSFFT_SYS_BOUSSINESQ ? 1 : 0;
        y.uhat = cur; y.ru = out; y.base_u = d_y_in;
        y.bhat = y.nv == 2 ? off(cur, 3 * C) : nullptr;
        y.rb = y.nv == 2 ? off(out, 3 * C) : nullptr;
        y.base_b = y.nv == 2 ? off(d_y_in, 3 * C) : nullptr;
        y.thhat = y.ns ? off(cur, 3 * C) : nullptr;
        y.rt = y.ns ? off(out, 3 * C) : nullptr;
        y.base_t = y.ns ? off(d_y_in, 3 * C) : nullptr;
        y.nu = params[0];
        y.eta = system == PSFFT_SYS_MHD ? params[1] : 0.0;
        y.kappa = system == PSFFT_SYS_BOUSSINESQ ? params[1] : 0.0;
        y.nbv = system == PSFFT_SYS_BOUSSINESQ ? params[2] : 0.0;
        y.cstep = dt / (double)(ord - j + 1);
        y.sparse_out = j < ord;   // only the last stage has to define the zeros of d_y_out
        const int rc = pl->lay.dtype == PSFFT_F64 ? rhs_fused_t<double>(pl, a, y, rhswork)
                                                  : rhs_fused_t<float>(pl, a, y, rhswork);
        if (rc) return rc;
        cur = out;
    }
    return PSFFT_OK;
}

int psfft_fft3d_r2c_host(psfft_plan plan, const void *h_real, void *h_spec, void *d_in, void *d_out, void *d_work,
                         void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!h_real || !h_spec || !d_in || !d_out) return PSFFT_E_NULL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const size_t nb = (size_t)pl->lay.batch;
    CU(cudaMemcpyAsync(d_in, h_real, nb * pl->lay.real_bytes, cudaMemcpyHostToDevice, st));
    int rc = psfft_fft3d_r2c(plan, d_in, d_out, d_work, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_spec, d_out, nb * pl->lay.spec_bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return PSFFT_OK;
}

int psfft_fft3d_c2r_host(psfft_plan plan, const void *h_spec, void *h_real, void *d_in, void *d_out, void *d_work,
                         void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!h_real || !h_spec || !d_in || !d_out) return PSFFT_E_NULL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const size_t nb = (size_t)pl->lay.batch;
    CU(cudaMemcpyAsync(d_in, h_spec, nb * pl->lay.spec_bytes, cudaMemcpyHostToDevice, st));
    int rc = psfft_fft3d_c2r(plan, d_in, d_out, d_work, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_real, d_out, nb * pl->lay.real_bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return PSFFT_OK;
}

int psfft_hd_rhs_host(psfft_plan plan, const void *h_uhat, void *h_rhs, double nu, void *d_in, void *d_out,
                      void *d_work, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!h_uhat || !h_rhs || !d_in || !d_out) return PSFFT_E_NULL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    CU(cudaMemcpyAsync(d_in, h_uhat, 3 * pl->lay.spec_bytes, cudaMemcpyHostToDevice, st));
    int rc = psfft_hd_rhs(plan, d_in, d_out, nu, d_work, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_rhs, d_out, 3 * pl->lay.spec_bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return PSFFT_OK;
}

// ---- host entry point that moves only the retained box (psfft_hd_rhs_host_box) -----------------------------------
// Index box around the 2/3-rule ellipsoid: kx in [0, bx), |ky| <= by, |kz| <= bz, from the plan's integer form of the
// rule (rx2 n^2 < lim on each axis with the other two indices 0).  A superset of the retained modes, and exact on the
// axes, so nothing the right-hand side reads or writes as non-zero lies outside it.
struct KeepBox { int bx, by, bz; };
static KeepBox keep_box(const Plan *pl)
{
    auto last = [&](int r2) { long n = 0; while ((long)r2 * (n + 1) * (n + 1) < (long)pl->lim) ++n; return (int)n; };
    return {last(pl->rx2) + 1, last(pl->ry2), last(pl->rz2)};
}

// The box of `fields` spectral fields [kz][ky][kx] between two dense arrays of the caller layout (same layout on both
// sides): per field four 3D copies, one per (ky, kz) index-range quadrant -- indices [0, b] and [N - b, N).
static int copy_box(const Plan *pl, void *dst, const void *src, int fields, cudaMemcpyKind kind, cudaStream_t st)
{
    const size_t cs = pl->lay.dtype == PSFFT_F64 ? 16 : 8, pitch = (size_t)pl->lay.ldk * cs;
    const KeepBox b = keep_box(pl);
    const int Ny = pl->lay.Ny, Nz = pl->lay.Nz;
    for (int f = 0; f < fields; ++f)
        for (int zq = 0; zq < 2; ++zq)
            for (int yq = 0; yq < 2; ++yq) {
                const int z0 = zq ? Nz - b.bz : 0, nz = zq ? b.bz : b.bz + 1;
                const int y0 = yq ? Ny - b.by : 0, ny = yq ? b.by : b.by + 1;
                if (nz <= 0 || ny <= 0) continue;
                cudaMemcpy3DParms p;
                memset(&p, 0, sizeof(p));
                p.srcPtr = make_cudaPitchedPtr(const_cast<char *>(off(src, (size_t)f * pl->lay.spec_bytes)), pitch, pitch, (size_t)Ny);
                p.dstPtr = make_cudaPitchedPtr(off(dst, (size_t)f * pl->lay.spec_bytes), pitch, pitch, (size_t)Ny);
                p.srcPos = make_cudaPos(0, (size_t)y0, (size_t)z0);
                p.dstPos = p.srcPos;
                p.extent = make_cudaExtent((size_t)b.bx * cs, (size_t)ny, (size_t)nz);
                p.kind = kind;
                CU(cudaMemcpy3DAsync(&p, st));
            }
    return PSFFT_OK;
}

size_t psfft_host_box_bytes(psfft_plan plan)
{
    Plan *pl = get(plan);
    if (!pl) return 0;
    const KeepBox b = keep_box(pl);
    return (size_t)b.bx * (size_t)(2 * b.by + 1) * (size_t)(2 * b.bz + 1) * (pl->lay.dtype == PSFFT_F64 ? 16 : 8);
}

int psfft_hd_rhs_host_box(psfft_plan plan, const void *h_uhat, void *h_rhs, double nu, void *d_in, void *d_out,
                          void *d_work, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!h_uhat || !h_rhs || !d_in || !d_out) return PSFFT_E_NULL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int rc = copy_box(pl, d_in, h_uhat, 3, cudaMemcpyHostToDevice, st);
    if (rc) return rc;
    rc = psfft_hd_rhs(plan, d_in, d_out, nu, d_work, stream);
    if (rc) return rc;
    rc = copy_box(pl, h_rhs, d_out, 3, cudaMemcpyDeviceToHost, st);
    if (rc) return rc;
    CU(cudaStreamSynchronize(st));
    return PSFFT_OK;
}

// ---- slab-decomposed transform (psfft_slab.cuh) --------------------------------------------------
static int slab_ranges(const Plan *pl, int P, int rank, psfft_slab_layout *o)
{
    if (P < 1 || P > PSFFT_MAX_RANKS || rank < 0 || rank >= P) return PSFFT_E_SIZE;
    if (pl->lay.Nz % P != 0 || P > pl->lay.ldk) return PSFFT_E_SIZE;
    const size_t s = pl->lay.dtype == PSFFT_F64 ? 8 : 4;
    memset(o, 0, sizeof(*o));
    o->P = P;
    o->rank = rank;
    o->Mz = pl->lay.Nz / P;
    o->z0 = rank * o->Mz;
    for (int q = 0; q <= P; ++q) o->x0[q] = (int)((long)q * pl->lay.ldk / P);
    o->w = o->x0[rank + 1] - o->x0[rank];
    o->real_elems = (size_t)o->Mz * pl->lay.Ny * pl->lay.N;
    o->zspec_elems = (size_t)o->Mz * pl->lay.Ny * pl->lay.ldk;
    o->xslab_elems = (size_t)pl->lay.Nz * pl->lay.Ny * o->w;
    o->real_bytes = o->real_elems * s;
    o->zspec_bytes = o->zspec_elems * 2 * s;
    o->xslab_bytes = o->xslab_elems * 2 * s;
    return PSFFT_OK;
}

static int slab_xdist(const Plan *pl, const psfft_slab_layout &sl, void *const *blocks, long zoff, XDistArgs *xd)
{
    // the planes [zoff, zoff + Mz) of every block must exist: a block has at most Nz planes (direct mode: it is the
    // x-slab of its rank, which may be peer memory -- a store past its end would land in someone else's data)
    if (zoff < 0 || zoff + sl.Mz > pl->lay.Nz) return PSFFT_E_SIZE;
    memset(xd, 0, sizeof(*xd));
    for (int q = 0; q < sl.P; ++q) {
        if (!blocks[q]) return PSFFT_E_NULL;
        // 8-byte alignment of every complex element is all the per-column accesses of this pass need in fp32
        if (reinterpret_cast<uintptr_t>(blocks[q]) & (pl->lay.dtype == PSFFT_F64 ? 15u : 7u)) return PSFFT_E_ALIGN;
        xd->base[q] = blocks[q];
    }
    for (int q = 0; q <= sl.P; ++q) xd->x0[q] = sl.x0[q];
    xd->P = sl.P;
    xd->zoff = zoff;
    return PSFFT_OK;
}

// Byte ranges a phase-1 / phase-2 call touches: the planes [zoff, zoff + Mz) of every block (written by r2c_xy, only
// read by c2r_yx) next to the call's other buffers.
static bool slab_spans_overlap(const Plan *pl, const psfft_slab_layout &sl, void *const *blocks, long zoff, bool blocks_written,
                               std::initializer_list<Span> others)
{
    const size_t cs = pl->lay.dtype == PSFFT_F64 ? 16 : 8;
    std::vector<Span> v(others);
    for (int q = 0; q < sl.P; ++q) {
        const size_t plane = (size_t)pl->lay.Ny * (size_t)(sl.x0[q + 1] - sl.x0[q]) * cs;
        v.push_back({static_cast<const char *>(blocks[q]) + (size_t)zoff * plane, (size_t)sl.Mz * plane, blocks_written});
    }
    return spans_overlap(v.data(), v.data() + v.size());
}

int psfft_slab_query(psfft_plan plan, int P, int rank, psfft_slab_layout *out)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!out) return PSFFT_E_NULL;
    return slab_ranges(pl, P, rank, out);
}

int psfft_slab_r2c_xy(psfft_plan plan, int P, int rank, const void *d_real_slab, void *d_zspec, void *const *d_blocks,
                      long zoff, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_real_slab || !d_zspec || !d_blocks) return PSFFT_E_NULL;
    if (misaligned(d_real_slab) || misaligned(d_zspec)) return PSFFT_E_ALIGN;
    psfft_slab_layout sl;
    int rc = slab_ranges(pl, P, rank, &sl);
    if (rc) return rc;
    XDistArgs xd;
    rc = slab_xdist(pl, sl, d_blocks, zoff, &xd);
    if (rc) return rc;
    if (slab_spans_overlap(pl, sl, d_blocks, zoff, true, {{d_real_slab, sl.real_bytes, false}, {d_zspec, sl.zspec_bytes, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    const long nrows = (long)sl.Mz * a.Ny;
    const double R = (double)sl.real_bytes, C = (double)sl.zspec_bytes;
    if (pl->lay.dtype == PSFFT_F64) {
        { ProfScope ps(pl, a.stream, K_XR2C, R + C); CU(launch_xpass_r2c<double>(a, d_real_slab, d_zspec, nrows, &pl->launches)); }
        { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass_xdist<double>(a, true, d_zspec, nullptr, xd, sl.Mz, &pl->launches)); }
    } else {
        { ProfScope ps(pl, a.stream, K_XR2C, R + C); CU(launch_xpass_r2c<float>(a, d_real_slab, d_zspec, nrows, &pl->launches)); }
        { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass_xdist<float>(a, true, d_zspec, nullptr, xd, sl.Mz, &pl->launches)); }
    }
    return PSFFT_OK;
}

int psfft_slab_z(psfft_plan plan, int P, int rank, int dir, void *d_xslab, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_xslab) return PSFFT_E_NULL;
    if (misaligned(d_xslab)) return PSFFT_E_ALIGN;
    if (dir != -1 && dir != 1) return PSFFT_E_SIZE;
    psfft_slab_layout sl;
    int rc = slab_ranges(pl, P, rank, &sl);
    if (rc) return rc;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    const long inner = (long)a.Ny * sl.w;   // columns (ky, kx) of the x-slab; z stride = inner
    ProfScope ps(pl, a.stream, K_CPZ, 2.0 * (double)sl.xslab_bytes);
    if (pl->lay.dtype == PSFFT_F64)
        CU(launch_cpass_raw<double>(a, dir, a.Nz, a.twZ, d_xslab, d_xslab, inner, inner, inner * a.Nz, 1, &pl->launches));
    else
        CU(launch_cpass_raw<float>(a, dir, a.Nz, a.twZ, d_xslab, d_xslab, inner, inner, inner * a.Nz, 1, &pl->launches));
    return PSFFT_OK;
}

int psfft_slab_c2r_yx(psfft_plan plan, int P, int rank, void *const *d_blocks, long zoff, void *d_zspec,
                      void *d_real_slab, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_real_slab || !d_zspec || !d_blocks) return PSFFT_E_NULL;
    if (misaligned(d_real_slab) || misaligned(d_zspec)) return PSFFT_E_ALIGN;
    psfft_slab_layout sl;
    int rc = slab_ranges(pl, P, rank, &sl);
    if (rc) return rc;
    XDistArgs xd;
    rc = slab_xdist(pl, sl, d_blocks, zoff, &xd);
    if (rc) return rc;
    if (slab_spans_overlap(pl, sl, d_blocks, zoff, false, {{d_zspec, sl.zspec_bytes, true}, {d_real_slab, sl.real_bytes, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    const long nrows = (long)sl.Mz * a.Ny;
    const double scale = 1.0 / ((double)a.N * a.Ny * a.Nz);
    const double R = (double)sl.real_bytes, C = (double)sl.zspec_bytes;
    if (pl->lay.dtype == PSFFT_F64) {
        { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass_xdist<double>(a, false, nullptr, d_zspec, xd, sl.Mz, &pl->launches)); }
        { ProfScope ps(pl, a.stream, K_XC2R, R + C); CU(launch_xpass_c2r<double>(a, d_zspec, d_real_slab, nrows, scale, &pl->launches)); }
    } else {
        { ProfScope ps(pl, a.stream, K_CPY, 2 * C); CU(launch_cpass_xdist<float>(a, false, nullptr, d_zspec, xd, sl.Mz, &pl->launches)); }
        { ProfScope ps(pl, a.stream, K_XC2R, R + C); CU(launch_xpass_c2r<float>(a, d_zspec, d_real_slab, nrows, scale, &pl->launches)); }
    }
    return PSFFT_OK;
}

int psfft_profile_enable(psfft_plan plan, int on)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    pl->prof = on != 0;
    return PSFFT_OK;
}

int psfft_profile_reset(psfft_plan plan)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    for (ProfRec &r : pl->recs) { pl->pool.push_back(r.start); pl->pool.push_back(r.stop); }
    pl->recs.clear();
    return PSFFT_OK;
}

int psfft_profile_count(psfft_plan plan)
{
    Plan *pl = get(plan);
    return pl ? (int)pl->recs.size() : PSFFT_E_PLAN;
}

int psfft_profile_get(psfft_plan plan, int i, int *kind, double *ms, double *bytes)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (i < 0 || i >= (int)pl->recs.size()) return PSFFT_E_SIZE;
    if (!kind || !ms || !bytes) return PSFFT_E_NULL;
    const ProfRec &r = pl->recs[i];
    CU(cudaEventSynchronize(r.stop));
    float t = 0.f;
    CU(cudaEventElapsedTime(&t, r.start, r.stop));
    *kind = r.kind;
    *ms = t;
    *bytes = r.bytes;
    return PSFFT_OK;
}

const char *psfft_kernel_name(int kind) { return (kind >= 0 && kind < K_COUNT) ? KERNEL_NAMES[kind] : "?"; }

int psfft_last_launch_count(psfft_plan plan)
{
    Plan *pl = get(plan);
    return pl ? pl->launches : PSFFT_E_PLAN;
}

const char *psfft_strerror(int code)
{
    switch (code) {
        case PSFFT_OK: return "success";
        case PSFFT_E_NULL: return "psfft: required pointer is NULL";
        case PSFFT_E_SIZE: return "psfft: unsupported grid size, batch, system, order or box length";
        case PSFFT_E_DTYPE: return "psfft: dtype must be PSFFT_F32 or PSFFT_F64";
        case PSFFT_E_ALIGN: return "psfft: device pointer not 16-byte aligned";
        case PSFFT_E_TABLE: return "psfft: table buffer too small";
        case PSFFT_E_PLAN: return "psfft: invalid plan handle";
        case PSFFT_E_BATCH: return "psfft: batch too large (batch * Nz must not exceed 65535)";
        case PSFFT_E_OVERLAP: return "psfft: input, output and workspace ranges of a call must not overlap";
        case PSFFT_E_SCRATCH:
            return "psfft: plan too large for the built-in workspace (work_bytes_fft > PSFFT_STATIC_SCRATCH_BYTES = 32 MiB); "
                   "call psfft_fft3d_c2r with a workspace of your own";
    }
    if (code > 0) return cudaGetErrorString((cudaError_t)code);
    return "psfft: unknown error code";
}

const char *psfft_version(void) { return "0.1"; }

}  // extern "C"

// ================================================================================================
// psfft_fft3d_c2r_static: the inverse transform for callers that cannot allocate device memory (psfft.h).
//
// Its workspace is this array.  It is part of the library image: the CUDA runtime gives it a home on every GPU
// that loads this file's device code and keeps it there until the process exits, so no call ever has to ask the
// driver for memory.  Everything that concerns it sits in this one file on purpose:
//   * In HOST code the name `g_static_scratch` is only a stand-in the runtime uses to find the symbol.  It is not
//     a device address.  Handing `g_static_scratch` (or `&g_static_scratch[0]`) to a kernel would make the kernel
//     fault, or -- on a system where the GPU can read host memory -- quietly work on the wrong bytes.  The device
//     address has to be asked for, per device, with cudaGetSymbolAddress; static_scratch_address() below does that
//     once per device, with that device current, and checks the return code.
//   * The array is shared by all plans and calls on a device and is never cleared.  The z-pass of the inverse
//     transform writes all batch * ldk * Ny * Nz elements before the y- and x-passes read any of them, so stale
//     contents of an earlier (possibly larger) call cannot leak into a result.  Calls that overlap on the GPU race.
static __device__ __align__(256) unsigned char g_static_scratch[PSFFT_STATIC_SCRATCH_BYTES];

namespace {

const int STATIC_SCRATCH_MAX_DEVICES = 64;
std::mutex g_static_scratch_mu;
void *g_static_scratch_addr[STATIC_SCRATCH_MAX_DEVICES];   // device address of the array per device; NULL = not asked yet

// Device address of g_static_scratch on the caller's current device.  The first call on a device asks the runtime
// (this is also what makes the runtime load this file's device image, and with it the array, on that device); the
// answer is kept, so later calls make no CUDA call here besides cudaGetDevice.
int static_scratch_address(void **out)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_SCRATCH_MAX_DEVICES) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_scratch_mu);
    if (!g_static_scratch_addr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return (int)cudaErrorInvalidSymbol;
        g_static_scratch_addr[dev] = p;
    }
    *out = g_static_scratch_addr[dev];
    return PSFFT_OK;
}

// The three passes of c2r_fields_inplace without its per-launch event hooks (creating an event allocates).
template <typename T> int c2r_fields_static(Plan *pl, const PassArgs &a, const void *d_spec, void *scratch, void *d_real)
{
    const int fields = pl->lay.batch;
    const long nrows = (long)fields * a.Ny * a.Nz;
    const double scale = 1.0 / ((double)a.N * a.Ny * a.Nz);
    CU(launch_cpass<T>(a, +1, 2, d_spec, scratch, fields, &pl->launches));    // z: input -> scratch (every element written)
    CU(launch_cpass<T>(a, +1, 1, scratch, scratch, fields, &pl->launches));   // y: in place
    CU(launch_xpass_c2r<T>(a, scratch, d_real, nrows, scale, &pl->launches)); // x: scratch -> output, scaled
    return PSFFT_OK;
}

}  // namespace

extern "C" int psfft_fft3d_c2r_static(psfft_plan plan, const void *d_spec, void *d_real, void *stream)
{
    Plan *pl = get(plan);
    if (!pl) return PSFFT_E_PLAN;
    if (!d_real || !d_spec) return PSFFT_E_NULL;
    if (misaligned(d_real) || misaligned(d_spec)) return PSFFT_E_ALIGN;
    if (pl->lay.work_bytes_fft > (size_t)PSFFT_STATIC_SCRATCH_BYTES) return PSFFT_E_SCRATCH;   // nothing enqueued
    void *scratch = nullptr;
    const int rc = static_scratch_address(&scratch);
    if (rc) return rc;
    if (spans_overlap({{d_spec, pl->lay.batch * pl->lay.spec_bytes, false}, {d_real, pl->lay.batch * pl->lay.real_bytes, true},
                       {scratch, pl->lay.work_bytes_fft, true}}))
        return PSFFT_E_OVERLAP;
    pl->launches = 0;
    PassArgs a = args_of(pl, stream);
    return pl->lay.dtype == PSFFT_F64 ? c2r_fields_static<double>(pl, a, d_spec, scratch, d_real)
                                      : c2r_fields_static<float>(pl, a, d_spec, scratch, d_real);
}
