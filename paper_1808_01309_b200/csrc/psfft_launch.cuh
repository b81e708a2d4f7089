// psfft_launch.cuh -- host-side launchers: pick the kernel instantiation for (dtype, N) and
// enqueue it.  Declared here, defined in psfft_launch_impl.cuh and instantiated per dtype in psfft_f{32,64}_*.cu.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace psfft {

// every supported grid size, in one place (psfft.h: 2^a 3^b, b <= 1, 8 <= N <= 1024, and 2048)
// (-D"PSFFT_SIZES(X)=X(32) X(512)" restricts the list for quick experimental builds)
#ifdef PSFFT_SIZES
#define PSFFT_FOR_EACH_N(X) PSFFT_SIZES(X)
#else
#define PSFFT_FOR_EACH_N(X) \
    X(8) X(12) X(16) X(24) X(32) X(48) X(64) X(96) X(128) X(192) X(256) X(384) X(512) X(768) X(1024) X(2048)
#endif

struct PassArgs {
    const void *tab;   // roots of unity exp(-2 pi i m/N), N complex of the plan dtype
    const void *twN;   // per-stage twiddle tables of the length-N transforms (y, z passes)
    const void *twX;   // per-stage twiddle tables of the length-N transforms in the symmetric schedule (x passes, mid_x)
    int N;             // grid points along x (and along y, z for the cubic plans every RHS call needs)
    int Ny, Nz;        // grid points along y, z (psfft_plan_create3: anisotropic grids, transforms only)
    const void *twY;   // per-stage tables of the length-Ny / length-Nz column transforms (= twN when cubic)
    const void *twZ;
    int ldk;
    cudaStream_t stream;
    // right-hand sides (psfft_rhs.cuh Geom; readings G24, G25): compact row pitch of the workspace fields,
    // retained kx count, integer weights of the 2/3-rule ellipsoid, wavenumber factors 2 pi / L_i
    int kxp, kxc, rx2, ry2, rz2, lim;
    double kf[3];
    bool unit_cube;    // Nx = Ny = Nz and the 2 pi box: the column passes run with compile-time geometry
};

// compact row pitch of the RHS workspace fields of an (Nx, Ny, Nz) plan with complex size csize (host)
int rhs_pitch3(int Nx, int Ny, int Nz, int csize);

// Each launcher returns cudaGetLastError() of its launch (or cudaErrorInvalidValue for an
// unsupported N) and increments *launches.
template <typename T> cudaError_t launch_xpass_r2c(const PassArgs &a, const void *in, void *out, long nrows, int *launches);
template <typename T> cudaError_t launch_xpass_c2r(const PassArgs &a, const void *in, void *out, long nrows, double scale, int *launches);
// dir = -1 forward, +1 backward; axis 1 = y, 2 = z; `fields` contiguous spectral fields
template <typename T> cudaError_t launch_cpass(const PassArgs &a, int dir, int axis, const void *in, void *out, int fields, int *launches);
template <typename T> cudaError_t launch_mask_curl(const PassArgs &a, const void *u, void *out6, int *launches);
template <typename T> cudaError_t launch_cross(const PassArgs &a, const void *pa, const void *pb, void *pc, int *launches);
template <typename T> cudaError_t launch_cross_mhd(const PassArgs &a, const void *u, const void *b, const void *w, const void *j, void *om, void *oe, int *launches);
template <typename T> cudaError_t launch_finish(const PassArgs &a, int mode, const void *f, const void *u, void *out, double nu, int *launches);

// fused right-hand side (psfft_rhs.cuh); nv = 1 (HD) or 2 (MHD); ns = 1 with nv = 1: Boussinesq
struct RhsArgs {
    int nv, ns;
    const void *src[2];   // u^, b^
    void *dst[2];         // rhs_u, rhs_b
    double diff[2];       // nu, eta
    const void *ssrc;     // ns = 1: theta^
    void *sdst;           // ns = 1: rhs_theta
    double sdiff, nbv;    // kappa, Brunt-Vaisala frequency N_bv
    // Runge-Kutta stage (psfft_rk_step): when base[0] != NULL the outputs are base + cstep * rhs on the retained
    // modes (base = the state y_n at the start of the step, in the same order as src / ssrc)
    const void *base[2];
    const void *sbase;
    double cstep;
    bool sparse_out;      // intermediate stage: skip the zero fill outside the truncation sphere
    void *zbuf;           // 5 nv + 2 ns compact fields (inv_z out; later mid_x out / fwd_y in place, 3 nv + ns fields)
    void *ybuf;           // 6 nv + 3 ns compact fields (inv_y out)
};
template <typename T> cudaError_t launch_rhs_mid_x(const PassArgs &a, const RhsArgs &r, int *launches);
// column passes: CUBE = compile-time geometry of the N^3 grid in the 2 pi box; false = the plan's run-time geometry
template <typename T, bool CUBE> cudaError_t launch_rhs_inv_z_g(const PassArgs &a, const RhsArgs &r, int *launches);
template <typename T, bool CUBE> cudaError_t launch_rhs_inv_y_g(const PassArgs &a, const RhsArgs &r, int *launches);
template <typename T, bool CUBE> cudaError_t launch_rhs_fwd_y_g(const PassArgs &a, const RhsArgs &r, int *launches);
template <typename T, bool CUBE> cudaError_t launch_rhs_fwd_z_g(const PassArgs &a, const RhsArgs &r, int *launches);
#define PSFFT_BY_GEOMETRY(name)                                                                          \
    template <typename T> inline cudaError_t launch_rhs_##name(const PassArgs &a, const RhsArgs &r, int *launches) \
    {                                                                                                    \
        return a.unit_cube ? launch_rhs_##name##_g<T, true>(a, r, launches) : launch_rhs_##name##_g<T, false>(a, r, launches); \
    }
PSFFT_BY_GEOMETRY(inv_z)
PSFFT_BY_GEOMETRY(inv_y)
PSFFT_BY_GEOMETRY(fwd_y)
#undef PSFFT_BY_GEOMETRY
// fwd_z takes the run-time geometry on every plan: measured on B200 it is the faster build of this pass (the epilogue
// spills less at the 64-register budget): 512^3 fp64 1.15 -> 1.09 ms, 768^3 fp32 2.73 -> 2.05 ms, 1024^3 fp32 MHD
// 10.8 -> 9.7 ms
template <typename T> inline cudaError_t launch_rhs_fwd_z(const PassArgs &a, const RhsArgs &r, int *launches)
{
    return launch_rhs_fwd_z_g<T, false>(a, r, launches);
}

// Gross-Pitaevskii right-hand side (psi = p + i q as two real fields): pass = 0 inv_z, 1 inv_y, 2 mid_x,
// 3 fwd_y, 4 fwd_z
struct GpeArgs {
    const void *psi;      // p^, q^ (caller layout)
    void *dst;            // R_p, R_q
    const void *base;     // Runge-Kutta stage: y_n, or NULL
    double alpha, beta, cstep;
    bool sparse_out;
    void *zbuf;           // 2 compact fields: inv_z out, inv_y in place
    void *obuf;           // 2 compact fields: mid_x out, fwd_y in place
};
template <typename T, bool CUBE> cudaError_t launch_gpe_pass_g(const PassArgs &a, const GpeArgs &g, int pass, int *launches);
template <typename T> inline cudaError_t launch_gpe_pass(const PassArgs &a, const GpeArgs &g, int pass, int *launches)
{
    return a.unit_cube ? launch_gpe_pass_g<T, true>(a, g, pass, launches) : launch_gpe_pass_g<T, false>(a, g, pass, launches);
}

// ---- slab-decomposed transform (psfft_slab.cuh) ------------------------------------------------
// x-distributed blocks of one exchange: block q holds kx in [x0[q], x0[q + 1]) as [rows][Ny][w_q]
struct XDistArgs {
    void *base[16];
    int x0[17];
    int P;
    long zoff;
};
// y-pass of the z-slab [mz][Ny][ldk] `slab` with the other side in the blocks: scatter (forward) or gather (inverse)
template <typename T> cudaError_t launch_cpass_xdist(const PassArgs &a, bool scatter, const void *slab_in, void *slab_out,
                                                     const XDistArgs &xd, int mz, int *launches);
// plain strided column pass of length `len` (table `tw`): element (i, col, o) at base[o outer_stride + i axis_stride + col]
template <typename T> cudaError_t launch_cpass_raw(const PassArgs &a, int dir, int len, const void *tw, const void *in, void *out,
                                                   long axis_stride, long inner, long outer_stride, long outer, int *launches);

// complex entries of the tables of an (Nx, Ny, Nz) plan: [roots of unity, Nx][stage tables Ny]
// [symmetric-schedule stage tables Nx (x passes, mid_x)][stage tables Nz, only when Nz != Ny]
struct TableOffsets { size_t y, x, z, total; };
TableOffsets table_entries(int Nx, int Ny, int Nz);
// symmetric radix schedule of the mid_x transforms (psfft_midxg.cuh): fills radix[], returns the stage count
int xsched_stages(int N, int *radix);

}  // namespace psfft
