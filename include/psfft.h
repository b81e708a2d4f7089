/*
 * psfft.h -- C ABI of libpsfft: the single-GPU hot path of arxiv 1808.01309 on B200 (sm_100a).
 *
 *   N^3 real-to-complex / complex-to-real 3D FFT on a periodic grid (Sec. 2,
 *   Eq. 8 and the three transform steps) and one pseudospectral Navier-Stokes (HD) or MHD
 *   right-hand-side evaluation (Eqs. 1, 3, 4-6).
 *
 * The calls follow the paper's plan concept -- create / execute forward / execute backward /
 * clean up, sizes derived from grid size and datatype, an integer return code from every call
 * (PAPER.md:146-159 Listing 1, :176-212 Sec. 3.2) -- but nothing else of its design: there is no
 * host staging, no cuFFT, no stream-chunking.  Every execute call is a handful of hand-written
 * kernels enqueued on the caller's stream.
 *
 * CONVENTIONS (all calls)
 *   Layout   real field      [b][z][y][x], x contiguous            (N^3 reals per field)
 *            half spectrum   [b][kz][ky][kx], kx in [0, N/2] contiguous, row stride ldk = N/2+1
 *                            (ldk*N*N complex per field); index q along y/z is wavenumber q for
 *                            q < N/2 and q-N otherwise; the box is 2*pi-periodic (integer k) unless
 *                            psfft_plan_set_box says otherwise.
 *            complex = interleaved (re, im) of the plan's dtype.
 *   Values   forward: X[r,q,p] = sum x[k,j,i] exp(-2 pi i (p i + q j + r k)/N), unnormalised
 *            (Eq. 8); inverse: sign +, scaled by 1/N^3 so c2r(r2c(x)) = x.
 *            Spectral fields handed to / returned by the RHS calls are such unnormalised
 *            spectra (N^3 x Fourier coefficient).
 *   Memory   "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.  The caller owns
 *            every buffer (inputs, outputs, workspace, tables); the library never allocates or
 *            frees device memory.  Device pointers must be 16-byte aligned (256 recommended).
 *            (16 bytes is what the widest vector access of the kernels needs and what the fields inside a
 *            multi-field array are aligned to: ldk*N*N*2s is in general not a multiple of 256.)
 *            Inputs are never modified.  Input and output of one call must not overlap; the
 *            workspace must overlap neither: every execute call checks the byte ranges it will touch
 *            (sizes from the plan's layout) and returns PSFFT_E_OVERLAP before enqueuing anything.
 *            Inputs may alias one another.  The workspace SIZE cannot be checked (the ABI passes no size).
 *   Streams  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Execute
 *            calls only enqueue work and return without synchronising; they are CUDA-graph
 *            capturable.  A plan may be used on one stream at a time.
 *   Errors   0 = success.  Negative = PSFFT_E_* argument errors detected on the host before
 *            anything is enqueued.  Positive = the cudaError_t of a failed CUDA call.
 *            There is no CPU fallback: without a CUDA device every execute call fails.
 */
#ifndef PSFFT_H
#define PSFFT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PSFFT_F32 0
#define PSFFT_F64 1

#define PSFFT_OK 0
#define PSFFT_E_NULL (-1)        /* a required pointer is NULL */
#define PSFFT_E_SIZE (-2)        /* unsupported N (see psfft_plan_query), batch < 1, bad system / order / box length */
#define PSFFT_E_DTYPE (-3)       /* dtype is not PSFFT_F32 / PSFFT_F64 */
#define PSFFT_E_ALIGN (-4)       /* a device pointer is not 16-byte aligned */
#define PSFFT_E_TABLE (-5)       /* table buffer smaller than layout.table_bytes */
#define PSFFT_E_PLAN (-6)        /* invalid or destroyed plan handle */
#define PSFFT_E_BATCH (-7)       /* batch * Nz exceeds 65535 (grid limit of the y-pass) */
#define PSFFT_E_OVERLAP (-8)     /* an output or workspace range of the call overlaps another range of the call */
#define PSFFT_E_SCRATCH (-9)     /* psfft_fft3d_c2r_static: the plan needs more workspace than PSFFT_STATIC_SCRATCH_BYTES */

typedef struct psfft_plan_s *psfft_plan;

/* Sizes implied by (N, dtype, batch); all element counts are per field. */
typedef struct psfft_layout {
    int N;                       /* grid points per direction */
    int dtype;                   /* PSFFT_F32 / PSFFT_F64 */
    int batch;                   /* fields per fft3d call */
    int ldk;                     /* leading dimension of the half spectrum (= N/2 + 1) */
    size_t real_elems;           /* N^3            reals   per real field */
    size_t spec_elems;           /* ldk * N * N    complex per spectral field */
    size_t real_bytes;           /* bytes of one real field */
    size_t spec_bytes;           /* bytes of one spectral field */
    size_t table_bytes;          /* size of the twiddle-table buffer for psfft_plan_create */
    size_t work_bytes_fft;       /* workspace for psfft_fft3d_r2c / c2r (batch fields) */
    size_t work_bytes_hd;        /* workspace for psfft_hd_rhs (cubic plans: also enough for psfft_hd_rhs_unfused) */
    size_t work_bytes_mhd;       /* workspace for psfft_mhd_rhs */
    size_t work_bytes_boussinesq; /* workspace for psfft_boussinesq_rhs */
    int Ny, Nz;                  /* grid points along y, z (= N except for psfft_plan_create3 plans) */
    size_t work_bytes_gpe;       /* workspace for psfft_gpe_rhs */
} psfft_layout;

/* Sizes for a prospective plan.  Supported N: 2^a * 3^b with b <= 1 and 8 <= N <= 1024
 * (8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024), and 2048 (the paper's largest grid is
 * 2048 x 2048 x 512; a cubic 2048^3 field does not fit one GPU).  Host-only. */
int psfft_plan_query(int N, int dtype, int batch, psfft_layout *out);

/* Create a plan ("create plan": sizes from the input size and datatype).
 * Computes the root-of-unity table exp(-2 pi i m/N), m = 0..N-1, on the host in long double,
 * rounds once to the plan dtype and copies it to `d_tables` (>= table_bytes) on `stream`;
 * returns after that copy has completed.  The plan keeps the pointer; the buffer must outlive
 * the plan. */
int psfft_plan_create(psfft_plan *plan, int N, int dtype, int batch, void *d_tables,
                      size_t table_bytes, void *stream);

/* Anisotropic grids ("we also update the formulation ... to accommodate anisotropic grids";
 * its largest runs are 1024 x 1024 x 256 and 2048 x 2048 x 512): a plan for an Nx x Ny x Nz grid,
 * each size from the supported list.  Real field [b][z][y][x] (Nx contiguous), half spectrum [b][kz][ky][kx]
 * with ldk = Nx/2 + 1; psfft_fft3d_r2c / c2r work as above (inverse scaled by 1/(Nx Ny Nz)).  layout.N is Nx.
 * Every right-hand-side and Runge-Kutta call works on such a plan (only the *_unfused cross-check variants need a
 * cubic one in the default 2 pi box and return PSFFT_E_SIZE otherwise); spectra are Nx Ny Nz x Fourier coefficient, and
 *   the 2/3 rule is the ellipsoidal truncation in index space, keep iff sum_i (n_i / N_i)^2 < 1/9, evaluated in
 *   integers as 9 sum_i (n_i L / N_i)^2 < L^2 with L = lcm(Nx, Ny, Nz) -- for a cube this is 9 |n|^2 < N^2;
 *   n_i = the integer index p (p < N_i / 2) or p - N_i. */
int psfft_plan_query3(int Nx, int Ny, int Nz, int dtype, int batch, psfft_layout *out);
int psfft_plan_create3(psfft_plan *plan, int Nx, int Ny, int Nz, int dtype, int batch, void *d_tables,
                       size_t table_bytes, void *stream);

/* Physical box (Sec. 2 below Eq. 8: "both the physical box size, L_i, and the number of physical space
 * points, N_i, may be specified independently in each direction").  Sets the box lengths of the plan; from then on
 * every derivative, projection and diffusion term of the right-hand-side calls uses the wavenumbers
 *     k_i = n_i * (2 pi / L_i),      2 pi / L_i evaluated once in fp64 and rounded to the plan dtype
 * (exactly 1, i.e. integer wavenumbers, for L_i = 2 pi -- the default of a new plan).  The dealiasing mask does not
 * depend on the box (see above); the transforms do not either.  Host-only, no device work.
 * Returns PSFFT_E_SIZE unless every length is positive and finite. */
int psfft_plan_set_box(psfft_plan plan, double Lx, double Ly, double Lz);

/* Free host-side state (PAPER.md:187 clean-up).  Never touches caller memory. */
int psfft_plan_destroy(psfft_plan plan);

/* Fill *out with the plan's layout. */
int psfft_plan_layout(psfft_plan plan, psfft_layout *out);

/* Forward transform of `batch` real fields (PAPER.md:70-77 steps 1-3; unnormalised, sign -).
 *   d_real  in   batch * N^3 reals
 *   d_spec  out  batch * ldk*N*N complex
 *   d_work       >= work_bytes_fft (may be NULL when that is 0)
 * Three kernels: x-pass (r2c) -> y-pass -> z-pass; the paper's transpose (step 2) is the
 * strided tile access of the y/z passes. */
int psfft_fft3d_r2c(psfft_plan plan, const void *d_real, void *d_spec, void *d_work, void *stream);

/* Inverse transform ("reverses these steps"; sign +, scaled by 1/N^3).
 * Defined for any half spectrum: imaginary parts of the kx = 0 and kx = N/2 entries that would
 * break Hermitian symmetry are ignored (x_i = Re Y_0 + (-1)^i Re Y_{N/2} + 2 sum Re(Y_p w^{pi})).
 *   d_spec  in   batch * ldk*N*N complex (not modified)
 *   d_real  out  batch * N^3 reals
 *   d_work       >= work_bytes_fft */
int psfft_fft3d_c2r(psfft_plan plan, const void *d_spec, void *d_real, void *d_work, void *stream);

/* Inverse transform for callers that have no device memory to give as workspace and cannot get any.
 *
 * psfft_fft3d_c2r needs a workspace of work_bytes_fft next to its input and output, because it must leave the
 * input spectrum untouched.  Normally the caller allocates that once.  Some callers cannot: a solver whose
 * host application handed it a fixed set of field buffers and forbids further device allocation (every byte of
 * HBM is already spoken for by the application's own arena, so a cudaMalloc would fail, or the time loop is not
 * allowed to stall on the device-wide synchronisation that cudaMalloc / cudaFree imply), or a plug-in that runs
 * inside someone else's process where it does not own the allocator at all.  For them this call takes the
 * workspace from an array that is part of the library image itself:
 *
 *     static __device__ __align__(256) unsigned char [PSFFT_STATIC_SCRATCH_BYTES]     (32 MiB)
 *
 * The CUDA runtime places that array on every GPU on which this library's device code gets loaded, and it stays
 * there until the process exits -- that is the price, and the reason the limit is modest.  The call itself
 * allocates nothing: no cudaMalloc / cudaFree, no event or stream creation, no allocating library routine; it
 * only enqueues the same three kernels as psfft_fft3d_c2r (z-pass, y-pass, c2r x-pass) with the array as d_work,
 * so the result is bit for bit that of psfft_fft3d_c2r.
 *
 *   d_spec  in   batch * ldk*Ny*Nz complex (not modified)
 *   d_real  out  batch * Nx*Ny*Nz reals
 *
 * Limit     the plan's layout.work_bytes_fft (= batch * spec_bytes) must not exceed PSFFT_STATIC_SCRATCH_BYTES:
 *           e.g. 128^3 fp64 batch 1 (17.0 MB), 128^3 fp32 batch 3 (25.6 MB), 192^3 fp32 batch 1 (28.6 MB).  A
 *           larger plan gets PSFFT_E_SCRATCH and nothing is enqueued; use psfft_fft3d_c2r with your own workspace.
 * Set-up    the first call on each device looks up where the array lives on that device (cudaGetSymbolAddress,
 *           with the caller's current device -- the one that holds d_spec and d_real -- and its return code
 *           checked) and remembers it; later calls on that device skip this.  Make that first call outside any
 *           stream capture.
 * Sharing   there is ONE array per device, shared by every plan and every call.  Two calls that can run on the
 *           GPU at the same time (different streams, different host threads) race on it and both produce
 *           garbage: serialise them on one stream, or order them with events.  The array keeps whatever the last
 *           call left in it; this call does not depend on that, because its first pass overwrites every element
 *           the later passes read, so nothing has to be cleared.
 * Profiling the per-launch event hooks below (psfft_profile_*) are not fed by this call, because creating events
 *           allocates.  psfft_last_launch_count works.
 * Errors    as psfft_fft3d_c2r, plus PSFFT_E_SCRATCH. */
#define PSFFT_STATIC_SCRATCH_BYTES (32u << 20)
int psfft_fft3d_c2r_static(psfft_plan plan, const void *d_spec, void *d_real, void *stream);

/* One Navier-Stokes right-hand side (Eq. 1 with theta = 0, Eq. 3):
 *     rhs = M P F[ F^-1(M u^) x F^-1(i k x M u^) ] - nu |k|^2 M u^
 * M = 2/3-rule spherical truncation, keep iff 9 |k|^2 < N^2 (integer test, masked outputs are
 * exactly +0); P = I - k k^T/|k|^2 (identity at k = 0).  6 inverse + 3 forward transforms.
 *   d_uhat  in   3 spectral fields [c][kz][ky][kx]
 *   d_rhs   out  3 spectral fields
 *   d_work       >= work_bytes_hd
 * Independent of the plan's batch. */
int psfft_hd_rhs(psfft_plan plan, const void *d_uhat, void *d_rhs, double nu, void *d_work,
                 void *stream);

/* One MHD right-hand side (Eqs. 4-6, v = u in Eq. 5):
 *     w = curl u, j = curl b;  rhs_u = M P F[u x w + j x b] - nu |k|^2 M u^
 *                              rhs_b = M i k x F[u x b]     - eta |k|^2 M b^
 * 12 inverse + 6 forward transforms.  d_work >= work_bytes_mhd. */
int psfft_mhd_rhs(psfft_plan plan, const void *d_uhat, const void *d_bhat, void *d_rhs_u,
                  void *d_rhs_b, double nu, double eta, void *d_work, void *stream);

/* One Boussinesq right-hand side, the paper's reference equations (Eqs. 1-3):
 *     d_t u     = -grad p - u.grad u - N_bv theta z^ + nu Lap u,   div u = 0
 *     d_t theta = -u.grad theta + N_bv w + kappa Lap theta          (w = u_z)
 * evaluated as (rotational form for the momentum term, as in psfft_hd_rhs)
 *     rhs_u  = M P ( F[u x w] - N_bv M theta^ z^ ) - nu |k|^2 M u^          (w = curl u)
 *     rhs_th = -M F[u . grad theta] + N_bv M u^_z - kappa |k|^2 M theta^
 * with u, w, grad theta = F^-1 of (M u^, i k x M u^, i k M theta^): 9 inverse + 4 forward transforms in
 * the definition; the fused passes need the equivalent of 8 inverse axis-pass sets (theta itself is
 * never needed in physical space).
 *   d_uhat    in   3 spectral fields     d_thhat   in   1 spectral field
 *   d_rhs_u   out  3 spectral fields     d_rhs_th  out  1 spectral field
 *   d_work         >= work_bytes_boussinesq
 * Independent of the plan's batch. */
int psfft_boussinesq_rhs(psfft_plan plan, const void *d_uhat, const void *d_thhat, void *d_rhs_u,
                         void *d_rhs_th, double nu, double kappa, double nbv, void *d_work,
                         void *stream);

/* Right-hand side of the Gross-Pitaevskii equation (Eq. 7),
 *     i hbar d_t psi = -hbar^2/(2m) Lap psi + g |psi|^2 psi   <=>   d_t psi = i alpha Lap psi - i beta |psi|^2 psi,
 * alpha = hbar/(2m), beta = g/hbar, for psi = p + i q carried as the two REAL fields p, q ("1 complex (or 2 real)"
 * primitive fields):
 *     rhs_p = beta M F[(p^2 + q^2) q] + alpha |k|^2 M q^,     rhs_q = -beta M F[(p^2 + q^2) p] - alpha |k|^2 M p^
 * with p, q = F^-1 of (M p^, M q^): 2 inverse + 2 forward transforms.  In the x pass the packed row P^ + i Q^
 * inverse-transforms to psi itself, so one complex transform per row and direction does both fields.
 *   d_psihat  in   2 spectral fields (p^, q^)      d_rhs  out  2 spectral fields
 *   d_work         >= work_bytes_gpe
 * psfft_rk_step takes PSFFT_SYS_GPE with params = { alpha, beta, - }. */
int psfft_gpe_rhs(psfft_plan plan, const void *d_psihat, void *d_rhs, double alpha, double beta, void *d_work,
                  void *stream);

/* One explicit Runge-Kutta time step around a right-hand side above ("the system of ODEs
 * is solved using an explicit Runge-Kutta scheme (of 2nd-4th order)"; the paper does not print the
 * scheme -- DESIGN.md reading G21: the low-storage form with `ord` stages
 *     y^(ord) = y_n;   y^(o-1) = M y_n + (dt / o) R(y^(o)),  o = ord, ..., 1;   y_{n+1} = y^(0) ).
 * Each stage is one fused right-hand-side evaluation whose last pass writes M y_n + (dt/o) R instead of
 * R (one more sparse read of y_n in its epilogue); there is no separate update kernel.
 *   system    PSFFT_SYS_HD (y = u^: 3 fields), PSFFT_SYS_MHD (u^, b^: 6), PSFFT_SYS_BOUSSINESQ (u^, theta^: 4),
 *             PSFFT_SYS_GPE (p^, q^ of psi = p + i q: 2 fields; R = psfft_gpe_rhs)
 *   d_y_in    in   the state y_n, fields contiguous in the order above (not modified)
 *   d_y_out   out  y_{n+1} (dealiased); must not overlap d_y_in
 *   ord       1..4 stages
 *   params    HOST pointer to 3 doubles: { nu, eta (MHD) or kappa (Boussinesq), N_bv };
 *             for PSFFT_SYS_GPE { alpha, beta, ignored }
 *   d_work         >= psfft_rk_work_bytes(plan, system) = one state-sized stage buffer + the RHS workspace
 * Returns PSFFT_E_SIZE for a bad system / ord, PSFFT_E_OVERLAP when d_y_in, d_y_out, d_work overlap. */
#define PSFFT_SYS_HD 0
#define PSFFT_SYS_MHD 1
#define PSFFT_SYS_BOUSSINESQ 2
#define PSFFT_SYS_GPE 3          /* y = (p^, q^): 2 fields; params = { alpha, beta, unused } */
size_t psfft_rk_work_bytes(psfft_plan plan, int system);
int psfft_rk_step(psfft_plan plan, int system, const void *d_y_in, void *d_y_out, int ord, double dt,
                  const double *params, void *d_work, void *stream);

/* The same two right-hand sides computed as the plain composition of the public passes: mask +
 * curl kernel, 6 (12) three-pass inverse transforms, pointwise product kernel, 3 (6) three-pass
 * forward transforms, mask + projection kernel.  Nothing is fused or pruned: every pass touches
 * the dense fields.  Same arguments, same results up to rounding; kept as the second CUDA path that
 * the full-size tests cross-check the fused one against, and as the "before" of DESIGN.md's
 * traffic comparison.  Their kernels use integer wavenumbers on a cube: a plan with Nx != Ny or Ny != Nz, or whose
 * box psfft_plan_set_box changed to anything but (2 pi, 2 pi, 2 pi), gets PSFFT_E_SIZE. */
int psfft_hd_rhs_unfused(psfft_plan plan, const void *d_uhat, void *d_rhs, double nu, void *d_work,
                         void *stream);
int psfft_mhd_rhs_unfused(psfft_plan plan, const void *d_uhat, const void *d_bhat, void *d_rhs_u,
                          void *d_rhs_b, double nu, double eta, void *d_work, void *stream);

/* End-to-end variants with HOST buffers (pinned memory recommended): copy the inputs host->device
 * into caller-provided device staging, run the call above, copy the result device->host, all on
 * `stream`, then synchronise the stream.
 *   d_in / d_out   device staging of the size of the input / output of the corresponding call */
int psfft_fft3d_r2c_host(psfft_plan plan, const void *h_real, void *h_spec, void *d_in, void *d_out,
                         void *d_work, void *stream);
int psfft_fft3d_c2r_host(psfft_plan plan, const void *h_spec, void *h_real, void *d_in, void *d_out,
                         void *d_work, void *stream);
int psfft_hd_rhs_host(psfft_plan plan, const void *h_uhat, void *h_rhs, double nu, void *d_in,
                      void *d_out, void *d_work, void *stream);

/* psfft_hd_rhs_host that moves only what the method defines (the cost of the
 * host <-> device transfers is the paper's own concern).  The right-hand side reads its input through the 2/3-rule
 * mask and its output is exactly zero outside the mask, so of each dense spectral field only the index box around the
 * retained ellipsoid,
 *     kx in [0, ceil(Nx/3)),   |ky| < Ny/3,   |kz| < Nz/3        (about 30 % of the field),
 * has to cross the bus.  Same arguments and same dense layouts as psfft_hd_rhs_host on both sides; per field and
 * direction the box goes as four cudaMemcpy3DAsync copies (the ky, kz index ranges [0, b] and [N - b, N)), all on
 * `stream`, which is synchronised before the call returns.  psfft_host_box_bytes = bytes per field and direction.
 *   h_uhat  in   3 dense spectral fields; only the box is read
 *   h_rhs   out  3 dense spectral fields; ONLY THE BOX IS WRITTEN.  Everything outside it is an exact zero of the
 *                result and is never touched: zero the array once before its first use (not once per call)
 *   d_in, d_out  device staging of 3 spectral fields each; need no initialisation (what lies outside the mask is
 *                never loaded by the kernels) */
size_t psfft_host_box_bytes(psfft_plan plan);
int psfft_hd_rhs_host_box(psfft_plan plan, const void *h_uhat, void *h_rhs, double nu, void *d_in,
                          void *d_out, void *d_work, void *stream);

/* ---- Slab-decomposed transform over P GPUs (Sec. 2, Fig. 1) ------------------------------------
 * The paper's decomposition: task p of P owns the z-slab of Mz = Nz / P planes.  Forward: (1) local 2D transform
 * (x, y) of the slab, (2) global transpose -- the all-to-all, "the only communication involved" -- (3)
 * local 1D transform along z of data that is now x-incomplete.  Here task q ends up with the x-slab
 *     [kz = 0..Nz)[ky = 0..Ny)[kx = x0[q]..x0[q+1])    (row pitch w_q = x0[q+1] - x0[q], x0[q] = floor(q ldk / P))
 * in the natural (not transposed) order.  Steps (1)+(2) are one call: the y-pass stores every finished column
 * straight into the block of the task that owns its kx -- no pack buffer, no local transpose, no unpack.
 *   d_blocks   HOST array of P DEVICE pointers; d_blocks[q] = where the block of rank q lives, addressed as
 *              [zoff + local plane][ky][kx - x0[q]] with pitch w_q.  Two ways to use it:
 *                direct:  d_blocks[q] = rank q's x-slab mapped into this process (NVLink peer / symmetric memory),
 *                         zoff = rank * Mz.  The stores are the all-to-all; the caller only has to make sure every
 *                         rank's phase 1 is complete (stream sync + barrier) before any rank starts phase 2.
 *                packed:  d_blocks[q] = a send buffer + sum_{q' < q} Mz Ny w_q' elements, zoff = 0; then ONE all-to-all of
 *                         contiguous slices (e.g. NCCL all_to_all_single with those split sizes) into the x-slab buffer,
 *                         whose layout [sender p][Mz][Ny][w] is already [Nz][Ny][w].
 * One field per call.  The results are bit for bit those of psfft_fft3d_r2c / c2r on the same data (same kernels,
 * same butterfly order per column).  Inverse: psfft_slab_z(dir = +1) on the x-slab, exchange (direct: nothing to do;
 * packed: all-to-all of the contiguous z-ranges [p Mz, (p+1) Mz) of the x-slabs), then psfft_slab_c2r_yx, whose y-pass
 * loads its columns from the blocks.
 * Returns PSFFT_E_SIZE unless 1 <= P <= PSFFT_MAX_RANKS, P divides Nz, P <= ldk, 0 <= rank < P, and (phase calls)
 * 0 <= zoff and zoff + Mz <= Nz: a block is at most an x-slab of Nz planes, and in direct mode it is another rank's
 * memory, so a plane range past its end is refused rather than stored.  The overlap check of these calls covers the
 * planes [zoff, zoff + Mz) of every block as well: the blocks must be disjoint from one another (r2c_xy writes them) and
 * from d_zspec / d_real_slab (PSFFT_E_OVERLAP otherwise). */
#define PSFFT_MAX_RANKS 16
typedef struct psfft_slab_layout {
    int P, rank;
    int Mz, z0;                  /* planes of this rank's z-slab, first global plane */
    int w;                       /* kx columns of this rank's x-slab */
    int x0[PSFFT_MAX_RANKS + 1]; /* kx range of every rank: [x0[q], x0[q+1]) */
    size_t real_elems, real_bytes;    /* z-slab in physical space: Mz Ny Nx reals */
    size_t zspec_elems, zspec_bytes;  /* z-slab after the x-pass: Mz Ny ldk complex (work buffer of phase 1) */
    size_t xslab_elems, xslab_bytes;  /* this rank's x-slab: Nz Ny w complex */
} psfft_slab_layout;
int psfft_slab_query(psfft_plan plan, int P, int rank, psfft_slab_layout *out);
/* forward phase 1: x-pass (r2c) of the z-slab into d_zspec (overwritten work buffer), y-pass from d_zspec into the blocks */
int psfft_slab_r2c_xy(psfft_plan plan, int P, int rank, const void *d_real_slab, void *d_zspec, void *const *d_blocks,
                      long zoff, void *stream);
/* forward phase 2 (dir = -1) / inverse phase 1 (dir = +1): z-pass of this rank's x-slab, in place, unnormalised */
int psfft_slab_z(psfft_plan plan, int P, int rank, int dir, void *d_xslab, void *stream);
/* inverse phase 2: y-pass loading from the blocks into d_zspec, then the c2r x-pass (scaled 1/(Nx Ny Nz)) into the z-slab */
int psfft_slab_c2r_yx(psfft_plan plan, int P, int rank, void *const *d_blocks, long zoff, void *d_zspec,
                      void *d_real_slab, void *stream);

/* Per-launch timing for measurement (bench.py's roofline object).  While enabled, every kernel an
 * execute call enqueues is bracketed by two CUDA events recorded on the launching stream (so the
 * call is then NOT graph-capturable).  psfft_profile_get synchronises on record i's stop event and
 * returns the kernel kind (name via psfft_kernel_name), its device time in ms and the ALGORITHMIC
 * bytes of that launch (compulsory reads + writes of the pass).
 * Records accumulate until psfft_profile_reset. */
int psfft_profile_enable(psfft_plan plan, int on);
int psfft_profile_reset(psfft_plan plan);
int psfft_profile_count(psfft_plan plan);
int psfft_profile_get(psfft_plan plan, int i, int *kind, double *ms, double *bytes);
const char *psfft_kernel_name(int kind);

/* Number of kernels the last execute call on this plan enqueued (bench.py's gpu_launches). */
int psfft_last_launch_count(psfft_plan plan);

/* Text for a return code (negative: PSFFT_E_*; positive: cudaGetErrorString). */
const char *psfft_strerror(int code);

/* Library version, "major.minor". */
const char *psfft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSFFT_H */
