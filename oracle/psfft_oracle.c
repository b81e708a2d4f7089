/*
 * psfft_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct double-precision implementation of what the hot path
 * of arxiv 1808.01309 computes: the unnormalised 3D real-to-complex DFT of PAPER.md:62
 * (Sec. 2, Eq. 8), its complex-to-real inverse, and one pseudospectral
 * Navier-Stokes / MHD / Boussinesq right-hand side (Eqs. 1-6).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code, header, table or helper with the CUDA path under
 * paper_1808_01309_b200/csrc/.  No blocking, no fusion, no real-FFT trick: every function
 * is the definition (or the paper's three-step algorithm) written out.
 * OpenMP is used only to spread independent pencils / output points over host cores.
 *
 * Parity pins (tests/test_oracle_*.py): brute-force O(N^6) DFT, single mode -> exact bin,
 * Parseval, round trip, numpy pocketfft, closed-form derivative, Taylor-Green closed form,
 * ABC null test, energy/helicity invariants, mask counts, grid independence; for the Boussinesq
 * right-hand side (tests/test_oracle_boussinesq.py): theta = 0 -> O6, Taylor-Green + sin x closed
 * form, hydrostatic balance, the N_bv w source, total-energy conservation, numpy restatement.  Every
 * exported function below is pinned by at least one of them; none is "parity unpinned".
 *
 * Conventions: real field [z][y][x], x contiguous; half spectrum
 * [kz][ky][kx], kx in [0, Nx/2]; forward sign -, unnormalised; inverse sign +, scaled by
 * 1/(Nx Ny Nz); wavenumbers k_i = n_i (2 pi / L_i) with n_i = p (p < N_i/2) or p - N_i (p >= N_i/2):
 * the integers themselves in the 2 pi-periodic box of every BASELINE.json config; the general grid
 * (Nx, Ny, Nz) and box (Lx, Ly, Lz) of PAPER.md:64 through the *3 entry points (pins:
 * tests/test_oracle_aniso.py).
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

static const double TWO_PI = 6.283185307179586476925286766559;

/* ---------------------------------------------------------------------------------------
 * thread control (bench.py reports the count it used)
 * ------------------------------------------------------------------------------------- */
int orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

int orc_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* w_n^m = exp(sign * 2 pi i m / n) from the REDUCED integer m (no recurrence). */
static cplx root(int n, long m, int sign)
{
    m %= n;
    if (m < 0) m += n;
    double a = TWO_PI * (double)m / (double)n;
    return cos(a) + I * (sign * sin(a));
}

/* table of w_n^m, m = 0..n-1, each entry computed directly as above */
static cplx *root_table(int n, int sign)
{
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (int m = 0; m < n; ++m) t[m] = root(n, m, sign);
    return t;
}

/* ---------------------------------------------------------------------------------------
 * O1  dft1d_direct: X[p] = sum_j x[j] w^(p j mod n), w = exp(sign 2 pi i / n).
 *     Eq. 8 restricted to one axis.  O(n^2).
 * ------------------------------------------------------------------------------------- */
void orc_dft1d_direct(int n, int sign, const cplx *x, long xs, cplx *X, long Xs)
{
    for (int p = 0; p < n; ++p) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) acc += x[j * xs] * root(n, (long)p * j, sign);
        X[p * Xs] = acc;
    }
}

/* ---------------------------------------------------------------------------------------
 * O2  fft1d: recursive decimation in time over the smallest prime factor; the p-point
 *     combination step is O1 with the root table of the top-level n; prime n falls back
 *     to O1.  ("naive radix-2 / mixed-radix FFT", BASELINE.json north_star.)
 *     tab = root_table(ntop, sign); step = ntop / n so that w_n^m = tab[(m*step) % ntop].
 * ------------------------------------------------------------------------------------- */
static int smallest_factor(int n)
{
    if (n % 2 == 0) return 2;
    for (int f = 3; (long)f * f <= n; f += 2)
        if (n % f == 0) return f;
    return n;
}

static void fft_rec(int n, const cplx *in, long is, cplx *out, cplx *scratch,
                    const cplx *tab, int ntop)
{
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_factor(n);
    int m = n / p;
    long step = ntop / n;
    if (p == n) { /* prime length: direct definition */
        for (int q = 0; q < n; ++q) {
            cplx acc = 0.0;
            for (int j = 0; j < n; ++j) acc += in[j * is] * tab[(((long)q * j) % n) * step];
            out[q] = acc;
        }
        return;
    }
    /* sub-transforms of the p decimated sequences x[r], x[r+p], ... -> scratch[r*m ..] */
    for (int r = 0; r < p; ++r)
        fft_rec(m, in + r * is, is * p, scratch + (long)r * m, out + (long)r * m, tab, ntop);
    /* X[k + m q] = sum_r w_n^{r (k + m q)} T_r[k] */
    for (int k = 0; k < m; ++k)
        for (int q = 0; q < p; ++q) {
            cplx acc = 0.0;
            long idx = k + (long)m * q;
            for (int r = 0; r < p; ++r) acc += scratch[(long)r * m + k] * tab[((r * idx) % n) * step];
            out[idx] = acc;
        }
}

/* public O2: strided in, strided out; allocates its own table and scratch */
void orc_fft1d(int n, int sign, const cplx *x, long xs, cplx *X, long Xs)
{
    cplx *tab = root_table(n, sign);
    cplx *out = (cplx *)malloc(sizeof(cplx) * (size_t)n * 2);
    fft_rec(n, x, xs, out, out + n, tab, n);
    for (int i = 0; i < n; ++i) X[i * Xs] = out[i];
    free(out);
    free(tab);
}

/* in-place transform of `count` pencils of length n, element stride es; pencil c starts at
 * base + off[c] where off is given by (c / inner)*outer_s + (c % inner)*inner_s */
static void fft_pencils(cplx *base, int n, int sign, long es, long count, long inner,
                        long inner_s, long outer_s)
{
    cplx *tab = root_table(n, sign);
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)n * 2);
#pragma omp for schedule(static)
        for (long c = 0; c < count; ++c) {
            cplx *p = base + (c / inner) * outer_s + (c % inner) * inner_s;
            fft_rec(n, p, es, buf, buf + n, tab, n);
            for (int i = 0; i < n; ++i) p[i * es] = buf[i];
        }
        free(buf);
    }
    free(tab);
}

/* ---------------------------------------------------------------------------------------
 * O3  r2c3d: X[r,q,p] = sum_{k,j,i} x[k,j,i] exp(-2 pi i (p i/Nx + q j/Ny + r k/Nz)),
 *     p in [0, Nx/2]  (Eq. 8; half spectrum PAPER.md:79).
 *     The paper's three steps: transform along x and y in every plane,
 *     then along z.  Real data is promoted to complex; no real-FFT trick.  Only the kept
 *     columns p <= Nx/2 are carried through the y and z steps.
 * ------------------------------------------------------------------------------------- */
void orc_r2c3d(int Nz, int Ny, int Nx, const double *x, cplx *X)
{
    int H = Nx / 2 + 1;
    cplx *tab = root_table(Nx, -1);
#pragma omp parallel
    {
        cplx *row = (cplx *)malloc(sizeof(cplx) * (size_t)Nx * 3);
#pragma omp for schedule(static)
        for (long zy = 0; zy < (long)Nz * Ny; ++zy) {
            const double *src = x + zy * Nx;
            for (int i = 0; i < Nx; ++i) row[i] = src[i];
            fft_rec(Nx, row, 1, row + Nx, row + 2 * Nx, tab, Nx);
            for (int p = 0; p < H; ++p) X[zy * H + p] = row[Nx + p];
        }
        free(row);
    }
    free(tab);
    /* y: pencils at fixed (z, p), element stride H */
    fft_pencils(X, Ny, -1, H, (long)Nz * H, H, 1, (long)Ny * H);
    /* z: pencils at fixed (q, p), element stride Ny*H */
    fft_pencils(X, Nz, -1, (long)Ny * H, (long)Ny * H, (long)Ny * H, 1, 0);
}

/* ---------------------------------------------------------------------------------------
 * O4  c2r3d: inverse along z, then y, on the half spectrum; then per row the real
 *     synthesis  x[i] = (1/Ntot) [ Re Y0 + (-1)^i Re Y_{Nx/2}
 *                                   + 2 sum_{p=1}^{Nx/2-1} Re( Y_p e^{+2 pi i p i/Nx} ) ],
 *     evaluated as the inverse complex transform of the Hermitian-extended row
 *     (Y_{Nx-p} = conj Y_p, imaginary parts of Y_0 and Y_{Nx/2} dropped), which is the
 *     same sum term by term.  PAPER.md:79 ("the reverse transform essentially reverses
 *     these steps to produce a real physical space field"); 1/N^3 from BASELINE.json
 *     config 1.  Defined for ANY half spectrum, Hermitian-consistent or not.
 *     X is not modified.
 * ------------------------------------------------------------------------------------- */
void orc_c2r3d(int Nz, int Ny, int Nx, const cplx *X, double *x)
{
    int H = Nx / 2 + 1;
    size_t nspec = (size_t)Nz * Ny * H;
    cplx *Y = (cplx *)malloc(sizeof(cplx) * nspec);
    memcpy(Y, X, sizeof(cplx) * nspec);
    fft_pencils(Y, Nz, +1, (long)Ny * H, (long)Ny * H, (long)Ny * H, 1, 0);
    fft_pencils(Y, Ny, +1, H, (long)Nz * H, H, 1, (long)Ny * H);
    double scale = 1.0 / ((double)Nx * (double)Ny * (double)Nz);
    cplx *tab = root_table(Nx, +1);
#pragma omp parallel
    {
        cplx *row = (cplx *)malloc(sizeof(cplx) * (size_t)Nx * 3);
#pragma omp for schedule(static)
        for (long zy = 0; zy < (long)Nz * Ny; ++zy) {
            const cplx *src = Y + zy * H;
            row[0] = creal(src[0]);
            for (int p = 1; p < H; ++p) {
                if (2 * p == Nx) row[p] = creal(src[p]);
                else { row[p] = src[p]; row[Nx - p] = conj(src[p]); }
            }
            fft_rec(Nx, row, 1, row + Nx, row + 2 * Nx, tab, Nx);
            for (int i = 0; i < Nx; ++i) x[zy * Nx + i] = creal(row[Nx + i]) * scale;
        }
        free(row);
    }
    free(tab);
    free(Y);
}

/* ---------------------------------------------------------------------------------------
 * O5  dft3d_bruteforce: the triple sum of Eq. 8 for every output, O(N^6).
 *     Full spectrum [r][q][p], p in [0, Nx).  Small grids only.
 *     orc_r2c3d_mode: the same triple sum for ONE output (sampled parity at full size).
 * ------------------------------------------------------------------------------------- */
static cplx dft3d_point(int Nz, int Ny, int Nx, const double *x, int r, int q, int p)
{
    cplx acc = 0.0;
    for (int k = 0; k < Nz; ++k) {
        cplx wk = root(Nz, (long)r * k, -1);
        cplx accy = 0.0;
        for (int j = 0; j < Ny; ++j) {
            cplx wj = root(Ny, (long)q * j, -1);
            cplx accx = 0.0;
            const double *row = x + ((long)k * Ny + j) * Nx;
            for (int i = 0; i < Nx; ++i) accx += row[i] * root(Nx, (long)p * i, -1);
            accy += accx * wj;
        }
        acc += accy * wk;
    }
    return acc;
}

void orc_r2c3d_mode(int Nz, int Ny, int Nx, const double *x, int r, int q, int p, double *out2)
{
    /* same sum as dft3d_point with the x-roots tabulated once (large grids) and the
     * z-planes spread over threads */
    cplx *tx = root_table(Nx, -1);
    double accr = 0.0, acci = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : accr, acci)
    for (int k = 0; k < Nz; ++k) {
        cplx wk = root(Nz, (long)r * k, -1);
        cplx accy = 0.0;
        for (int j = 0; j < Ny; ++j) {
            cplx wj = root(Ny, (long)q * j, -1);
            cplx accx = 0.0;
            const double *row = x + ((long)k * Ny + j) * Nx;
            for (int i = 0; i < Nx; ++i) accx += row[i] * tx[((long)p * i) % Nx];
            accy += accx * wj;
        }
        cplx t = accy * wk;
        accr += creal(t);
        acci += cimag(t);
    }
    free(tx);
    out2[0] = accr;
    out2[1] = acci;
}

void orc_dft3d_bruteforce(int Nz, int Ny, int Nx, const double *x, cplx *X)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int r = 0; r < Nz; ++r)
        for (int q = 0; q < Ny; ++q)
            for (int p = 0; p < Nx; ++p)
                X[((long)r * Ny + q) * Nx + p] = dft3d_point(Nz, Ny, Nx, x, r, q, p);
}

/* brute-force inverse for ONE physical point from a FULL complex spectrum [r][q][p]:
 * x[k,j,i] = (1/Ntot) sum X[r,q,p] e^{+2 pi i (...)}  (Eq. 8 with the sign changed) */
void orc_idft3d_point(int Nz, int Ny, int Nx, const cplx *X, int k, int j, int i, double *out2)
{
    cplx acc = 0.0;
    for (int r = 0; r < Nz; ++r)
        for (int q = 0; q < Ny; ++q)
            for (int p = 0; p < Nx; ++p)
                acc += X[((long)r * Ny + q) * Nx + p] * root(Nz, (long)r * k, +1) *
                       root(Ny, (long)q * j, +1) * root(Nx, (long)p * i, +1);
    acc /= ((double)Nx * Ny * Nz);
    out2[0] = creal(acc);
    out2[1] = cimag(acc);
}

/* ---------------------------------------------------------------------------------------
 * Grid and box.  PAPER.md:64 (Sec. 2, below Eq. 8): "both the physical box size, L_i, and the number of
 * physical space points, N_i, may be specified independently in each direction".
 *   wavenumbers   k_i = n_i (2 pi / L_i), n_i the integer index p (p < N_i/2) or p - N_i (DESIGN.md
 *                 reading G24; the factor 2 pi / L_i is evaluated once in fp64 and is exactly 1 for L_i = 2 pi)
 *   2/3 rule      ellipsoidal truncation in INDEX space, sum_i (n_i / N_i)^2 < 1/9, whatever the box
 *                 (reading G25), evaluated in integers: with L = lcm(Nx, Ny, Nz) and r_i = L / N_i,
 *                 keep iff 9 sum_i (r_i n_i)^2 < L^2.  For Nx = Ny = Nz = N this is 9 |n|^2 < N^2 (G4).
 * The cubic 2 pi box (every BASELINE.json config) is the special case r_i = 1, k_i = n_i.
 * ------------------------------------------------------------------------------------- */
typedef struct {
    int Nx, Ny, Nz, H;      /* H = Nx/2 + 1 */
    long nf, nr;            /* modes of a half spectrum, points of a real field */
    double kfx, kfy, kfz;   /* 2 pi / L_i */
    long rx, ry, rz, L;     /* L = lcm(Nx, Ny, Nz), r_i = L / N_i */
} grid_t;

static long gcd_l(long a, long b) { while (b) { long t = a % b; a = b; b = t; } return a; }

static grid_t grid_make(int Nz, int Ny, int Nx, const double *box /* Lx, Ly, Lz; NULL = 2 pi each */)
{
    grid_t g;
    g.Nx = Nx; g.Ny = Ny; g.Nz = Nz; g.H = Nx / 2 + 1;
    g.nf = (long)Nz * Ny * g.H;
    g.nr = (long)Nz * Ny * Nx;
    g.kfx = box ? TWO_PI / box[0] : 1.0;
    g.kfy = box ? TWO_PI / box[1] : 1.0;
    g.kfz = box ? TWO_PI / box[2] : 1.0;
    long l = (long)Nx / gcd_l(Nx, Ny) * Ny;
    g.L = l / gcd_l(l, Nz) * Nz;
    g.rx = g.L / Nx; g.ry = g.L / Ny; g.rz = g.L / Nz;
    return g;
}

static inline int wavenumber(int idx, int n) { return idx < n / 2 ? idx : idx - n; } /* n/2 -> -n/2 (G8) */

/* a9: 2/3-rule truncation, integer arithmetic (G4, G25) */
static inline int keep_mode(const grid_t *g, int nx, int ny, int nz)
{
    long a = g->rx * nx, b = g->ry * ny, c = g->rz * nz;
    return 9 * (a * a + b * b + c * c) < g->L * g->L;
}

/* loop over the half spectrum: o = linear index, (kx, ky, kz) = real wavenumbers, keep = mask bit */
#define FOR_MODES(g)                                                         \
    _Pragma("omp parallel for schedule(static)")                             \
    for (int r = 0; r < (g)->Nz; ++r)                                        \
        for (int q = 0; q < (g)->Ny; ++q)                                    \
            for (int p = 0; p < (g)->H; ++p)
#define MODE_VARS(g)                                                         \
    const long o = ((long)r * (g)->Ny + q) * (g)->H + p;                     \
    const int nx = p, ny = wavenumber(q, (g)->Ny), nz = wavenumber(r, (g)->Nz); \
    const double kx = nx * (g)->kfx, ky = ny * (g)->kfy, kz = nz * (g)->kfz; \
    (void)o; (void)kx; (void)ky; (void)kz;

static void dealias_mask_g(const grid_t *g, unsigned char *mask)
{
    FOR_MODES(g) { MODE_VARS(g) mask[o] = (unsigned char)keep_mode(g, nx, ny, nz); }
}

/* step 1 / step 6 of O6: f <- M f; masked entries become +0.0 (both parts) */
static void apply_mask_g(const grid_t *g, int ncomp, cplx *f)
{
    FOR_MODES(g) {
        MODE_VARS(g)
        if (!keep_mode(g, nx, ny, nz))
            for (int c = 0; c < ncomp; ++c) f[c * g->nf + o] = 0.0;
    }
}

/* a7: w = i k x u  (w_x = i (k_y u_z - k_z u_y), cyclic) */
static void curl_g(const grid_t *g, const cplx *u, cplx *w)
{
    const long nf = g->nf;
    FOR_MODES(g) {
        MODE_VARS(g)
        cplx ux = u[o], uy = u[nf + o], uz = u[2 * nf + o];
        w[o] = I * (ky * uz - kz * uy);
        w[nf + o] = I * (kz * ux - kx * uz);
        w[2 * nf + o] = I * (kx * uy - ky * ux);
    }
}

/* a10: f <- f - k (k.f)/|k|^2 for k != 0; identity at k = 0 (G6, G7) */
static void project_g(const grid_t *g, cplx *f)
{
    const long nf = g->nf;
    FOR_MODES(g) {
        MODE_VARS(g)
        double k2 = kx * kx + ky * ky + kz * kz;
        if (k2 == 0.0) continue;
        cplx d = (kx * f[o] + ky * f[nf + o] + kz * f[2 * nf + o]) / k2;
        f[o] -= kx * d;
        f[nf + o] -= ky * d;
        f[2 * nf + o] -= kz * d;
    }
}

/* a11: f <- f - nu |k|^2 u */
static void add_diffusion(const grid_t *g, double nu, const cplx *u, cplx *f)
{
    const long nf = g->nf;
    FOR_MODES(g) {
        MODE_VARS(g)
        double k2 = kx * kx + ky * ky + kz * kz;
        for (int c = 0; c < 3; ++c) f[c * nf + o] -= nu * k2 * u[c * nf + o];
    }
}

/* a8: c = a x b pointwise on n points, 3-component fields laid out [3][n] */
static void cross_add(long n, const double *a, const double *b, double *c, int accumulate)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) {
        double ax = a[i], ay = a[n + i], az = a[2 * n + i];
        double bx = b[i], by = b[n + i], bz = b[2 * n + i];
        double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;
        if (accumulate) { c[i] += cx; c[n + i] += cy; c[2 * n + i] += cz; }
        else { c[i] = cx; c[n + i] = cy; c[2 * n + i] = cz; }
    }
}

static void inv3(const grid_t *g, const cplx *X, double *x) { orc_c2r3d(g->Nz, g->Ny, g->Nx, X, x); }
static void fwd3(const grid_t *g, const double *x, cplx *X) { orc_r2c3d(g->Nz, g->Ny, g->Nx, x, X); }

/* ---------------------------------------------------------------------------------------
 * O6  hd_rhs(uhat, nu) = M P F[ F^-1(M uhat) x F^-1(i k x M uhat) ] - nu |k|^2 M uhat
 *     (Eq. 1 with theta = 0, Eq. 3; nonlinear term in physical
 *     space, projection in spectral space; rotational form, 2/3 rule and the transform
 *     count 6 + 3 from BASELINE.json config 2).  Steps 1-8 of SURVEY.md §8(c) O6.
 *     uhat, rhs: [3][kz][ky][kx], values = (Nx Ny Nz) x Fourier coefficient.
 * ------------------------------------------------------------------------------------- */
static void hd_rhs_g(const grid_t *g, const cplx *uhat, double nu, cplx *rhs)
{
    const long nf = g->nf, nr = g->nr;
    cplx *um = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    cplx *wh = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    double *u = (double *)malloc(sizeof(double) * 3 * nr);
    double *w = (double *)malloc(sizeof(double) * 3 * nr);
    memcpy(um, uhat, sizeof(cplx) * 3 * nf);
    apply_mask_g(g, 3, um);                                     /* 1 */
    curl_g(g, um, wh);                                          /* 2 */
    for (int c = 0; c < 3; ++c) {                               /* 3 */
        inv3(g, um + c * nf, u + c * nr);
        inv3(g, wh + c * nf, w + c * nr);
    }
    free(wh);
    double *n = (double *)malloc(sizeof(double) * 3 * nr);
    cross_add(nr, u, w, n, 0);                                  /* 4 */
    free(u);
    free(w);
    for (int c = 0; c < 3; ++c) fwd3(g, n + c * nr, rhs + c * nf); /* 5 */
    free(n);
    apply_mask_g(g, 3, rhs);                                    /* 6 */
    project_g(g, rhs);                                          /* 7 */
    if (nu != 0.0) add_diffusion(g, nu, um, rhs);               /* 8 */
    free(um);
}

/* ---------------------------------------------------------------------------------------
 * O7  mhd_rhs (Eqs. 4-6, "v" in Eq. 5 read as u; BASELINE.json config 5):
 *     w = curl u, j = curl b;  m = u x w + j x b;  e = u x b;
 *     R_u = M P F[m] - nu |k|^2 M uhat;   R_b = M i k x F[e] - eta |k|^2 M bhat.
 *     (B.grad B - grad(p + |B|^2/2) = j x b under the projection, as for u.)
 * ------------------------------------------------------------------------------------- */
static void mhd_rhs_g(const grid_t *g, const cplx *uhat, const cplx *bhat, double nu, double eta, cplx *ru,
                      cplx *rb)
{
    const long nf = g->nf, nr = g->nr;
    cplx *um = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    cplx *bm = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    cplx *th = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    double *u = (double *)malloc(sizeof(double) * 3 * nr);
    double *b = (double *)malloc(sizeof(double) * 3 * nr);
    double *t = (double *)malloc(sizeof(double) * 3 * nr);
    double *m = (double *)malloc(sizeof(double) * 3 * nr);
    memcpy(um, uhat, sizeof(cplx) * 3 * nf);
    memcpy(bm, bhat, sizeof(cplx) * 3 * nf);
    apply_mask_g(g, 3, um);
    apply_mask_g(g, 3, bm);
    for (int c = 0; c < 3; ++c) {
        inv3(g, um + c * nf, u + c * nr);
        inv3(g, bm + c * nf, b + c * nr);
    }
    curl_g(g, um, th);                                     /* w^ */
    for (int c = 0; c < 3; ++c) inv3(g, th + c * nf, t + c * nr);
    cross_add(nr, u, t, m, 0);                             /* m = u x w */
    curl_g(g, bm, th);                                     /* j^ */
    for (int c = 0; c < 3; ++c) inv3(g, th + c * nf, t + c * nr);
    cross_add(nr, t, b, m, 1);                             /* m += j x b */
    cross_add(nr, u, b, t, 0);                             /* e = u x b */
    free(u);
    free(b);
    for (int c = 0; c < 3; ++c) fwd3(g, m + c * nr, ru + c * nf);
    for (int c = 0; c < 3; ++c) fwd3(g, t + c * nr, th + c * nf);
    free(m);
    free(t);
    apply_mask_g(g, 3, ru);
    project_g(g, ru);
    if (nu != 0.0) add_diffusion(g, nu, um, ru);
    apply_mask_g(g, 3, th);
    curl_g(g, th, rb);
    if (eta != 0.0) add_diffusion(g, eta, bm, rb);
    free(th);
    free(um);
    free(bm);
}

/* ---------------------------------------------------------------------------------------
 * O8  boussinesq_rhs (Eqs. 1-3, the paper's reference equations):
 *       d_t u     = -grad p - u.grad u - N_bv theta z^ + nu Lap u      (Eq. 1)
 *       d_t theta = -u.grad theta + N_bv w + kappa Lap theta           (Eq. 2),  div u = 0 (Eq. 3)
 *     Nonlinear terms in physical space, pressure by projection in spectral space.
 *     Step by step (rotational form for the momentum term as in O6, reading G5):
 *       1. um = M u^, tm = M theta^                       (2/3-rule mask on load)
 *       2. w^ = i k x um;  g^ = i k tm                    (curl and gradient in spectral space)
 *       3. u, w, g = c2r3d(.)                             (9 inverse transforms)
 *       4. n = u x w;  s = u . g                          (pointwise)
 *       5. n^ = r2c3d(n) (3), s^ = r2c3d(s) (1)           (4 forward transforms)
 *       6. n^ <- M n^, s^ <- M s^
 *       7. n^_z <- n^_z - N_bv tm;  n^ <- P n^            (buoyancy is inside the projection: Eq. 1)
 *       8. R_u = n^ - nu |k|^2 um
 *       9. R_th = -s^ + N_bv um_z - kappa |k|^2 tm
 *     uhat, ru: [3][kz][ky][kx]; thhat, rt: [kz][ky][kx]; values = (Nx Ny Nz) x Fourier coefficient.
 * ------------------------------------------------------------------------------------- */
static void boussinesq_rhs_g(const grid_t *g, const cplx *uhat, const cplx *thhat, double nu, double kappa,
                             double nbv, cplx *ru, cplx *rt)
{
    const long nf = g->nf, nr = g->nr;
    cplx *um = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    cplx *tm = (cplx *)malloc(sizeof(cplx) * nf);
    cplx *wh = (cplx *)malloc(sizeof(cplx) * 3 * nf);
    double *u = (double *)malloc(sizeof(double) * 3 * nr);
    double *w = (double *)malloc(sizeof(double) * 3 * nr);
    memcpy(um, uhat, sizeof(cplx) * 3 * nf);
    memcpy(tm, thhat, sizeof(cplx) * nf);
    apply_mask_g(g, 3, um);                                     /* 1 */
    apply_mask_g(g, 1, tm);
    curl_g(g, um, wh);                                          /* 2 (curl) */
    for (int c = 0; c < 3; ++c) {                               /* 3 (u, w) */
        inv3(g, um + c * nf, u + c * nr);
        inv3(g, wh + c * nf, w + c * nr);
    }
    double *n = (double *)malloc(sizeof(double) * 3 * nr);
    cross_add(nr, u, w, n, 0);                                  /* 4 (n = u x w) */
    FOR_MODES(g) {                                              /* 2 (gradient), reusing wh */
        MODE_VARS(g)
        wh[o] = I * kx * tm[o];
        wh[nf + o] = I * ky * tm[o];
        wh[2 * nf + o] = I * kz * tm[o];
    }
    for (int c = 0; c < 3; ++c) inv3(g, wh + c * nf, w + c * nr);   /* 3 (g) */
    free(wh);
    double *s = (double *)malloc(sizeof(double) * nr);
#pragma omp parallel for schedule(static)                       /* 4 (s = u . g) */
    for (long i = 0; i < nr; ++i) s[i] = u[i] * w[i] + u[nr + i] * w[nr + i] + u[2 * nr + i] * w[2 * nr + i];
    free(u);
    free(w);
    for (int c = 0; c < 3; ++c) fwd3(g, n + c * nr, ru + c * nf);   /* 5 */
    fwd3(g, s, rt);
    free(n);
    free(s);
    apply_mask_g(g, 3, ru);                                     /* 6 */
    apply_mask_g(g, 1, rt);
    for (long o = 0; o < nf; ++o) ru[2 * nf + o] -= nbv * tm[o];               /* 7 */
    project_g(g, ru);
    if (nu != 0.0) add_diffusion(g, nu, um, ru);                /* 8 */
    FOR_MODES(g) {                                              /* 9 */
        MODE_VARS(g)
        double k2 = kx * kx + ky * ky + kz * kz;
        rt[o] = -rt[o] + nbv * um[2 * nf + o] - kappa * k2 * tm[o];
    }
    free(um);
    free(tm);
}

/* ---------------------------------------------------------------------------------------
 * O10 gpe_rhs: the Gross-Pitaevskii equation, Eq. 7,
 *         i hbar d_t psi = -hbar^2/(2m) Lap psi + g |psi|^2 psi
 *     <=> d_t psi = i alpha Lap psi - i beta |psi|^2 psi,   alpha = hbar/(2m), beta = g/hbar.
 *     The paper counts GPE as "1 complex (or 2 real)" primitive fields: psi = p + i q with
 *     p, q REAL fields carried as two half spectra, like every other field of the framework:
 *         d_t p = -alpha Lap q + beta (p^2 + q^2) q,      d_t q = alpha Lap p - beta (p^2 + q^2) p.
 *     Step by step (nonlinear term in physical space; 2/3-rule mask as for the other
 *     solvers, reading G23):
 *       1. pm = M p^, qm = M q^
 *       2. p, q = c2r3d(pm), c2r3d(qm)                        (2 inverse transforms)
 *       3. a = (p^2 + q^2) q,  b = (p^2 + q^2) p              (pointwise)
 *       4. a^ = M r2c3d(a),  b^ = M r2c3d(b)                  (2 forward transforms)
 *       5. R_p = beta a^ + alpha |k|^2 qm,   R_q = -beta b^ - alpha |k|^2 pm
 *     psihat, rhs: [2][kz][ky][kx] = (p^, q^); values = (Nx Ny Nz) x Fourier coefficient.
 * ------------------------------------------------------------------------------------- */
static void gpe_rhs_g(const grid_t *g, const cplx *psihat, double alpha, double beta, cplx *rhs)
{
    const long nf = g->nf, nr = g->nr;
    cplx *pm = (cplx *)malloc(sizeof(cplx) * 2 * nf);
    double *p = (double *)malloc(sizeof(double) * 2 * nr);
    double *a = (double *)malloc(sizeof(double) * 2 * nr);
    memcpy(pm, psihat, sizeof(cplx) * 2 * nf);
    apply_mask_g(g, 2, pm);                                              /* 1 */
    for (int c = 0; c < 2; ++c) inv3(g, pm + c * nf, p + c * nr);        /* 2 */
#pragma omp parallel for schedule(static)                                /* 3 */
    for (long i = 0; i < nr; ++i) {
        double rho = p[i] * p[i] + p[nr + i] * p[nr + i];
        a[i] = rho * p[nr + i];
        a[nr + i] = rho * p[i];
    }
    free(p);
    for (int c = 0; c < 2; ++c) fwd3(g, a + c * nr, rhs + c * nf);       /* 4 */
    free(a);
    apply_mask_g(g, 2, rhs);
    FOR_MODES(g) {                                                       /* 5 */
        MODE_VARS(g)
        double k2 = kx * kx + ky * ky + kz * kz;
        cplx ra = rhs[o], rb = rhs[nf + o];
        rhs[o] = beta * ra + alpha * k2 * pm[nf + o];
        rhs[nf + o] = -beta * rb - alpha * k2 * pm[o];
    }
    free(pm);
}

/* ---------------------------------------------------------------------------------------
 * O9  rk_step: one explicit Runge-Kutta time step around the right-hand sides above.
 *     "the system of ODEs is solved using an explicit Runge-Kutta scheme (of
 *     2nd-4th order); explicit time stepping is used to resolve all wave modes".  The paper does
 *     not print the scheme; reading G21 takes the low-storage form with `ord` stages
 *         y^(ord) = y_n;   y^(o-1) = M y_n + (dt / o) R(y^(o)),  o = ord, ..., 1;   y_{n+1} = y^(0)
 *     (R = O6 / O7 / O8 / O10, M = the 2/3 mask).  For a linear R = L y this is the degree-`ord` Taylor
 *     polynomial of exp(dt L), i.e. order `ord`; for the nonlinear terms it is second order.
 *     sys: 0 = HD (y = u^, 3 fields), 1 = MHD (y = u^, b^: 6 fields), 2 = Boussinesq (y = u^, theta^: 4),
 *     3 = GPE (y = p^, q^: 2 fields).  par = { nu, eta (MHD) or kappa (Boussinesq), N_bv }; GPE: { alpha, beta }.
 * ------------------------------------------------------------------------------------- */
static void rk_rhs(const grid_t *g, int sys, const double *par, const cplx *y, cplx *r)
{
    const long nf = g->nf;
    if (sys == 0) hd_rhs_g(g, y, par[0], r);
    else if (sys == 1) mhd_rhs_g(g, y, y + 3 * nf, par[0], par[1], r, r + 3 * nf);
    else if (sys == 3) gpe_rhs_g(g, y, par[0], par[1], r);
    else boussinesq_rhs_g(g, y, y + 3 * nf, par[0], par[1], par[2], r, r + 3 * nf);
}

static void rk_step_g(const grid_t *g, int sys, int ord, double dt, const double *par, const cplx *y0, cplx *y1)
{
    int nfields = sys == 0 ? 3 : sys == 1 ? 6 : sys == 3 ? 2 : 4;
    long n = nfields * g->nf;
    cplx *ym = (cplx *)malloc(sizeof(cplx) * n);   /* M y_n */
    cplx *r = (cplx *)malloc(sizeof(cplx) * n);
    memcpy(ym, y0, sizeof(cplx) * n);
    apply_mask_g(g, nfields, ym);
    memcpy(y1, y0, sizeof(cplx) * n);              /* y^(ord) = y_n */
    for (int o = ord; o >= 1; --o) {
        rk_rhs(g, sys, par, y1, r);
        for (long i = 0; i < n; ++i) y1[i] = ym[i] + (dt / o) * r[i];
    }
    free(ym);
    free(r);
}

/* ---------------------------------------------------------------------------------------
 * exported entry points: the cubic 2 pi box (N) and the general grid and box (Nz, Ny, Nx, box = {Lx, Ly, Lz})
 * ------------------------------------------------------------------------------------- */
void orc_dealias_mask(int N, unsigned char *mask) { grid_t g = grid_make(N, N, N, NULL); dealias_mask_g(&g, mask); }
void orc_apply_mask(int N, int ncomp, cplx *f) { grid_t g = grid_make(N, N, N, NULL); apply_mask_g(&g, ncomp, f); }
void orc_curl(int N, const cplx *u, cplx *w) { grid_t g = grid_make(N, N, N, NULL); curl_g(&g, u, w); }
void orc_project(int N, cplx *f) { grid_t g = grid_make(N, N, N, NULL); project_g(&g, f); }
void orc_hd_rhs(int N, const cplx *uhat, double nu, cplx *rhs) { grid_t g = grid_make(N, N, N, NULL); hd_rhs_g(&g, uhat, nu, rhs); }
void orc_mhd_rhs(int N, const cplx *uhat, const cplx *bhat, double nu, double eta, cplx *ru, cplx *rb)
{
    grid_t g = grid_make(N, N, N, NULL);
    mhd_rhs_g(&g, uhat, bhat, nu, eta, ru, rb);
}
void orc_boussinesq_rhs(int N, const cplx *uhat, const cplx *thhat, double nu, double kappa, double nbv, cplx *ru,
                        cplx *rt)
{
    grid_t g = grid_make(N, N, N, NULL);
    boussinesq_rhs_g(&g, uhat, thhat, nu, kappa, nbv, ru, rt);
}
void orc_gpe_rhs(int N, const cplx *psihat, double alpha, double beta, cplx *rhs)
{
    grid_t g = grid_make(N, N, N, NULL);
    gpe_rhs_g(&g, psihat, alpha, beta, rhs);
}
void orc_rk_step(int N, int sys, int ord, double dt, const double *par, const cplx *y0, cplx *y1)
{
    grid_t g = grid_make(N, N, N, NULL);
    rk_step_g(&g, sys, ord, dt, par, y0, y1);
}

void orc_dealias_mask3(int Nz, int Ny, int Nx, unsigned char *mask) { grid_t g = grid_make(Nz, Ny, Nx, NULL); dealias_mask_g(&g, mask); }
void orc_curl3(int Nz, int Ny, int Nx, const double *box, const cplx *u, cplx *w) { grid_t g = grid_make(Nz, Ny, Nx, box); curl_g(&g, u, w); }
void orc_project3(int Nz, int Ny, int Nx, const double *box, cplx *f) { grid_t g = grid_make(Nz, Ny, Nx, box); project_g(&g, f); }
void orc_hd_rhs3(int Nz, int Ny, int Nx, const double *box, const cplx *uhat, double nu, cplx *rhs)
{
    grid_t g = grid_make(Nz, Ny, Nx, box);
    hd_rhs_g(&g, uhat, nu, rhs);
}
void orc_mhd_rhs3(int Nz, int Ny, int Nx, const double *box, const cplx *uhat, const cplx *bhat, double nu, double eta,
                  cplx *ru, cplx *rb)
{
    grid_t g = grid_make(Nz, Ny, Nx, box);
    mhd_rhs_g(&g, uhat, bhat, nu, eta, ru, rb);
}
void orc_boussinesq_rhs3(int Nz, int Ny, int Nx, const double *box, const cplx *uhat, const cplx *thhat, double nu,
                         double kappa, double nbv, cplx *ru, cplx *rt)
{
    grid_t g = grid_make(Nz, Ny, Nx, box);
    boussinesq_rhs_g(&g, uhat, thhat, nu, kappa, nbv, ru, rt);
}
void orc_gpe_rhs3(int Nz, int Ny, int Nx, const double *box, const cplx *psihat, double alpha, double beta, cplx *rhs)
{
    grid_t g = grid_make(Nz, Ny, Nx, box);
    gpe_rhs_g(&g, psihat, alpha, beta, rhs);
}
void orc_rk_step3(int Nz, int Ny, int Nx, const double *box, int sys, int ord, double dt, const double *par,
                  const cplx *y0, cplx *y1)
{
    grid_t g = grid_make(Nz, Ny, Nx, box);
    rk_step_g(&g, sys, ord, dt, par, y0, y1);
}
