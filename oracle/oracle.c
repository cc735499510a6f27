/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path of
 * arxiv/paper_2502_06296 computes: the second-order finite-difference pressure
 * Poisson solve (Eq. 12; steps PAPER.md:124-131) and the
 * wall-normal implicit-diffusion Helmholtz solve (Eq. 11).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header,
 * table or constant generator with the CUDA path under
 * paper_2502_06296_b200/csrc/ and neither includes the other.
 *
 * Both solves are DIRECT solvers of a linear system, so the oracle is the
 * definition of that system written out (readings R1-R6):
 *
 *   Poisson  (L_h phi)_ijk = f_ijk,  sum_ijk dzf_k phi_ijk = 0          [O-P]
 *   (L_h phi)_ijk = (phi_{i+1}-2phi_i+phi_{i-1})/dx^2 + (same in j)/dy^2
 *                 + A_k (phi_{k-1}-phi_k) + C_k (phi_{k+1}-phi_k)
 *   periodic in i,j; A_0 = C_{nz-1} = 0 (zero wall-normal gradient).
 *
 *   Helmholtz  u_k - a [A_k(u_{k-1}-u_k) + C_k(u_{k+1}-u_k) - W_k u_k] = r_k  [O-H]
 *   per (i,j) column, Dirichlet u = 0 on both wall faces (W_k: ghost = -interior).
 *
 * Arrays are C-order p[k][j][i], x fastest.  A_k = 1/(dzf_k dzc_{k-1}),
 * C_k = 1/(dzf_k dzc_k), dzf_k = zf[k+1]-zf[k], dzc_k = zc[k+1]-zc[k].
 *
 * The Poisson route is the paper's own (eigenfunction expansion, Eq. 12):
 * DFT along x, DFT along y, one real tridiagonal solve per (qx,qy) for the real
 * and for the imaginary part, inverse DFTs.  The DFT is either the O(n^2)
 * definition (variant 0) or a textbook recursive radix-2 FFT (variant 1) that
 * tests/ pins against the definition and against numpy.fft.  No blocking,
 * fusion or reordering beyond that.
 *
 * Parity pins (tests/test_oracle_*.py): closed-form discrete eigenfunctions,
 * dense LU on <= 8^3 grids, apply-then-solve round trips, residual and
 * weighted-mean invariants, numpy.fft, Parseval.  No function here is
 * "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ tables */

/* z-metric tables from the double inputs zc[nz], zf[nz+1] (one division each).
 * PAPER.md:88 ("the set of coefficients eta represent the finite-difference
 * discretization of L_z"); reading R2 in DESIGN.md: cell-centred MAC Laplacian,
 * flux difference over cell width.  dzc has nz-1 entries. */
void orc_z_tables(int nz, const double *zc, const double *zf,
                  double *dzf, double *dzc, double *A, double *C)
{
    for (int k = 0; k < nz; ++k) dzf[k] = zf[k + 1] - zf[k];
    for (int k = 0; k + 1 < nz; ++k) dzc[k] = zc[k + 1] - zc[k];
    for (int k = 0; k < nz; ++k) {
        A[k] = (k >= 1) ? 1.0 / (dzf[k] * dzc[k - 1]) : 0.0;
        C[k] = (k + 1 < nz) ? 1.0 / (dzf[k] * dzc[k]) : 0.0;
    }
}

/* Modified wavenumbers, PAPER.md:88 ("second-order accurate eigenvalues"),
 * natural order q = 0..n-1:  lambda_q / Delta^2 = -4 sin^2(pi q / n) / Delta^2
 * (reading R1/R6: never the 2cos-2 form).  Delta = L / n. */
void orc_lambda(int n, double L, double *lam)
{
    const double delta = L / (double)n;
    for (int q = 0; q < n; ++q) {
        /* lambda_{n-q} = lambda_q exactly; fold so the sine argument stays in [0, pi/2] */
        const int qf = (q <= n - q) ? q : n - q;
        const double s = sin(ORC_PI * (double)qf / (double)n);
        lam[q] = -4.0 * s * s / (delta * delta);
    }
}

/* --------------------------------------------------------------------- DFT */

/* Definition-level DFT of one complex line with stride:
 *   X_q = sum_i x_i exp(sign * 2 pi i (q*i mod n) / n),  sign = -1 forward, +1 inverse
 * (no 1/n).  O(n^2).  Scratch-free: out must not alias in. */
void orc_dft_naive(int n, int sign, const double *in_re, const double *in_im,
                   double *out_re, double *out_im)
{
    for (int q = 0; q < n; ++q) {
        double sr = 0.0, si = 0.0;
        for (int i = 0; i < n; ++i) {
            const long long m = ((long long)q * (long long)i) % n;
            const double ang = 2.0 * ORC_PI * (double)m / (double)n;
            const double c = cos(ang), s = sign * sin(ang);
            sr += in_re[i] * c - in_im[i] * s;
            si += in_re[i] * s + in_im[i] * c;
        }
        out_re[q] = sr;
        out_im[q] = si;
    }
}

/* Textbook recursive radix-2 decimation-in-time FFT (n a power of two):
 *   X_q = E_q + w^q O_q,  X_{q+n/2} = E_q - w^q O_q,  w = exp(sign 2 pi i / n),
 * E, O the DFTs of the even- and odd-indexed samples.  In place on (re, im);
 * tmp has 2n doubles. */
static void fft_rec(int n, int sign, double *re, double *im, double *tmp)
{
    if (n == 1) return;
    const int h = n / 2;
    double *er = tmp, *ei = tmp + h, *orr = tmp + n, *oi = tmp + n + h;
    for (int i = 0; i < h; ++i) {
        er[i] = re[2 * i];      ei[i] = im[2 * i];
        orr[i] = re[2 * i + 1]; oi[i] = im[2 * i + 1];
    }
    for (int i = 0; i < h; ++i) {
        re[i] = er[i];      im[i] = ei[i];
        re[h + i] = orr[i]; im[h + i] = oi[i];
    }
    fft_rec(h, sign, re, im, tmp);
    fft_rec(h, sign, re + h, im + h, tmp);
    for (int q = 0; q < h; ++q) {
        const double ang = 2.0 * ORC_PI * (double)q / (double)n;
        const double c = cos(ang), s = sign * sin(ang);
        const double tr = re[h + q] * c - im[h + q] * s;
        const double ti = re[h + q] * s + im[h + q] * c;
        const double ar = re[q], ai = im[q];
        re[q] = ar + tr;     im[q] = ai + ti;
        re[h + q] = ar - tr; im[h + q] = ai - ti;
    }
}

void orc_fft_radix2(int n, int sign, double *re, double *im)
{
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    fft_rec(n, sign, re, im, tmp);
    free(tmp);
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* One DFT of a strided complex line inside planar arrays, in place.
 * variant 0: definition; variant 1: radix-2 FFT (power-of-two n only). */
static void dft_line(int n, int sign, int variant, double *re, double *im, size_t stride,
                     double *buf /* 4n doubles */, double *tmp /* 2n doubles */)
{
    double *lr = buf, *li = buf + n, *outr = buf + 2 * n, *outi = buf + 3 * n;
    for (int i = 0; i < n; ++i) { lr[i] = re[i * stride]; li[i] = im[i * stride]; }
    if (variant == 1 && is_pow2(n)) {
        fft_rec(n, sign, lr, li, tmp);
        for (int i = 0; i < n; ++i) { re[i * stride] = lr[i]; im[i * stride] = li[i]; }
    } else {
        orc_dft_naive(n, sign, lr, li, outr, outi);
        for (int i = 0; i < n; ++i) { re[i * stride] = outr[i]; im[i * stride] = outi[i]; }
    }
}

/* 2-D DFT (x then y) of every z-plane of a planar complex field, in place.
 * PAPER.md:125-126 (steps 2-3) forward, :130-131 (steps 7-8) inverse.
 * No normalisation here. */
void orc_dft_xy(int nx, int ny, int nz, int sign, int variant, double *re, double *im)
{
    const size_t plane = (size_t)nx * (size_t)ny;
    const int nmax = nx > ny ? nx : ny;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 4 * (size_t)nmax);
        double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)nmax);
#pragma omp for schedule(static)
        for (long long l = 0; l < (long long)ny * nz; ++l)       /* lines along x */
            dft_line(nx, sign, variant, re + (size_t)l * nx, im + (size_t)l * nx, 1, buf, tmp);
#pragma omp for schedule(static)
        for (long long l = 0; l < (long long)nx * nz; ++l) {     /* lines along y */
            const size_t k = (size_t)(l / nx), i = (size_t)(l % nx);
            dft_line(ny, sign, variant, re + k * plane + i, im + k * plane + i, (size_t)nx, buf, tmp);
        }
        free(buf);
        free(tmp);
    }
}

/* ------------------------------------------------------- tridiagonal solves */

/* One Poisson column for horizontal eigenvalue lam = lam_x + lam_y < 0
 * (Eq. 12):
 *     A_k phi_{k-1} + (-(A_k+C_k) + lam) phi_k + C_k phi_{k+1} = d_k .
 * Serial Thomas ("serially performs operations along the third
 * direction") written with the pivot in the form p_k = C_k + e_k so that the
 * exact diagonal -(A_k+C_k)+lam of the double tables is used without ever
 * forming it (reading R5 in DESIGN.md):  sigma = -lam,
 *     e_0 = sigma,  p_k = C_k + e_k,  e_k = sigma + A_k e_{k-1} / p_{k-1},
 *     g_k = (-d_k + A_k g_{k-1}) / p_k,
 *     phi_{nz-1} = g_{nz-1},  phi_k = g_k + (C_k / p_k) phi_{k+1}.
 * stride = distance between consecutive k in d and phi.  work: 2 nz doubles. */
void orc_thomas_poisson(int nz, const double *A, const double *C, double sigma,
                        const double *d, double *phi, size_t stride, double *work)
{
    double *p = work, *g = work + nz;
    double e = sigma;
    p[0] = C[0] + e;
    g[0] = -d[0] / p[0];
    for (int k = 1; k < nz; ++k) {
        e = sigma + A[k] * e / p[k - 1];
        p[k] = C[k] + e;
        g[k] = (-d[(size_t)k * stride] + A[k] * g[k - 1]) / p[k];
    }
    phi[(size_t)(nz - 1) * stride] = g[nz - 1];
    for (int k = nz - 2; k >= 0; --k)
        phi[(size_t)k * stride] = g[k] + (C[k] / p[k]) * phi[(size_t)(k + 1) * stride];
}

/* The singular (0,0) column (lam = 0), reading R4: in flux form
 *   (phi_{k+1}-phi_k)/dzc_k - (phi_k-phi_{k-1})/dzc_{k-1} = dzf_k d_k
 * so with S_k = sum_{l<=k} dzf_l d_l :  phi_{k+1} = phi_k + dzc_k S_k, phi_0 = 0;
 * the gauge is then fixed by removing the dzf-weighted mean (zero volume mean
 * of the whole field, reading R3).  The last equation (S_{nz-1} = 0, the
 * compatibility condition) is the one not enforced. */
void orc_zero_mode_column(int nz, const double *dzf, const double *dzc,
                          const double *d, double *phi, size_t stride)
{
    double S = 0.0, v = 0.0, wsum = 0.0, lz = 0.0;
    double *dd = (double *)malloc(sizeof(double) * (size_t)nz);   /* d may alias phi */
    for (int k = 0; k < nz; ++k) dd[k] = d[(size_t)k * stride];
    phi[0] = 0.0;
    for (int k = 0; k + 1 < nz; ++k) {
        S += dzf[k] * dd[k];
        v += dzc[k] * S;
        phi[(size_t)(k + 1) * stride] = v;
    }
    free(dd);
    for (int k = 0; k < nz; ++k) { wsum += dzf[k] * phi[(size_t)k * stride]; lz += dzf[k]; }
    const double mean = wsum / lz;
    for (int k = 0; k < nz; ++k) phi[(size_t)k * stride] -= mean;
}

/* Plain Thomas algorithm for a general tridiagonal system
 *   lo_k x_{k-1} + di_k x_k + up_k x_{k+1} = d_k   (lo_0, up_{n-1} ignored).
 * work: 2 n doubles. */
void orc_thomas(int n, const double *lo, const double *di, const double *up,
                const double *d, double *x, size_t stride, double *work)
{
    double *cp = work, *dp = work + n;
    cp[0] = up[0] / di[0];
    dp[0] = d[0] / di[0];
    for (int k = 1; k < n; ++k) {
        const double m = di[k] - lo[k] * cp[k - 1];
        cp[k] = up[k] / m;
        dp[k] = (d[(size_t)k * stride] - lo[k] * dp[k - 1]) / m;
    }
    x[(size_t)(n - 1) * stride] = dp[n - 1];
    for (int k = n - 2; k >= 0; --k)
        x[(size_t)k * stride] = dp[k] - cp[k] * x[(size_t)(k + 1) * stride];
}

/* ------------------------------------------------------------ the operators */

/* phi -> L_h phi, definition O-P written out (difference form), double.
 * Used by tests for round trips and by bench for nothing. */
void orc_apply_poisson_operator(int nx, int ny, int nz, double lx, double ly,
                                const double *zc, const double *zf,
                                const double *phi, double *out)
{
    double *dzf = (double *)malloc(sizeof(double) * 4 * (size_t)nz);
    double *dzc = dzf + nz, *A = dzf + 2 * nz, *C = dzf + 3 * nz;
    orc_z_tables(nz, zc, zf, dzf, dzc, A, C);
    const double dx = lx / nx, dy = ly / ny;
    const double rdx2 = 1.0 / (dx * dx), rdy2 = 1.0 / (dy * dy);
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t c = (size_t)k * plane + (size_t)j * nx + i;
                const int ip = (i + 1) % nx, im = (i + nx - 1) % nx;
                const int jp = (j + 1) % ny, jm = (j + ny - 1) % ny;
                const double pc = phi[c];
                double v = (phi[c - i + ip] - 2.0 * pc + phi[c - i + im]) * rdx2
                         + (phi[c - (size_t)j * nx + (size_t)jp * nx] - 2.0 * pc
                            + phi[c - (size_t)j * nx + (size_t)jm * nx]) * rdy2;
                if (k > 0)      v += A[k] * (phi[c - plane] - pc);
                if (k + 1 < nz) v += C[k] * (phi[c + plane] - pc);
                out[c] = v;
            }
    free(dzf);
}

/* Helmholtz column matrix of O-H:  lo_k = -a A_k, up_k = -a C_k,
 * di_k = 1 + a (A_k + C_k + W_k),  W_0 = 2/(dzf_0 dzw_0), W_{nz-1} = 2/(dzf_{nz-1} dzw_1),
 * dzw_0 = 2 (zc_0 - zf_0), dzw_1 = 2 (zf_nz - zc_{nz-1})   (reading R7). */
void orc_helmholtz_matrix(int nz, const double *zc, const double *zf, double a,
                          double *lo, double *di, double *up)
{
    double *dzf = (double *)malloc(sizeof(double) * 4 * (size_t)nz);
    double *dzc = dzf + nz, *A = dzf + 2 * nz, *C = dzf + 3 * nz;
    orc_z_tables(nz, zc, zf, dzf, dzc, A, C);
    for (int k = 0; k < nz; ++k) {
        double W = 0.0;
        if (k == 0)      W += 2.0 / (dzf[0] * (2.0 * (zc[0] - zf[0])));
        if (k == nz - 1) W += 2.0 / (dzf[nz - 1] * (2.0 * (zf[nz] - zc[nz - 1])));
        lo[k] = -a * A[k];
        up[k] = -a * C[k];
        di[k] = 1.0 + a * (A[k] + C[k] + W);
    }
    free(dzf);
}

/* ---------------------------------------------------------------- the solves */

/* Poisson solve, out of place: f[N] -> phi[N].  variant 0 = O(n^2) DFT,
 * variant 1 = radix-2 FFT (nx, ny powers of two; otherwise falls back to 0).
 * Returns 0, or 1 on allocation failure.
 * (2) transforms along x, (3) along y, (4-6) tridiagonal
 * systems along z, (7-8) inverse transforms. */
int orc_poisson_solve(int nx, int ny, int nz, double lx, double ly,
                      const double *zc, const double *zf,
                      const double *f, double *phi, int variant)
{
    const size_t plane = (size_t)nx * ny, N = plane * (size_t)nz;
    double *re = (double *)malloc(sizeof(double) * N);
    double *im = (double *)calloc(N, sizeof(double));
    double *tab = (double *)malloc(sizeof(double) * (4 * (size_t)nz + nx + ny));
    if (!re || !im || !tab) { free(re); free(im); free(tab); return 1; }
    double *dzf = tab, *dzc = tab + nz, *A = tab + 2 * nz, *C = tab + 3 * nz;
    double *lamx = tab + 4 * nz, *lamy = lamx + nx;
    orc_z_tables(nz, zc, zf, dzf, dzc, A, C);
    orc_lambda(nx, lx, lamx);
    orc_lambda(ny, ly, lamy);
    memcpy(re, f, sizeof(double) * N);

    orc_dft_xy(nx, ny, nz, -1, variant, re, im);

#pragma omp parallel
    {
        double *work = (double *)malloc(sizeof(double) * 2 * (size_t)nz);
#pragma omp for schedule(static)
        for (long long c = 0; c < (long long)plane; ++c) {
            const int qy = (int)(c / nx), qx = (int)(c % nx);
            if (qx == 0 && qy == 0) {
                orc_zero_mode_column(nz, dzf, dzc, re + c, re + c, plane);
                orc_zero_mode_column(nz, dzf, dzc, im + c, im + c, plane);
            } else {
                const double sigma = -(lamx[qx] + lamy[qy]);
                orc_thomas_poisson(nz, A, C, sigma, re + c, re + c, plane, work);
                orc_thomas_poisson(nz, A, C, sigma, im + c, im + c, plane, work);
            }
        }
        free(work);
    }

    orc_dft_xy(nx, ny, nz, +1, variant, re, im);
    const double scale = 1.0 / ((double)nx * (double)ny);
#pragma omp parallel for schedule(static)
    for (long long c = 0; c < (long long)N; ++c) phi[c] = re[c] * scale;
    free(re); free(im); free(tab);
    return 0;
}

/* Helmholtz solve, out of place: r[N] -> u[N]; a >= 0.  One plain Thomas
 * solve of O-H per (i,j) column. */
int orc_helmholtz_z_solve(int nx, int ny, int nz, const double *zc, const double *zf,
                          double a, const double *r, double *u)
{
    const size_t plane = (size_t)nx * ny;
    double *m = (double *)malloc(sizeof(double) * 3 * (size_t)nz);
    if (!m) return 1;
    double *lo = m, *di = m + nz, *up = m + 2 * nz;
    orc_helmholtz_matrix(nz, zc, zf, a, lo, di, up);
#pragma omp parallel
    {
        double *work = (double *)malloc(sizeof(double) * 2 * (size_t)nz);
#pragma omp for schedule(static)
        for (long long c = 0; c < (long long)plane; ++c)
            orc_thomas(nz, lo, di, up, r + c, u + c, plane, work);
        free(work);
    }
    free(m);
    return 0;
}

/* Helmholtz on a list of sampled columns only (full-size parity on sampled
 * outputs): cols[ncols] are flat (j*nx+i) indices, rcols/ucols are
 * [ncols][nz] contiguous. */
int orc_helmholtz_z_solve_columns(int nz, const double *zc, const double *zf, double a,
                                  long long ncols, const double *rcols, double *ucols)
{
    double *m = (double *)malloc(sizeof(double) * 5 * (size_t)nz);
    if (!m) return 1;
    double *lo = m, *di = m + nz, *up = m + 2 * nz, *work = m + 3 * nz;
    orc_helmholtz_matrix(nz, zc, zf, a, lo, di, up);
    for (long long c = 0; c < ncols; ++c)
        orc_thomas(nz, lo, di, up, rcols + (size_t)c * nz, ucols + (size_t)c * nz, 1, work);
    free(m);
    return 0;
}

/* --------------------------- wall-normal diffusion of the FACE-centred component w */

/* Matrix of (I - a L_z^w) for the wall-normal velocity, which lives on the z FACES of the
 * staggered grid ("staggered ... grid"; reading R16): w_k on the face
 * zf[k+1], k = 0..nz-1; the bottom wall face zf[0] carries w = 0 and is not stored, the top
 * wall face is k = nz-1 and keeps its value (identity row).  For k = 0..nz-2
 *   (L_z^w w)_k = [ (w_{k+1} - w_k)/dzf_{k+1} - (w_k - w_{k-1})/dzf_k ] / dzc_k,
 * the second difference of the face values across the two neighbouring cells, with
 * w_{-1} = 0 and w_{nz-1} = 0 (the walls):
 *   lo_k = -a Aw_k,  up_k = -a Cw_k,  di_k = 1 + a (1/(dzc_k dzf_k) + 1/(dzc_k dzf_{k+1})),
 *   Aw_k = 1/(dzc_k dzf_k) (k >= 1, else 0),  Cw_k = 1/(dzc_k dzf_{k+1}) (k <= nz-3, else 0). */
void orc_helmholtz_w_matrix(int nz, const double *zc, const double *zf, double a,
                            double *lo, double *di, double *up)
{
    for (int k = 0; k < nz; ++k) {
        if (k == nz - 1) { lo[k] = 0.0; up[k] = 0.0; di[k] = 1.0; continue; }
        const double dzc = zc[k + 1] - zc[k];
        const double dzm = zf[k + 1] - zf[k], dzp = zf[k + 2] - zf[k + 1];
        const double Aw = 1.0 / (dzc * dzm), Cw = 1.0 / (dzc * dzp);
        lo[k] = (k >= 1) ? -a * Aw : 0.0;
        up[k] = (k <= nz - 3) ? -a * Cw : 0.0;
        di[k] = 1.0 + a * (Aw + Cw);
    }
}

/* r[N] -> w[N]: one plain Thomas solve per (i,j) column (Eq. 11 for the third component). */
int orc_helmholtz_w_solve(int nx, int ny, int nz, const double *zc, const double *zf,
                          double a, const double *r, double *w)
{
    const size_t plane = (size_t)nx * ny;
    double *m = (double *)malloc(sizeof(double) * 3 * (size_t)nz);
    if (!m) return 1;
    double *lo = m, *di = m + nz, *up = m + 2 * nz;
    orc_helmholtz_w_matrix(nz, zc, zf, a, lo, di, up);
#pragma omp parallel
    {
        double *work = (double *)malloc(sizeof(double) * 2 * (size_t)nz);
#pragma omp for schedule(static)
        for (long long c = 0; c < (long long)plane; ++c)
            orc_thomas(nz, lo, di, up, r + c, w + c, plane, work);
        free(work);
    }
    free(m);
    return 0;
}

/* ------------------------------------------- fully implicit diffusion, Eq. (8) */

/* u -> (I - a L_h) u with periodic x, y and Dirichlet walls in z (definition O-H3):
 *   u - a [ (u_{i+1} - 2u + u_{i-1})/dx^2 + (u_{j+1} - 2u + u_{j-1})/dy^2
 *           + A_k (u_{k-1} - u) + C_k (u_{k+1} - u) - W_k u ],
 * W_k as in orc_helmholtz_matrix (reading R7).  PAPER.md:63 (Eq. 8): "a Helmholtz equation for
 * the prediction velocity, implicit in the three spatial directions". */
void orc_apply_helmholtz3d_operator(int nx, int ny, int nz, double lx, double ly,
                                    const double *zc, const double *zf, double a,
                                    const double *u, double *out)
{
    double *dzf = (double *)malloc(sizeof(double) * 4 * (size_t)nz);
    double *dzc = dzf + nz, *A = dzf + 2 * nz, *C = dzf + 3 * nz;
    orc_z_tables(nz, zc, zf, dzf, dzc, A, C);
    const double dx = lx / nx, dy = ly / ny;
    const double rdx2 = 1.0 / (dx * dx), rdy2 = 1.0 / (dy * dy);
    const double W0 = 2.0 / (dzf[0] * (2.0 * (zc[0] - zf[0])));
    const double W1 = 2.0 / (dzf[nz - 1] * (2.0 * (zf[nz] - zc[nz - 1])));
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t c = (size_t)k * plane + (size_t)j * nx + i;
                const int ip = (i + 1) % nx, im = (i + nx - 1) % nx;
                const int jp = (j + 1) % ny, jm = (j + ny - 1) % ny;
                const double pc = u[c];
                double v = (u[c - i + ip] - 2.0 * pc + u[c - i + im]) * rdx2
                         + (u[c - (size_t)j * nx + (size_t)jp * nx] - 2.0 * pc
                            + u[c - (size_t)j * nx + (size_t)jm * nx]) * rdy2;
                if (k > 0)      v += A[k] * (u[c - plane] - pc);
                if (k + 1 < nz) v += C[k] * (u[c + plane] - pc);
                if (k == 0)      v -= W0 * pc;
                if (k == nz - 1) v -= W1 * pc;
                out[c] = pc - a * v;
            }
    free(dzf);
}

/* 3-D Helmholtz solve, out of place: r[N] -> u[N], (I - a L_h) u = r.  The same eigenfunction
 * expansion as the Poisson solve ("Poisson/Helmholtz equation"): transforms
 * along x and y, then per (qx, qy) one plain Thomas solve of
 *   -a A_k u_{k-1} + (1 + a (A_k + C_k + W_k + sigma)) u_k - a C_k u_{k+1} = r~_k,
 * sigma = -(lambda_x + lambda_y) >= 0, inverse transforms.  The matrix is strictly diagonally
 * dominant with positive diagonal: no cancellation, no pin. */
int orc_helmholtz3d_solve(int nx, int ny, int nz, double lx, double ly,
                          const double *zc, const double *zf, double a,
                          const double *r, double *u, int variant)
{
    const size_t plane = (size_t)nx * ny, N = plane * (size_t)nz;
    double *re = (double *)malloc(sizeof(double) * N);
    double *im = (double *)calloc(N, sizeof(double));
    double *tab = (double *)malloc(sizeof(double) * (3 * (size_t)nz + nx + ny));
    if (!re || !im || !tab) { free(re); free(im); free(tab); return 1; }
    double *lo = tab, *di = tab + nz, *up = tab + 2 * nz;
    double *lamx = tab + 3 * nz, *lamy = lamx + nx;
    orc_helmholtz_matrix(nz, zc, zf, a, lo, di, up);
    orc_lambda(nx, lx, lamx);
    orc_lambda(ny, ly, lamy);
    memcpy(re, r, sizeof(double) * N);

    orc_dft_xy(nx, ny, nz, -1, variant, re, im);

#pragma omp parallel
    {
        double *work = (double *)malloc(sizeof(double) * 3 * (size_t)nz);
        double *dk = work + 2 * nz;
#pragma omp for schedule(static)
        for (long long c = 0; c < (long long)plane; ++c) {
            const int qy = (int)(c / nx), qx = (int)(c % nx);
            const double sigma = -(lamx[qx] + lamy[qy]);
            for (int k = 0; k < nz; ++k) dk[k] = di[k] + a * sigma;
            orc_thomas(nz, lo, dk, up, re + c, re + c, plane, work);
            orc_thomas(nz, lo, dk, up, im + c, im + c, plane, work);
        }
        free(work);
    }

    orc_dft_xy(nx, ny, nz, +1, variant, re, im);
    const double scale = 1.0 / ((double)nx * (double)ny);
#pragma omp parallel for schedule(static)
    for (long long c = 0; c < (long long)N; ++c) u[c] = re[c] * scale;
    free(re); free(im); free(tab);
    return 0;
}
