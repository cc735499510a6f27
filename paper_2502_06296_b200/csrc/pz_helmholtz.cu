// pz_helmholtz.cu -- step a6 of the hot path: wall-normal implicit diffusion (Eq. 11,
// PAPER.md:74-78) with the paper's split of cyclic reduction into pre-processing and runtime
// (Algorithm 2).
//
// Pre-processing (helmholtz_build_tables, host, long double -> double): the matrix I - a L_z is
// the same for every (i,j) column ("identical for all (i,j) indexes"), so the
// coefficient sub-arrays (a, b, c) of Algorithm 2 Step 1 are 1-D arrays in k.  The z direction is
// cut into P sub-domains of m rows (padded with identity rows to P*m); for the boundary system of
// size 2P the multipliers of every parallel-cyclic-reduction level are precomputed too, so the
// runtime applies numbers and never divides ("store 1/b").
//
// Runtime (helmholtz_kernel): a CTA owns TX neighbouring columns (TX*8 contiguous bytes per row);
// thread (column, sub-domain) loads its m rows straight into registers (one coalesced HBM read),
// runs Step 2 (forward / backward sweeps touching only d), exchanges the two boundary rows through
// shared memory, applies the precomputed PCR levels (Step 3), reconstructs (Step 4) and stores
// (one HBM write): 16 bytes and about 5 FMAs per point.
#include "pz_internal.h"

#include <cmath>
#include <cstring>

namespace pz {

namespace {

// Table layout (doubles), nzp = P*m, n2 = 2P, LV = levels:
//   [0, nzp)        fA_k  = A_i / b_{i-1}          (Step 2 forward, i = 2..m-1, else 0)
//   [nzp, 2nzp)     bC_k  = C_i / b_{i+1}          (Step 2 backward, i = 0..m-3, else 0)
//   [2nzp, 3nzp)    rb_k  = 1 / b_i                (Step 4)
//   [3nzp, 4nzp)    ra_k  = a_i / b_i
//   [4nzp, 5nzp)    rc_k  = c_i / b_i
//   [5nzp, +LV*2*n2)   per level l and reduced row r: k1, k2 (d_r += k1 d_{r-h} + k2 d_{r+h})
//   then n2         rbr_r = 1 / b_r after the last level
// Threads per CTA = tx * P.  Register budget per sub-domain size (whole tile lives in registers):
// m <= 16: 64 registers (up to 1024 threads per SM), m = 32: 128 registers.
template <int M> struct HelmLimits {
    static constexpr int kMaxThreads = (M >= 32) ? 256 : 512;
    static constexpr int kMinBlocks = 2;
};

template <int M, bool FULL>
__global__ void __launch_bounds__(HelmLimits<M>::kMaxThreads, HelmLimits<M>::kMinBlocks)
    helmholtz_kernel(double *__restrict__ u, const double *__restrict__ tab, size_t plane, int nz, int P,
                     int levels, int tx)
{
    extern __shared__ double smem_h[]; // 2 buffers x (2P rows) x tx
    const int c = threadIdx.x % tx, s = threadIdx.x / tx;
    const int nzp = P * M, n2 = 2 * P;
    const int k0 = s * M;
    const double *fA = tab + k0, *bC = tab + nzp + k0, *rb = tab + 2 * nzp + k0;
    const double *ra = tab + 3 * nzp + k0, *rc = tab + 4 * nzp + k0;
    const double *pcr = tab + 5 * (size_t)nzp;
    double *up = u + ((size_t)blockIdx.x * tx + c) + (size_t)k0 * plane;

    double d[M];
#pragma unroll
    for (int i = 0; i < M; ++i) d[i] = (FULL || k0 + i < nz) ? up[(size_t)i * plane] : 0.0;

    // Step 2: runtime reduction, d only
#pragma unroll
    for (int i = 2; i < M; ++i) d[i] = fma(-__ldg(&fA[i]), d[i - 1], d[i]);
#pragma unroll
    for (int i = M - 3; i >= 0; --i) d[i] = fma(-__ldg(&bC[i]), d[i + 1], d[i]);

    // Step 3: boundary system, rows (2s, 2s+1) = (first, last) row of sub-domain s
    double *cur = smem_h, *nxt = smem_h + (size_t)n2 * tx;
    double x0 = d[0], x1 = d[M - 1];
    const int r0 = 2 * s, r1 = 2 * s + 1;
    cur[r0 * tx + c] = x0;
    cur[r1 * tx + c] = x1;
    __syncthreads();
    int h = 1;
    for (int l = 0; l < levels; ++l, h *= 2) {
        const double *kk = pcr + (size_t)l * 2 * n2;
        // multipliers are zero where the partner row does not exist; clamp the index instead of branching
        const int a0 = max(r0 - h, 0), b0 = min(r0 + h, n2 - 1), a1 = max(r1 - h, 0), b1 = min(r1 + h, n2 - 1);
        const double2 k0v = __ldg(reinterpret_cast<const double2 *>(kk) + r0);
        const double2 k1v = __ldg(reinterpret_cast<const double2 *>(kk) + r1);
        x0 = fma(k0v.x, cur[a0 * tx + c], fma(k0v.y, cur[b0 * tx + c], x0));
        x1 = fma(k1v.x, cur[a1 * tx + c], fma(k1v.y, cur[b1 * tx + c], x1));
        if (l + 1 < levels) {
            nxt[r0 * tx + c] = x0;
            nxt[r1 * tx + c] = x1;
            __syncthreads();
            double *t = cur; cur = nxt; nxt = t;
        }
    }
    {
        const double2 rbr = __ldg(reinterpret_cast<const double2 *>(pcr + (size_t)levels * 2 * n2) + s);
        x0 *= rbr.x;
        x1 *= rbr.y;
    }

    // Step 4: reconstruct in place and store
    if (FULL || k0 < nz) up[0] = x0;
#pragma unroll
    for (int i = 1; i < M - 1; ++i) {
        const double v = fma(-__ldg(&rc[i]), x1, fma(-__ldg(&ra[i]), x0, __ldg(&rb[i]) * d[i]));
        if (FULL || k0 + i < nz) up[(size_t)i * plane] = v;
    }
    if (FULL || k0 + M - 1 < nz) up[(size_t)(M - 1) * plane] = x1;
}

int ilog2_ceil(int n)
{
    int l = 0;
    while ((1 << l) < n) ++l;
    return l;
}

} // namespace

// Choose the sub-domain size m and count P for this nz (and the CTA width) -- launch geometry.
static void helm_geometry(pz_plan *pl)
{
    int variant = pl->opt.helm_variant;
    // variant 1 up to nz = 1920 with two chunks per column and up to 3584 with four: beyond, the tile
    // of a chunk plus the tables exceed shared memory
    const int zopt = pl->opt.helm_zsplit;
    const int vmax = (zopt == 1) ? 1024 : (zopt == 2) ? 1920 : 3584;
    if (variant != 0 && variant != 1) variant = (pl->nz <= vmax) ? 1 : 0;
    if (variant == 1 && pl->nz > vmax) variant = 0;
    if (variant == 0 && pl->nz > 2048 && pl->nz <= vmax) variant = 1;   // the register tile stops at 2048 planes
    pl->helm_variant = variant;
    int m = pl->opt.helm_m;
    pl->helm_zs = 1;
    if (variant == 1) {
        // TX / 2 column pairs x P sub-domains per CTA, at most 512 threads, m in {4, 8, 16}
        if (m != 4 && m != 8 && m != 16) m = (pl->nz <= 128) ? 4 : (pl->nz <= 256 ? 8 : 16);
        while (m < 16 && (pl->nz + m - 1) / m > 64) m *= 2;
        pl->helm_m = m;
        int P = (pl->nz + m - 1) / m;
        const bool even64 = ((size_t)pl->nx * pl->ny) % 64 == 0;
        // m = 16 (nz > 256): the column is cut in two chunks owned by the two CTAs of a cluster (the
        // paper's own decomposition, with CTAs for its MPI tasks): half the rows per
        // tile leave room for 256-byte rows up to nz = 1024, for two resident CTAs per SM up to
        // nz = 512 and for nz up to 1920 at all.  Measured, 3 fields: 512^3 5.96 TB/s against 5.73
        // (whole columns, 32-column tiles) and 5.45 (16-column tiles); 1024^3 5.80 against 5.13 TB/s.
        int zs = pl->opt.helm_zsplit;
        // (four chunks were measured slower than two wherever two fit: 1.17 against 1.09 ms at 512^3 x 3,
        // 9.8 against 9.0 ms at 1024^3 x 3; they serve 1920 < nz <= 3584)
        if (zs != 1 && zs != 2 && zs != 4) zs = (m != 16) ? 1 : (pl->nz > 1920 ? 4 : 2);
        if (zs >= 2 && (m != 16 || pl->nz < 4 * m)) zs = 1;
        if (zs == 4 && pl->nz < 8 * m) zs = 2;   // at least two sub-domains per chunk
        if (zs >= 2) P = (P + zs - 1) / zs;      // sub-domains per chunk
        pl->helm_zs = zs;
        pl->helm_P = P;
        // wide tiles (32 columns, 256-byte rows) where one of them fits shared memory and 512 threads
        // (measured: 5.76 against 5.45 TB/s at 512^3 x 3 fields, 5.81 against 5.17 TB/s at 1024 x 1024 x 512 x 3)
        pl->helm_tx = (pl->opt.helm_tx != 16 && m == 16 && P <= 32 && even64) ? 32 : 16;
        if (zs == 4 && pl->opt.helm_tx == 64 && P <= 16 && ((size_t)pl->nx * pl->ny) % 128 == 0) pl->helm_tx = 64;
        pl->helm_levels = ilog2_ceil(2 * P);
        return;
    }
    if (m != 4 && m != 8 && m != 16 && m != 32) m = (pl->nz <= 128) ? 4 : (pl->nz <= 256) ? 8 : (pl->nz <= 512 ? 16 : 32);
    int P = (pl->nz + m - 1) / m;
    int tx = pl->opt.helm_tx;
    if (tx != 4 && tx != 8 && tx != 16 && tx != 32) tx = 8;
    while (m < 32 && 4 * P > 512) { m *= 2; P = (pl->nz + m - 1) / m; }
    const int limit = (m >= 32) ? 256 : 512; // __launch_bounds__ of helmholtz_kernel<m>
    while (tx > 4 && tx * P > limit) tx /= 2;
    pl->helm_m = m;
    pl->helm_P = P;
    pl->helm_tx = tx;
    pl->helm_levels = ilog2_ceil(2 * P);
}

namespace {

typedef long double ld;

// Algorithm 2 Step 1 for the P sub-domains of m rows of ONE tridiagonal matrix
// (A, B, C: sub-diagonal, diagonal, super-diagonal of P*m rows), plus the precomputed parallel
// cyclic reduction of its boundary system.  out: [fA | bC | rb | ra | rc] (5 P m) + LV*2*2P + 2P.
void build_chunk_tables(const ld *A, const ld *B, const ld *C, int m, int P, int LV, double *out)
{
    const int nzp = P * m, n2 = 2 * P;
    double *fA = out, *bC = fA + nzp, *rb = bC + nzp, *ra = rb + nzp, *rc = ra + nzp;
    double *pcr = rc + nzp;
    std::vector<ld> ra2(n2), rbd(n2), rc2(n2); // boundary system
    std::vector<ld> ca(m), cb(m), cc(m);
    for (int s = 0; s < P; ++s) {
        const ld *As = &A[s * m], *Bs = &B[s * m], *Cs = &C[s * m];
        for (int i = 0; i < m; ++i) ca[i] = cb[i] = cc[i] = 0;
        ca[1] = As[1];
        cb[1] = Bs[1];
        for (int i = 2; i < m; ++i) {
            cb[i] = Bs[i] - As[i] * Cs[i - 1] / cb[i - 1];
            ca[i] = -As[i] * ca[i - 1] / cb[i - 1];
        }
        cc[m - 1] = Cs[m - 1];
        cc[m - 2] = Cs[m - 2];
        for (int i = m - 3; i >= 1; --i) {
            ca[i] = ca[i] - Cs[i] * ca[i + 1] / cb[i + 1];
            cc[i] = -Cs[i] * cc[i + 1] / cb[i + 1];
        }
        ca[0] = As[0];
        cb[0] = Bs[0] - Cs[0] * ca[1] / Bs[1];
        cc[0] = -Cs[0] * cc[1] / Bs[1];
        for (int i = 0; i < m; ++i) {
            const int k = s * m + i;
            fA[k] = (i >= 2) ? (double)(As[i] / cb[i - 1]) : 0.0;
            bC[k] = (i <= m - 3) ? (double)(Cs[i] / cb[i + 1]) : 0.0;
            rb[k] = ra[k] = rc[k] = 0.0;
            if (i >= 1 && i <= m - 2) {
                rb[k] = (double)((ld)1 / cb[i]);
                ra[k] = (double)(ca[i] / cb[i]);
                rc[k] = (double)(cc[i] / cb[i]);
            }
        }
        ra2[2 * s] = ca[0];         rbd[2 * s] = cb[0];         rc2[2 * s] = cc[0];
        ra2[2 * s + 1] = ca[m - 1]; rbd[2 * s + 1] = cb[m - 1]; rc2[2 * s + 1] = cc[m - 1];
    }
    ra2[0] = 0;
    rc2[n2 - 1] = 0;
    // PCR of the boundary system with the multipliers recorded per level
    std::vector<ld> na(n2), nb(n2), nc(n2);
    int h = 1;
    for (int l = 0; l < LV; ++l, h *= 2) {
        double *kk = pcr + (size_t)l * 2 * n2;
        for (int r = 0; r < n2; ++r) {
            ld k1 = 0, k2 = 0;
            ld b = rbd[r], an = 0, cn = 0;
            if (r - h >= 0) { k1 = ra2[r] / rbd[r - h]; b -= k1 * rc2[r - h]; an = -k1 * ra2[r - h]; }
            if (r + h < n2) { k2 = rc2[r] / rbd[r + h]; b -= k2 * ra2[r + h]; cn = -k2 * rc2[r + h]; }
            kk[2 * r] = (double)(-k1);
            kk[2 * r + 1] = (double)(-k2);
            na[r] = an; nb[r] = b; nc[r] = cn;
        }
        ra2 = na; rbd = nb; rc2 = nc;
    }
    double *rbr = pcr + (size_t)LV * 2 * n2;
    for (int r = 0; r < n2; ++r) rbr[r] = (double)((ld)1 / rbd[r]);
}

// x = T^{-1} e_j by plain elimination in long double (T diagonally dominant: no pivoting)
void unit_response(const ld *A, const ld *B, const ld *C, int n, int j, std::vector<ld> &x)
{
    std::vector<ld> cp(n), dp(n);
    for (int k = 0; k < n; ++k) {
        const ld rhs = (k == j) ? (ld)1 : (ld)0;
        const ld den = (k == 0) ? B[0] : B[k] - A[k] * cp[k - 1];
        cp[k] = C[k] / den;
        dp[k] = (k == 0) ? rhs / den : (rhs - A[k] * dp[k - 1]) / den;
    }
    x.assign(n, 0);
    x[n - 1] = dp[n - 1];
    for (int k = n - 2; k >= 0; --k) x[k] = dp[k] - cp[k] * x[k + 1];
}

} // namespace

// Doubles of one chunk's table block: [5 nzc | PCR | corr (nzc) | wOwn, wPeer]
// (four chunks: [5 nzc | PCR | corrP (nzc) | corrN (nzc) | wP (8) | wN (8)])
static size_t chunk_doubles(int nzc, int P, int LV, int ZS = 1)
{
    return (ZS > 2 ? 7 : 6) * (size_t)nzc + (size_t)LV * 4 * P + 2 * P + (ZS > 2 ? 4 * ZS : 2);
}

// Algorithm 2 Step 1 on the host, plus the precomputed PCR of the boundary system.
int helmholtz_build_tables(pz_plan *pl, double a, int kind)
{
    helm_geometry(pl);
    const int nz = pl->nz, m = pl->helm_m, P = pl->helm_P, ZS = pl->helm_zs, nzc = P * m, LV = pl->helm_levels;
    const int nzp = ZS * nzc;
    if (pl->helm_variant == 1) {
        const int rc = helmholtz_tma_prepare(pl);
        if (rc != PZ_OK) return rc;
    } else if (pl->helm_tx * P > ((m >= 32) ? 256 : 512)) {
        set_error("helmholtz: nz = %d is too large for the register-tile kernel (P = %d sub-domains)", nz, P);
        return PZ_EUNSUPPORTED;
    }
    const size_t cstride = chunk_doubles(nzc, P, LV, ZS);
    pl->helm_cstride = cstride;
    // the one-kernel step of Eq. (11) (helmholtz_z_step) takes whole columns: its own table block
    // behind the chunks' where the columns are cut and a whole one still fits the kernel (nz <= 1024)
    pl->helm_cn_P = 0; pl->helm_cn_levels = 0; pl->helm_cn_off = 0;
    size_t cn_doubles = 0;
    if (pl->helm_variant == 1) {
        if (ZS == 1) { pl->helm_cn_P = P; pl->helm_cn_levels = LV; }
        else if ((nz + m - 1) / m <= 64) {
            pl->helm_cn_P = (nz + m - 1) / m;
            pl->helm_cn_levels = ilog2_ceil(2 * pl->helm_cn_P);
            pl->helm_cn_off = ZS * cstride;
            cn_doubles = chunk_doubles(pl->helm_cn_P * m, pl->helm_cn_P, pl->helm_cn_levels);
        }
    }
    const size_t ndbl = ZS * cstride + cn_doubles;
    const size_t bytes = ndbl * sizeof(double);

    // matrix of I - a L_z with Dirichlet walls, padded with identity rows
    const int nzw = (cn_doubles > 0 && pl->helm_cn_P * m > nzp) ? pl->helm_cn_P * m : nzp;
    std::vector<ld> A(nzw, 0), B(nzw, 1), C(nzw, 0);
    for (int k = 0; k < nz && kind == 0; ++k) {
        ld W = 0;
        if (k == 0) W += (ld)2 / ((ld)pl->dzf[0] * ((ld)2 * ((ld)pl->zc[0] - (ld)pl->zf[0])));
        if (k == nz - 1) W += (ld)2 / ((ld)pl->dzf[nz - 1] * ((ld)2 * ((ld)pl->zf[nz] - (ld)pl->zc[nz - 1])));
        A[k] = -(ld)a * (ld)pl->A[k];
        C[k] = -(ld)a * (ld)pl->C[k];
        B[k] = (ld)1 + (ld)a * ((ld)pl->A[k] + (ld)pl->C[k] + W);
    }
    // kind 1: the face-centred component w (w_k on the face zf[k+1]; both wall faces 0, the top one
    // is row nz-1 and keeps its value): second difference of the face values,
    //   (L w)_k = [ (w_{k+1} - w_k)/dzf_{k+1} - (w_k - w_{k-1})/dzf_k ] / dzc_k   (reading R16)
    for (int k = 0; k + 1 < nz && kind == 1; ++k) {
        const ld Aw = (ld)1 / ((ld)pl->dzc[k] * (ld)pl->dzf[k]), Cw = (ld)1 / ((ld)pl->dzc[k] * (ld)pl->dzf[k + 1]);
        A[k] = (k >= 1) ? -(ld)a * Aw : (ld)0;
        C[k] = (k <= nz - 3) ? -(ld)a * Cw : (ld)0;
        B[k] = (ld)1 + (ld)a * (Aw + Cw);
    }
    std::vector<double> host(ndbl, 0.0);
    if (ZS == 1) {
        build_chunk_tables(A.data(), B.data(), C.data(), m, P, LV, host.data());
    } else if (ZS > 2) {
        // ZS chunks (ZS CTAs of a cluster).  With y = T_c^{-1} r on every chunk,
        //   u_c = y_c - corrP_c L_{c-1} - corrN_c F_{c+1},  corrP_c = A_cut,c T_c^{-1} e_first,  corrN_c = C_cut,c T_c^{-1} e_last,
        // L_c / F_c the last / first value of u on chunk c; evaluated at the chunks' ends that is a
        // linear system for the 2 (ZS - 1) interface values, inverted here once: every chunk gets the
        // weights that turn the 2 ZS end values of y (F_0.., L_0..) into its L_{c-1} and F_{c+1}.
        const int nu = 2 * (ZS - 1);
        std::vector<std::vector<ld>> cP(ZS), cN(ZS);
        for (int c = 0; c < ZS; ++c) {
            std::vector<ld> Ac(A.begin() + c * nzc, A.begin() + (c + 1) * nzc), Bc(B.begin() + c * nzc, B.begin() + (c + 1) * nzc),
                Cc(C.begin() + c * nzc, C.begin() + (c + 1) * nzc);
            const ld Acut = Ac[0], Ccut = Cc[nzc - 1];
            Ac[0] = 0;
            Cc[nzc - 1] = 0;
            build_chunk_tables(Ac.data(), Bc.data(), Cc.data(), m, P, LV, host.data() + c * cstride);
            std::vector<ld> pr, qr;
            unit_response(Ac.data(), Bc.data(), Cc.data(), nzc, 0, pr);
            unit_response(Ac.data(), Bc.data(), Cc.data(), nzc, nzc - 1, qr);
            cP[c].resize(nzc);
            cN[c].resize(nzc);
            for (int k = 0; k < nzc; ++k) { cP[c][k] = (c > 0 ? Acut : (ld)0) * pr[k]; cN[c][k] = (c + 1 < ZS ? Ccut : (ld)0) * qr[k]; }
        }
        // unknown index: F_c (c = 1..ZS-1) -> c - 1;  L_c (c = 0..ZS-2) -> ZS - 1 + c
        auto iF = [&](int c) { return c - 1; };
        auto iL = [&](int c) { return ZS - 1 + c; };
        std::vector<std::vector<ld>> Mx(nu, std::vector<ld>(nu + 2 * ZS, 0)); // [matrix | selection of the y values]
        for (int c = 1; c < ZS; ++c) {            // F_c + kPF L_{c-1} + kNF F_{c+1} = yF_c
            auto &row = Mx[iF(c)];
            row[iF(c)] += 1;
            row[iL(c - 1)] += cP[c][0];
            if (c + 1 < ZS) row[iF(c + 1)] += cN[c][0];
            row[nu + c] = 1;                      // yF_c
        }
        for (int c = 0; c + 1 < ZS; ++c) {        // L_c + kPL L_{c-1} + kNL F_{c+1} = yL_c
            auto &row = Mx[iL(c)];
            row[iL(c)] += 1;
            if (c > 0) row[iL(c - 1)] += cP[c][nzc - 1];
            row[iF(c + 1)] += cN[c][nzc - 1];
            row[nu + ZS + c] = 1;                 // yL_c
        }
        for (int col = 0; col < nu; ++col) {      // Gauss-Jordan with partial pivoting (diagonally dominant: benign)
            int piv = col;
            for (int r = col + 1; r < nu; ++r)
                if (fabsl(Mx[r][col]) > fabsl(Mx[piv][col])) piv = r;
            std::swap(Mx[col], Mx[piv]);
            const ld inv = (ld)1 / Mx[col][col];
            for (auto &v : Mx[col]) v *= inv;
            for (int r = 0; r < nu; ++r) {
                if (r == col) continue;
                const ld f = Mx[r][col];
                if (f == 0) continue;
                for (int q = 0; q < nu + 2 * ZS; ++q) Mx[r][q] -= f * Mx[col][q];
            }
        }
        const size_t ocorr = 5 * (size_t)nzc + (size_t)LV * 4 * P + 2 * P;
        for (int c = 0; c < ZS; ++c) {
            double *blk = host.data() + c * cstride + ocorr;
            for (int k = 0; k < nzc; ++k) { blk[k] = (double)cP[c][k]; blk[nzc + k] = (double)cN[c][k]; }
            for (int q = 0; q < 2 * ZS; ++q) {
                blk[2 * nzc + q] = (c > 0) ? (double)Mx[iL(c - 1)][nu + q] : 0.0;               // L_{c-1}
                blk[2 * nzc + 2 * ZS + q] = (c + 1 < ZS) ? (double)Mx[iF(c + 1)][nu + q] : 0.0; // F_{c+1}
            }
        }
        if (cn_doubles > 0) build_chunk_tables(A.data(), B.data(), C.data(), m, pl->helm_cn_P, pl->helm_cn_levels, host.data() + pl->helm_cn_off);
    } else {
        // two chunks, couplings across the cut moved to the interface (PAPER.md:120-135 with the
        // two CTAs of a cluster for its MPI tasks; the matrix is k-only, so everything the
        // interface needs is precomputed here): with y = T_c^{-1} r on each chunk,
        //   u_0 = y_0 - (C_cut F1) q_0,  u_1 = y_1 - (A_cut L0) p_1,   q_0 = T_0^{-1} e_last, p_1 = T_1^{-1} e_first,
        //   L0 = u_0[last] = (y0L - k0 y1F) / (1 - k0 k1),  F1 = u_1[first] = (y1F - k1 y0L) / (1 - k0 k1),
        //   k0 = C_cut q_0[last],  k1 = A_cut p_1[first].
        const ld Ccut = C[nzc - 1], Acut = A[nzc];
        std::vector<ld> A0(A.begin(), A.begin() + nzc), B0(B.begin(), B.begin() + nzc), C0(C.begin(), C.begin() + nzc);
        std::vector<ld> A1(A.begin() + nzc, A.begin() + nzp), B1(B.begin() + nzc, B.begin() + nzp), C1(C.begin() + nzc, C.begin() + nzp);
        C0[nzc - 1] = 0;
        A1[0] = 0;
        build_chunk_tables(A0.data(), B0.data(), C0.data(), m, P, LV, host.data());
        build_chunk_tables(A1.data(), B1.data(), C1.data(), m, P, LV, host.data() + cstride);
        std::vector<ld> q0, p1;
        unit_response(A0.data(), B0.data(), C0.data(), nzc, nzc - 1, q0);
        unit_response(A1.data(), B1.data(), C1.data(), nzc, 0, p1);
        const ld k0 = Ccut * q0[nzc - 1], k1 = Acut * p1[0], g = (ld)1 / ((ld)1 - k0 * k1);
        const size_t ocorr = 5 * (size_t)nzc + (size_t)LV * 4 * P + 2 * P;
        for (int k = 0; k < nzc; ++k) {
            host[ocorr + k] = (double)(Ccut * q0[k]);
            host[cstride + ocorr + k] = (double)(Acut * p1[k]);
        }
        // X of a chunk = wOwn * (its own interface value of y) + wPeer * (the peer's)
        host[ocorr + nzc] = (double)(-g * k1);            host[ocorr + nzc + 1] = (double)g;
        host[cstride + ocorr + nzc] = (double)(-g * k0);  host[cstride + ocorr + nzc + 1] = (double)g;
        if (cn_doubles > 0) build_chunk_tables(A.data(), B.data(), C.data(), m, pl->helm_cn_P, pl->helm_cn_levels, host.data() + pl->helm_cn_off);
    }

    // upload into a table set that no in-flight solve reads and no captured graph refers to (a
    // captured helmholtz_z_solve keeps the address of the set that was current at capture time: such
    // a set is never rewritten or freed before the plan is destroyed, so replays stay valid -- and
    // keep solving with the coefficient of capture time -- across any number of later set-ups)
    int nb = -1;
    for (int i = 0; i < (int)pl->helm.size(); ++i)
        if (i != pl->helm_cur && i != pl->helm_w_cur && !pl->helm[i].captured) { nb = i; break; }
    if (nb < 0) {
        HelmTables fresh;
        PZ_CUDA(cudaEventCreateWithFlags(&fresh.uploaded, cudaEventDisableTiming));
        PZ_CUDA(cudaEventCreateWithFlags(&fresh.last_use, cudaEventDisableTiming));
        pl->helm.push_back(fresh);
        nb = (int)pl->helm.size() - 1;
    }
    HelmTables &t = pl->helm[nb];
    if (t.used) PZ_CUDA(cudaEventSynchronize(t.uploaded)); // this set's previous upload has left its staging buffer
    if (t.bytes < bytes) {
        if (t.used) PZ_CUDA(cudaEventSynchronize(t.last_use));
        if (t.dev) PZ_CUDA(cudaFree(t.dev));
        t.dev = nullptr;
        cudaError_t e = cudaMalloc(&t.dev, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); set_error("helmholtz tables: %s", cudaGetErrorString(e)); return PZ_ENOMEM; }
        t.bytes = bytes;
    }
    if (t.host_bytes < bytes) {
        if (t.host) PZ_CUDA(cudaFreeHost(t.host));
        t.host = nullptr;
        cudaError_t e = cudaMallocHost(&t.host, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); set_error("helmholtz staging: %s", cudaGetErrorString(e)); return PZ_ENOMEM; }
        t.host_bytes = bytes;
    }
    if (t.used) PZ_CUDA(cudaStreamWaitEvent(pl->upload_stream, t.last_use, 0)); // old readers done
    std::memcpy(t.host, host.data(), bytes);
    PZ_CUDA(cudaMemcpyAsync(t.dev, t.host, bytes, cudaMemcpyHostToDevice, pl->upload_stream));
    PZ_CUDA(cudaEventRecord(t.uploaded, pl->upload_stream));
    t.upload_seen = false;
    t.used = true;
    if (kind == 1) { pl->helm_w_cur = nb; pl->helm_w_a = a; }
    else { pl->helm_cur = nb; pl->helm_a = a; }
    return PZ_OK;
}

// Eq. (11) in one kernel where the variant-1 pipeline can hold the tiles of u** and u^k;
// PZ_EUNSUPPORTED otherwise (no launch made).
// Orders a solve on `st` after the upload of table set t.  While `st` is being captured into a
// graph the set is pinned for the plan's lifetime (see helmholtz_build_tables) and the upload,
// a few kilobytes on another stream, is waited for on the host, so the graph needs no dependency
// on it.
static int order_after_upload(HelmTables &t, cudaStream_t st, bool *capturing)
{
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    PZ_CUDA(cudaStreamIsCapturing(st, &cap));
    *capturing = (cap != cudaStreamCaptureStatusNone);
    if (*capturing) {
        t.captured = true;
        if (!t.upload_seen) {
            // event calls on another stream are "potentially unsafe" under global capture mode:
            // make this one in relaxed mode (the upload stream is not part of the capture)
            cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
            PZ_CUDA(cudaThreadExchangeStreamCaptureMode(&mode));
            const cudaError_t q = cudaEventSynchronize(t.uploaded);
            cudaThreadExchangeStreamCaptureMode(&mode);
            if (q != cudaSuccess) return cuda_fail(q, "helmholtz table upload");
            t.upload_seen = true;
        }
    } else if (t.upload_seen) {
        // nothing to order
    } else if (cudaEventQuery(t.uploaded) == cudaSuccess) {
        t.upload_seen = true;
    } else {
        cudaGetLastError();
        PZ_CUDA(cudaStreamWaitEvent(st, t.uploaded, 0));
    }
    return PZ_OK;
}

int launch_helmholtz_step(pz_plan *pl, double *u2, const double *uk, cudaStream_t st)
{
    if (pl->helm_variant != 1 || pl->opt.step_fused == 0) return PZ_EUNSUPPORTED;
    HelmTables &t = pl->helm[pl->helm_cur];
    bool capturing = false;
    {
        const int rc0 = order_after_upload(t, st, &capturing);
        if (rc0 != PZ_OK) return rc0;
    }
    int rc;
    {
        ProfScope prof(pl, PZ_K_HELMHOLTZ, st);
        rc = launch_helmholtz_tma_cn(pl, u2, uk, t.dev, st);
    }
    if (rc == PZ_OK && !capturing) PZ_CUDA(cudaEventRecord(t.last_use, st));
    return rc;
}

int launch_helmholtz_n(pz_plan *pl, double *const *u, int n, cudaStream_t st, int kind)
{
    if (n == 0) return PZ_OK;
    HelmTables &t = pl->helm[kind == 1 ? pl->helm_w_cur : pl->helm_cur];
    bool capturing = false;
    {
        const int rc0 = order_after_upload(t, st, &capturing);
        if (rc0 != PZ_OK) return rc0;
    }
    const size_t plane = (size_t)pl->nx * pl->ny;
    const int tx = pl->helm_tx, P = pl->helm_P;
    if (pl->helm_variant == 1) {
        for (int f0 = 0; f0 < n; f0 += 4) {
            const int nf = (n - f0 < 4) ? n - f0 : 4;
            ProfScope prof(pl, PZ_K_HELMHOLTZ, st);
            const int rc = launch_helmholtz_tma(pl, u + f0, nf, t.dev, st);
            if (rc != PZ_OK) return rc;
        }
    } else {
        const unsigned blocks = (unsigned)(plane / tx);
        const size_t smem = 2 * (size_t)(2 * P) * tx * sizeof(double);
        const int threads = tx * P;
        const bool full = (P * pl->helm_m == pl->nz);
#define PZ_HELM_LAUNCH(MM)                                                                                       \
    do {                                                                                                         \
        if (full) helmholtz_kernel<MM, true><<<blocks, threads, smem, st>>>(u[f], t.dev, plane, pl->nz, P, pl->helm_levels, tx); \
        else helmholtz_kernel<MM, false><<<blocks, threads, smem, st>>>(u[f], t.dev, plane, pl->nz, P, pl->helm_levels, tx);    \
    } while (0)
        for (int f = 0; f < n; ++f) {
            ProfScope prof(pl, PZ_K_HELMHOLTZ, st);
            switch (pl->helm_m) {
            case 4: PZ_HELM_LAUNCH(4); break;
            case 8: PZ_HELM_LAUNCH(8); break;
            case 16: PZ_HELM_LAUNCH(16); break;
            case 32: PZ_HELM_LAUNCH(32); break;
            default: set_error("helmholtz: bad sub-domain size %d", pl->helm_m); return PZ_EINVAL;
            }
            count_launch();
            PZ_CUDA(cudaGetLastError());
        }
#undef PZ_HELM_LAUNCH
    }
    if (!capturing) PZ_CUDA(cudaEventRecord(t.last_use, st));
    return PZ_OK;
}

} // namespace pz
