// pz_zslab.cu -- the z direction of ONE Poisson problem spread over G ranks by z-slabs: the
// paper's parallel tridiagonal solver (PAPER.md:120-135 steps 4-6, :139-155) across GPUs.
//
// Rank g owns the planes [kb[g], kb[g+1]); x and y transforms are plane-local.  Per spectral column
// the nz unknowns are cut at the slab boundaries:
//   reduce     every rank solves its slab-local system T_g (the slab's rows with the couplings to
//              the rows outside moved away) for the right-hand side: y = T_g^{-1} (-d).  Only the
//              first and last value of y leave the rank: 2 nx ny doubles ("pack 2 Nx Ny boundary
//              values").  The local solve is the warp-level algorithm of
//              pz_zsolve_pair.cuh (32 lanes = 32 sub-domains, Algorithm 1 in M-matrix form, PCR of
//              the lane boundaries), stopped before the reconstruction.
//   exchange   ONE all-gather of those rows (the caller's, over NCCL).
//   interface  phi_first / phi_last of every slab satisfy, with phi_prev = the previous slab's last
//              and phi_next = the next slab's first value,
//                  F_g = RF_g + PF_g phi_prev + QF_g phi_next,   L_g = RL_g + PL_g phi_prev + QL_g phi_next
//              (superposition; P, Q = T_g^{-1} applied to the two removed couplings): a system of
//              size 2G per column ("reduced systems ... with local size 2 p_z"),
//              solved redundantly by every rank.  Its coefficients do not depend on the right-hand
//              side (exchanged "only once as an initialization step"); here every
//              rank computes all G sets itself at plan creation, as the paper does for the
//              Helmholtz coefficients ("each GPU computing the global (a',b',c') coefficients",
//              PAPER.md:199): no plan-time collective at all.
//   finish     with phi_prev, phi_next known, the slab is solved once more with the removed
//              couplings on the right-hand side (solve_pair, OPEN) and reconstructed in place.
//
// Numerics: on stretched grids the low modes have P + Q = 1 - O(1e-9); 1 - PF QL would cancel.  The
// excess E = 1 - P - Q = sigma T_g^{-1} 1 >= 0 is therefore computed as a third coefficient solve and
// the interface elimination only ever adds non-negative numbers (the M-matrix form of pz_zsolve.cu).
// The singular (0,0) column is not part of the interface system: its nz right-hand-side values are
// gathered with the boundary rows and every rank solves it whole by the two prefix sums of the
// closed form, volume mean removed.
#include "pz_internal.h"
#include "pz_zsolve_pair.cuh"

namespace pz {

namespace {

constexpr int kTX = 16;    // real columns per tile (128-byte rows)
constexpr int kPairs = 8;  // complex pairs per tile = warps per CTA
constexpr int kMaxG = 16;  // slabs

struct RowAcc {
    double2 *d;
    __device__ __forceinline__ double2 &operator()(int i) const { return d[i * (kTX / 2)]; }
};

// Shared-memory coefficient tables of one slab [kb, kb + nk) of the global grid, one sub-domain
// of M rows per lane (stride CS): al / ga = sub- / super-diagonal magnitudes with the couplings
// across the slab boundaries removed, ex = the diagonal excess those leave behind.
template <int M>
__device__ __forceinline__ void stage_slab_tables(double *s_al, double *s_ga, double *s_ex, const double *__restrict__ A,
                                                  const double *__restrict__ C, int kb, int nk)
{
    constexpr int CS = M + 1;
    for (int k = threadIdx.x; k < kLanes * M; k += blockDim.x) {
        double al = 0.0, ga = 0.0, ex = 0.0;
        if (k < nk) {
            al = A[kb + k];
            ga = C[kb + k];
            if (k == 0) { ex += al; al = 0.0; }
            if (k == nk - 1) { ex += ga; ga = 0.0; }
        }
        s_al[(k / M) * CS + (k % M)] = al;
        s_ga[(k / M) * CS + (k % M)] = ga;
        s_ex[(k / M) * CS + (k % M)] = ex;
    }
}

__device__ __forceinline__ double sigma_of(size_t col, int nx, const double *lamx, const double *lamy_nat,
                                           const double *lamy_pk)
{
    const int i = (int)(col % nx), j = (int)(col / nx);
    return -(lamx[i] + ((i < 2) ? lamy_pk[j] : lamy_nat[j]));
}

// Plan time: the interface coefficients (PF, QF, EF, PL, QL, EL) of slab [kb, kb + nk) for every
// real column; coef[c * plane + col].  No field is read.
template <int M>
__global__ void __launch_bounds__(kPairs *kLanes)
    slab_coef_kernel(double *__restrict__ coef, const double *__restrict__ A, const double *__restrict__ C,
                     const double *__restrict__ lamx, const double *__restrict__ lamy_nat,
                     const double *__restrict__ lamy_pk, int nx, size_t plane, int kb, int nk)
{
    constexpr int CS = M + 1;
    __shared__ double s_tab[3 * kLanes * CS];
    double *s_al = s_tab, *s_ga = s_al + kLanes * CS, *s_ex = s_ga + kLanes * CS;
    stage_slab_tables<M>(s_al, s_ga, s_ex, A, C, kb, nk);
    __syncthreads();
    const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
    const size_t col = ((size_t)blockIdx.x * kPairs + q) * 2;
    const double *al = s_al + lane * CS, *ga = s_ga + lane * CS, *ex = s_ex + lane * CS;
    const int k0 = lane * M;
    const double aopen = A[kb], copen = C[kb + nk - 1];
#pragma unroll
    for (int comp = 0; comp < 2; ++comp) {
        const double sig = sigma_of(col + comp, nx, lamx, lamy_nat, lamy_pk);
        double F[3], L[3];
        reduce_pair<M, 3>(al, ga, ex, sig, k0, nk,
                          [&](int i, double(&o)[3]) {
                              const int k = k0 + i;
                              o[0] = (k == 0) ? aopen : 0.0;
                              o[1] = (k == nk - 1) ? copen : 0.0;
                              o[2] = (k < nk) ? sig : 0.0;
                          },
                          F, L);
        if (lane == 0) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                coef[(size_t)c * plane + col + comp] = F[c];
                coef[(size_t)(3 + c) * plane + col + comp] = L[c];
            }
        }
    }
}

// Runtime, first half: the boundary values RF, RL of y = T_g^{-1}(-d) for every real column, and
// the slab's rows of the (0,0) column.  bout = [RF (plane) | RL (plane) | d00 (nk)].
template <int M>
__global__ void __launch_bounds__(kPairs *kLanes, (M <= 8) ? 3 : (M == 16 ? 2 : 1))
    slab_reduce_kernel(const double *__restrict__ p, const BoutSet bouts, const double *__restrict__ A,
                       const double *__restrict__ C, const double *__restrict__ lamx,
                       const double *__restrict__ lamy_nat, const double *__restrict__ lamy_pk, int nx, size_t plane,
                       int kb, int nk)
{
    constexpr int CH = M * kTX + 2, CS = M + 1;
    extern __shared__ double smem_zs[];
    double *tile = smem_zs;
    double *s_al = tile + kLanes * CH, *s_ga = s_al + kLanes * CS, *s_ex = s_ga + kLanes * CS;
    const size_t col0 = (size_t)blockIdx.x * kTX;
    {
        const int c2 = (threadIdx.x & 7) * 2;
        for (int k = threadIdx.x >> 3; k < nk; k += 32) {
            const double2 v = *reinterpret_cast<const double2 *>(p + (size_t)k * plane + col0 + c2);
            *reinterpret_cast<double2 *>(tile + (k / M) * CH + (k % M) * kTX + c2) = v;
        }
        stage_slab_tables<M>(s_al, s_ga, s_ex, A, C, kb, nk);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
    const size_t col = col0 + 2 * q;
    const RowAcc d{reinterpret_cast<double2 *>(tile + lane * CH + 2 * q)};
    const double *al = s_al + lane * CS, *ga = s_ga + lane * CS, *ex = s_ex + lane * CS;
    const int k0 = lane * M;
    const double sig0 = sigma_of(col, nx, lamx, lamy_nat, lamy_pk), sig1 = sigma_of(col + 1, nx, lamx, lamy_nat, lamy_pk);
    double2 rf, rl;
    if (sig0 == sig1) {
        double F[2], L[2];
        reduce_pair<M, 2>(al, ga, ex, sig0, k0, nk,
                          [&](int i, double(&o)[2]) {
                              const bool live = k0 + i < nk;
                              const double2 v = d(i);
                              o[0] = live ? -v.x : 0.0;
                              o[1] = live ? -v.y : 0.0;
                          },
                          F, L);
        rf = make_double2(F[0], F[1]);
        rl = make_double2(L[0], L[1]);
    } else {
        double F[1], L[1];
        reduce_pair<M, 1>(al, ga, ex, sig0, k0, nk, [&](int i, double(&o)[1]) { o[0] = (k0 + i < nk) ? -d(i).x : 0.0; }, F, L);
        rf.x = F[0]; rl.x = L[0];
        reduce_pair<M, 1>(al, ga, ex, sig1, k0, nk, [&](int i, double(&o)[1]) { o[0] = (k0 + i < nk) ? -d(i).y : 0.0; }, F, L);
        rf.y = F[0]; rl.y = L[0];
    }
    for (int dst = 0; dst < bouts.n; ++dst) {
        double *bout = bouts.p[dst];
        if (lane == 0) {
            *reinterpret_cast<double2 *>(bout + col) = rf;
            *reinterpret_cast<double2 *>(bout + plane + col) = rl;
        }
        if (blockIdx.x == 0)
            for (int k = threadIdx.x; k < nk; k += blockDim.x) bout[2 * plane + k] = tile[(k / M) * CH + (k % M) * kTX];
    }
}

// The reduced systems of size 2G, one per real column (PAPER.md:128 step 5), every rank for itself.
// ball = G gathered boundary buffers of stride bstride; coef = [G][6][plane].  Unknowns L_j (last
// value of slab j) and F_{j+1} (first value of slab j+1), j = 0..G-2, eliminated slab by slab:
//   L_j     = rl' + q' F_{j+1},   q' = QL_j + PL_j mu,  excess e' = EL_j + PL_j nu,  rl' = RL_j + PL_j lambda
//   F_{j+1} = rho + tau F_{j+2},  den = EF + QF + PF e'  (= 1 - PF q', formed without subtraction)
//   L_j     = lambda + mu F_{j+2},  lambda = rl' + q' rho,  mu = q' tau,  nu = 1 - mu = e' + q' eta
// Output: phi_prev = L_{g-1} and phi_next = F_{g+1} of this rank's slab g (0 where there is none).
__global__ void __launch_bounds__(256)
    slab_interface_kernel(const double *__restrict__ ball, size_t bstride, const double *__restrict__ coef, size_t plane,
                          int G, int g, double *__restrict__ phi_prev, double *__restrict__ phi_next)
{
    const size_t col = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= plane) return;
    double pv = 0.0, nv = 0.0;
    if (col != 0 && G > 1) { // (0,0): solved whole from the gathered column
        double rho[kMaxG], tau[kMaxG], rlp[kMaxG], qp[kMaxG];
        double lam = 0.0, mu = 0.0, nu = 1.0;
        for (int j = 0; j + 1 < G; ++j) {
            const double *cj = coef + (size_t)j * 6 * plane + col, *cn = coef + (size_t)(j + 1) * 6 * plane + col;
            const double PL = cj[3 * plane], QL = cj[4 * plane], EL = cj[5 * plane];
            const double PF = cn[0], QF = cn[plane], EF = cn[2 * plane];
            const double RL = ball[(size_t)j * bstride + plane + col], RF = ball[(size_t)(j + 1) * bstride + col];
            const double rl1 = fma(PL, lam, RL), q1 = fma(PL, mu, QL), e1 = fma(PL, nu, EL);
            const double rden = 1.0 / (EF + QF + PF * e1);
            const double rh = fma(PF, rl1, RF) * rden, ta = QF * rden, et = fma(PF, e1, EF) * rden;
            rho[j] = rh; tau[j] = ta; rlp[j] = rl1; qp[j] = q1;
            lam = fma(q1, rh, rl1);
            mu = q1 * ta;
            nu = fma(q1, et, e1);
        }
        double fn = 0.0; // F_{j+2}
        for (int j = G - 2; j >= 0; --j) {
            const double f = fma(tau[j], fn, rho[j]); // F_{j+1}
            const double l = fma(qp[j], f, rlp[j]);   // L_j
            if (j + 1 == g + 1) nv = f;
            if (j == g - 1) pv = l;
            fn = f;
        }
    }
    phi_prev[col] = pv;
    phi_next[col] = nv;
}

// Runtime, second half: the slab solved with the neighbours' boundary values on the right-hand
// side (solve_pair, OPEN), in place.
template <int M>
__global__ void __launch_bounds__(kPairs *kLanes, (M <= 8) ? 3 : (M == 16 ? 2 : 1))
    slab_finish_kernel(double *__restrict__ p, const double *__restrict__ phi_prev, const double *__restrict__ phi_next,
                       const double *__restrict__ A, const double *__restrict__ C, const double *__restrict__ lamx,
                       const double *__restrict__ lamy_nat, const double *__restrict__ lamy_pk, int nx, size_t plane,
                       int kb, int nk)
{
    constexpr int CH = M * kTX + 2, CS = M + 1;
    extern __shared__ double smem_zs[];
    double *tile = smem_zs;
    double *s_al = tile + kLanes * CH, *s_ga = s_al + kLanes * CS, *s_ex = s_ga + kLanes * CS;
    const size_t col0 = (size_t)blockIdx.x * kTX;
    {
        const int c2 = (threadIdx.x & 7) * 2;
        for (int k = threadIdx.x >> 3; k < nk; k += 32) {
            const double2 v = *reinterpret_cast<const double2 *>(p + (size_t)k * plane + col0 + c2);
            *reinterpret_cast<double2 *>(tile + (k / M) * CH + (k % M) * kTX + c2) = v;
        }
        stage_slab_tables<M>(s_al, s_ga, s_ex, A, C, kb, nk);
    }
    __syncthreads();
    {
        const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
        const size_t col = col0 + 2 * q;
        const RowAcc d{reinterpret_cast<double2 *>(tile + lane * CH + 2 * q)};
        const double *al = s_al + lane * CS, *ga = s_ga + lane * CS, *ex = s_ex + lane * CS;
        const int k0 = lane * M;
        const double sig0 = sigma_of(col, nx, lamx, lamy_nat, lamy_pk), sig1 = sigma_of(col + 1, nx, lamx, lamy_nat, lamy_pk);
        const double aopen = A[kb], copen = C[kb + nk - 1];
        const double2 pp = *reinterpret_cast<const double2 *>(phi_prev + col), pn = *reinterpret_cast<const double2 *>(phi_next + col);
        const double2 bp = make_double2(aopen * pp.x, aopen * pp.y), bn = make_double2(copen * pn.x, copen * pn.y);
        if (sig0 == sig1) {
            solve_pair<M, 3, false, false, false, true>(d, al, ga, sig0, k0, nk, nullptr, 0.0, ex, bp, bn);
        } else {
            solve_pair<M, 1, false, false, false, true>(d, al, ga, sig0, k0, nk, nullptr, 0.0, ex, bp, bn);
            solve_pair<M, 2, false, false, false, true>(d, al, ga, sig1, k0, nk, nullptr, 0.0, ex, bp, bn);
        }
    }
    __syncthreads();
    {
        const int c2 = (threadIdx.x & 7) * 2;
        for (int k = threadIdx.x >> 3; k < nk; k += 32) {
            const double2 v = *reinterpret_cast<const double2 *>(tile + (k / M) * CH + (k % M) * kTX + c2);
            *reinterpret_cast<double2 *>(p + (size_t)k * plane + col0 + c2) = v;
        }
    }
}

// The (0,0) column, whole, from the gathered right-hand side (closed form of the singular Neumann
// system: S_k = sum_{l<=k} dzf_l d_l, phi_{k+1} = phi_k + dzc_k S_k, then zero volume mean); this
// rank's rows are written into its slab (g >= 0) or, for the plan's own cut, all rows (g < 0, p =
// the whole field).  One CTA of 1024 threads: two block-wide prefix sums per chunk of 1024 rows
// with running carries (fixed summation tree: deterministic, the same on every rank).
__device__ __forceinline__ double block_scan_incl(double v, double *wsum, double *total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o *= 2) {
        const double t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    __syncthreads(); // wsum free again
    if (lane == 31) wsum[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double w = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o *= 2) {
            const double t = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += t;
        }
        wsum[lane] = w;
    }
    __syncthreads();
    *total = wsum[31];
    return v + (warp > 0 ? wsum[warp - 1] : 0.0);
}

constexpr int kZmChunks = 16; // rows per column <= 16 * 1024

__global__ void __launch_bounds__(1024)
    slab_zero_mode_kernel(double *__restrict__ p, const double *__restrict__ ball, size_t bstride, size_t plane,
                          const int *__restrict__ kb, int G, int g, const double *__restrict__ dzf,
                          const double *__restrict__ zc, double inv_lz)
{
    __shared__ double wsum[32];
    const int nz = kb[G];
    double phi[kZmChunks];
    double carryS = 0.0, carryP = 0.0, acc = 0.0;
#pragma unroll
    for (int c = 0; c < kZmChunks; ++c) {
        phi[c] = 0.0;
        if (c * 1024 < nz) {
            const int k = c * 1024 + (int)threadIdx.x;
            double t = 0.0;
            if (k < nz) {
                int j = 0;
                while (k >= kb[j + 1]) ++j;
                t = dzf[k] * ball[(size_t)j * bstride + 2 * plane + (k - kb[j])];
            }
            double totS, totP;
            const double S = carryS + block_scan_incl(t, wsum, &totS);
            const double u = (k + 1 < nz) ? (zc[k + 1] - zc[k]) * S : 0.0;
            const double incl = block_scan_incl(u, wsum, &totP);
            phi[c] = carryP + (incl - u); // exclusive: phi_k = sum_{l<k} dzc_l S_l
            if (k < nz) acc = fma(dzf[k], phi[c], acc);
            carryS += totS;
            carryP += totP;
        }
    }
    double tot;
    block_scan_incl(acc, wsum, &tot);
    const double mean = tot * inv_lz;
#pragma unroll
    for (int c = 0; c < kZmChunks; ++c) {
        const int k = c * 1024 + (int)threadIdx.x;
        if (k < nz) {
            if (g < 0) p[(size_t)k * plane] = phi[c] - mean;
            else if (k >= kb[g] && k < kb[g + 1]) p[(size_t)(k - kb[g]) * plane] = phi[c] - mean;
        }
    }
}

int m_for(int nk) { return nk <= 128 ? 4 : nk <= 256 ? 8 : nk <= 512 ? 16 : 32; }
template <int M> constexpr size_t slab_smem() { return ((size_t)kLanes * (M * kTX + 2) + 3 * (size_t)kLanes * (M + 1)) * sizeof(double); }

#define PZ_SLAB_DISPATCH(nk, ...)                                                                  \
    switch (m_for(nk)) {                                                                           \
    case 4: { constexpr int MM = 4; __VA_ARGS__; } break;                                          \
    case 8: { constexpr int MM = 8; __VA_ARGS__; } break;                                          \
    case 16: { constexpr int MM = 16; __VA_ARGS__; } break;                                        \
    default: { constexpr int MM = 32; __VA_ARGS__; } break;                                        \
    }

} // namespace

// plan time: coefficient planes of every slab into pl->slab_coef ([G][6][plane])
int launch_slab_coefficients(pz_plan *pl, cudaStream_t st)
{
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)(plane / kTX);
    for (int j = 0; j < pl->slab_G; ++j) {
        const int kb = pl->slab_kb[j], nk = pl->slab_kb[j + 1] - kb;
        double *coef = pl->slab_coef + (size_t)j * 6 * plane;
        PZ_SLAB_DISPATCH(nk, (slab_coef_kernel<MM><<<blocks, kPairs * kLanes, 0, st>>>(coef, pl->d_A, pl->d_C, pl->d_lamx, pl->d_lamy_nat,
                                                                                       pl->d_lamy_pk, pl->nx, plane, kb, nk)));
        count_launch();
        PZ_CUDA(cudaGetLastError());
    }
    return PZ_OK;
}

// Slab g of the plan's cut: p_slab points at its first plane.  Slabs of more than 128 planes take the
// TMA pipeline of pz_zsolve_tma.cu (slab modes), thinner ones the kernels above.
static int slab_reduce_g(pz_plan *pl, double *p_slab, int g, const BoutSet &bout, cudaStream_t st)
{
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)(plane / kTX);
    const int kb = pl->slab_kb[g], nk = pl->slab_kb[g + 1] - kb;
    if (nk > 128 && pl->opt.zsolve_variant != 1) return launch_zslab_tma(pl, p_slab, kb, nk, &bout, nullptr, nullptr, st);
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    PZ_SLAB_DISPATCH(nk, {
        { const int rc = smem_optin(pl, slab_reduce_kernel<MM>, slab_smem<MM>()); if (rc != PZ_OK) return rc; }
        slab_reduce_kernel<MM><<<blocks, kPairs * kLanes, slab_smem<MM>(), st>>>(p_slab, bout, pl->d_A, pl->d_C, pl->d_lamx, pl->d_lamy_nat,
                                                                                 pl->d_lamy_pk, pl->nx, plane, kb, nk);
    });
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

static int slab_finish_g(pz_plan *pl, double *p_slab, int g, const double *ball, cudaStream_t st)
{
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)(plane / kTX);
    const int G = pl->slab_G, kb = pl->slab_kb[g], nk = pl->slab_kb[g + 1] - kb;
    {
        ProfScope prof(pl, PZ_K_Z_SOLVE, st);
        slab_interface_kernel<<<(unsigned)((plane + 255) / 256), 256, 0, st>>>(ball, pl->slab_bstride, pl->slab_coef, plane, G, g,
                                                                             pl->slab_phi, pl->slab_phi + plane);
        count_launch();
        PZ_CUDA(cudaGetLastError());
    }
    if (nk > 128 && pl->opt.zsolve_variant != 1) {
        const int rc = launch_zslab_tma(pl, p_slab, kb, nk, nullptr, pl->slab_phi, pl->slab_phi + plane, st);
        if (rc != PZ_OK) return rc;
    } else {
        ProfScope prof(pl, PZ_K_Z_SOLVE, st);
        PZ_SLAB_DISPATCH(nk, {
            { const int rc = smem_optin(pl, slab_finish_kernel<MM>, slab_smem<MM>()); if (rc != PZ_OK) return rc; }
            slab_finish_kernel<MM><<<blocks, kPairs * kLanes, slab_smem<MM>(), st>>>(p_slab, pl->slab_phi, pl->slab_phi + plane, pl->d_A, pl->d_C,
                                                                                     pl->d_lamx, pl->d_lamy_nat, pl->d_lamy_pk, pl->nx, plane, kb, nk);
        });
        count_launch();
        PZ_CUDA(cudaGetLastError());
    }
    if (pl->slab_internal) return PZ_OK; // the plan's own cut writes the whole (0,0) column once (launch_zsolve_islab)
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    slab_zero_mode_kernel<<<1, 1024, 0, st>>>(p_slab, ball, pl->slab_bstride, plane, pl->d_slab_kb, G, g, pl->d_dzf, pl->d_zc, pl->inv_lz);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

// Peer-memory exchange: after the reduction kernel has stored this rank's block into every rank's
// gathered buffer, one thread makes those stores visible system-wide and raises this rank's flag in
// every rank's flag array; a finish first waits until all ranks' flags of its own array carry the epoch.
struct FlagSet { long long *p[16]; int n; };
__global__ void slab_signal_kernel(const FlagSet fl, int slot, long long epoch)
{
    __threadfence_system();
    for (int r = threadIdx.x; r < fl.n; r += blockDim.x) {
        long long *f = fl.p[r] + slot;
        asm volatile("st.release.sys.global.s64 [%0], %1;" ::"l"(f), "l"(epoch) : "memory");
    }
}
__global__ void slab_wait_kernel(const long long *__restrict__ flags, int n, long long epoch)
{
    for (int r = threadIdx.x; r < n; r += blockDim.x) {
        long long v;
        do {
            asm volatile("ld.acquire.sys.global.s64 %0, [%1];" : "=l"(v) : "l"(flags + r) : "memory");
            if (v < epoch) __nanosleep(200);
        } while (v < epoch);
    }
    __threadfence_system();
}

int launch_slab_signal(pz_plan *pl, long long *const *flags, int n, int slot, long long epoch, cudaStream_t st)
{
    (void)pl;
    FlagSet fl;
    fl.n = n;
    for (int r = 0; r < n; ++r) fl.p[r] = flags[r];
    slab_signal_kernel<<<1, 32, 0, st>>>(fl, slot, epoch);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

int launch_slab_wait(pz_plan *pl, const long long *flags, int n, long long epoch, cudaStream_t st)
{
    (void)pl;
    slab_wait_kernel<<<1, 32, 0, st>>>(flags, n, epoch);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

int launch_slab_reduce(pz_plan *pl, double *p, const BoutSet &bout, cudaStream_t st) { return slab_reduce_g(pl, p, pl->slab_g, bout, st); }
int launch_slab_finish(pz_plan *pl, double *p, const double *ball, cudaStream_t st) { return slab_finish_g(pl, p, pl->slab_g, ball, st); }

// A whole column of more than 1024 rows on ONE GPU (the paper's wall-normal size is 1594,
// PAPER.md:268): the plan cuts z into slabs of at most 1024 planes itself and runs the distributed
// algorithm locally -- every slab's reduction, the interface systems, every slab's finish; the
// "exchange" is the plan's own boundary buffer.  24 instead of 16 bytes per point cross HBM, against
// 32 and an N-double workspace for the thread-per-column sweep of pz_zsolve.cu.
int launch_zsolve_islab(pz_plan *pl, double *p, cudaStream_t st)
{
    const size_t plane = (size_t)pl->nx * pl->ny;
    for (int g = 0; g < pl->slab_G; ++g) {
        BoutSet one;
        one.n = 1;
        one.p[0] = pl->islab_ball + (size_t)g * pl->slab_bstride;
        const int rc = slab_reduce_g(pl, p + (size_t)pl->slab_kb[g] * plane, g, one, st);
        if (rc != PZ_OK) return rc;
    }
    for (int g = 0; g < pl->slab_G; ++g) {
        const int rc = slab_finish_g(pl, p + (size_t)pl->slab_kb[g] * plane, g, pl->islab_ball, st);
        if (rc != PZ_OK) return rc;
    }
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    slab_zero_mode_kernel<<<1, 1024, 0, st>>>(p, pl->islab_ball, pl->slab_bstride, plane, pl->d_slab_kb, pl->slab_G, -1, pl->d_dzf, pl->d_zc,
                                              pl->inv_lz);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace pz
