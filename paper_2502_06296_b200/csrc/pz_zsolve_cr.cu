// pz_zsolve_cr.cu -- step a3, variant 1: the paper's parallel tridiagonal algorithm
// (Algorithm 1 at :157-197) applied INSIDE one GPU.
//
// In the paper the z direction is cut into p_z sub-domains owned by different GPUs: each reduces
// its rows to the two boundary unknowns, a small system of size 2 p_z is solved, and the interior
// is reconstructed.  Here a CTA stages a tile of 16 neighbouring spectral columns x all nz rows in
// shared memory (one coalesced HBM read, one write: 16 B/point), a warp owns one complex column
// (the packed pair (2q, 2q+1): Re and Im share the matrix, so pivots are computed once for both),
// and its 32 lanes are the 32 "sub-domains" of m = nz/32 rows.  The boundary system is solved
// with warp-shuffle parallel cyclic reduction.  Coefficients depend on (i,j,k) for the Poisson
// problem, so Algorithm 1's private a', c' arrays live in registers and are
// recomputed every solve; storing them would cost 8-16 more HBM bytes per point.
//
// All rows are kept in M-matrix form with an explicit diagonal excess (see pz_zsolve.cu): the
// sub-domain sweeps, the reduced system and the PCR levels only add non-negative numbers.
#include "pz_internal.h"
#include "pz_zsolve_pair.cuh"

namespace pz {

namespace {

constexpr int kTX = 16;    // real columns per tile (128-byte rows)
constexpr int kPairs = 8;  // complex pairs per tile = warps per CTA

// rows of one sub-domain inside the manually staged tile: stride kTX doubles
struct RowAcc {
    double2 *d;
    __device__ __forceinline__ double2 &operator()(int i) const { return d[i * (kTX / 2)]; }
};

template <int M, bool HELM>
__global__ void __launch_bounds__(kPairs *kLanes, (M <= 8) ? 3 : (M == 16 ? 2 : 1))
    zsolve_cr_kernel(double *__restrict__ p, const double *__restrict__ A, const double *__restrict__ C,
                     const double *__restrict__ dzf, const double *__restrict__ lamx,
                     const double *__restrict__ lamy_nat, const double *__restrict__ lamy_pk, int nx, int ny,
                     int nz, double inv_lz, double ha, double hw0, double hw1, int zflags)
{
    constexpr int CH = M * kTX + 2;  // doubles per sub-domain in the tile (+2: bank spread, 16-B aligned)
    constexpr int CS = M + 1;        // coefficient stride per lane (bank spread)
    extern __shared__ double smem_z[];
    double *tile = smem_z;                     // kLanes * CH
    double *s_al = tile + kLanes * CH;         // kLanes * CS
    double *s_ga = s_al + kLanes * CS;
    double *s_e0 = s_ga + kLanes * CS;

    const size_t plane = (size_t)nx * ny;
    const size_t col0 = (size_t)blockIdx.x * kTX;

    // stage the tile: 8 threads x 16 B per row, 32 rows per sweep
    {
        const int c2 = (threadIdx.x & 7) * 2;
        for (int k = threadIdx.x >> 3; k < nz; k += 32) {
            const double2 v = *reinterpret_cast<const double2 *>(p + (size_t)k * plane + col0 + c2);
            *reinterpret_cast<double2 *>(tile + (k / M) * CH + (k % M) * kTX + c2) = v;
        }
        for (int k = threadIdx.x; k < kLanes * M; k += blockDim.x) {
            const double sc = HELM ? ha : 1.0;
            s_al[(k / M) * CS + (k % M)] = (k < nz) ? sc * A[k] : 0.0;
            s_ga[(k / M) * CS + (k % M)] = (k < nz) ? sc * C[k] : 0.0;
            const double wk = (k == 0 ? hw0 : 0.0) + (k == nz - 1 ? hw1 : 0.0);
            s_e0[(k / M) * CS + (k % M)] = HELM ? 1.0 + ha * wk : wk;
        }
    }
    __syncthreads();

    {
        const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
        const size_t col = col0 + 2 * q;
        const int i = (int)(col % nx), j = (int)(col / nx);
        const double ly = (i < 2) ? lamy_pk[j] : lamy_nat[j];
        const double sig0 = -(lamx[i] + ly), sig1 = -(lamx[i + 1] + ly);
        const RowAcc d{reinterpret_cast<double2 *>(tile + lane * CH + 2 * q)};
        const double *al = s_al + lane * CS, *ga = s_ga + lane * CS;
        const int k0 = lane * M;
        if constexpr (HELM) {
            const double *e0 = s_e0 + lane * CS;
            if (sig0 == sig1) {
                solve_pair<M, 3, false, false, true>(d, al, ga, ha * sig0, k0, nz, dzf, inv_lz, e0);
            } else {
                solve_pair<M, 1, false, false, true>(d, al, ga, ha * sig0, k0, nz, dzf, inv_lz, e0);
                solve_pair<M, 2, false, false, true>(d, al, ga, ha * sig1, k0, nz, dzf, inv_lz, e0);
            }
        } else if (zflags & 1) {
            // Dirichlet wall(s): the wall rows carry the excess W (s_e0); no column is singular
            const double *ex = s_e0 + lane * CS;
            const double2 z2 = make_double2(0.0, 0.0);
            if (sig0 == sig1) {
                solve_pair<M, 3, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, z2, z2);
            } else {
                solve_pair<M, 1, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, z2, z2);
                solve_pair<M, 2, false, false, false, true>(d, al, ga, sig1, k0, nz, nullptr, 0.0, ex, z2, z2);
            }
        } else if (sig0 == sig1) {
            solve_pair<M, 3, false>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
        } else {
            // pair 0 of a row: x-modes 0 and nx/2 have different eigenvalues; (0,0) is singular
            if (i == 0 && j == 0 && (zflags & 2))
                solve_pair<M, 1, true>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
            else
                solve_pair<M, 1, false>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
            solve_pair<M, 2, false>(d, al, ga, sig1, k0, nz, dzf, inv_lz);
        }
    }
    __syncthreads();

    {
        const int c2 = (threadIdx.x & 7) * 2;
        for (int k = threadIdx.x >> 3; k < nz; k += 32) {
            const double2 v = *reinterpret_cast<const double2 *>(tile + (k / M) * CH + (k % M) * kTX + c2);
            *reinterpret_cast<double2 *>(p + (size_t)k * plane + col0 + c2) = v;
        }
    }
}

template <int M, bool HELM>
int launch_m(pz_plan *pl, double *p, cudaStream_t st, double ha)
{
    constexpr size_t smem = ((size_t)kLanes * (M * kTX + 2) + 3 * (size_t)kLanes * (M + 1)) * sizeof(double);
    if (smem > 48 * 1024) {
        const int rc = smem_optin(pl, zsolve_cr_kernel<M, HELM>, smem);
        if (rc != PZ_OK) return rc;
    }
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)(plane / kTX);
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    zsolve_cr_kernel<M, HELM><<<blocks, kPairs * kLanes, smem, st>>>(p, pl->d_A, pl->d_C, pl->d_dzf, pl->d_lamx,
                                                                      pl->d_lamy_nat, pl->d_lamy_pk, pl->nx, pl->ny,
                                                                      pl->nz, pl->inv_lz, ha, HELM ? pl->wall_w0 : pl->pw0,
                                                                      HELM ? pl->wall_w1 : pl->pw1, pl->zflags());
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace

int launch_zsolve_cr(pz_plan *pl, double *p, cudaStream_t st, double helm_a)
{
    const int nz = pl->nz;
#define PZ_ZC(MM) (helm_a >= 0.0 ? launch_m<MM, true>(pl, p, st, helm_a) : launch_m<MM, false>(pl, p, st, 0.0))
    if (nz <= 32 * 4) return PZ_ZC(4);
    if (nz <= 32 * 8) return PZ_ZC(8);
    if (nz <= 32 * 16) return PZ_ZC(16);
    if (nz <= 32 * 32) return PZ_ZC(32);
#undef PZ_ZC
    set_error("z-solve variant 1 supports nz <= 1024 (got %d); use zsolve_variant = 0", nz);
    return PZ_EUNSUPPORTED;
}

} // namespace pz
