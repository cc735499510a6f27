// pz_zsolve_tma.cu -- step a3, variant 2 (default for nz <= 512): the chunked cyclic reduction of
// pz_zsolve_cr.cu (Algorithm 1 inside one GPU) fed by an asynchronous pipeline.
//
// Variant 1 stages its tile with ordinary loads, solves, and writes back: the three phases of a
// CTA do not overlap and only two CTAs fit an SM (ncu r01b: 35 % of DRAM peak, 24 % of the warp
// slots active, every pipe below 55 %).  Here one CTA per SM stays resident:
//   * a producer warp drives the TMA unit: the tile {16 columns x nz rows} of spectral column
//     block t is fetched into one of S shared-memory stages as 32 boxes {16 columns x m rows}, one
//     per sub-domain; a stage that has been solved is written back by TMA stores straight from
//     shared memory, and is refilled as soon as the store has read it;
//   * eight solver warps, one per complex column pair, wait for "stage full", solve their pair in
//     place (lanes = the 32 sub-domains; warp-shuffle PCR for the boundary system) and signal
//     "stage done".  Solver warps never wait for one another: each walks the tile sequence at its
//     own pace, so loads, solves and stores of neighbouring tiles overlap.
//   * Shared-memory layout: a warp reads the same 16-byte slot (its pair) of 32 different rows,
//     which in a dense [row][128 B] tile is a 32-way bank conflict.  The boxes use the TMA
//     128-byte swizzle (the 16-byte slot index is XORed with the row index mod 8) and each
//     sub-domain slot is m+1 rows long, so the 8 lanes of a shared-memory wavefront sit in 8
//     different rows mod 8: conflict-free.
#include "pz_internal.h"
#include "pz_tma.cuh"
#include "pz_zsolve_pair.cuh"

namespace pz {

namespace {

constexpr int kTX = 16;      // real columns per tile (128-byte rows)
constexpr int kSolvers = 8;  // solver warps = complex pairs per tile
constexpr int kThreads = (kSolvers + 1) * 32;

// Row i of a sub-domain whose slot starts at absolute row R0 of a 1024-byte aligned stage:
// byte offset (R0+i)*128 + ((pair ^ ((R0+i) & 7)) << 4).
struct SwzAcc {
    unsigned char *slot; // stage base + R0*128
    int off[8];          // ((pair ^ ((R0 + j) & 7)) << 4), j = 0..7
    __device__ __forceinline__ double2 &operator()(int i) const
    {
        return *reinterpret_cast<double2 *>(slot + i * 128 + off[i & 7]);
    }
};

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int M> struct Geo {
    static constexpr int SLOT = M + 1;                       // rows per sub-domain slot
    static constexpr size_t STAGE = (size_t)kLanes * SLOT * 128;
    static constexpr int CS = M + 1;                         // coefficient stride per lane
    static constexpr size_t COEF = (size_t)3 * kLanes * CS * sizeof(double);   // alpha, gamma, e0
    __host__ __device__ static size_t bytes(int stages) { return 1024 + stages * STAGE + COEF + 64; }
};

// z-slab of a cut column (pz_zslab.cu): what the slab modes need beside the tile
struct SlabArgs {
    int kb = 0;                       // first global row of the slab (the tile holds rows kb .. kb + nz - 1)
    BoutSet bout;                     // reduce: destinations of [RF (plane) | RL (plane) | (0,0) column (nz)]
    const double *phi_prev = nullptr; // finish: value of the row below the slab, per real column
    const double *phi_next = nullptr; //         and of the row above
    size_t plane = 0;
};

// HELM = false: the Poisson systems (diagonal excess sigma = -(lambda_x + lambda_y), rhs -d, (0,0)
// pinned).  HELM = true: the fully implicit Helmholtz systems of Eq. (8) with a = ha and the
// Dirichlet wall terms hw0, hw1 (solve_pair, HELM).
// MODE 0: whole columns.  MODE 1 / 2: one z-slab of cut columns -- 1 = slab-local reduction (the
// slab's boundary values of T^{-1}(-d) go to sa.bout, nothing is stored back), 2 = the slab solved
// with its neighbours' boundary values on the right-hand side (solve_pair, OPEN), in place.
template <int M, bool HELM, int MODE = 0>
__global__ void __launch_bounds__(kThreads, 1)
    zsolve_tma_kernel(const __grid_constant__ CUtensorMap map, const double *__restrict__ A,
                      const double *__restrict__ C, const double *__restrict__ dzf, const double *__restrict__ lamx,
                      const double *__restrict__ lamy_nat, const double *__restrict__ lamy_pk, int nx, int ny, int nz,
                      double inv_lz, int ntiles, int stages, double ha, double hw0, double hw1, int probe, const SlabArgs sa, int zflags)
{
    static_assert(!(HELM && MODE != 0), "slabs of cut columns are Poisson systems");
    using G = Geo<M>;
    extern __shared__ unsigned char smem_zt[];
    // 1024-byte aligned stage area (the swizzle pattern is a function of the address)
    unsigned char *base = smem_zt + ((1024u - (smem_u32(smem_zt) & 1023u)) & 1023u);
    double *s_al = reinterpret_cast<double *>(base + stages * G::STAGE);
    double *s_ga = s_al + kLanes * G::CS;
    double *s_e0 = s_ga + kLanes * G::CS;
    uint64_t *full = reinterpret_cast<uint64_t *>(s_e0 + kLanes * G::CS);
    uint64_t *done = full + 4;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int b = 0; b < stages; ++b) {
            mbar_init(&full[b], 1);
            mbar_init(&done[b], kSolvers);
        }
        mbar_fence_init();
    }
    for (int k = threadIdx.x; k < kLanes * M; k += blockDim.x) {
        const double sc = HELM ? ha : 1.0;
        double al = (k < nz) ? sc * A[sa.kb + k] : 0.0, ga = (k < nz) ? sc * C[sa.kb + k] : 0.0;
        // HELM: 1 + a W_k; Poisson with Dirichlet walls (zflags bit 0): W_k, the wall rows' extra diagonal
        const double wk = (k == 0 ? hw0 : 0.0) + (k == nz - 1 ? hw1 : 0.0);
        double ex = HELM ? 1.0 + ha * wk : wk;
        if constexpr (MODE != 0) {
            // couplings across the slab's ends leave the matrix; their magnitude stays on the diagonal
            ex = 0.0;
            if (k == 0) { ex += al; al = 0.0; }
            if (k == nz - 1) { ex += ga; ga = 0.0; }
        }
        s_al[(k / M) * G::CS + (k % M)] = al;
        s_ga[(k / M) * G::CS + (k % M)] = ga;
        s_e0[(k / M) * G::CS + (k % M)] = ex;
    }
    __syncthreads();

    const int my_tiles = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    constexpr unsigned kStageTx = (unsigned)(kLanes * M * 128);

    if (warp == kSolvers) {
        // ---------------------------------------------------------------- producer
        if (lane == 0) {
            auto load = [&](int it) {
                const int b = it % stages, col0 = ((int)blockIdx.x + it * (int)gridDim.x) * kTX;
                mbar_arrive_expect_tx(&full[b], kStageTx);
                for (int l = 0; l < kLanes; ++l)
                    tma_load_2d(base + b * G::STAGE + (size_t)l * G::SLOT * 128, &map, col0, l * M, &full[b]);
            };
            for (int it = 0; it < stages && it < my_tiles; ++it) load(it);
            for (int it = 0; it < my_tiles; ++it) {
                const int b = it % stages, col0 = ((int)blockIdx.x + it * (int)gridDim.x) * kTX;
                mbar_wait(&done[b], (it / stages) & 1);
                if constexpr (MODE != 1) {
                    for (int l = 0; l < kLanes; ++l)
                        if (l * M < nz) tma_store_2d(&map, base + b * G::STAGE + (size_t)l * G::SLOT * 128, col0, l * M);
                    tma_store_commit();
                }
                if (it + stages < my_tiles) {
                    if constexpr (MODE != 1) tma_store_wait_read<0>();
                    load(it + stages);
                }
            }
            tma_store_wait_all<0>();
        }
        return;
    }

    // -------------------------------------------------------------------- solvers
    const int q = warp;
    const bool no_pad = (nz == kLanes * M);
    const double *al = s_al + lane * G::CS, *ga = s_ga + lane * G::CS;
    const int k0 = lane * M, R0 = lane * G::SLOT;
    SwzAcc d;
#pragma unroll
    for (int j = 0; j < 8; ++j) d.off[j] = (q ^ ((R0 + j) & 7)) << 4;

    for (int it = 0; it < my_tiles; ++it) {
        const int b = it % stages;
        const size_t col = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * kTX + 2 * q;
        const int i = (int)(col % nx), j = (int)(col / nx);
        const double ly = (i < 2) ? lamy_pk[j] : lamy_nat[j];
        const double sig0 = -(lamx[i] + ly), sig1 = -(lamx[i + 1] + ly);
        d.slot = base + b * G::STAGE + (size_t)R0 * 128;
        mbar_wait(&full[b], (it / stages) & 1);
        if constexpr (MODE == 1) {
            const double *ex = s_e0 + lane * G::CS;
            double2 rf, rl;
            if (sig0 == sig1) {
                double F[2], L[2];
                reduce_pair<M, 2>(al, ga, ex, sig0, k0, nz,
                                  [&](int r, double(&o)[2]) {
                                      const bool live = k0 + r < nz;
                                      const double2 v = d(r);
                                      o[0] = live ? -v.x : 0.0;
                                      o[1] = live ? -v.y : 0.0;
                                  },
                                  F, L);
                rf = make_double2(F[0], F[1]);
                rl = make_double2(L[0], L[1]);
            } else {
                double F[1], L[1];
                reduce_pair<M, 1>(al, ga, ex, sig0, k0, nz, [&](int r, double(&o)[1]) { o[0] = (k0 + r < nz) ? -d(r).x : 0.0; }, F, L);
                rf.x = F[0]; rl.x = L[0];
                reduce_pair<M, 1>(al, ga, ex, sig1, k0, nz, [&](int r, double(&o)[1]) { o[0] = (k0 + r < nz) ? -d(r).y : 0.0; }, F, L);
                rf.y = F[0]; rl.y = L[0];
            }
            for (int dst = 0; dst < sa.bout.n; ++dst) {
                double *bo = sa.bout.p[dst];
                if (lane == 0) {
                    *reinterpret_cast<double2 *>(bo + col) = rf;
                    *reinterpret_cast<double2 *>(bo + sa.plane + col) = rl;
                }
                if (col == 0) // the slab's rows of the singular (0,0) column travel whole
#pragma unroll
                    for (int r = 0; r < M; ++r)
                        if (k0 + r < nz) bo[2 * sa.plane + k0 + r] = d(r).x;
            }
        } else if constexpr (MODE == 2) {
            const double *ex = s_e0 + lane * G::CS;
            const double aopen = A[sa.kb], copen = C[sa.kb + nz - 1];
            const double2 pp = *reinterpret_cast<const double2 *>(sa.phi_prev + col), pn = *reinterpret_cast<const double2 *>(sa.phi_next + col);
            const double2 bp = make_double2(aopen * pp.x, aopen * pp.y), bn = make_double2(copen * pn.x, copen * pn.y);
            if (sig0 == sig1) {
                solve_pair<M, 3, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, bp, bn);
            } else {
                solve_pair<M, 1, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, bp, bn);
                solve_pair<M, 2, false, false, false, true>(d, al, ga, sig1, k0, nz, nullptr, 0.0, ex, bp, bn);
            }
        } else if (kProbes && probe == 2) {
            // diagnostic: pipeline skeleton only (TMA load, TMA store), no arithmetic
        } else if constexpr (HELM) {
            const double *e0 = s_e0 + lane * G::CS;
            if (sig0 == sig1) {
                solve_pair<M, 3, false, false, true>(d, al, ga, ha * sig0, k0, nz, dzf, inv_lz, e0);
            } else {
                solve_pair<M, 1, false, false, true>(d, al, ga, ha * sig0, k0, nz, dzf, inv_lz, e0);
                solve_pair<M, 2, false, false, true>(d, al, ga, ha * sig1, k0, nz, dzf, inv_lz, e0);
            }
        } else if (zflags & 1) {
            // Dirichlet wall(s): the wall rows carry the excess W (s_e0); no column is singular
            const double *ex = s_e0 + lane * G::CS;
            const double2 z2 = make_double2(0.0, 0.0);
            if (sig0 == sig1) {
                solve_pair<M, 3, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, z2, z2);
            } else {
                solve_pair<M, 1, false, false, false, true>(d, al, ga, sig0, k0, nz, nullptr, 0.0, ex, z2, z2);
                solve_pair<M, 2, false, false, false, true>(d, al, ga, sig1, k0, nz, nullptr, 0.0, ex, z2, z2);
            }
        } else if (sig0 == sig1) {
            if (no_pad) solve_pair<M, 3, false, true>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
            else solve_pair<M, 3, false>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
        } else {
            // pair 0 of a row: x-modes 0 and nx/2 have different eigenvalues; (0,0) is singular
            if (i == 0 && j == 0 && (zflags & 2))
                solve_pair<M, 1, true>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
            else
                solve_pair<M, 1, false>(d, al, ga, sig0, k0, nz, dzf, inv_lz);
            solve_pair<M, 2, false>(d, al, ga, sig1, k0, nz, dzf, inv_lz);
        }
        fence_proxy_async_smem(); // this lane's shared-memory writes -> visible to the TMA store
        __syncwarp();
        if (lane == 0) mbar_arrive(&done[b]);
    }
}

// nk: rows of the tile (the plan's nz for whole columns, the slab's for MODE 1 / 2)
template <int M, bool HELM, int MODE = 0>
int launch_m(pz_plan *pl, double *p, cudaStream_t st, double ha, int nk, const SlabArgs &sa)
{
    using G = Geo<M>;
    int stages = (int)((227 * 1024 - 1024 - G::COEF - 64) / G::STAGE);
    if (stages > 3) stages = 3;
    if (pl->opt.zsolve_stages > 0 && pl->opt.zsolve_stages < stages) stages = pl->opt.zsolve_stages;
    if (stages < 1) { set_error("z-solve variant 2: nz = %d does not fit shared memory", nk); return PZ_EUNSUPPORTED; }
    const size_t smem = G::bytes(stages);
    const size_t plane = (size_t)pl->nx * pl->ny;
    const int ntiles = (int)(plane / kTX);
    // per plan (= per device): shared-memory opt-in and resident CTAs, queried once
    constexpr int mi = (M == 4) ? 0 : (M == 8) ? 1 : (M == 16) ? 2 : 3;
    pz_plan::ZtGeo &g = pl->zt[mi][HELM ? 1 : (MODE == 0 ? 0 : MODE + 1)];
    if (g.blocks == 0 || g.stages != stages) {
        { const int rc = smem_optin(pl, zsolve_tma_kernel<M, HELM, MODE>, 227 * 1024); if (rc != PZ_OK) return rc; }
        int occ = 1;
        if (smem * 2 <= 227 * 1024) PZ_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, zsolve_tma_kernel<M, HELM, MODE>, kThreads, smem));
        if (occ < 1) occ = 1;
        g.blocks = pl->num_sms * occ;
        g.stages = stages;
    }
    int blocks = g.blocks;
    if (blocks > ntiles) blocks = ntiles;
    const CUtensorMap *mapp = nullptr;
    const int rc = cached_column_map(pl, &mapp, p, plane, nk, kTX, M, 1, /*swizzle128=*/true);
    if (rc != PZ_OK) return rc;
    const CUtensorMap &map = *mapp;
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    zsolve_tma_kernel<M, HELM, MODE><<<blocks, kThreads, smem, st>>>(map, pl->d_A, pl->d_C, pl->d_dzf, pl->d_lamx,
                                                                      pl->d_lamy_nat, pl->d_lamy_pk, pl->nx, pl->ny, nk,
                                                                      pl->inv_lz, ntiles, stages, ha, HELM ? pl->wall_w0 : pl->pw0,
                                                                      HELM ? pl->wall_w1 : pl->pw1, pl->opt.zsolve_probe, sa, pl->zflags());
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace

// helm_a < 0: the Poisson systems; helm_a >= 0: the fully implicit Helmholtz systems with a = helm_a.
int launch_zsolve_tma(pz_plan *pl, double *p, cudaStream_t st, double helm_a)
{
    const int nz = pl->nz;
    const SlabArgs none{};
#define PZ_ZT(MM) (helm_a >= 0.0 ? launch_m<MM, true>(pl, p, st, helm_a, nz, none) : launch_m<MM, false>(pl, p, st, 0.0, nz, none))
    if (nz <= 32 * 4) return PZ_ZT(4);
    if (nz <= 32 * 8) return PZ_ZT(8);
    if (nz <= 32 * 16) return PZ_ZT(16);
    if (nz <= 32 * 32) return PZ_ZT(32);
#undef PZ_ZT
    set_error("z-solve variant 2 supports nz <= 1024 (got %d); use zsolve_variant = 0", nz);
    return PZ_EUNSUPPORTED;
}

// One z-slab [kb, kb + nk) of cut columns through the same pipeline (pz_zslab.cu): p points at the
// slab's first plane.  reduce: boundary values into bout; finish: in place with phi_prev / phi_next.
int launch_zslab_tma(pz_plan *pl, double *p, int kb, int nk, const BoutSet *bout, const double *phi_prev, const double *phi_next,
                     cudaStream_t st)
{
    SlabArgs sa;
    sa.kb = kb; if (bout) sa.bout = *bout; sa.phi_prev = phi_prev; sa.phi_next = phi_next; sa.plane = (size_t)pl->nx * pl->ny;
#define PZ_ZS(MM) (bout ? launch_m<MM, false, 1>(pl, p, st, 0.0, nk, sa) : launch_m<MM, false, 2>(pl, p, st, 0.0, nk, sa))
    if (nk <= 32 * 4) return PZ_ZS(4);
    if (nk <= 32 * 8) return PZ_ZS(8);
    if (nk <= 32 * 16) return PZ_ZS(16);
    if (nk <= 32 * 32) return PZ_ZS(32);
#undef PZ_ZS
    set_error("z-slab: %d planes per slab (at most 1024)", nk);
    return PZ_EUNSUPPORTED;
}

} // namespace pz
