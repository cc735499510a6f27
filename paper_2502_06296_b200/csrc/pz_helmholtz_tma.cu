// pz_helmholtz_tma.cu -- step a6, variant 1 (default): the runtime half of Algorithm 2
// as a persistent, TMA-fed pipeline.
//
// pz_helmholtz.cu explains the pre-processing / runtime split and builds the k-only tables; its
// own kernel (variant 0) loads the column tile straight into registers, which leaves the memory
// system idle while a CTA computes (ncu r01b: 40 % of DRAM peak, L1 wavefront-bound on 64-byte
// rows).  Here one CTA per tile slot stays resident and walks over the column tiles of all n
// fields:
//   * the tile {16 columns x all nz rows} (128-byte rows, zero-filled past nz) is fetched by the
//     TMA unit into shared memory and signalled on an mbarrier;
//   * thread (c, s) copies the m rows of sub-domain s of column c into registers, the CTA
//     synchronises once and thread 0 immediately issues the fetch of the NEXT tile into the same
//     buffer, so loads stay in flight through Steps 2-4 and the stores of this tile;
//   * Step 2 (forward / backward sweeps on d only), Step 3 (boundary system: precomputed
//     parallel-cyclic-reduction multipliers applied through a small shared-memory exchange),
//     Step 4 (reconstruction) run in registers; results go back with coalesced 128-byte stores;
//   * the k-only tables are staged once per CTA in shared memory with a padded stride, so the
//     two sub-domains that share a warp read them without bank conflicts.
// 16 bytes and five FMAs per point; the paper's "store 1/b" makes it division-free.
#include "pz_internal.h"
#include "pz_tma.cuh"

namespace pz {

namespace {

constexpr int kTX = 16;        // columns per tile
constexpr int kMaxFields = 4;  // fields per launch

struct HelmArgs {
    CUtensorMap map[kMaxFields];
    double *u[kMaxFields];
};

template <int M> struct Limits {
    static constexpr int kMaxThreads = 512;                // P <= 32 sub-domains
    static constexpr int kMinBlocks = (M >= 32) ? 1 : 2;   // m = 32 keeps 64 doubles of d + addresses
};

template <int M, bool FULL>
__global__ void __launch_bounds__(Limits<M>::kMaxThreads, Limits<M>::kMinBlocks)
    helmholtz_tma_kernel(const __grid_constant__ HelmArgs args, const double *__restrict__ tab, size_t plane, int nz,
                         int P, int levels, int box_rows, int nbox, int tiles_per_field, int total_tiles)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int TS = M + 1; // padded table stride per sub-domain
    const int nzp = P * M, n2 = 2 * P;
    const int rows_alloc = box_rows * nbox;
    double *tile = reinterpret_cast<double *>(smem_raw);                  // rows_alloc x 16
    double *xch = tile + (size_t)rows_alloc * kTX;                        // 2 buffers x 2 x P x 16
    double *stab = xch + (size_t)2 * n2 * kTX;                            // 5 x P x TS
    uint64_t *bar = reinterpret_cast<uint64_t *>(stab + (size_t)5 * P * TS);

    const int tid = threadIdx.x, c = tid & (kTX - 1), s = tid >> 4;
    const int k0 = s * M;
    const unsigned tile_bytes = (unsigned)rows_alloc * kTX * sizeof(double);

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    for (int q = tid; q < 5 * nzp; q += blockDim.x) {
        const int t = q / nzp, k = q - t * nzp;
        stab[(size_t)t * P * TS + (k / M) * TS + (k % M)] = tab[q];
    }
    __syncthreads();

    auto fetch = [&](int t) {
        const int f = t / tiles_per_field, col0 = (t - f * tiles_per_field) * kTX;
        mbar_arrive_expect_tx(bar, tile_bytes);
        for (int b = 0; b < nbox; ++b) tma_load_2d(tile + (size_t)b * box_rows * kTX, &args.map[f], col0, b * box_rows, bar);
    };

    int t = blockIdx.x;
    if (tid == 0 && t < total_tiles) fetch(t);

    const double *fA = stab + s * TS, *bC = fA + P * TS, *rb = bC + P * TS, *ra = rb + P * TS, *rc = ra + P * TS;
    const double *pcr = tab + 5 * (size_t)nzp;
    const int sm1 = max(s - 1, 0), sp1 = min(s + 1, P - 1);
    unsigned phase = 0;

    for (; t < total_tiles; t += gridDim.x) {
        double d[M];
        mbar_wait(bar, phase);
        phase ^= 1;
#pragma unroll
        for (int i = 0; i < M; ++i) d[i] = tile[(k0 + i) * kTX + c];
        __syncthreads(); // every thread holds its rows: the buffer is free again
        if (tid == 0 && t + (int)gridDim.x < total_tiles) fetch(t + gridDim.x);

        // Step 2: runtime reduction, d only
#pragma unroll
        for (int i = 2; i < M; ++i) d[i] = fma(-fA[i], d[i - 1], d[i]);
#pragma unroll
        for (int i = M - 3; i >= 0; --i) d[i] = fma(-bC[i], d[i + 1], d[i]);

        // Step 3: boundary system.  Row 2s = first row of sub-domain s (x0), row 2s+1 = last (x1);
        // shared layout [buffer][first/last][s][c].
        double x0 = d[0], x1 = d[M - 1];
        double *cur = xch, *nxt = xch + (size_t)n2 * kTX;
        cur[(s)*kTX + c] = x0;
        cur[(P + s) * kTX + c] = x1;
        __syncthreads();
        {
            // level 0 (h = 1): partners of x0 are (x1 of s-1, own x1), of x1 (own x0, x0 of s+1)
            const double2 ka = __ldg(reinterpret_cast<const double2 *>(pcr) + 2 * s);
            const double2 kb = __ldg(reinterpret_cast<const double2 *>(pcr) + 2 * s + 1);
            const double n0 = fma(ka.x, cur[(P + sm1) * kTX + c], fma(ka.y, x1, x0));
            const double n1 = fma(kb.x, x0, fma(kb.y, cur[sp1 * kTX + c], x1));
            x0 = n0;
            x1 = n1;
        }
        for (int l = 1, hs = 1; l < levels; ++l, hs *= 2) {
            nxt[s * kTX + c] = x0;
            nxt[(P + s) * kTX + c] = x1;
            __syncthreads();
            double *tmp = cur; cur = nxt; nxt = tmp;
            const double2 ka = __ldg(reinterpret_cast<const double2 *>(pcr + (size_t)l * 2 * n2) + 2 * s);
            const double2 kb = __ldg(reinterpret_cast<const double2 *>(pcr + (size_t)l * 2 * n2) + 2 * s + 1);
            const int sa = max(s - hs, 0), sb = min(s + hs, P - 1);
            x0 = fma(ka.x, cur[sa * kTX + c], fma(ka.y, cur[sb * kTX + c], x0));
            x1 = fma(kb.x, cur[(P + sa) * kTX + c], fma(kb.y, cur[(P + sb) * kTX + c], x1));
        }
        {
            const double2 rbr = __ldg(reinterpret_cast<const double2 *>(pcr + (size_t)levels * 2 * n2) + s);
            x0 *= rbr.x;
            x1 *= rbr.y;
        }

        // Step 4: reconstruct and store
        const int f = t / tiles_per_field;
        double *up = args.u[f] + (size_t)(t - f * tiles_per_field) * kTX + c + (size_t)k0 * plane;
        if (FULL || k0 < nz) up[0] = x0;
#pragma unroll
        for (int i = 1; i < M - 1; ++i) {
            const double v = fma(-rc[i], x1, fma(-ra[i], x0, rb[i] * d[i]));
            if (FULL || k0 + i < nz) up[(size_t)i * plane] = v;
        }
        if (FULL || k0 + M - 1 < nz) up[(size_t)(M - 1) * plane] = x1;
    }
}

template <int M>
size_t smem_bytes(int P)
{
    const int nzp = P * M, box_rows = nzp <= 256 ? nzp : 256, nbox = (nzp + box_rows - 1) / box_rows;
    return ((size_t)box_rows * nbox * kTX + (size_t)2 * 2 * P * kTX + (size_t)5 * P * (M + 1)) * sizeof(double) + 16;
}

template <int M, bool FULL>
int prepare_mf(pz_plan *pl)
{
    const size_t smem = smem_bytes<M>(pl->helm_P);
    auto kern = helmholtz_tma_kernel<M, FULL>;
    if (smem > 227 * 1024) { set_error("helmholtz (TMA variant): tile of %zu bytes does not fit shared memory", smem); return PZ_EUNSUPPORTED; }
    PZ_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    int bps = 0;
    PZ_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, kTX * pl->helm_P, smem));
    if (bps < 1) { set_error("helmholtz (TMA variant): kernel does not fit an SM"); return PZ_ECUDA; }
    pl->helm_bps = bps;
    return PZ_OK;
}

template <int M, bool FULL>
int launch_mf(pz_plan *pl, double *const *u, int n, const double *tab, cudaStream_t st)
{
    const int P = pl->helm_P, nzp = P * M;
    const int box_rows = nzp <= 256 ? nzp : 256;
    const int nbox = (nzp + box_rows - 1) / box_rows;
    const size_t plane = (size_t)pl->nx * pl->ny;
    const size_t smem = smem_bytes<M>(P);
    HelmArgs args;
    for (int f = 0; f < n; ++f) {
        const int rc = encode_column_tile_map(&args.map[f], u[f], plane, pl->nz, kTX, box_rows);
        if (rc != PZ_OK) return rc;
        args.u[f] = u[f];
    }
    for (int f = n; f < kMaxFields; ++f) { args.map[f] = args.map[0]; args.u[f] = u[0]; }
    const int tiles_per_field = (int)(plane / kTX);
    const long long total = (long long)tiles_per_field * n;
    long long blocks = (long long)pl->num_sms * pl->helm_bps;
    if (blocks > total) blocks = total;
    helmholtz_tma_kernel<M, FULL><<<(unsigned)blocks, kTX * P, smem, st>>>(args, tab, plane, pl->nz, P, pl->helm_levels,
                                                                            box_rows, nbox, tiles_per_field, (int)total);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace

// Called when the launch geometry (m, P) changes: shared-memory opt-in and resident CTAs per SM.
int helmholtz_tma_prepare(pz_plan *pl)
{
    const bool full = (pl->helm_P * pl->helm_m == pl->nz);
#define PZ_HP(MM) (full ? prepare_mf<MM, true>(pl) : prepare_mf<MM, false>(pl))
    switch (pl->helm_m) {
    case 4: return PZ_HP(4);
    case 8: return PZ_HP(8);
    case 16: return PZ_HP(16);
    case 32: return PZ_HP(32);
    default: set_error("helmholtz: bad sub-domain size %d", pl->helm_m); return PZ_EINVAL;
    }
#undef PZ_HP
}

// n <= 4 fields in one persistent launch.  The caller (launch_helmholtz_n) has ordered the stream
// after the table upload and records the table's last use.
int launch_helmholtz_tma(pz_plan *pl, double *const *u, int n, const double *tab, cudaStream_t st)
{
    if (n < 1 || n > kMaxFields) { set_error("helmholtz (TMA variant): 1..4 fields per launch"); return PZ_EINVAL; }
    const bool full = (pl->helm_P * pl->helm_m == pl->nz);
#define PZ_HT(MM) (full ? launch_mf<MM, true>(pl, u, n, tab, st) : launch_mf<MM, false>(pl, u, n, tab, st))
    switch (pl->helm_m) {
    case 4: return PZ_HT(4);
    case 8: return PZ_HT(8);
    case 16: return PZ_HT(16);
    case 32: return PZ_HT(32);
    default: set_error("helmholtz: bad sub-domain size %d", pl->helm_m); return PZ_EINVAL;
    }
#undef PZ_HT
}

} // namespace pz
