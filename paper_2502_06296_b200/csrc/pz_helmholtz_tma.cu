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
//   * thread (cp, s) copies the m rows of sub-domain s of the column PAIR cp into registers with
//     16-byte shared-memory loads (one k-only table value then serves two points and every load /
//     store instruction moves 16 bytes: with one column per thread the kernel is bound by LSU
//     instruction issue, ncu r01c), the CTA synchronises once and thread 0 immediately issues
//     the fetch of the NEXT tile into the same buffer, so loads stay in flight through Steps 2-4
//     and the stores of this tile;
//   * Step 2 (forward / backward sweeps on d only), Step 3 (boundary system: precomputed
//     parallel-cyclic-reduction multipliers applied through a small shared-memory exchange),
//     Step 4 (reconstruction) run in registers; results go back with 16-byte stores, 128
//     contiguous bytes per 8 lanes;
//   * the k-only tables and the PCR multipliers are staged once per CTA in shared memory; the
//     table stride per sub-domain is padded so that the four sub-domains of a warp hit different
//     bank groups.
// 16 bytes and five FMAs per point; the paper's "store 1/b" makes it division-free.
#include "pz_internal.h"
#include "pz_tma.cuh"

namespace pz {

namespace {

constexpr int kTX = 16;        // columns per tile (32 in the wide variant: 256-byte rows)
constexpr int kMaxFields = 4;  // fields per launch

struct HelmArgs {
    CUtensorMap map[kMaxFields];
    double *u[kMaxFields];
    // CN mode (helmholtz_z_step, one field): tiles of u^k and what the operator L_z needs
    CUtensorMap qmap;
    const double *q;
    const double *A, *C;
    double a, w0, w1;
};

__host__ __device__ constexpr int nzp_of(int P, int M) { return P * M; }

template <int M> struct Limits {
    static constexpr int kMaxThreads = 512;                // 8 column pairs x P <= 64 sub-domains
    static constexpr int kMinBlocks = (M >= 16) ? 1 : 2;   // m = 16: 2 x 16 doubles of d per thread
};

__device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void st2(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }
__device__ __forceinline__ void st2g(double *p, double2 v) { __stcs(reinterpret_cast<double2 *>(p), v); }

// Shared-memory carve-up in doubles; host and device agree through these helpers.
template <int M, int TX = kTX, int ZS = 1> struct Smem {
    static constexpr int kTX = TX;
    static constexpr int TS = M + 2; // table stride per sub-domain: even (16-byte pairs)
    // as few boxes of at most 256 rows as cover the P M rows, all of one size (a multiple of 8 rows)
    __host__ __device__ static int nbox(int P) { return (P * M + 255) / 256; }
    __host__ __device__ static int box_rows(int P) { return (((P * M + nbox(P) - 1) / nbox(P)) + 7) & ~7; }
    __host__ __device__ static size_t tile(int P) { return (size_t)box_rows(P) * nbox(P) * kTX; }
    __host__ __device__ static size_t xch(int P) { return (size_t)2 * 2 * P * kTX; }
    __host__ __device__ static size_t tab(int P) { return (size_t)(ZS > 2 ? 7 : ZS > 1 ? 6 : 5) * P * TS; }   // 6th / 7th table: z-split corrections
    __host__ __device__ static size_t pcr(int P, int levels) { return (size_t)levels * 4 * P + 2 * P; }
    // z-split interface values: ZS = 2 [parity][own / peer][TX]; ZS = 4 [parity][chunk][first / last][TX]
    __host__ __device__ static size_t zx() { return ZS > 2 ? (size_t)2 * ZS * 2 * TX : ZS > 1 ? (size_t)2 * 2 * TX : 0; }
    __host__ __device__ static size_t bytes(int P, int levels, bool cn = false)
    {
        return ((cn ? 2 : 1) * tile(P) + xch(P) + tab(P) + pcr(P, levels) + zx()) * sizeof(double) + 16;
    }
};

// Thread (cp, s): columns (2cp, 2cp+1) of the tile, sub-domain s (rows s*M .. s*M+M-1).
// CN: the whole of Eq. (11), PAPER.md:76 -- a second tile holds u^k and the right-hand side
// u** - a L_z u^k is formed in registers while the rows are copied out (the separate pass of
// helmholtz_z_rhs and its 16 B/point round trip disappear); one CTA per SM.
// ZS = 2: the column is cut into two chunks of P sub-domains each, owned by the two CTAs of a
// cluster (PAPER.md:120-135 with CTAs for MPI tasks): each solves its chunk with the couplings
// across the cut removed (tables of that chunk), the two interface values cross through
// distributed shared memory, and the reconstruction adds the precomputed k-only correction.
template <int M, bool FULL, int CN, int TX = 16, int ZS = 1>
__global__ void __launch_bounds__(Limits<M>::kMaxThreads, CN != 0 ? 1 : Limits<M>::kMinBlocks)
    helmholtz_tma_kernel(const __grid_constant__ HelmArgs args, const double *__restrict__ tab_all, size_t plane, int nz,
                         int P, int levels, int tiles_per_field, int total_tiles, int probe, int box_rows, int nbox, int csz,
                         size_t cstride)
{
    static_assert(ZS == 1 || CN == 0, "the fused step kernel takes whole columns");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    using L = Smem<M, TX, ZS>;
    constexpr int TS = L::TS;
    constexpr int kTX = TX; // shadows the file-level default
    const int nzp = P * M, n2 = 2 * P;
    double *tile = reinterpret_cast<double *>(smem_raw);   // rows x 16
    double *qtile = tile + L::tile(P);                     // CN only: rows x 16 of u^k
    double *xch = qtile + (CN == 1 ? L::tile(P) : 0);           // [buffer][first/last][s][16]
    double *stab = xch + L::xch(P);                        // [table][s][TS]
    double *spcr = stab + L::tab(P);                       // [level][s][4], then [s][2]
    double *zx = spcr + L::pcr(P, levels);                 // ZS = 2: interface values [parity][own / peer][TX]
    uint64_t *bar = reinterpret_cast<uint64_t *>(zx + L::zx());

    const int tid = threadIdx.x, c2 = 2 * (tid % (TX / 2)), s = tid / (TX / 2);
    // z-split: chunk of this CTA (rank in the cluster), its first global row and its table block
    // cluster of csz = ZS * TP CTAs: rank = tp * ZS + chunk; TP neighbouring tiles walk in step
    const int cl_rank = (ZS > 1) ? (int)(blockIdx.x % csz) : 0;
    const int crank = cl_rank % ZS, ctile = cl_rank / ZS, TP = (ZS > 1) ? csz / ZS : 1;
    const int kc0 = crank * nzp_of(P, M);
    const double *tab = tab_all + (size_t)crank * cstride;
    const int k0 = s * M;                                  // row inside the chunk
    const unsigned tile_bytes = (unsigned)((CN == 1 ? 2 : 1) * L::tile(P) * sizeof(double));

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    for (int q = tid; q < 5 * nzp; q += blockDim.x) {
        const int t = q / nzp, k = q - t * nzp;
        stab[(size_t)t * P * TS + (k / M) * TS + (k % M)] = tab[q];
    }
    for (int q = tid; q < (int)L::pcr(P, levels); q += blockDim.x) spcr[q] = tab[5 * (size_t)nzp + q];
    double w_own = 0.0, w_peer = 0.0;
    double wP[ZS > 2 ? 2 * ZS : 1], wN[ZS > 2 ? 2 * ZS : 1]; // ZS = 4: weights of the 2 ZS end values of y
    if constexpr (ZS == 2) {
        const double *corr = tab + 5 * (size_t)nzp + L::pcr(P, levels);
        for (int k = tid; k < nzp; k += blockDim.x) stab[(size_t)5 * P * TS + (k / M) * TS + (k % M)] = corr[k];
        w_own = corr[nzp];
        w_peer = corr[nzp + 1];
    } else if constexpr (ZS > 2) {
        const double *corr = tab + 5 * (size_t)nzp + L::pcr(P, levels);
        for (int k = tid; k < 2 * nzp; k += blockDim.x) {
            const int t6 = k / nzp, kk = k - t6 * nzp;
            stab[(size_t)(5 + t6) * P * TS + (kk / M) * TS + (kk % M)] = corr[k];
        }
#pragma unroll
        for (int q = 0; q < 2 * ZS; ++q) { wP[q] = corr[2 * nzp + q]; wN[q] = corr[2 * nzp + 2 * ZS + q]; }
    }
    __syncthreads();

    const uint64_t pol = l2_policy_evict_first(); // every tile is read once
    auto fetch = [&](int t) {
        const int f = t / tiles_per_field, tt = t - f * tiles_per_field, col0 = tt * kTX;
        mbar_arrive_expect_tx(bar, tile_bytes);
        if (kProbes && probe == 3) { // diagnostic: same bytes fetched as 32-column boxes (256-byte rows)
            for (int b = 0; b < nbox; ++b)
                tma_load_2d(tile + (size_t)b * box_rows * 32, &args.map[f], (tt >> 1) * 32, (tt & 1) * (nzp / 2) + b * box_rows, bar);
            return;
        }
        for (int b = 0; b < nbox; ++b)
            tma_load_2d_hint(tile + (size_t)b * box_rows * kTX, &args.map[f], col0, kc0 + b * box_rows, bar, pol);
        if constexpr (CN == 1)
            for (int b = 0; b < nbox; ++b)
                tma_load_2d_hint(qtile + (size_t)b * box_rows * kTX, &args.qmap, col0, b * box_rows, bar, pol);
    };

    // tiles walk by CTA (ZS = 1) or by cluster (ZS = 2: both CTAs own the same columns)
    const int tstep = (ZS > 1) ? ((int)gridDim.x / csz) * TP : (int)gridDim.x;
    int t = (ZS > 1) ? ((int)blockIdx.x / csz) * TP + ctile : (int)blockIdx.x;
    if (tid == 0 && t < total_tiles) fetch(t);

    const double *fA = stab + s * TS, *bC = fA + P * TS, *rb = bC + P * TS, *ra = rb + P * TS, *rc = ra + P * TS;
    const int sm1 = max(s - 1, 0), sp1 = min(s + 1, P - 1);
    unsigned phase = 0;

    const double *rx = stab + (size_t)5 * P * TS + s * TS; // ZS = 2: correction per row
    int zpar = 0;
    for (; t < total_tiles; t += tstep) {
        double da[M], db[M]; // the two columns
        mbar_wait(bar, phase);
        phase ^= 1;
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double2 v = ld2(tile + (k0 + i) * kTX + c2);
            da[i] = v.x;
            db[i] = v.y;
        }
        if constexpr (CN != 0) {
            // d <- u** - a L_z u^k, (L_z q)_k = A_k (q_{k-1} - q_k) + C_k (q_{k+1} - q_k) - W_k q_k.
            // CN == 1: u^k from the second shared-memory tile; CN == 2 (the tile pair does not fit):
            // straight from global memory, row stride `plane`.
            const size_t qs = (CN == 1) ? (size_t)kTX : plane;
            const double *qt = (CN == 1) ? qtile + c2 : args.q + (size_t)t * kTX + c2;
            double2 qm = make_double2(0.0, 0.0), qc = make_double2(0.0, 0.0);
            if (FULL || k0 < nz) qc = ld2(qt + k0 * qs);
            if (k0 > 0 && (FULL || k0 - 1 < nz)) qm = ld2(qt + (k0 - 1) * qs);
#pragma unroll
            for (int i = 0; i < M; ++i) {
                const int k = k0 + i;
                double2 qn = make_double2(0.0, 0.0);
                if (k + 1 < nz) qn = ld2(qt + (k + 1) * qs);
                if (FULL || k < nz) {
                    double2 lz = make_double2(0.0, 0.0);
                    if (k > 0) {
                        const double ak = __ldg(args.A + k);
                        lz.x += ak * (qm.x - qc.x);
                        lz.y += ak * (qm.y - qc.y);
                    }
                    if (k + 1 < nz) {
                        const double ck = __ldg(args.C + k);
                        lz.x += ck * (qn.x - qc.x);
                        lz.y += ck * (qn.y - qc.y);
                    }
                    const double wk = (k == 0 ? args.w0 : 0.0) + (k == nz - 1 ? args.w1 : 0.0);
                    lz.x -= wk * qc.x;
                    lz.y -= wk * qc.y;
                    da[i] -= args.a * lz.x;
                    db[i] -= args.a * lz.y;
                }
                qm = qc;
                qc = qn;
            }
        }
        // every thread holds its rows: the buffer is free again.  With a cluster (csz > 1) the
        // CTAs of the cluster, which own neighbouring tiles, also meet here, so that their next
        // fetches (and their stores) reach DRAM together as 128*csz contiguous bytes per row.
        if (csz > 1 && ZS == 1) {
            asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
        } else {
            __syncthreads();
        }
        if (tid == 0 && t + tstep < total_tiles) fetch(t + tstep);

        if (kProbes && probe == 2) { // diagnostic: pipeline skeleton only (load, store)
            const int f = t / tiles_per_field;
            double *up = args.u[f] + (size_t)(t - f * tiles_per_field) * kTX + c2 + (size_t)(kc0 + k0) * plane;
#pragma unroll
            for (int i = 0; i < M; ++i)
                if (FULL || kc0 + k0 + i < nz) st2g(up + (size_t)i * plane, make_double2(da[i], db[i]));
            continue;
        }
        // Step 2: runtime reduction, d only (forward i = 2..M-1, backward i = M-3..0)
#pragma unroll
        for (int i = 2; i < M; i += 2) {
            const double2 f = ld2(fA + i);
            da[i] = fma(-f.x, da[i - 1], da[i]);
            db[i] = fma(-f.x, db[i - 1], db[i]);
            da[i + 1] = fma(-f.y, da[i], da[i + 1]);
            db[i + 1] = fma(-f.y, db[i], db[i + 1]);
        }
#pragma unroll
        for (int i = M - 4; i >= 0; i -= 2) {
            const double2 g = ld2(bC + i);
            da[i + 1] = fma(-g.y, da[i + 2], da[i + 1]);
            db[i + 1] = fma(-g.y, db[i + 2], db[i + 1]);
            da[i] = fma(-g.x, da[i + 1], da[i]);
            db[i] = fma(-g.x, db[i + 1], db[i]);
        }

        // Step 3: boundary system.  Row 2s = first row of sub-domain s (x0), row 2s+1 = last (x1).
        double2 x0 = make_double2(da[0], db[0]), x1 = make_double2(da[M - 1], db[M - 1]);
        double *cur = xch, *nxt = xch + (size_t)n2 * kTX;
        st2(cur + s * kTX + c2, x0);
        st2(cur + (P + s) * kTX + c2, x1);
        __syncthreads();
        {
            // level 0 (h = 1): partners of x0 are (x1 of s-1, own x1), of x1 (own x0, x0 of s+1)
            const double2 ka = ld2(spcr + 4 * s), kb = ld2(spcr + 4 * s + 2);
            const double2 pm = ld2(cur + (P + sm1) * kTX + c2), pp = ld2(cur + sp1 * kTX + c2);
            const double2 n0 = make_double2(fma(ka.x, pm.x, fma(ka.y, x1.x, x0.x)), fma(ka.x, pm.y, fma(ka.y, x1.y, x0.y)));
            const double2 n1 = make_double2(fma(kb.x, x0.x, fma(kb.y, pp.x, x1.x)), fma(kb.x, x0.y, fma(kb.y, pp.y, x1.y)));
            x0 = n0;
            x1 = n1;
        }
        for (int l = 1, hs = 1; l < levels; ++l, hs *= 2) {
            st2(nxt + s * kTX + c2, x0);
            st2(nxt + (P + s) * kTX + c2, x1);
            __syncthreads();
            double *tmp = cur; cur = nxt; nxt = tmp;
            const double *kk = spcr + (size_t)l * 4 * P + 4 * s;
            const double2 ka = ld2(kk), kb = ld2(kk + 2);
            const int sa = max(s - hs, 0), sb = min(s + hs, P - 1);
            const double2 am = ld2(cur + sa * kTX + c2), ap = ld2(cur + sb * kTX + c2);
            const double2 bm = ld2(cur + (P + sa) * kTX + c2), bp = ld2(cur + (P + sb) * kTX + c2);
            x0.x = fma(ka.x, am.x, fma(ka.y, ap.x, x0.x));
            x0.y = fma(ka.x, am.y, fma(ka.y, ap.y, x0.y));
            x1.x = fma(kb.x, bm.x, fma(kb.y, bp.x, x1.x));
            x1.y = fma(kb.x, bm.y, fma(kb.y, bp.y, x1.y));
        }
        {
            const double2 rbr = ld2(spcr + (size_t)levels * 4 * P + 2 * s);
            x0.x *= rbr.x; x0.y *= rbr.x;
            x1.x *= rbr.y; x1.y *= rbr.y;
        }

        // z-split: x0 / x1 are the chunk-local solution y at the sub-domain ends.  The chunk's
        // interface value (last row of chunk 0, first row of chunk 1) goes to both CTAs; the value
        // of the neighbouring chunk's interface row follows from the precomputed 2 x 2 system.
        double2 X = make_double2(0.0, 0.0), Xn = make_double2(0.0, 0.0);
        if constexpr (ZS > 2) {
            // every chunk's first and last value of y go to all CTAs of the cluster; the values of the
            // neighbouring chunks' interface rows are precomputed linear combinations of them
            double *slot = zx + (size_t)zpar * (ZS * 2 * TX);
            const int cbase = (cl_rank / ZS) * ZS;
            if (s == 0 || s == P - 1) {
#pragma unroll
                for (int r = 0; r < ZS; ++r) {
                    if (s == 0) {
                        unsigned ra;
                        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(slot + (crank * 2 + 0) * TX + c2)), "r"(cbase + r));
                        asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(ra), "d"(x0.x), "d"(x0.y) : "memory");
                    }
                    if (s == P - 1) {
                        unsigned ra;
                        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(slot + (crank * 2 + 1) * TX + c2)), "r"(cbase + r));
                        asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(ra), "d"(x1.x), "d"(x1.y) : "memory");
                    }
                }
            }
            asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
#pragma unroll
            for (int r = 0; r < ZS; ++r) {
                const double2 yf = ld2(slot + (r * 2 + 0) * TX + c2), yl = ld2(slot + (r * 2 + 1) * TX + c2);
                X.x = fma(wP[r], yf.x, fma(wP[ZS + r], yl.x, X.x));
                X.y = fma(wP[r], yf.y, fma(wP[ZS + r], yl.y, X.y));
                Xn.x = fma(wN[r], yf.x, fma(wN[ZS + r], yl.x, Xn.x));
                Xn.y = fma(wN[r], yf.y, fma(wN[ZS + r], yl.y, Xn.y));
            }
            zpar ^= 1;
        } else if constexpr (ZS > 1) {
            double *slot = zx + (size_t)zpar * 2 * TX;
            if ((crank == 0 && s == P - 1) || (crank == 1 && s == 0)) {
                const double2 mine = (crank == 0) ? x1 : x0;
                st2(slot + c2, mine);
                unsigned remote;
                asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(slot + TX + c2)), "r"(cl_rank ^ 1));
                asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(remote), "d"(mine.x), "d"(mine.y) : "memory");
            }
            // (an st.async + mbarrier hand-over without this barrier was measured SLOWER, 1.17 against
            // 1.08 ms at 512^3 x 3: the barrier also keeps the two CTAs' fetches and stores in step)
            asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
            const double2 own = ld2(slot + c2), peer = ld2(slot + TX + c2);
            X = make_double2(fma(w_own, own.x, w_peer * peer.x), fma(w_own, own.y, w_peer * peer.y));
            zpar ^= 1;
        }

        // Step 4: reconstruct and store
        if (kProbes && (probe == 1 || probe == 3) && x0.x != 1.2345e300) continue; // diagnostic: no stores
        const int f = t / tiles_per_field;
        double *up = args.u[f] + (size_t)(t - f * tiles_per_field) * kTX + c2 + (size_t)(kc0 + k0) * plane;
#pragma unroll
        for (int i = 0; i < M; i += 2) {
            const double2 qb = ld2(rb + i), qa = ld2(ra + i), qc = ld2(rc + i);
            double2 v, w;
            if (i == 0) {
                v = x0;
            } else {
                v.x = fma(-qc.x, x1.x, fma(-qa.x, x0.x, qb.x * da[i]));
                v.y = fma(-qc.x, x1.y, fma(-qa.x, x0.y, qb.x * db[i]));
            }
            if (i + 1 == M - 1) {
                w = x1;
            } else {
                w.x = fma(-qc.y, x1.x, fma(-qa.y, x0.x, qb.y * da[i + 1]));
                w.y = fma(-qc.y, x1.y, fma(-qa.y, x0.y, qb.y * db[i + 1]));
            }
            if constexpr (ZS > 1) {
                const double2 cr = ld2(rx + i);
                v.x = fma(-cr.x, X.x, v.x); v.y = fma(-cr.x, X.y, v.y);
                w.x = fma(-cr.y, X.x, w.x); w.y = fma(-cr.y, X.y, w.y);
            }
            if constexpr (ZS > 2) {
                const double2 cn = ld2(rx + (size_t)P * TS + i);
                v.x = fma(-cn.x, Xn.x, v.x); v.y = fma(-cn.x, Xn.y, v.y);
                w.x = fma(-cn.y, Xn.x, w.x); w.y = fma(-cn.y, Xn.y, w.y);
            }
            if (FULL || kc0 + k0 + i < nz) st2g(up + (size_t)i * plane, v);
            if (FULL || kc0 + k0 + i + 1 < nz) st2g(up + (size_t)(i + 1) * plane, w);
        }
    }
    // no CTA of the cluster leaves while its peer may still write into its shared memory
    if constexpr (ZS > 1) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int M, bool FULL, int TX = kTX, int ZS = 1>
int prepare_mf(pz_plan *pl)
{
    const size_t smem = Smem<M, TX, ZS>::bytes(pl->helm_P, pl->helm_levels);
    auto kern = helmholtz_tma_kernel<M, FULL, 0, TX, ZS>;
    if (smem > 227 * 1024) { set_error("helmholtz (TMA variant): tile of %zu bytes does not fit shared memory", smem); return PZ_EUNSUPPORTED; }
    {
        const int rc = smem_optin(pl, kern, 227 * 1024);
        if (rc != PZ_OK) return rc;
    }
    int bps = 0;
    PZ_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, (TX / 2) * pl->helm_P, smem));
    if (bps < 1) { set_error("helmholtz (TMA variant): kernel does not fit an SM"); return PZ_ECUDA; }
    pl->helm_bps = bps;
    pl->helm_nclusters[0] = pl->helm_nclusters[1] = pl->helm_nclusters[2] = 0;
    return PZ_OK;
}

template <int M, bool FULL, int TX = kTX, int ZS = 1>
int launch_mf(pz_plan *pl, double *const *u, int n, const double *tab, cudaStream_t st)
{
    constexpr int kTX = TX; // shadows the file-level default
    const int P = pl->helm_P;
    const size_t plane = (size_t)pl->nx * pl->ny;
    const size_t smem = Smem<M, TX, ZS>::bytes(P, pl->helm_levels);
    const bool wide = (pl->opt.helm_probe == 3) && (P * M) % 512 == 0 && TX == 16;
    int box_rows = Smem<M, TX>::box_rows(P), nbox = Smem<M, TX>::nbox(P);
    if (pl->opt.helm_box_rows > 0 && (P * M) % pl->opt.helm_box_rows == 0 && pl->opt.helm_box_rows <= 256) {
        box_rows = pl->opt.helm_box_rows;
        nbox = P * M / box_rows;
    }
    if (wide) { box_rows = 256; nbox = P * M / 512; }
    HelmArgs args;
    for (int f = 0; f < n; ++f) {
        const CUtensorMap *mf = nullptr;
        const int rc = cached_column_map(pl, &mf, u[f], plane, pl->nz, wide ? 32 : kTX, box_rows, pl->opt.helm_l2promo, false);
        if (rc != PZ_OK) return rc;
        args.map[f] = *mf;
        args.u[f] = u[f];
    }
    for (int f = n; f < kMaxFields; ++f) { args.map[f] = args.map[0]; args.u[f] = u[0]; }
    const int tiles_per_field = (int)(plane / kTX);
    const long long total = (long long)tiles_per_field * n;
    long long blocks = (long long)pl->num_sms * pl->helm_bps;
    if (blocks > total * ZS) blocks = total * ZS;
    // CTAs of a cluster own neighbouring tiles and meet once per tile, so their fetches and stores
    // reach DRAM together (256 contiguous bytes per row for a pair).  Measured (profiles/r01c):
    // +15-20 % with m = 16, a loss with the smaller sub-domains (two or more CTAs per SM).
    int csz = pl->opt.helm_cluster;
    if (csz == 0) csz = (M == 16) ? 2 : 1;
    if (csz != 2 && csz != 4 && csz != 8) csz = 1;
    while (csz > 1 && (tiles_per_field % csz != 0 || blocks < csz)) csz /= 2;
    if (ZS > 1) {
        // the cluster is the pair of chunks of one tile; helm_cluster = 4 adds a neighbouring tile in
        // step (measured slower: 1.18 against 1.10 ms at 512^3 x 3, 10.0 against 9.0 ms at 1024^3 x 3)
        const int tp = (pl->opt.helm_cluster == 4 && total % 2 == 0) ? 2 : 1;
        csz = ZS * tp;
    }
    const int probe = wide ? 3 : (pl->opt.helm_probe == 3 ? 1 : pl->opt.helm_probe);
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3((kTX / 2) * P);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = csz;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (csz > 1) {
        // resident clusters: queried once per geometry (helmholtz_tma_prepare resets it)
        if (pl->helm_nclusters[csz == 2 ? 0 : csz == 4 ? 1 : 2] == 0) {
            cfg.gridDim = dim3((unsigned)((long long)pl->num_sms * pl->helm_bps / csz * csz));
            int nclusters = 0;
            PZ_CUDA(cudaOccupancyMaxActiveClusters(&nclusters, helmholtz_tma_kernel<M, FULL, 0, TX, ZS>, &cfg));
            if (nclusters < 1) { set_error("helmholtz (TMA variant): no cluster of %d CTAs fits", csz); return PZ_ECUDA; }
            pl->helm_nclusters[csz == 2 ? 0 : csz == 4 ? 1 : 2] = nclusters;
        }
        const int nclusters = pl->helm_nclusters[csz == 2 ? 0 : csz == 4 ? 1 : 2];
        if ((long long)nclusters * csz < blocks) blocks = (long long)nclusters * csz;
    }
    blocks = blocks / csz * csz;
    cfg.gridDim = dim3((unsigned)blocks);
    PZ_CUDA(cudaLaunchKernelEx(&cfg, helmholtz_tma_kernel<M, FULL, 0, TX, ZS>, args, tab, plane, pl->nz, P, pl->helm_levels,
                               tiles_per_field, (int)total, probe, box_rows, nbox, csz, pl->helm_cstride));
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

// helmholtz_z_step: one field, u** in u2 (in place), u^k in uk.  Returns PZ_EUNSUPPORTED when the two
// tiles do not fit shared memory (the caller then runs the right-hand side as a separate pass).
template <int M, bool FULL, int CN>
int launch_cn_mfc(pz_plan *pl, double *u2, const double *uk, const double *tab, cudaStream_t st)
{
    const int P = pl->helm_cn_P;
    const size_t plane = (size_t)pl->nx * pl->ny;
    const size_t smem = Smem<M>::bytes(P, pl->helm_cn_levels, CN == 1);
    auto kern = helmholtz_tma_kernel<M, FULL, CN>;
    int rc = smem_optin(pl, kern, 227 * 1024);
    if (rc != PZ_OK) return rc;
    const int box_rows = Smem<M>::box_rows(P), nbox = Smem<M>::nbox(P);
    HelmArgs args;
    const CUtensorMap *m0 = nullptr, *m1 = nullptr;
    if ((rc = cached_column_map(pl, &m0, u2, plane, pl->nz, kTX, box_rows, pl->opt.helm_l2promo, false)) != PZ_OK) return rc;
    args.map[0] = *m0;
    if ((rc = cached_column_map(pl, &m1, uk, plane, pl->nz, kTX, box_rows, pl->opt.helm_l2promo, false)) != PZ_OK) return rc;
    args.qmap = *m1;
    for (int f = 0; f < kMaxFields; ++f) { args.map[f] = args.map[0]; args.u[f] = u2; }
    args.q = uk;
    args.A = pl->d_A; args.C = pl->d_C; args.a = pl->helm_a; args.w0 = pl->wall_w0; args.w1 = pl->wall_w1;
    const int tiles = (int)(plane / kTX);
    int blocks = pl->num_sms < tiles ? pl->num_sms : tiles;
    kern<<<blocks, (kTX / 2) * P, smem, st>>>(args, tab + pl->helm_cn_off, plane, pl->nz, P, pl->helm_cn_levels, tiles, tiles, 0, box_rows, nbox, 1,
                                              (size_t)0);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

// helmholtz_z_step: one field, u** in u2 (in place), u^k in uk.  u^k comes through a second
// shared-memory tile where the pair fits, from global memory otherwise.
template <int M, bool FULL>
int launch_cn_mf(pz_plan *pl, double *u2, const double *uk, const double *tab, cudaStream_t st)
{
    if (Smem<M>::bytes(pl->helm_cn_P, pl->helm_cn_levels, true) <= 227 * 1024 && pl->opt.step_fused != 2)
        return launch_cn_mfc<M, FULL, 1>(pl, u2, uk, tab, st);
    if (Smem<M>::bytes(pl->helm_cn_P, pl->helm_cn_levels, false) > 227 * 1024) return PZ_EUNSUPPORTED;
    return launch_cn_mfc<M, FULL, 2>(pl, u2, uk, tab, st);
}

} // namespace

int launch_helmholtz_tma_cn(pz_plan *pl, double *u2, const double *uk, const double *tab, cudaStream_t st)
{
    if (pl->helm_cn_P <= 0) return PZ_EUNSUPPORTED; // no whole-column tables (nz > 1024): the caller runs the right-hand side as its own pass
    const bool full = (pl->helm_cn_P * pl->helm_m == pl->nz);
#define PZ_HC(MM) (full ? launch_cn_mf<MM, true>(pl, u2, uk, tab, st) : launch_cn_mf<MM, false>(pl, u2, uk, tab, st))
    switch (pl->helm_m) {
    case 4: return PZ_HC(4);
    case 8: return PZ_HC(8);
    case 16: return PZ_HC(16);
    default: return PZ_EUNSUPPORTED;
    }
#undef PZ_HC
}

// Called when the launch geometry (m, P) changes: shared-memory opt-in and resident CTAs per SM.
int helmholtz_tma_prepare(pz_plan *pl)
{
    const bool full = (pl->helm_zs * pl->helm_P * pl->helm_m == pl->nz);
#define PZ_HP(MM) (full ? prepare_mf<MM, true>(pl) : prepare_mf<MM, false>(pl))
    switch (pl->helm_m) {
    case 4: return PZ_HP(4);
    case 8: return PZ_HP(8);
    case 16:
        if (pl->helm_zs == 4 && pl->helm_tx == 64) return full ? prepare_mf<16, true, 64, 4>(pl) : prepare_mf<16, false, 64, 4>(pl);
        if (pl->helm_zs == 4 && pl->helm_tx == 32) return full ? prepare_mf<16, true, 32, 4>(pl) : prepare_mf<16, false, 32, 4>(pl);
        if (pl->helm_zs == 4) return full ? prepare_mf<16, true, 16, 4>(pl) : prepare_mf<16, false, 16, 4>(pl);
        if (pl->helm_zs == 2 && pl->helm_tx == 32) return full ? prepare_mf<16, true, 32, 2>(pl) : prepare_mf<16, false, 32, 2>(pl);
        if (pl->helm_zs == 2) return full ? prepare_mf<16, true, 16, 2>(pl) : prepare_mf<16, false, 16, 2>(pl);
        if (pl->helm_tx == 32) return full ? prepare_mf<16, true, 32>(pl) : prepare_mf<16, false, 32>(pl);
        return PZ_HP(16);
    default: set_error("helmholtz: bad sub-domain size %d", pl->helm_m); return PZ_EINVAL;
    }
#undef PZ_HP
}

// n <= 4 fields in one persistent launch.  The caller (launch_helmholtz_n) has ordered the stream
// after the table upload and records the table's last use.
int launch_helmholtz_tma(pz_plan *pl, double *const *u, int n, const double *tab, cudaStream_t st)
{
    if (n < 1 || n > kMaxFields) { set_error("helmholtz (TMA variant): 1..4 fields per launch"); return PZ_EINVAL; }
    for (int f = 0; f < n; ++f)
        if (((uintptr_t)u[f] & 15) != 0) { set_error("helmholtz_z_solve: u must be 16-byte aligned"); return PZ_EINVAL; }
    const bool full = (pl->helm_zs * pl->helm_P * pl->helm_m == pl->nz);
#define PZ_HT(MM) (full ? launch_mf<MM, true>(pl, u, n, tab, st) : launch_mf<MM, false>(pl, u, n, tab, st))
    switch (pl->helm_m) {
    case 4: return PZ_HT(4);
    case 8: return PZ_HT(8);
    case 16:
        if (pl->helm_zs == 4 && pl->helm_tx == 64) return full ? launch_mf<16, true, 64, 4>(pl, u, n, tab, st) : launch_mf<16, false, 64, 4>(pl, u, n, tab, st);
        if (pl->helm_zs == 4 && pl->helm_tx == 32) return full ? launch_mf<16, true, 32, 4>(pl, u, n, tab, st) : launch_mf<16, false, 32, 4>(pl, u, n, tab, st);
        if (pl->helm_zs == 4) return full ? launch_mf<16, true, 16, 4>(pl, u, n, tab, st) : launch_mf<16, false, 16, 4>(pl, u, n, tab, st);
        if (pl->helm_zs == 2 && pl->helm_tx == 32) return full ? launch_mf<16, true, 32, 2>(pl, u, n, tab, st) : launch_mf<16, false, 32, 2>(pl, u, n, tab, st);
        if (pl->helm_zs == 2) return full ? launch_mf<16, true, 16, 2>(pl, u, n, tab, st) : launch_mf<16, false, 16, 2>(pl, u, n, tab, st);
        if (pl->helm_tx == 32) return full ? launch_mf<16, true, 32>(pl, u, n, tab, st) : launch_mf<16, false, 32>(pl, u, n, tab, st);
        return PZ_HT(16);
    default: set_error("helmholtz: bad sub-domain size %d", pl->helm_m); return PZ_EINVAL;
    }
#undef PZ_HT
}

} // namespace pz
