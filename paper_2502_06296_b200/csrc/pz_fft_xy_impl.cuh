// pz_fft_xy_impl.cuh -- steps a1+a2 (and a4+a5) as ONE persistent kernel per direction.
//
// The x and y transforms of a plane need the whole plane, so as two kernels they cost two HBM
// round trips (32 B/point).  Here the plane makes the second trip through L2 only: resident CTAs
// draw work items from a ticket counter in an order that runs the first-phase items of plane k+D
// right behind the second-phase items of plane k,
//     forward:  X(0) .. X(D-1) | Y(0) X(D) | Y(1) X(D+1) | ...      (X = x lines, Y = y columns)
//     inverse:  Y'(0) .. Y'(D-1) | X'(0) Y'(D) | ...
// and a second-phase item waits on a per-plane counter until all first-phase items of its plane
// have been published (release/acquire at GPU scope).  A ticket is only handed out after every
// earlier ticket has been taken by a resident CTA, so the wait cannot deadlock; D is chosen so
// that it practically never spins while D planes (tens of MB) stay far below the 126 MB L2.  The
// in-flight planes are written by phase one, read and re-written by phase two while still dirty
// in L2: DRAM sees one read and one write per point (16 B/point).  Measured on this pool's B200
// (L2-resident working sets): 18 TB/s of reads, 7.7 TB/s of writes, 12.8 TB/s of a copy, so the L2
// leg costs about as much as the DRAM leg and overlaps with it.
//
// Items (pz_fft2.cuh: 32 complex points per thread, two passes, ONE shared-memory exchange per
// transform, split / merge of the real transform in registers).  The on-SM work bounds this kernel,
// not DRAM: the 16-point items of pz_fft_x.cu / pz_fft_y.cu put 1.04 M wavefronts per SM per
// direction through the L1 / shared-memory data pipe at 512^3 (0.53 ms at one per clock), and with
// 64 registers of data per thread only 12 warps fit an SM, too few to hide global-load latency
// (ncu r02: 0.56 + 0.48 ms for the two item types fed by ordinary loads).  So the input of an item
// is fetched by the TMA unit into the CTA's ONE shared-memory buffer while the previous item is
// still in its second pass:
//     wait(full) | pass 1: buffer -> registers | sync | exchange -> buffer | sync | buffer -> registers
//     | sync | thread 0: TMA of the NEXT item into the buffer | pass 2, split, global stores
// (x items: one bulk copy of LPB contiguous lines; y items: boxes {TC pairs x 256 rows} of a 2-D
// tensor map over the field).  Second-phase reads therefore come from L2 through the async proxy
// and never touch L1.  The pair-0 split of pz_fft_y.cu is folded into the y item that owns pair 0.
// Sizes: nx in {256, 512, 1024, 2048}, ny in {256, 512, 1024}; other sizes take the separate kernels.
#pragma once
#include <type_traits>

#include "pz_fft2.cuh"
#include "pz_internal.h"
#include "pz_tma.cuh"

namespace pz {

namespace {

constexpr int kThreads = 128;

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

__device__ __forceinline__ void bulk_load_1d(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load_1d_hint(void *dst, const void *src, unsigned bytes, uint64_t *bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 16-byte global store with an L2 eviction policy: first-phase results are kept (evict_last) until
// the second phase has read them, second-phase results leave first (evict_first)
__device__ __forceinline__ void st2h(double2 *p, double2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// Per-CTA twiddle tables in shared memory (the look-ups of a thread never change):
//   xp[m * TX + t] = w_M^(t 2^m), m < 5   powers of the x lines' radix-32 twiddle base
//   xs[j]          = w_n^j, j < 32        class factor of the split / merge twiddle (n = 2M)
//   yp[m * TY + t] = w_L^(t 2^m), m < 5   powers of the y columns' radix-32 twiddle base
template <int TX, int TY> struct TwTab {
    static constexpr int XP = 0, XS = 5 * TX, YP = XS + 32, COUNT = YP + 5 * TY;
};

// ------------------------------------------------------------------------------------------------
// x item, forward: LPB = 128 / T lines of one plane, T = M / 32 threads per line (M = nx / 2).
// pass 1: radix 32, butterfly j1 = t, twiddle w_M^{t r'} on its outputs;  pass 2: radix M / 32 on
// the residue classes (+-t) of the thread, then the real-to-complex split in registers.
// `in` holds the LPB lines back to back (M complex each); the exchange re-uses the buffer, in place
// (Xchg2X).  next() is called by every thread once the buffer is free again.
template <int M, class Next>
__device__ __forceinline__ void x_item_fwd(double *__restrict__ plane_base, const double2 *__restrict__ tw,
                                           const double2 *xp, const double2 *xs, int idx, double2 *smem, uint64_t pol, Next next)
{
    constexpr int R1 = 32, R2 = M / 32, T = R2, NB = 32 / R2, LPB = kThreads / T;
    constexpr bool IP = x_fwd_inplace<M>();
    constexpr int LD = xline_elems<M, R1, IP>();
    const int t = threadIdx.x % T, ll = threadIdx.x / T;
    double2 *lp = reinterpret_cast<double2 *>(plane_base + ((size_t)idx * LPB + ll) * (2 * (size_t)M));
    const double2 *in = smem + (size_t)ll * M;
    Xchg2X<R1, IP> xc{smem + (size_t)ll * LD};

    double2 v[kE2];
#pragma unroll
    for (int r = 0; r < R1; ++r) v[r] = in[t + r * T];
    dif<R1, 1>(v);
    apply_twiddles32<true>(v, xp + t, T);
    xc.sync(); // every line has been read: the exchange may overwrite it
#pragma unroll
    for (int rp = 0; rp < R1; ++rp) xc.put(t * R1 + rp, v[slot_of<R1>(rp)]);
    xc.sync();

    if constexpr (NB >= 2) {
        constexpr int NP = NB / 2;
        int jc[NB];
#pragma unroll
        for (int p = 0; p < NP; ++p) { jc[2 * p] = sym_ja<T>(t, p); jc[2 * p + 1] = sym_jb<T>(t, p); }
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int r = 0; r < R2; ++r) v[b * R2 + r] = xc.get(jc[b] + r * R1);
        next();
#pragma unroll
        for (int b = 0; b < NB; ++b) dif<R2, 1>(v + b * R2);
        // Z[jc[b] + 32 r'] = v[b R2 + slot(r')].  Split: the partner of k = ja + 32 r' is
        // M - k = jb + 32 (R2-1-r') (regular pair); thread 0's pair 0 holds the self-paired classes
        // 0 (partner index (R2 - r') mod R2) and 16 (partner index R2-1-r').
        const bool t0 = (t == 0);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const double2 *za = v + (2 * p) * R2, *zb = v + (2 * p + 1) * R2;
            const double2 wja = xs[jc[2 * p]], wjb = xs[jc[2 * p + 1]];
            static_for<0, R2>([&](auto ic) {
                constexpr int rp = decltype(ic)::value;
                double2 pa = zb[slot_of<R2>(R2 - 1 - rp)], pb = za[slot_of<R2>(R2 - 1 - rp)];
                if (p == 0 && t0) {
                    pa = za[slot_of<R2>((R2 - rp) % R2)];
                    pb = zb[slot_of<R2>(R2 - 1 - rp)];
                }
                double2 oa = r2c_split<2 * R2, rp>(za[slot_of<R2>(rp)], pa, wja);
                const double2 ob = r2c_split<2 * R2, rp>(zb[slot_of<R2>(rp)], pb, wjb);
                if (p == 0 && rp == 0 && t0) oa = make_double2(za[0].x + za[0].y, za[0].x - za[0].y); // Re X_0, Re X_{n/2}
                st2h(&lp[jc[2 * p] + 32 * rp], oa, pol);
                st2h(&lp[jc[2 * p + 1] + 32 * rp], ob, pol);
            });
        }
    } else {
        // M = 1024: one class per lane (j2 = t), a line is one warp; the partner of
        // k = t + 32 r' sits in lane (32 - t) mod 32, slot 31 - r' (lane 0: own slot (32 - r') mod 32)
        static_assert(T == 32, "one warp per line");
#pragma unroll
        for (int r = 0; r < R2; ++r) v[r] = xc.get(t + r * R1);
        next();
        dif<R2, 1>(v);
        // every result goes to global memory as soon as it is formed: nothing but v is held (an
        // array of the 32 results beside v spilled 800 bytes per thread)
        const int src = (32 - t) & 31;
        const double2 wt = __ldg(&tw[t]);   // w_n^t; w_n^{t + 32 r'} = wt w_64^{r'}
        static_for<0, R2>([&](auto ic) {
            constexpr int rp = decltype(ic)::value;
            const double2 mine = v[slot_of<R2>(R2 - 1 - rp)];
            double2 pa;
            pa.x = __shfl_sync(0xffffffffu, mine.x, src);
            pa.y = __shfl_sync(0xffffffffu, mine.y, src);
            if (t == 0) pa = v[slot_of<R2>((R2 - rp) % R2)];
            double2 o = r2c_split64<rp>(v[slot_of<R2>(rp)], pa, wt);
            if (rp == 0 && t == 0) o = make_double2(v[0].x + v[0].y, v[0].x - v[0].y);
            st2h(&lp[t + 32 * rp], o, pol);
        });
    }
}

// elements of a warp's region in the inverse x items: its 1024 points + the padding of their exchange
template <int M> constexpr int kWarpPitchInv = (32 / (M / 32)) * xline_elems<M, M / 32>();

// x item, inverse: merge in registers on the classes (+-t), pass 1 radix M / 32, pass 2 radix 32
// with butterfly j2 = t and the twiddle w_M^{t r} on its inputs; output x[t + r' T], natural order.
// The packed lines arrive per warp (see below).
template <int M, class Next>
__device__ __forceinline__ void x_item_inv(double *__restrict__ plane_base, const double2 *__restrict__ tw,
                                           const double2 *xp, const double2 *xs, int idx, double scale, double2 *smem,
                                           uint64_t pol, Next next)
{
    constexpr int R1 = M / 32, R2 = 32, T = R1, NB = 32 / R1, LPB = kThreads / T;
    constexpr int LD = xline_elems<M, R1>();
    const int t = threadIdx.x % T, ll = threadIdx.x / T;
    double2 *lp = reinterpret_cast<double2 *>(plane_base + ((size_t)idx * LPB + ll) * (2 * (size_t)M));
    // A warp's lines (1024 points in all) arrive back to back in the warp's own region of
    // kWarpPitchInv<M> elements (one bulk copy per warp); the padded exchange of a line reaches into
    // the next line's input and, for the last line, into the region's tail: only this warp's
    // threads ever touch the region, so the exchange is ordered by __syncwarp alone.
    constexpr int LPW = 32 / T;   // lines per warp
    double2 *region = smem + (size_t)(ll / LPW) * kWarpPitchInv<M>;
    const double2 *in = region + (size_t)(ll % LPW) * M;
    Xchg2X<R1> xc{region + (size_t)(ll % LPW) * LD};

    double2 v[kE2];
    if constexpr (NB >= 2) {
        constexpr int NP = NB / 2;
        int jc[NB];
#pragma unroll
        for (int p = 0; p < NP; ++p) { jc[2 * p] = sym_ja<T>(t, p); jc[2 * p + 1] = sym_jb<T>(t, p); }
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int r = 0; r < R1; ++r) v[b * R1 + r] = in[jc[b] + 32 * r];
        const bool t0 = (t == 0);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            double2 *xa = v + (2 * p) * R1, *xb = v + (2 * p + 1) * R1;
            const double2 wja = xs[jc[2 * p]], wjb = xs[jc[2 * p + 1]];
            double2 za[R1], zb[R1];
            static_for<0, R1>([&](auto ic) {
                constexpr int r = decltype(ic)::value;
                double2 pa = xb[R1 - 1 - r], pb = xa[R1 - 1 - r];
                if (p == 0 && t0) {
                    pa = xa[(R1 - r) % R1];
                    pb = xb[R1 - 1 - r];
                }
                za[r] = c2r_merge_conj<2 * R1, r>(xa[r], pa, wja);
                zb[r] = c2r_merge_conj<2 * R1, r>(xb[r], pb, wjb);
            });
            if (p == 0 && t0) za[0] = make_double2(xa[0].x + xa[0].y, -(xa[0].x - xa[0].y));
#pragma unroll
            for (int r = 0; r < R1; ++r) { xa[r] = za[r]; xb[r] = zb[r]; }
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) dif<R1, 1>(v + b * R1);
        __syncwarp(); // every packed line of the warp has been read
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int rp = 0; rp < R1; ++rp) xc.put(jc[b] * R1 + rp, v[b * R1 + slot_of<R1>(rp)]);
    } else {
        static_assert(T == 32, "one warp per line");
#pragma unroll
        for (int r = 0; r < R1; ++r) v[r] = in[t + 32 * r];
        // merged in place, indices r and R1-1-r together (partners of each other in the other lanes);
        // lane 0 pairs r with (R1 - r) mod R1 instead, whose old value is carried along in `hi`
        const int src = (32 - t) & 31;
        double2 hi = v[0];   // old v[(R1 - r) % R1] for lane 0 at step r
        const double2 wt = __ldg(&tw[t]);   // w_n^t; w_n^{t + 32 r} = wt w_64^r
        static_for<0, R1 / 2>([&](auto ic) {
            constexpr int r = decltype(ic)::value, q = R1 - 1 - r;
            const double2 a = v[r], b = v[q];
            double2 pa, pb;   // partners of index r and of index q
            pa.x = __shfl_sync(0xffffffffu, b.x, src);
            pa.y = __shfl_sync(0xffffffffu, b.y, src);
            pb.x = __shfl_sync(0xffffffffu, a.x, src);
            pb.y = __shfl_sync(0xffffffffu, a.y, src);
            if (t == 0) { pa = hi; pb = v[r + 1]; }   // (R1 - q) mod R1 = r + 1: not yet overwritten
            double2 za = c2r_merge_conj64<r>(a, pa, wt);
            const double2 zb = c2r_merge_conj64<q>(b, pb, wt);
            if (r == 0 && t == 0) za = make_double2(a.x + a.y, -(a.x - a.y));
            hi = b;           // = old v[R1 - (r + 1)]
            v[r] = za;
            v[q] = zb;
        });
        dif<R1, 1>(v);
        __syncwarp();
#pragma unroll
        for (int rp = 0; rp < R1; ++rp) xc.put(t * R1 + rp, v[slot_of<R1>(rp)]);
    }
    __syncwarp();
#pragma unroll
    for (int r = 0; r < R2; ++r) v[r] = xc.get(t + r * R1);
    next();
    apply_twiddles32<false>(v, xp + t, T);
    dif<R2, 1>(v);
#pragma unroll
    for (int rp = 0; rp < R2; ++rp) {
        const double2 x = v[slot_of<R2>(rp)];
        st2h(&lp[t + rp * T], make_double2(x.x * scale, -x.y * scale), pol);
    }
}

// ------------------------------------------------------------------------------------------------
// y item: TC = 128 / T neighbouring complex pairs of one plane, all ny rows, T = L / 32 threads per
// column.  pass 1: radix 32, butterfly j1 = t, twiddle w_L^{t r'} on its outputs; pass 2: radix
// L / 32, butterflies j2 = t + b T.  `smem` holds the tile [row][TC] (what the TMA boxes deliver);
// the exchange uses the same layout.  P0: the item that owns pair 0 (two real sequences: x-modes 0
// and nx/2) also converts between W_r = A_r + i B_r and the packed spectra of the two real columns
// (see pz_fft_y.cu).
template <int L, bool INV, bool P0, class Next>
__device__ __forceinline__ void y_item(double *__restrict__ plane_base, const double2 *yp, int idx, int nx,
                                       double2 *smem, uint64_t pol, Next next)
{
    constexpr int R1 = 32, R2 = L / 32, T = R2, NB = 32 / R2, TC = kThreads / T;
    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    double *base = plane_base + 2 * ((size_t)idx * TC + c);
    Xchg2Y<TC, (TC < 8)> xc{smem, c};   // the exchange; the tile the TMA boxes deliver is dense
    constexpr int h = L / 2;

    double2 v[kE2];
#pragma unroll
    for (int r = 0; r < R1; ++r) {
        const int row = t + r * T;
        double2 x = smem[row * TC + c];
        if (INV && P0 && c == 0) {
            // re-merge the packed spectra of columns 0 and 1 into W_row = A + i B
            if (row == 0 || row == h) {
                x = smem[(row == 0 ? 0 : 1) * TC];
            } else {
                const int rr = row < h ? row : L - row;
                const double2 lo = smem[(2 * rr) * TC], hi = smem[(2 * rr + 1) * TC];
                x = row < h ? make_double2(lo.x - hi.y, hi.x + lo.y) : make_double2(lo.x + hi.y, lo.y - hi.x);
            }
        }
        v[r] = INV ? cconj(x) : x;
    }
    dif<R1, 1>(v);
    apply_twiddles32<true>(v, yp + t, T);
    __syncthreads();
#pragma unroll
    for (int rp = 0; rp < R1; ++rp) xc.put(t * R1 + rp, v[slot_of<R1>(rp)]);
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int r = 0; r < R2; ++r) v[b * R2 + r] = xc.get(t + b * T + r * R1);
    if constexpr (!(P0 && !INV)) next();
#pragma unroll
    for (int b = 0; b < NB; ++b) dif<R2, 1>(v + b * R2);
    // W[t + b T + 32 r'] = v[b R2 + slot(r')]
    if constexpr (P0 && !INV) {
        __syncthreads();
        if (c == 0)
#pragma unroll
            for (int b = 0; b < NB; ++b)
#pragma unroll
                for (int rp = 0; rp < R2; ++rp) smem[t + b * T + 32 * rp] = v[b * R2 + slot_of<R2>(rp)];
        __syncthreads();
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int rp = 0; rp < R2; ++rp) {
                const int row = t + b * T + 32 * rp;
                const double2 w = v[b * R2 + slot_of<R2>(rp)];
                if (c != 0) {
                    st2h(reinterpret_cast<double2 *>(base + (size_t)row * nx), w, pol);
                } else if (row == 0 || row == h) {
                    st2h(reinterpret_cast<double2 *>(base + (size_t)(row == 0 ? 0 : 1) * nx), w, pol);
                } else if (row < h) {
                    const double2 wc = cconj(smem[L - row]);
                    const double2 a = make_double2(0.5 * (w.x + wc.x), 0.5 * (w.y + wc.y));
                    const double2 d = csub(w, wc);
                    const double2 bb = make_double2(0.5 * d.y, -0.5 * d.x);
                    st2h(reinterpret_cast<double2 *>(base + (size_t)(2 * row) * nx), make_double2(a.x, bb.x), pol);
                    st2h(reinterpret_cast<double2 *>(base + (size_t)(2 * row + 1) * nx), make_double2(a.y, bb.y), pol);
                }
            }
        next(); // one item in ny / TC: the buffer is released after the stores
    } else {
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int rp = 0; rp < R2; ++rp) {
                const double2 w = v[b * R2 + slot_of<R2>(rp)];
                st2h(reinterpret_cast<double2 *>(base + (size_t)(t + b * T + 32 * rp) * nx), INV ? cconj(w) : w, pol);
            }
    }
}

// ------------------------------------------------------------------------------------------------
struct XYArgs {
    double *p;
    const double2 *twx, *twy;
    int *ctr;      // [kC1] first-phase ticket counter, [kC2] second-phase, [kPub + k] first-phase items of plane k published
    int nx, ny, nz;
    int n1, n2;    // first- / second-phase items per plane
    int D;         // planes by which the first phase may run ahead of the second
    int pf;        // planes by which first-phase inputs are prefetched into L2
    int xshare, group; // SMs with (index mod 2 group) < xshare prefer the first phase
    double scale;
};
constexpr int kC1 = 0, kC2 = 32, kPub = 64; // counters on separate 128-byte lines

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_relaxed(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

template <int MX, int LY> struct XYGeo {
    static constexpr int TX = MX / 32, TY = LY / 32;
    static constexpr int LPB = kThreads / TX;   // x lines per item
    static constexpr int TC = kThreads / TY;    // complex pairs per y item
    static constexpr int BOXR = LY < 256 ? LY : 256; // rows per TMA box of a y tile
    // x exchange: R1 = 32 forward, R1 = MX / 32 inverse
    static constexpr size_t SMEM_XF = (size_t)LPB * xline_elems<MX, 32, x_fwd_inplace<MX>()>() * sizeof(double2);
    static constexpr size_t SMEM_XI = (size_t)LPB * xline_elems<MX, MX / 32>() * sizeof(double2);
    static constexpr size_t SMEM_X = SMEM_XF > SMEM_XI ? SMEM_XF : SMEM_XI;
    static constexpr size_t SMEM_Y = (size_t)(TC < 8 ? LY + LY / 32 : LY) * TC * sizeof(double2);   // padded exchange (Xchg2Y)
    static constexpr size_t SMEM = (SMEM_X > SMEM_Y ? SMEM_X : SMEM_Y) + 128; // + alignment slack
    static constexpr unsigned X_BYTES = (unsigned)((size_t)LPB * MX * sizeof(double2));
    static constexpr unsigned Y_BYTES = (unsigned)((size_t)LY * TC * sizeof(double2));
};

// Work distribution.  Two ticket counters (atomicAdd: pipelined in L2, unlike a compare-and-swap
// chain), one per phase, drawn in plane order.  A drawn item may have to wait:
//   * first-phase item of plane k >= D: until the second phase has drawn every ticket of plane
//     k - D (bounds the planes in flight, i.e. the L2 footprint, to about D);
//   * second-phase item of plane k: until all n1 first-phase items of plane k are published.
// The CTAs of an SM prefer ONE phase (by SM index): the unrolled code of an item type is about
// 32 KB, both types do not fit the instruction cache (ncu r02: 1.3-1.9 stall cycles per issue on
// instruction fetch with mixed roles).  First-phase CTAs switch to the second phase only when the
// first is drawn out; second-phase CTAs never switch.  No deadlock: by induction over planes, the
// first-phase items of planes < D never wait, so the second-phase tickets of plane 0 can be served
// and drawn, which releases plane D, and so on; a waiting CTA holds nothing but its own ticket.
struct Item { int phase, k, idx; }; // phase 0 = nothing left

template <int MX, int LY, bool INV>
__global__ void __launch_bounds__(kThreads, 3) fft_xy_kernel(const __grid_constant__ CUtensorMap ymap, const XYArgs a)
{
    using G = XYGeo<MX, LY>;
    using TT = TwTab<G::TX, G::TY>;
    extern __shared__ unsigned char smem_raw_xy[];
    double2 *smem = reinterpret_cast<double2 *>(smem_raw_xy + ((128u - (smem_u32(smem_raw_xy) & 127u)) & 127u));
    __shared__ double2 s_tw[TT::COUNT];
    __shared__ Item s_item;
    __shared__ int s_deferred;
    __shared__ __align__(8) uint64_t s_bar;
    const size_t plane_sz = (size_t)a.nx * a.ny;

    if (threadIdx.x == 0) {
        mbar_init(&s_bar, 1);
        mbar_fence_init();
    }
    for (int q = threadIdx.x; q < TT::COUNT; q += kThreads) {
        double2 w;
        if (q < TT::XS) w = a.twx[2 * (q % G::TX) * (1 << (q / G::TX))];
        else if (q < TT::YP) w = a.twx[q - TT::XS];
        else w = a.twy[((q - TT::YP) % G::TY) * (1 << ((q - TT::YP) / G::TY))];
        s_tw[q] = w;
    }
    // first-phase results stay in L2 until the second phase has read them; everything else streams
    const uint64_t pol_keep = l2_policy_evict_last(), pol_stream = l2_policy_evict_first();
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    int role = ((int)(smid % (2u * a.group)) < a.xshare) ? 1 : 2; // thread 0's current phase preference
    Item pend;                                          // thread 0: ticket drawn but not started yet
    pend.phase = -1; pend.k = 0; pend.idx = 0;

    // thread 0: draw the next ticket (if none is pending) and, when its item can start, start the
    // fetch.  block = false: one look only (called in the middle of an item, whose publication the
    // pending item's plane may be waiting for); returns false if the item cannot start yet.
    auto acquire = [&](bool block) -> bool {
        if (pend.phase < 0) {
            pend.phase = 0;
            if (role == 1) {
                const int t = atomicAdd(&a.ctr[kC1], 1);
                if (t < a.nz * a.n1) { pend.phase = 1; pend.k = t / a.n1; pend.idx = t - pend.k * a.n1; }
                else role = 2;
            }
            if (role == 2) {
                const int t = atomicAdd(&a.ctr[kC2], 1);
                if (t < a.nz * a.n2) { pend.phase = 2; pend.k = t / a.n2; pend.idx = t - pend.k * a.n2; }
            }
        }
        if (pend.phase == 1) {
            while (pend.k >= a.D && ld_relaxed(&a.ctr[kC2]) < (pend.k - a.D + 1) * a.n2) {
                if (!block) return false;
                __nanosleep(100);
            }
        } else if (pend.phase == 2) {
            while (ld_acquire(&a.ctr[kPub + pend.k]) < a.n1) {
                if (!block) return false;
                __nanosleep(100);
            }
            fence_proxy_async_global(); // generic-proxy writes of other SMs (acquired) -> async-proxy reads
        }
        const Item it = pend;
        pend.phase = -1;
        s_item = it;
        if (it.phase == 0) return true;
        const bool is_x = (it.phase == 1) != INV;
        if (is_x) {
            const double *src = a.p + (size_t)it.k * plane_sz + (size_t)it.idx * G::LPB * (2 * (size_t)MX);
            mbar_arrive_expect_tx(&s_bar, G::X_BYTES);
            if constexpr (INV) {
                // one copy per warp: its 1024 points into its own region (x_item_inv)
#pragma unroll
                for (int w = 0; w < kThreads / 32; ++w)
                    bulk_load_1d_hint(smem + (size_t)w * kWarpPitchInv<MX>, src + (size_t)w * 2048, 1024 * sizeof(double2), &s_bar, pol_stream);
            } else {
                bulk_load_1d_hint(smem, src, G::X_BYTES, &s_bar, pol_stream);
            }
            if (it.phase == 1 && it.k + a.pf < a.nz) bulk_prefetch_l2(src + (size_t)a.pf * plane_sz, G::X_BYTES);
        } else {
            mbar_arrive_expect_tx(&s_bar, G::Y_BYTES);
#pragma unroll
            for (int b = 0; b < LY / G::BOXR; ++b)
                tma_load_2d_hint(smem + (size_t)b * G::BOXR * G::TC, &ymap, 2 * it.idx * G::TC, it.k * a.ny + b * G::BOXR, &s_bar, pol_stream);
            if (it.phase == 1 && it.k + a.pf < a.nz)
#pragma unroll
                for (int b = 0; b < LY / G::BOXR; ++b)
                    tma_prefetch_l2_2d(&ymap, 2 * it.idx * G::TC, (it.k + a.pf) * a.ny + b * G::BOXR);
        }
        return true;
    };

    if (threadIdx.x == 0) acquire(true);
    __syncthreads();
    Item it = s_item;
    unsigned parity = 0;

    while (it.phase != 0) {
        double *pb = a.p + (size_t)it.k * plane_sz;
        // Called by every thread when its last read of the buffer is done: after the barrier the
        // buffer is free and thread 0 draws the next item and, if it can start right now, starts
        // its fetch; otherwise the fetch is deferred to the end of this item.  (Drawing tickets
        // earlier hides the L2 round trips but leaves the last items of a plane waiting in CTAs
        // that are still busy, which stalls the second phase: measured slower.)
        auto next = [&]() {
            __syncthreads();
            if (threadIdx.x == 0) s_deferred = acquire(false) ? 0 : 1;
        };
        mbar_wait(&s_bar, parity);
        parity ^= 1;
        const bool is_x = (it.phase == 1) != INV;
        const uint64_t pol = (it.phase == 1) ? pol_keep : pol_stream;
        if (is_x) {
            if constexpr (!INV) x_item_fwd<MX>(pb, a.twx, s_tw + TT::XP, s_tw + TT::XS, it.idx, smem, pol, next);
            else x_item_inv<MX>(pb, a.twx, s_tw + TT::XP, s_tw + TT::XS, it.idx, a.scale, smem, pol, next);
        } else {
            if (it.idx == 0) y_item<LY, INV, true>(pb, s_tw + TT::YP, it.idx, a.nx, smem, pol, next);
            else y_item<LY, INV, false>(pb, s_tw + TT::YP, it.idx, a.nx, smem, pol, next);
        }
        __syncthreads(); // every store of this item precedes its publication; s_item / s_deferred are visible
        const Item done = it;
        const bool deferred = s_deferred != 0;
        if (!deferred) it = s_item;
        if (threadIdx.x == 0 && done.phase == 1) {
            // publication; the fence overlaps the wait for the next item's data
            __threadfence();
            atomicAdd(&a.ctr[kPub + done.k], 1);
        }
        if (deferred) {
            if (threadIdx.x == 0) acquire(true);
            __syncthreads();
            it = s_item;
        }
    }
}

template <int MX, int LY, bool INV>
int launch_xy(pz_plan *pl, double *p, cudaStream_t st)
{
    using G = XYGeo<MX, LY>;
    XYArgs a;
    a.p = p; a.twx = pl->d_twx; a.twy = pl->d_twy;
    a.ctr = pl->d_xyctr + (INV ? pl->nz + 64 : 0);
    a.nx = pl->nx; a.ny = pl->ny; a.nz = pl->nz;
    const int nxi = pl->ny / G::LPB, nyi = (pl->nx / 2) / G::TC;
    a.scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    auto kern = fft_xy_kernel<MX, LY, INV>;
    int &bps = pl->xy_bps[INV ? 1 : 0];
    if (bps == 0) {
        { const int rc = smem_optin(pl, kern, G::SMEM); if (rc != PZ_OK) return rc; }
        PZ_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, kThreads, G::SMEM));
        if (bps < 1) { bps = 0; set_error("fft_xy: kernel does not fit an SM"); return PZ_ECUDA; }
    }
    // y tiles: the field as {nx doubles} x {ny nz rows}, boxes of TC pairs x BOXR rows
    CUtensorMap ymap;
    const int rc = encode_column_tile_map(&ymap, p, (size_t)pl->nx, pl->ny * pl->nz, 2 * G::TC, G::BOXR, 1, false);
    if (rc != PZ_OK) return rc;
    a.n1 = INV ? nyi : nxi;
    a.n2 = INV ? nxi : nyi;
    long long total = (long long)pl->nz * (a.n1 + a.n2);
    int use_bps = bps;
    if (pl->opt.xy_bps > 0 && pl->opt.xy_bps < bps) use_bps = pl->opt.xy_bps;
    long long blocks = (long long)pl->num_sms * use_bps;
    if (blocks > total) blocks = total;
    // D: the first phase may run this many planes ahead (what is in flight stays in L2); enough
    // that half the CTAs find first-phase work while the other half runs the second phase
    // Planes of 16 MB: what is in flight between the phases must still fit L2 (126 MB) beside the
    // streams: at most three planes ahead, one plane of prefetch (2048 x 1024 x 512: 6.3 + 6.0 ms
    // against 6.4 + 8.0 ms with the defaults below)
    const bool big_planes = (size_t)pl->nx * pl->ny * sizeof(double) >= ((size_t)16 << 20);
    int D = pl->opt.xy_lag;
    if (D <= 0) {
        D = 2 + (int)((blocks + a.n1 - 1) / a.n1);
        if (big_planes && D > 3) D = 3;
    }
    if (D > pl->nz) D = pl->nz;
    a.D = D;
    a.pf = pl->opt.xy_prefetch > 0 ? pl->opt.xy_prefetch : (big_planes ? 1 : 3);
    // SMs of a role group run the same phase (the two SMs of a TPC share an instruction-cache level);
    // measured at 512^3: forward 0.598 ms with groups of 4 against 0.612 with 2, inverse 0.572 with 2 against 0.582
    a.group = pl->opt.xy_group > 0 ? pl->opt.xy_group : (INV ? 2 : 4);
    a.xshare = (pl->opt.xy_xshare > 0 && pl->opt.xy_xshare < 2 * a.group) ? pl->opt.xy_xshare : a.group;
    ProfScope prof(pl, INV ? PZ_K_FFT_XY_INV : PZ_K_FFT_XY_FWD, st);
    kern<<<(unsigned)blocks, kThreads, G::SMEM, st>>>(ymap, a);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

template <int MX, bool INV>
int dispatch_y(pz_plan *pl, double *p, cudaStream_t st)
{
    switch (pl->ny) {
    case 256: return launch_xy<MX, 256, INV>(pl, p, st);
    case 512: return launch_xy<MX, 512, INV>(pl, p, st);
    case 1024: return launch_xy<MX, 1024, INV>(pl, p, st);
    default: set_error("fft_xy: unsupported ny = %d", pl->ny); return PZ_EUNSUPPORTED;
    }
}

template <bool INV>
int dispatch_xy(pz_plan *pl, double *p, cudaStream_t st)
{
    switch (pl->nx) {
    case 256: return dispatch_y<128, INV>(pl, p, st);
    case 512: return dispatch_y<256, INV>(pl, p, st);
    case 1024: return dispatch_y<512, INV>(pl, p, st);
    case 2048: return dispatch_y<1024, INV>(pl, p, st);
    default: set_error("fft_xy: unsupported nx = %d", pl->nx); return PZ_EUNSUPPORTED;
    }
}

} // namespace
} // namespace pz
