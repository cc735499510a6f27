// pz_fft_xy_impl.cuh -- steps a1+a2 (and a4+a5) as ONE persistent kernel per direction.
//
// The x and y transforms of a plane need the whole plane, so as two kernels they cost two HBM
// round trips (32 B/point).  Here the plane makes the second trip through L2 only: resident CTAs
// draw work items from a ticket counter in an order that runs the first-phase items of plane k+D
// right behind the second-phase items of plane k,
//     forward:  X(0) .. X(D-1) | Y(0) X(D) | Y(1) X(D+1) | ...      (X = x lines, Y = y columns)
//     inverse:  Y'(0) .. Y'(D-1) | X'(0) Y'(D) | ...
// and a second-phase item waits on a per-plane counter until all first-phase items of its plane
// have been published (release/acquire at GPU scope; second-phase loads bypass L1).  A ticket is
// only handed out after every earlier ticket has been taken by a resident CTA, so the wait cannot
// deadlock; D is chosen so that it practically never spins while D planes (tens of MB) stay far
// below the 126 MB L2.  The in-flight planes are written by phase one, read and re-written by
// phase two while still dirty in L2: DRAM sees one read and one write per point (16 B/point).
//
// The items are the bodies of pz_fft_x.cu / pz_fft_y.cu; the pair-0 split of pz_fft_y.cu's small
// kernel is folded into the y item that owns pair 0.  Sizes: nx, ny in {256, 512, 1024, 2048}
// (every BASELINE configuration); other sizes take the separate kernels.
#pragma once
#include "pz_fft.cuh"
#include "pz_internal.h"

namespace pz {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ int padx(int pos) { return pos + (pos >> 4); }
__host__ __device__ constexpr int line_ld(int M) { return M + M / 16 + 1; }

struct XchgX {
    double *re, *im;
    __device__ __forceinline__ void put(int pos, double2 v) const
    {
        const int q = padx(pos);
        re[q] = v.x;
        im[q] = v.y;
    }
    __device__ __forceinline__ double2 get(int pos) const
    {
        const int q = padx(pos);
        return make_double2(re[q], im[q]);
    }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
};

template <int TC>
struct XchgY {
    double2 *buf; // [pos][TC]
    int c;
    __device__ __forceinline__ void put(int pos, double2 v) const { buf[pos * TC + c] = v; }
    __device__ __forceinline__ double2 get(int pos) const { return buf[pos * TC + c]; }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
};

// loads that must see what other SMs published during this kernel go to L2
template <bool CG> __device__ __forceinline__ double2 ldg2(const double2 *p)
{
    if constexpr (CG) return __ldcg(p);
    else return *p;
}

// ---- x item: LPB lines of one plane (see pz_fft_x.cu for the split / merge algebra)
template <int M, bool INV, bool CG>
__device__ __forceinline__ void x_item(double *__restrict__ plane_base, const double2 *__restrict__ tw, int idx,
                                       double scale, double *smem)
{
    using P = FftPlan<M>;
    constexpr int E = P::E, T = P::T, LD = line_ld(M), LPB = kThreads / T;
    const int tid = threadIdx.x % T, ll = threadIdx.x / T;
    double2 *lp = reinterpret_cast<double2 *>(plane_base + ((size_t)idx * LPB + ll) * (2 * (size_t)M));
    XchgX xc{smem + (size_t)ll * 2 * LD, smem + (size_t)ll * 2 * LD + LD};
    double2 v[E];
    if constexpr (!INV) {
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = ldg2<CG>(&lp[tid + e * T]);
        fft_line<M, 2, 1>(v, tid, tw, xc);
        if constexpr (P::R2 > 1) xc.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) xc.put(tid + e * T, v[e]);
        xc.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = tid + e * T;
            double2 out;
            if (k == 0) {
                out = make_double2(v[e].x + v[e].y, v[e].x - v[e].y);
            } else {
                const double2 zm = cconj(xc.get(M - k));
                const double2 w = __ldg(&tw[k]);
                const double2 ev = make_double2(0.5 * (v[e].x + zm.x), 0.5 * (v[e].y + zm.y));
                const double2 d = csub(v[e], zm);
                const double2 od = make_double2(0.5 * d.y, -0.5 * d.x);
                out = cadd(ev, cmul(od, w));
            }
            lp[k] = out;
        }
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = tid + e * T;
            const double2 xk = ldg2<CG>(&lp[k]);
            double2 z;
            if (k == 0) {
                z = make_double2(xk.x + xk.y, xk.x - xk.y);
            } else {
                const double2 xm = cconj(ldg2<CG>(&lp[M - k]));
                const double2 w = __ldg(&tw[k]);
                const double2 s = cadd(xk, xm);
                const double2 c = cmul_conj(csub(xk, xm), w);
                z = make_double2(s.x - c.y, s.y + c.x);
            }
            v[e] = cconj(z);
        }
        fft_line<M, 2, 1>(v, tid, tw, xc);
#pragma unroll
        for (int e = 0; e < E; ++e) lp[tid + e * T] = make_double2(v[e].x * scale, -v[e].y * scale);
    }
}

// ---- y item: TC neighbouring complex pairs of one plane, all ny rows (see pz_fft_y.cu)
template <int L, bool INV, bool CG>
__device__ __forceinline__ void y_item(double *__restrict__ plane_base, const double2 *__restrict__ tw, int idx, int nx,
                                       double2 *smem)
{
    using P = FftPlan<L>;
    constexpr int E = P::E, T = P::T, TC = kThreads / T;
    const int c = threadIdx.x % TC, tid = threadIdx.x / TC;
    double *base = plane_base + 2 * ((size_t)idx * TC + c);
    XchgY<TC> xc{smem, c};
    const bool p0 = (idx == 0); // this CTA owns pair 0 (two real sequences, packed along y)
    constexpr int h = L / 2;

    double2 v[E];
    if (INV && p0) {
        // re-merge the packed spectra of columns 0 and 1 into W_r = A_r + i B_r
        if (c == 0)
#pragma unroll
            for (int e = 0; e < E; ++e) smem[tid + e * T] = ldg2<CG>(reinterpret_cast<const double2 *>(base + (size_t)(tid + e * T) * nx));
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int r = tid + e * T;
            if (c == 0) {
                double2 w;
                if (r == 0 || r == h) {
                    w = smem[r == 0 ? 0 : 1];
                } else {
                    const int rr = r < h ? r : L - r;
                    const double2 lo = smem[2 * rr], hi = smem[2 * rr + 1];
                    w = r < h ? make_double2(lo.x - hi.y, hi.x + lo.y) : make_double2(lo.x + hi.y, lo.y - hi.x);
                }
                v[e] = cconj(w);
            } else {
                v[e] = cconj(ldg2<CG>(reinterpret_cast<const double2 *>(base + (size_t)r * nx)));
            }
        }
        __syncthreads(); // the merge buffer is the exchange buffer
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double2 t = ldg2<CG>(reinterpret_cast<const double2 *>(base + (size_t)(tid + e * T) * nx));
            v[e] = INV ? cconj(t) : t;
        }
    }
    fft_line<L, 1, (L >= 1024) ? 1 : 0>(v, tid, tw, xc);
    if (!INV && p0) {
        // split W_r = A_r + i B_r into the packed spectra of the two real columns
        __syncthreads();
        if (c == 0)
#pragma unroll
            for (int e = 0; e < E; ++e) smem[tid + e * T] = v[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int r = tid + e * T;
            if (c != 0) {
                *reinterpret_cast<double2 *>(base + (size_t)r * nx) = v[e];
            } else if (r == 0 || r == h) {
                *reinterpret_cast<double2 *>(base + (size_t)(r == 0 ? 0 : 1) * nx) = v[e];
            } else if (r < h) {
                const double2 w = v[e], wm = cconj(smem[L - r]);
                const double2 a = make_double2(0.5 * (w.x + wm.x), 0.5 * (w.y + wm.y));
                const double2 d = csub(w, wm);
                const double2 b = make_double2(0.5 * d.y, -0.5 * d.x);
                *reinterpret_cast<double2 *>(base + (size_t)(2 * r) * nx) = make_double2(a.x, b.x);
                *reinterpret_cast<double2 *>(base + (size_t)(2 * r + 1) * nx) = make_double2(a.y, b.y);
            }
        }
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e)
            *reinterpret_cast<double2 *>(base + (size_t)(tid + e * T) * nx) = INV ? cconj(v[e]) : v[e];
    }
}

struct XYArgs {
    double *p;
    const double2 *twx, *twy;
    int *ctr;      // [0] ticket counter, [1 + k] first-phase items of plane k published
    int nx, ny, nz;
    int n1, n2;    // first- / second-phase items per plane
    int D;         // planes by which the first phase runs ahead
    double scale;
};

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <int MX, int LY> struct XYGeo {
    static constexpr int LPB = kThreads / FftPlan<MX>::T;   // x lines per item
    static constexpr int TC = kThreads / FftPlan<LY>::T;    // complex pairs per y item
    static constexpr size_t SMEM_X = (size_t)LPB * 2 * line_ld(MX) * sizeof(double);
    static constexpr size_t SMEM_Y = (size_t)LY * TC * sizeof(double2);
    static constexpr size_t SMEM = SMEM_X > SMEM_Y ? SMEM_X : SMEM_Y;
};

template <int MX, int LY, bool INV>
__global__ void __launch_bounds__(kThreads, 2) fft_xy_kernel(const XYArgs a)
{
    extern __shared__ __align__(16) double smem_xy[];
    __shared__ int s_ticket;
    const size_t plane_sz = (size_t)a.nx * a.ny;
    const int total = a.nz * (a.n1 + a.n2), head = a.D * a.n1, B = a.n1 + a.n2, kfull = a.nz - a.D;
    // Thread 0 draws the NEXT ticket while the current item runs (the atomic's round trip to L2 is
    // off the critical path); a CTA therefore holds two tickets, which the choice of D allows for.
    int next = 0;
    if (threadIdx.x == 0) next = atomicAdd(&a.ctr[0], 1);
    for (;;) {
        if (threadIdx.x == 0) {
            s_ticket = next;
            next = atomicAdd(&a.ctr[0], 1);
        }
        __syncthreads();
        const int t = s_ticket;
        if (t >= total) break;
        int phase, k, idx;
        if (t < head) {
            phase = 1; k = t / a.n1; idx = t - k * a.n1;
        } else {
            const int u = t - head;
            if (u < kfull * B) {
                k = u / B;
                const int r = u - k * B;
                if (r < a.n2) { phase = 2; idx = r; } else { phase = 1; k += a.D; idx = r - a.n2; }
            } else {
                const int v = u - kfull * B;
                phase = 2; k = kfull + v / a.n2; idx = v % a.n2;
            }
        }
        double *pb = a.p + (size_t)k * plane_sz;
        if (phase == 1) {
            if constexpr (!INV) x_item<MX, false, false>(pb, a.twx, idx, a.scale, smem_xy);
            else y_item<LY, true, false>(pb, a.twy, idx, a.nx, reinterpret_cast<double2 *>(smem_xy));
            __syncthreads(); // every store of this item precedes the publication
            if (threadIdx.x == 0) {
                __threadfence();
                atomicAdd(&a.ctr[1 + k], 1);
            }
        } else {
            if (threadIdx.x == 0)
                while (ld_acquire(&a.ctr[1 + k]) < a.n1) __nanosleep(64);
            __syncthreads();
            if constexpr (!INV) y_item<LY, false, true>(pb, a.twy, idx, a.nx, reinterpret_cast<double2 *>(smem_xy));
            else x_item<MX, true, true>(pb, a.twx, idx, a.scale, smem_xy);
        }
        __syncthreads(); // s_ticket and the exchange buffer are reused by the next item
    }
}

template <int MX, int LY, bool INV>
int launch_xy(pz_plan *pl, double *p, cudaStream_t st)
{
    using G = XYGeo<MX, LY>;
    auto kern = fft_xy_kernel<MX, LY, INV>;
    static int bps = 0;
    if (bps == 0) {
        PZ_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM));
        PZ_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, kThreads, G::SMEM));
        if (bps < 1) { bps = 0; set_error("fft_xy: kernel does not fit an SM"); return PZ_ECUDA; }
    }
    XYArgs a;
    a.p = p; a.twx = pl->d_twx; a.twy = pl->d_twy;
    a.ctr = pl->d_xyctr + (INV ? pl->nz + 1 : 0);
    a.nx = pl->nx; a.ny = pl->ny; a.nz = pl->nz;
    const int nxi = pl->ny / G::LPB, nyi = (pl->nx / 2) / G::TC;
    a.n1 = INV ? nyi : nxi;
    a.n2 = INV ? nxi : nyi;
    a.scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    long long total = (long long)pl->nz * (a.n1 + a.n2);
    long long blocks = (long long)pl->num_sms * bps;
    if (blocks > total) blocks = total;
    int D = pl->opt.xy_lag;
    if (D <= 0) D = 1 + (int)((2 * blocks * 12 / 10 + a.n1 + a.n2 - 1) / (a.n1 + a.n2));
    if (D > pl->nz) D = pl->nz;
    a.D = D;
    ProfScope prof(pl, INV ? PZ_K_FFT_XY_INV : PZ_K_FFT_XY_FWD, st);
    kern<<<(unsigned)blocks, kThreads, G::SMEM, st>>>(a);
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
    case 2048: return launch_xy<MX, 2048, INV>(pl, p, st);
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
