// pz_fft_x.cu -- steps a1 / a5 of the hot path: real-to-complex and complex-to-real FFT along
// the contiguous x direction (PAPER.md:125 step 2, :131 step 8), output in the packed
// half-complex layout of Appendix A (reading R8):
//     line[0] = Re X_0, line[1] = Re X_{n/2}, line[2q], line[2q+1] = Re X_q, Im X_q  (0 < q < n/2)
// so an n-real line stays n reals and the transform is in place.
//
// One real line of n = 2M points is transformed as ONE complex FFT of length M on
// z_m = x_{2m} + i x_{2m+1} (a 16-byte load per point) followed by the split
//     X_k = (Z_k + conj Z_{M-k})/2 - (i/2) w_n^k (Z_k - conj Z_{M-k}),   w_n = exp(-2 pi i/n).
// The inverse builds Z'_k = (X_k + conj X_{M-k}) + i conj(w_n^k)(X_k - conj X_{M-k}) (no 1/2:
// the result is n x) and runs the same forward FFT on conj(Z').
#include "pz_fft.cuh"
#include "pz_internal.h"

namespace pz {

namespace {

// Shared-memory exchange buffer of one line: split re / im arrays of doubles, one pad double
// every 16 so that the stride-R writes of a Stockham pass spread over the banks.
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
    // unpadded access for the split exchange: written ascending, read descending, both contiguous
    // (the Stockham padding would put positions q and q-15 of a 16-lane group into the same bank)
    __device__ __forceinline__ void put_lin(int pos, double2 v) const
    {
        re[pos] = v.x;
        im[pos] = v.y;
    }
    __device__ __forceinline__ double2 get_lin(int pos) const { return make_double2(re[pos], im[pos]); }
};

// DIV (forward only): the lines are not read from p but formed on the fly as the right-hand side of
// Eq. (4), D u* / (gamma dt), from the staggered velocity (pz_projection.cu, same arithmetic in the
// same order, so the result is bitwise the one of pz_divergence_rhs followed by this kernel); the
// 16 B/point round trip of the right-hand side through HBM disappears.
template <int M, int LPB, bool INV, bool DIV>
__global__ void __launch_bounds__(FftPlan<M>::T *LPB, (FftPlan<M>::T * LPB <= 128) ? 5 : 1)
    fft_x_kernel(double *__restrict__ p, const double2 *__restrict__ tw, long long nlines, double scale, const DivSrc ds)
{
    static_assert(!(INV && DIV), "the divergence is fused into the forward transform only");
    using P = FftPlan<M>;
    constexpr int E = P::E, T = P::T, LD = line_ld(M);
    extern __shared__ double smem_x[];

    const int tid = threadIdx.x % T, ll = threadIdx.x / T;
    const long long line = (long long)blockIdx.x * LPB + ll;
    const bool active = line < nlines;
    double2 *lp = reinterpret_cast<double2 *>(p + (active ? line : 0) * (2LL * M));
    XchgX xc{smem_x + (size_t)ll * 2 * LD, smem_x + (size_t)ll * 2 * LD + LD};

    double2 v[E];
    if constexpr (!INV) {
        if constexpr (DIV) {
            const long long ln = active ? line : 0;
            const int j = (int)(ln % ds.ny), k = (int)(ln / ds.ny);
            const size_t c0 = (size_t)ln * (2 * (size_t)M);
            const double *ul = ds.u + c0;
            const double2 *vl = reinterpret_cast<const double2 *>(ds.v + c0);
            const double2 *vp = reinterpret_cast<const double2 *>(ds.v + (j == 0 ? c0 + (size_t)(ds.ny - 1) * 2 * M : c0 - 2 * (size_t)M));
            const double2 *wl = reinterpret_cast<const double2 *>(ds.w + c0);
            const double2 *wp = reinterpret_cast<const double2 *>(ds.w + (k > 0 ? c0 - (size_t)ds.ny * 2 * M : c0));
            const double rdz = 1.0 / ds.dzf[k];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int m = tid + e * T;
                const double2 uc = reinterpret_cast<const double2 *>(ul)[m], vc = vl[m], wc = wl[m];
                const double um = ul[m == 0 ? 2 * M - 1 : 2 * m - 1];
                const double2 vm = vp[m];
                double2 wm = make_double2(0.0, 0.0);
                if (k > 0) wm = wp[m];
                double2 d;
                d.x = ((uc.x - um) * ds.rdx + (vc.x - vm.x) * ds.rdy + (wc.x - wm.x) * rdz) * ds.scale;
                d.y = ((uc.y - uc.x) * ds.rdx + (vc.y - vm.y) * ds.rdy + (wc.y - wm.y) * rdz) * ds.scale;
                v[e] = active ? d : make_double2(0.0, 0.0);
            }
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = active ? lp[tid + e * T] : make_double2(0.0, 0.0);
        }
        fft_line<M, 2, 2>(v, tid, tw, xc);
        if constexpr (P::R2 > 1) xc.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) xc.put_lin(tid + e * T, v[e]);
        xc.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = tid + e * T;
            double2 out;
            if (k == 0) {
                out = make_double2(v[e].x + v[e].y, v[e].x - v[e].y);
            } else {
                const double2 zm = cconj(xc.get_lin(M - k));
                const double2 w = __ldg(&tw[k]);
                const double2 ev = make_double2(0.5 * (v[e].x + zm.x), 0.5 * (v[e].y + zm.y));
                const double2 d = csub(v[e], zm);
                const double2 od = make_double2(0.5 * d.y, -0.5 * d.x); // -(i/2) d
                const double2 t = cmul(od, w);
                out = cadd(ev, t);
            }
            if (active) lp[k] = out;
        }
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = tid + e * T;
            double2 z = make_double2(0.0, 0.0);
            if (active) {
                const double2 xk = lp[k];
                if (k == 0) {
                    z = make_double2(xk.x + xk.y, xk.x - xk.y);
                } else {
                    const double2 xm = cconj(lp[M - k]);
                    const double2 w = __ldg(&tw[k]);
                    const double2 s = cadd(xk, xm);
                    const double2 c = cmul_conj(csub(xk, xm), w);
                    z = make_double2(s.x - c.y, s.y + c.x); // s + i c
                }
            }
            v[e] = cconj(z);
        }
        // every global read of the line precedes the first barrier inside fft_line (or, for a
        // single-pass transform, is done by the one thread that owns the line): in place is safe
        fft_line<M, 2, 2>(v, tid, tw, xc);
        if (active) {
#pragma unroll
            for (int e = 0; e < E; ++e) lp[tid + e * T] = make_double2(v[e].x * scale, -v[e].y * scale);
        }
    }
}

template <int M, bool INV>
int launch_m(const pz_plan *pl, double *p, long long nlines, cudaStream_t st, const DivSrc *div)
{
    using P = FftPlan<M>;
    constexpr int LPB = (P::T >= 128) ? 1 : 128 / P::T;
    constexpr int threads = P::T * LPB;
    constexpr size_t smem = (size_t)LPB * 2 * line_ld(M) * sizeof(double);
    static_assert(smem <= 48 * 1024, "x-FFT exchange buffer must fit the default shared-memory limit");
    const long long blocks = (nlines + LPB - 1) / LPB;
    const double scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    ProfScope prof(pl, INV ? PZ_K_FFT_X_INV : PZ_K_FFT_X_FWD, st);
    if constexpr (!INV) {
        if (div) {
            fft_x_kernel<M, LPB, false, true><<<(unsigned)blocks, threads, smem, st>>>(p, pl->d_twx, nlines, scale, *div);
            count_launch();
            PZ_CUDA(cudaGetLastError());
            return PZ_OK;
        }
    }
    fft_x_kernel<M, LPB, INV, false><<<(unsigned)blocks, threads, smem, st>>>(p, pl->d_twx, nlines, scale, DivSrc{});
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

template <bool INV>
int dispatch(const pz_plan *pl, double *p, long long nlines, cudaStream_t st, const DivSrc *div)
{
    switch (pl->nx / 2) {
    case 4: return launch_m<4, INV>(pl, p, nlines, st, div);
    case 8: return launch_m<8, INV>(pl, p, nlines, st, div);
    case 16: return launch_m<16, INV>(pl, p, nlines, st, div);
    case 32: return launch_m<32, INV>(pl, p, nlines, st, div);
    case 64: return launch_m<64, INV>(pl, p, nlines, st, div);
    case 128: return launch_m<128, INV>(pl, p, nlines, st, div);
    case 256: return launch_m<256, INV>(pl, p, nlines, st, div);
    case 512: return launch_m<512, INV>(pl, p, nlines, st, div);
    case 1024: return launch_m<1024, INV>(pl, p, nlines, st, div);
    case 2048: return launch_m<2048, INV>(pl, p, nlines, st, div);
    default: set_error("fft_x: unsupported nx = %d", pl->nx); return PZ_EUNSUPPORTED;
    }
}

} // namespace

// Transform the x lines of planes k0 .. k0+nk-1, in place.
// div != NULL (forward, whole field only): transform the right-hand side of Eq. (4) formed from *div
int launch_fft_x(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st, const DivSrc *div)
{
    double *base = p + (size_t)k0 * pl->nx * pl->ny;
    const long long nlines = (long long)nk * pl->ny;
    if (div && (inverse || k0 != 0 || nk != pl->nz)) { set_error("fft_x: the fused divergence needs the whole field, forward"); return PZ_EINVAL; }
    if (pl->bcx != PZ_PERIODIC) {
        if (div) { set_error("fft_x: the fused divergence needs periodic x"); return PZ_EUNSUPPORTED; }
        return launch_r2r_x(pl, base, nlines, inverse, st);
    }
    if (!fast_fft_len(pl->nx)) {
        if (div) { set_error("fft_x: the fused divergence needs a power-of-two nx"); return PZ_EUNSUPPORTED; }
        return launch_fft_x_generic(pl, base, nlines, inverse, st);
    }
    return inverse ? dispatch<true>(pl, base, nlines, st, nullptr) : dispatch<false>(pl, base, nlines, st, div);
}

} // namespace pz
