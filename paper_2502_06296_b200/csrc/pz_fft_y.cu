// pz_fft_y.cu -- steps a2 / a4 of the hot path: FFT along y (PAPER.md:126 step 3, :130 step 7).
//
// In the paper the y transform sits behind an x->y pencil transpose, which takes 81.7-90.5 % of
// the Poisson time at scale.  On one GPU the transpose is removed: a CTA
// transforms TC neighbouring columns at once, reading and writing rows of TC*16 contiguous
// bytes with stride nx, so every access is coalesced and the field is never re-laid-out.
//
// After the packed x transform, the two reals at (2q, 2q+1) of a line are Re/Im of x-mode q, so
// along y the data is already a COMPLEX sequence per q: one complex-to-complex FFT of length ny
// per pair gives the 2-D spectrum F(q, r), r = 0..ny-1, in the same storage.  Pair q = 0 holds
// two real sequences (x-modes 0 and nx/2) instead; a tiny kernel separates their spectra into
// the packed layout along y (and re-merges them before the inverse), DESIGN.md "Spectral layout".
#include "pz_fft.cuh"
#include "pz_internal.h"

namespace pz {

namespace {

template <int TC>
struct XchgY {
    double2 *buf; // [pos][TC]
    int c;
    __device__ __forceinline__ void put(int pos, double2 v) const { buf[pos * TC + c] = v; }
    __device__ __forceinline__ double2 get(int pos) const { return buf[pos * TC + c]; }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
};

template <int L, int TC, bool INV, bool FUSE_P0>
__global__ void __launch_bounds__(FftPlan<L>::T *TC, (FftPlan<L>::T * TC <= 256) ? 2 : 1)
    fft_y_kernel(double *__restrict__ p, const double2 *__restrict__ tw, int nx)
{
    using P = FftPlan<L>;
    constexpr int E = P::E, T = P::T;
    extern __shared__ double2 smem_y[];

    const int c = threadIdx.x % TC, tid = threadIdx.x / TC;
    const size_t pair = (size_t)blockIdx.x * TC + c;
    double *base = p + (size_t)blockIdx.y * L * nx + 2 * pair;
    XchgY<TC> xc{smem_y, c};

    // The CTA that owns pair 0 (x-modes 0 and nx/2: two real sequences) also converts between
    // W_r = A_r + i B_r and the packed spectra of the two real columns (rows (2r, 2r+1) hold
    // (Re A_r, Re B_r), (Im A_r, Im B_r); rows 0, 1 hold r = 0, ny/2) -- see pair0_kernel below,
    // which does the same as a separate pass (fft_y_p0 = 0).
    const bool p0 = FUSE_P0 && blockIdx.x == 0;
    constexpr int h = L / 2;
    double2 v[E];
    if (INV && p0) {
        if (c == 0)
#pragma unroll
            for (int e = 0; e < E; ++e)
                smem_y[tid + e * T] = *reinterpret_cast<const double2 *>(base + (size_t)(tid + e * T) * nx);
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int r = tid + e * T;
            if (c == 0) {
                double2 w;
                if (r == 0 || r == h) {
                    w = smem_y[r == 0 ? 0 : 1];
                } else {
                    const int rr = r < h ? r : L - r;
                    const double2 lo = smem_y[2 * rr], hi = smem_y[2 * rr + 1];
                    w = r < h ? make_double2(lo.x - hi.y, hi.x + lo.y) : make_double2(lo.x + hi.y, lo.y - hi.x);
                }
                v[e] = cconj(w);
            } else {
                v[e] = cconj(*reinterpret_cast<const double2 *>(base + (size_t)r * nx));
            }
        }
        __syncthreads(); // the merge buffer is the exchange buffer
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double2 t = *reinterpret_cast<const double2 *>(base + (size_t)(tid + e * T) * nx);
            v[e] = INV ? cconj(t) : t;
        }
    }
    fft_line<L, 1, (L >= 1024) ? 2 : 0>(v, tid, tw, xc); // long lines: factored twiddles (fewer L1 look-ups)
    if (!INV && p0) {
        __syncthreads();
        if (c == 0)
#pragma unroll
            for (int e = 0; e < E; ++e) smem_y[tid + e * T] = v[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int r = tid + e * T;
            if (c != 0) {
                *reinterpret_cast<double2 *>(base + (size_t)r * nx) = v[e];
            } else if (r == 0 || r == h) {
                *reinterpret_cast<double2 *>(base + (size_t)(r == 0 ? 0 : 1) * nx) = v[e];
            } else if (r < h) {
                const double2 w = v[e], wm = cconj(smem_y[L - r]);
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

// Pair q = 0: W_r = A_r + i B_r with A, B the spectra of the real sequences in columns 0 and 1.
// Forward: rows (2r, 2r+1) <- (Re A_r, Re B_r), (Im A_r, Im B_r); rows 0, 1 <- r = 0, ny/2.
// Inverse: the reverse.  One CTA per plane; the whole column pair is staged in shared memory.
template <bool INV>
__global__ void pair0_kernel(double *__restrict__ p, int nx, int ny)
{
    extern __shared__ double2 smem_p0[];
    double *base = p + (size_t)blockIdx.x * ny * nx;
    for (int r = threadIdx.x; r < ny; r += blockDim.x)
        smem_p0[r] = *reinterpret_cast<const double2 *>(base + (size_t)r * nx);
    __syncthreads();
    const int h = ny / 2;
    for (int r = threadIdx.x; r <= h; r += blockDim.x) {
        if constexpr (!INV) {
            double2 lo, hi;
            if (r == 0 || r == h) {
                const double2 w = smem_p0[r];
                *reinterpret_cast<double2 *>(base + (size_t)(r == 0 ? 0 : 1) * nx) = w;
                continue;
            }
            const double2 w = smem_p0[r], wm = cconj(smem_p0[ny - r]);
            const double2 a = make_double2(0.5 * (w.x + wm.x), 0.5 * (w.y + wm.y));
            const double2 d = csub(w, wm);
            const double2 b = make_double2(0.5 * d.y, -0.5 * d.x);
            lo = make_double2(a.x, b.x);
            hi = make_double2(a.y, b.y);
            *reinterpret_cast<double2 *>(base + (size_t)(2 * r) * nx) = lo;
            *reinterpret_cast<double2 *>(base + (size_t)(2 * r + 1) * nx) = hi;
        } else {
            if (r == 0 || r == h) {
                const double2 w = smem_p0[r == 0 ? 0 : 1];
                *reinterpret_cast<double2 *>(base + (size_t)r * nx) = w;
                continue;
            }
            const double2 lo = smem_p0[2 * r], hi = smem_p0[2 * r + 1];
            const double2 a = make_double2(lo.x, hi.x), b = make_double2(lo.y, hi.y);
            // W_r = A + iB,  W_{ny-r} = conj(A) + i conj(B)
            *reinterpret_cast<double2 *>(base + (size_t)r * nx) = make_double2(a.x - b.y, a.y + b.x);
            *reinterpret_cast<double2 *>(base + (size_t)(ny - r) * nx) = make_double2(a.x + b.y, b.x - a.y);
        }
    }
}

template <int L, int TC, bool INV>
int launch_ltc(const pz_plan *pl, double *p, int nk, cudaStream_t st)
{
    using P = FftPlan<L>;
    constexpr int threads = P::T * TC;
    // exchange tile; at least one column pair for the pair-0 conversion of single-pass lengths
    constexpr size_t smem = (P::R2 > 1) ? (size_t)L * TC * sizeof(double2) : (size_t)L * sizeof(double2);
    if (smem > 48 * 1024) {
        int rc;
        if ((rc = smem_optin(pl, fft_y_kernel<L, TC, INV, true>, smem)) != PZ_OK) return rc;
        if ((rc = smem_optin(pl, fft_y_kernel<L, TC, INV, false>, smem)) != PZ_OK) return rc;
    }
    dim3 grid((unsigned)(pl->nx / 2 / TC), (unsigned)nk);
    ProfScope prof(pl, INV ? PZ_K_FFT_Y_INV : PZ_K_FFT_Y_FWD, st);
    if (pl->opt.fft_y_p0 != 0)
        fft_y_kernel<L, TC, INV, true><<<grid, threads, smem, st>>>(p, pl->d_twy, pl->nx);
    else
        fft_y_kernel<L, TC, INV, false><<<grid, threads, smem, st>>>(p, pl->d_twy, pl->nx);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

// TC (complex pairs per CTA): 128-byte rows (TC = 8) while the exchange tile stays <= 64 KB,
// narrower for long lines; never more pairs than the field has.  A (L, TC) combination is
// instantiated only if its CTA has at most 512 threads and its tile at most 128 KB.
template <int L, int TC>
constexpr bool tc_valid() { return FftPlan<L>::T * TC <= 512 && (size_t)L * TC * sizeof(double2) <= 128 * 1024; }

template <int L, int TC, bool INV>
int try_ltc(const pz_plan *pl, double *p, int nk, cudaStream_t st)
{
    if constexpr (tc_valid<L, TC>()) {
        return launch_ltc<L, TC, INV>(pl, p, nk, st);
    } else {
        set_error("fft_y: no kernel for ny = %d with %d pairs per CTA", L, TC);
        return PZ_EUNSUPPORTED;
    }
}

template <int L, bool INV>
int launch_l(const pz_plan *pl, double *p, int nk, cudaStream_t st)
{
    const int npairs = pl->nx / 2;
    int tc = pl->opt.fft_y_tc;
    if (tc == 0) tc = (L <= 256) ? 16 : (L <= 512) ? 8 : 4; // 256 threads and <= 64 KB of exchange tile per CTA
    if (tc > npairs) tc = npairs;
    // the pairs of a row must split evenly over the CTAs (nx / 2 need not be a power of two)
    if (tc >= 16 && npairs % 16 == 0 && tc_valid<L, 16>()) return try_ltc<L, 16, INV>(pl, p, nk, st);
    if (tc >= 8 && npairs % 8 == 0 && tc_valid<L, 8>()) return try_ltc<L, 8, INV>(pl, p, nk, st);
    if (tc >= 4 && npairs % 4 == 0 && tc_valid<L, 4>()) return try_ltc<L, 4, INV>(pl, p, nk, st);
    return try_ltc<L, 2, INV>(pl, p, nk, st);
}

template <bool INV>
int dispatch(const pz_plan *pl, double *p, int nk, cudaStream_t st)
{
    switch (pl->ny) {
    case 8: return launch_l<8, INV>(pl, p, nk, st);
    case 16: return launch_l<16, INV>(pl, p, nk, st);
    case 32: return launch_l<32, INV>(pl, p, nk, st);
    case 64: return launch_l<64, INV>(pl, p, nk, st);
    case 128: return launch_l<128, INV>(pl, p, nk, st);
    case 256: return launch_l<256, INV>(pl, p, nk, st);
    case 512: return launch_l<512, INV>(pl, p, nk, st);
    case 1024: return launch_l<1024, INV>(pl, p, nk, st);
    case 2048: return launch_l<2048, INV>(pl, p, nk, st);
    case 4096: return launch_l<4096, INV>(pl, p, nk, st);
    default: set_error("fft_y: unsupported ny = %d", pl->ny); return PZ_EUNSUPPORTED;
    }
}

} // namespace

int launch_fft_y(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st)
{
    double *base = p + (size_t)k0 * pl->nx * pl->ny;
    if (pl->bcy != PZ_PERIODIC) return launch_r2r_y(pl, base, nk, inverse, st);
    // x in cosines / sines: no pair is special, the separate conversion pass handles all of them
    if (!fast_fft_len(pl->ny) || (pl->nx / 2) % 2 != 0 || pl->bcx != PZ_PERIODIC) return launch_fft_y_generic(pl, base, nk, inverse, st);
    return inverse ? dispatch<true>(pl, base, nk, st) : dispatch<false>(pl, base, nk, st);
}

int launch_pair0(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st)
{
    if (pl->bcy != PZ_PERIODIC) return PZ_OK; // cosine / sine coefficients of real sequences are real: nothing is packed
    if (pl->bcx != PZ_PERIODIC) return launch_allpairs(pl, p + (size_t)k0 * pl->nx * pl->ny, nk, inverse, st);
    if (pl->opt.fft_y_p0 != 0 && fast_fft_len(pl->ny) && (pl->nx / 2) % 2 == 0) return PZ_OK; // done inside fft_y_kernel
    double *base = p + (size_t)k0 * pl->nx * pl->ny;
    const size_t smem = (size_t)pl->ny * sizeof(double2);
    const int threads = pl->ny / 2 >= 256 ? 256 : (pl->ny / 2 < 32 ? 32 : pl->ny / 2);
    if (smem > 48 * 1024) {
        int rc;
        if ((rc = smem_optin(pl, pair0_kernel<false>, 128 * 1024)) != PZ_OK) return rc;
        if ((rc = smem_optin(pl, pair0_kernel<true>, 128 * 1024)) != PZ_OK) return rc;
    }
    ProfScope prof(pl, inverse ? PZ_K_PAIR0_INV : PZ_K_PAIR0_FWD, st);
    if (inverse)
        pair0_kernel<true><<<(unsigned)nk, threads, smem, st>>>(base, pl->nx, pl->ny);
    else
        pair0_kernel<false><<<(unsigned)nk, threads, smem, st>>>(base, pl->nx, pl->ny);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace pz
