// pz_fft2.cuh -- two-pass register-resident FFT items (32 complex points per thread) for the fused
// x/y transform (pz_fft_xy.cu), steps a1+a2 / a4+a5 of the hot path (
// packed half-complex layout of Appendix A, reading R8).
//
// Why a second FFT core next to pz_fft.cuh.  With 16 points per thread a line of 512 complex points
// takes three register passes (two shared-memory exchanges) and the real-to-complex split of an x
// line a third exchange; at 512^3 that is 96 bytes per grid point through the 128 B/clk
// shared-memory / L1 path per transform direction, 0.35 ms of a 0.33 ms DRAM budget.  Here a
// thread keeps 32 complex points: every length up to 1024 is TWO passes (L = R1 R2, one exchange),
// and on the x lines a thread owns the residue classes +-t of the spectral index, so the split
// X_k <- (Z_k, Z_{M-k}) (and the merge of the inverse) pairs values the thread already holds: no
// exchange.  64 bytes per point per direction instead of 96.
//
// Index convention (Stockham, decimation in frequency, as pz_fft.cuh), L = R1 R2:
//   pass 1, butterfly j1 < R2:  y[j1 R1 + r'] = sum_r x[j1 + r R2] w_R1^{r r'}
//   twiddle:                    y[j1 R1 + r'] *= w_L^{j1 r'}
//   pass 2, butterfly j2 < R1:  X[j2 + r' R1] = sum_r y[j2 + r R1] w_R2^{r r'}
// The twiddle is applied on the radix-32 side, where a thread holds ONE butterfly and every
// factor is a power of a single base.
#pragma once
#include "pz_fft.cuh"

namespace pz {

constexpr int kE2 = 32; // complex points per thread

// result r' of an in-register butterfly of radix R (dif<R, 1>) sits in slot bitrev(r')
template <int R> __host__ __device__ constexpr int slot_of(int rp) { return bitrev(rp, ilog2(R)); }

// v[slot(r)] *= w^r, r = 1..31, for the radix-32 side of a transform, w a single base per thread.  Only w, w^2, w^4, w^8, w^16 are looked
// up; every other power is a product of at most two factors w^{4a} w^{b} (the table look-ups of a
// 16-byte twiddle cost as many L1 wavefronts as the data they multiply, ncu r02: the transforms are
// bound by the L1 / shared-memory data pipe, not by FP64).
// BITREV: value r sits in slot bitrev(r) (outputs of a butterfly) or in slot r (inputs).
// The five looked-up powers come from a small table base[m * pitch] = w^(2^m) of this thread
// (staged in shared memory once per CTA: the thread's base never changes).
template <bool BITREV>
__device__ __forceinline__ void apply_twiddles32(double2 *v, const double2 *base, int pitch)
{
    auto slot = [](int r) { return BITREV ? slot_of<32>(r) : r; };
    double2 wl[4], wh[8];
    wl[1] = base[0];
    wl[2] = base[pitch];
    wl[3] = cmul(wl[1], wl[2]);
    wh[1] = base[2 * pitch];
    wh[2] = base[3 * pitch];
    wh[4] = base[4 * pitch];
    wh[3] = cmul(wh[1], wh[2]);
    wh[5] = cmul(wh[4], wh[1]);
    wh[6] = cmul(wh[4], wh[2]);
    wh[7] = cmul(wh[4], wh[3]);
#pragma unroll
    for (int r = 1; r < 32; ++r) {
        const int a = r / 4, b = r % 4;
        double2 x = v[slot(r)];
        if (a) x = cmul(x, wh[a]);
        if (b) x = cmul(x, wl[b]);
        v[slot(r)] = x;
    }
}

// d * conj(w_R^r)
template <int R, int r>
__device__ __forceinline__ double2 mul_wc(double2 d) { return cconj(mul_w<R, r>(cconj(d))); }

// ---- exchange buffers
// x lines: one line per T <= 32 threads, 16-byte elements.  Lanes of pass 1 (consecutive
// j1 = pos / R1) write with a stride of R1 elements, lanes of pass 2 (consecutive j2 = pos % R1) read
// consecutive elements.
// PADDED (INPLACE = false): element pos at (pos / R1)(R1 + 1) + pos % R1; both accesses are
//   conflict-free (8 lanes x 16 B per wavefront); the padded line reaches into the space of the next
//   line's input, so the exchange is bracketed by CTA barriers.
// IN PLACE (R1 >= 8): element pos at pos ^ ((pos / R1) & 7) -- the 16-byte chunk index is swizzled
//   with the butterfly index: conflict-free as well, and a line stays inside its own M elements; the
//   lines of a warp being its own, the exchange needs __syncwarp only (ncu r02: the CTA barriers are
//   the largest stall of the fused kernel).  Used by the forward items (R1 = 32: 0.599 -> 0.572 ms at
//   512^3); in the inverse items of 256-point lines (R1 = 8) the 32 run-time store addresses per
//   thread spilled 400 bytes and lost more than the barriers cost.
template <int R1, bool INPLACE = false>
struct Xchg2X {
    static_assert(!INPLACE || R1 >= 8, "the swizzle permutes the low three bits of the position");
    double2 *buf;
    __device__ __forceinline__ static int idx(int pos)
    {
        if constexpr (INPLACE) return pos ^ ((pos / R1) & 7);
        else return (pos / R1) * (R1 + 1) + (pos % R1);
    }
    __device__ __forceinline__ void put(int pos, double2 v) const { buf[idx(pos)] = v; }
    __device__ __forceinline__ double2 get(int pos) const { return buf[idx(pos)]; }
    // orders the accesses of the threads that may touch the same elements
    __device__ __forceinline__ static void sync()
    {
        if constexpr (INPLACE) __syncwarp();
        else __syncthreads();
    }
};
template <int L, int R1, bool INPLACE = false> __host__ __device__ constexpr int xline_elems() { return INPLACE ? L : (L / R1) * (R1 + 1); }
// forward x items of the fused kernel: in place from 256-point lines (128-point lines measured slower)
template <int M> __host__ __device__ constexpr bool x_fwd_inplace() { return M >= 256; }

// y columns: TC neighbouring complex columns side by side, c fastest: 8 lanes = 128 contiguous bytes
// With TC = 4 (columns of 1024 points) a quarter warp holds two butterflies j1 whose pass-1 outputs
// lie 32 rows = 2 KB apart: the same banks.  PAD skips one row every 32 (as Xchg2X does), which puts
// them 64 bytes apart modulo 128: conflict-free (ncu r02: 606 M shared-memory wavefronts per launch at
// 2048 x 1024 x 512 where 470 M are needed).
template <int TC, bool PAD = false>
struct Xchg2Y {
    double2 *buf;
    int c;
    __device__ __forceinline__ static int idx(int pos) { return PAD ? pos + (pos >> 5) : pos; }
    __device__ __forceinline__ void put(int pos, double2 v) const { buf[idx(pos) * TC + c] = v; }
    __device__ __forceinline__ double2 get(int pos) const { return buf[idx(pos) * TC + c]; }
};

// Residue classes mod 32 closed under negation for thread t of T (x lines): 32 / T classes per
// thread in pairs (ja, jb = -ja mod 32).
//   t >= 1: pair p = (t + 2 T p, 32 - t - 2 T p)
//   t == 0: pair 0 = (0, 16), the two self-paired classes; pair p >= 1 = (T p, 32 - T p)
template <int T> __device__ __forceinline__ int sym_ja(int t, int p) { return t ? t + 2 * T * p : T * p; }
template <int T> __device__ __forceinline__ int sym_jb(int t, int p) { return t ? 32 - t - 2 * T * p : (p ? 32 - T * p : 16); }

// split of the real-to-complex transform: X_k from Z_k, Z_{M-k} and w_n^k, n = 2M,
//   X_k = (Z_k + conj Z_{M-k})/2 - (i/2) w_n^k (Z_k - conj Z_{M-k}),
// with k = j + 32 r': w_n^k = w_n^j w_{n/32}^{r'}; wj = w_n^j is one look-up per residue class and
// the second factor a compile-time constant (R2X = n / 32 <= 32) or, for n = 2048, wj itself is
// the full twiddle (ROT = 0).
template <int R2X, int ROT>
__device__ __forceinline__ double2 r2c_split(double2 zk, double2 zmk, double2 wj)
{
    const double2 zm = cconj(zmk);
    const double2 ev = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y + zm.y));
    const double2 d = csub(zk, zm);
    const double2 od = make_double2(0.5 * d.y, -0.5 * d.x);
    return cadd(ev, cmul(mul_w<R2X, ROT>(od), wj));
}
// merge of the complex-to-real transform: conj(Z'_k), Z'_k = (X_k + conj X_{M-k}) + i conj(w_n^k)(X_k - conj X_{M-k})
template <int R2X, int ROT>
__device__ __forceinline__ double2 c2r_merge_conj(double2 xk, double2 xmk, double2 wj)
{
    const double2 xm = cconj(xmk);
    const double2 s = cadd(xk, xm);
    const double2 c = cmul_conj(mul_wc<R2X, ROT>(csub(xk, xm)), wj);
    return make_double2(s.x - c.y, -(s.y + c.x));
}

// ---- lines of n = 2048 reals (M = 1024): w_n^k with k = t + 32 r' is w_n^t w_64^{r'}; the first
// factor is one look-up per thread, the second a compile-time constant (32 look-ups per thread and
// line cost as many L1 wavefronts as an exchange and their latency was the kernel's second stall).
__host__ __device__ constexpr double cos64(int m) // cos(2 pi m / 64), m = 0..16
{
    constexpr double c[17] = {1.0,
                              0.995184726672196886245, 0.980785280403230449126, 0.956940335732208864936, 0.923879532511286756128,
                              0.881921264348355029713, 0.831469612302545237079, 0.773010453362736960811, 0.707106781186547524401,
                              0.634393284163645498215, 0.555570233019602224743, 0.471396736825997648556, 0.382683432365089771728,
                              0.290284677254462367636, 0.195090322016128267848, 0.0980171403295606019942, 0.0};
    return c[m];
}
__host__ __device__ constexpr double c64(int m) { return m <= 16 ? cos64(m) : -cos64(32 - m); } // cos(2 pi m / 64), m <= 32
__host__ __device__ constexpr double s64(int m) { return m <= 16 ? cos64(16 - m) : cos64(m - 16); } // sin
// d * w_64^r (CONJ: d * conj(w_64^r)), r = 0..31
template <int r, bool CONJ>
__device__ __forceinline__ double2 rot64(double2 d)
{
    static_assert(r >= 0 && r < 32, "w_64^r with r < 32");
    if constexpr (r == 0) {
        return d;
    } else if constexpr (r == 16) {
        return CONJ ? make_double2(-d.y, d.x) : make_double2(d.y, -d.x);
    } else {
        constexpr double c = c64(r), sg = CONJ ? -s64(r) : s64(r);
        // (d.x + i d.y)(c - i sg)
        return make_double2(fma(d.x, c, d.y * sg), fma(d.y, c, -(d.x * sg)));
    }
}
// r2c_split / c2r_merge_conj with the twiddle w_n^{t + 32 r} = wt w_64^r
template <int r>
__device__ __forceinline__ double2 r2c_split64(double2 zk, double2 zmk, double2 wt)
{
    const double2 zm = cconj(zmk);
    const double2 ev = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y + zm.y));
    const double2 d = csub(zk, zm);
    const double2 od = make_double2(0.5 * d.y, -0.5 * d.x);
    return cadd(ev, cmul(rot64<r, false>(od), wt));
}
template <int r>
__device__ __forceinline__ double2 c2r_merge_conj64(double2 xk, double2 xmk, double2 wt)
{
    const double2 xm = cconj(xmk);
    const double2 s = cadd(xk, xm);
    const double2 c = cmul_conj(rot64<r, true>(csub(xk, xm)), wt);
    return make_double2(s.x - c.y, -(s.y + c.x));
}

} // namespace pz
