// pz_fft.cuh -- register-resident Stockham FFT building blocks (FP64, sm_100a).
//
// The paper's in-house FFT is a mixed-radix R2C/C2R transform written as a plain CUDA/HIP
// function with auto-tuned launch parameters whose output is kept in the packed
// half-complex layout of Appendix A.  This is a B200-first restatement:
// every thread keeps E complex points in registers, a pass of radix R is E/R decimation-in-
// frequency butterflies done entirely in registers, and the only shared-memory traffic is one
// exchange between passes (FP64 Stockham with an smem round trip per radix-2/4 stage would be
// bound by the 128 B/clk shared-memory pipe, not by HBM).
//
// Index convention of one pass (complex length L, radix R, Ns = product of the previous
// radices, butterfly j in [0, L/R)):
//     in : x[j + r L/R] * w_{Ns R}^{r (j mod Ns)},  r = 0..R-1
//     out: y[(j div Ns) Ns R + (j mod Ns) + r' Ns] = sum_r in_r exp(-2 pi i r r'/R)
// A thread with index tid in [0, T), T = L/E, always owns the points tid + e T (e < E), so
// butterfly b of a pass uses registers e = b + r E/R and the last pass leaves the natural-order
// result in the same slots.
#pragma once
#include <cuda_runtime.h>

namespace pz {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 w)
{
    return make_double2(fma(a.x, w.x, -(a.y * w.y)), fma(a.x, w.y, a.y * w.x));
}
__device__ __forceinline__ double2 cmul_conj(double2 a, double2 w) // a * conj(w)
{
    return make_double2(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -(a.x * w.y)));
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }

// cos(m pi/16), m = 0..8
__host__ __device__ constexpr double cos_pi16(int m)
{
    return m == 0 ? 1.0
         : m == 1 ? 0.98078528040323044913
         : m == 2 ? 0.92387953251128675613
         : m == 3 ? 0.83146961230254523708
         : m == 4 ? 0.70710678118654752440
         : m == 5 ? 0.55557023301960222474
         : m == 6 ? 0.38268343236508977173
         : m == 7 ? 0.19509032201612826785
                  : 0.0;
}
// cos / sin of 2 pi m / 32 for m in [0, 16]
__host__ __device__ constexpr double cos32(int m) { return m <= 8 ? cos_pi16(m) : -cos_pi16(16 - m); }
__host__ __device__ constexpr double sin32(int m) { return m <= 8 ? cos_pi16(8 - m) : cos_pi16(m - 8); }

// d * w_R^r with w_R = exp(-2 pi i / R), r < R/2, R <= 32: compile-time special cases.
template <int R, int r>
__device__ __forceinline__ double2 mul_w(double2 d)
{
    static_assert(R <= 32 && r < R / 2 + 1, "radix too large");
    if constexpr (r == 0) {
        return d;
    } else if constexpr (4 * r == R) { // -i
        return make_double2(d.y, -d.x);
    } else if constexpr (8 * r == R) { // (1 - i)/sqrt2
        constexpr double h = 0.70710678118654752440;
        return make_double2((d.x + d.y) * h, (d.y - d.x) * h);
    } else if constexpr (8 * r == 3 * R) { // (-1 - i)/sqrt2
        constexpr double h = 0.70710678118654752440;
        return make_double2((d.y - d.x) * h, -(d.x + d.y) * h);
    } else {
        constexpr int m = r * (32 / R);
        constexpr double c = cos32(m), s = -sin32(m);
        return make_double2(fma(d.x, c, -(d.y * s)), fma(d.x, s, d.y * c));
    }
}

// One radix-2 decimation-in-frequency level over the R points v[r*S], then recurse.
// Result X[r'] ends up at v[bitrev_R(r') * S].
template <int R, int S, int r>
__device__ __forceinline__ void dif_level(double2 *v)
{
    if constexpr (r < R / 2) {
        const double2 a = v[r * S], b = v[(r + R / 2) * S];
        v[r * S] = cadd(a, b);
        v[(r + R / 2) * S] = mul_w<R, r>(csub(a, b));
        dif_level<R, S, r + 1>(v);
    }
}
template <int R, int S>
__device__ __forceinline__ void dif(double2 *v)
{
    if constexpr (R > 1) {
        dif_level<R, S, 0>(v);
        dif<R / 2, S>(v);
        dif<R / 2, S>(v + (R / 2) * S);
    }
}

__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n / 2); }
__host__ __device__ constexpr int bitrev(int p, int bits)
{
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((p >> b) & 1) << (bits - 1 - b);
    return r;
}

// Twiddle + butterflies of one pass, in registers.  tw[k] = exp(-2 pi i k / LT), k < LT, where
// LT is a multiple of L (table stride LT/L lets the x kernels share the length-n table).
// TWMODE 0: every twiddle w^{r jm} is looked up (cheap when all lanes of a warp share jm: the y
// kernels).  TWMODE 1: only w^{jm}, w^{2jm}, w^{4jm}, w^{8jm} are looked up and the other powers are
// products of two of them (one rounding more; the x kernels, whose lanes hit 16-32 different
// table lines per lookup and would otherwise be bound by L1 wavefronts).  TWMODE 2: ONE look-up,
// w^{jm}; w^2, w^4, w^8 by squaring (at most three roundings more; the x kernels and the y kernels
// from 1024 points: 3.69 -> 3.27 ms for the x transform at nx = 2048, 19.1 -> 18.2 ms per c3 solve).
template <int L, int E, int R, int NS, int TWSTRIDE, int TWMODE>
__device__ __forceinline__ void pass_butterflies(double2 (&v)[E], int tid, const double2 *__restrict__ tw)
{
    constexpr int T = L / E, S = E / R;
    static_assert(T * E == L && S * R == E, "bad FFT factorisation");
#pragma unroll
    for (int b = 0; b < S; ++b) {
        if constexpr (NS > 1) {
            const int jm = (tid + b * T) & (NS - 1);
            constexpr int STEP = (L / (NS * R)) * TWSTRIDE;
            if constexpr (TWMODE == 0 || R <= 2) {
#pragma unroll
                for (int r = 1; r < R; ++r) {
                    const double2 w = __ldg(&tw[r * jm * STEP]);
                    v[b + r * S] = cmul(v[b + r * S], w);
                }
            } else {
                double2 w[R];
                if constexpr (TWMODE == 2) {
                    // ONE look-up; w^2, w^4, w^8 by squaring (two roundings more on the highest power)
                    w[1] = __ldg(&tw[jm * STEP]);
#pragma unroll
                    for (int r = 2; r < R; r *= 2) w[r] = cmul(w[r / 2], w[r / 2]);
                } else {
#pragma unroll
                    for (int r = 1; r < R; r *= 2) w[r] = __ldg(&tw[r * jm * STEP]);
                }
#pragma unroll
                for (int r = 3; r < R; ++r) {
                    if ((r & (r - 1)) != 0) { // not a power of two: highest set bit times the rest
                        int hb = 1;
                        while (hb * 2 <= r) hb *= 2;
                        w[r] = cmul(w[hb], w[r - hb]);
                    }
                }
#pragma unroll
                for (int r = 1; r < R; ++r) v[b + r * S] = cmul(v[b + r * S], w[r]);
            }
        }
        dif<R, S>(&v[b]);
    }
}

// Output position of result r' of butterfly b (element index into the length-L line).
template <int L, int E, int R, int NS>
__device__ __forceinline__ int pass_out_pos(int tid, int b, int rp)
{
    constexpr int T = L / E;
    const int j = tid + b * T;
    return (j / NS) * (NS * R) + (j & (NS - 1)) + rp * NS;
}

// After the LAST pass the natural-order result of slot e' = b + r' S sits in register
// b + bitrev(r') S: undo the bit reversal in registers (compile-time permutation).
template <int E, int R>
__device__ __forceinline__ void unscramble(double2 (&v)[E])
{
    constexpr int S = E / R, bits = ilog2(R);
    double2 t[E];
#pragma unroll
    for (int e = 0; e < E; ++e) t[e] = v[e];
#pragma unroll
    for (int b = 0; b < S; ++b)
#pragma unroll
        for (int rp = 0; rp < R; ++rp) v[b + rp * S] = t[b + bitrev(rp, bits) * S];
}

// Factorisation of a power-of-two complex length L into at most three register passes.
template <int L> struct FftPlan;
#define PZ_FFT_PLAN(L_, E_, R1_, R2_, R3_)                                                        \
    template <> struct FftPlan<L_> {                                                              \
        static constexpr int E = E_, R1 = R1_, R2 = R2_, R3 = R3_, T = L_ / E_;                   \
        static_assert(R1_ * R2_ * R3_ == L_, "radices must multiply to L");                       \
    };
PZ_FFT_PLAN(4, 4, 4, 1, 1)
PZ_FFT_PLAN(8, 8, 8, 1, 1)
PZ_FFT_PLAN(16, 16, 16, 1, 1)
PZ_FFT_PLAN(32, 8, 8, 4, 1)
PZ_FFT_PLAN(64, 8, 8, 8, 1)
PZ_FFT_PLAN(128, 16, 16, 8, 1)
PZ_FFT_PLAN(256, 16, 16, 16, 1)
PZ_FFT_PLAN(512, 16, 16, 8, 4)
PZ_FFT_PLAN(1024, 16, 16, 16, 4)
PZ_FFT_PLAN(2048, 16, 16, 16, 8)
PZ_FFT_PLAN(4096, 16, 16, 16, 16)
#undef PZ_FFT_PLAN

// Forward complex FFT of one length-L line held as v[e] = x[tid + e T], cooperating threads
// tid = 0..T-1 exchanging through `Xchg` (a functor pair supplied by the kernel):
//   xchg.put(pos, value)  store one point of this line at line position pos
//   xchg.get(pos)         load it back
//   xchg.sync()           barrier covering every thread that shares the buffer
// On return v[e] = X[tid + e T] (natural order).
template <int L, int TWSTRIDE, int TWMODE, class Xchg>
__device__ __forceinline__ void fft_line(double2 (&v)[FftPlan<L>::E], int tid, const double2 *__restrict__ tw,
                                         Xchg &xchg)
{
    using P = FftPlan<L>;
    constexpr int E = P::E, T = P::T, R1 = P::R1, R2 = P::R2, R3 = P::R3;

    pass_butterflies<L, E, R1, 1, TWSTRIDE, TWMODE>(v, tid, tw);
    if constexpr (R2 == 1) {
        unscramble<E, R1>(v);
        return;
    } else {
        {
            constexpr int S = E / R1, bits = ilog2(R1);
#pragma unroll
            for (int b = 0; b < S; ++b)
#pragma unroll
                for (int rp = 0; rp < R1; ++rp)
                    xchg.put(pass_out_pos<L, E, R1, 1>(tid, b, rp), v[b + bitrev(rp, bits) * S]);
        }
        xchg.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = xchg.get(tid + e * T);
        pass_butterflies<L, E, R2, R1, TWSTRIDE, TWMODE>(v, tid, tw);
        if constexpr (R3 == 1) {
            unscramble<E, R2>(v);
            return;
        } else {
            xchg.sync(); // everyone has read pass-1 data before it is overwritten
            {
                constexpr int S = E / R2, bits = ilog2(R2);
#pragma unroll
                for (int b = 0; b < S; ++b)
#pragma unroll
                    for (int rp = 0; rp < R2; ++rp)
                        xchg.put(pass_out_pos<L, E, R2, R1>(tid, b, rp), v[b + bitrev(rp, bits) * S]);
            }
            xchg.sync();
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = xchg.get(tid + e * T);
            pass_butterflies<L, E, R3, R1 * R2, TWSTRIDE, TWMODE>(v, tid, tw);
            unscramble<E, R3>(v);
        }
    }
}

} // namespace pz
