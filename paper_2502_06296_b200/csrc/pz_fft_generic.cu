// pz_fft_generic.cu -- steps a1/a2/a4/a5 for lengths that are not powers of two: mixed-radix
// (2, 3, 4, 5, 7, 8) Stockham transforms.  The paper's in-house FFT is mixed-radix
// and every grid it runs has such lengths: 7168 = 2^10 7, 3200 x 3456 (:278),
// 3456 x 3072 (:280).  Same data layout as the power-of-two kernels (pz_fft_x.cu, pz_fft_y.cu):
// real-to-complex along x through one complex transform of length M = nx / 2 plus the split,
// output packed into the nx reals of the line (Appendix A, reading R8);
// along y one complex transform of length ny per packed pair, TC neighbouring pairs per CTA.
//
// One pass of radix R (Ns = product of the earlier radices, butterfly j < L / R), as in pz_fft.cuh:
//     in : x[j + r L/R] w_{Ns R}^{r (j mod Ns)},   r < R
//     out: y[(j div Ns) Ns R + (j mod Ns) + r' Ns] = sum_r in_r exp(-2 pi i r r' / R)
// The lines of a CTA live in ONE shared-memory buffer; a pass reads all its butterflies' inputs into
// registers (at most kE points per thread), synchronises, and writes the results back in place, so
// the buffer is as large as shared memory allows (8192 points) and rows stay as wide as possible.
#include "pz_internal.h"
#include "pz_fft.cuh"

namespace pz {

namespace {

constexpr int kE = 16;    // complex points per thread, at most
constexpr int kMaxT = 512;        // threads per CTA, at most (128 registers each)
constexpr int kPts = kMaxT * kE;  // largest buffer
// Threads per CTA: 512 (8192-point buffer, one CTA per SM) where a line or a useful tile needs it,
// else 256 (4096 points, two CTAs per SM: the loads of one overlap the passes of the other).

struct Radices { int n; int r[20]; };

// ---- small DFTs, forward sign, natural order in and out
__device__ __forceinline__ double2 mul_mi(double2 a) { return make_double2(a.y, -a.x); } // a * (-i)
__device__ __forceinline__ double2 axpy(double c, double2 x, double2 y) { return make_double2(fma(c, x.x, y.x), fma(c, x.y, y.y)); }
__device__ __forceinline__ double2 scal(double c, double2 x) { return make_double2(c * x.x, c * x.y); }

template <int R> __device__ __forceinline__ void dft(double2 (&v)[R]);

template <> __device__ __forceinline__ void dft<2>(double2 (&v)[2])
{
    const double2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
}
template <> __device__ __forceinline__ void dft<4>(double2 (&v)[4])
{
    dif<4, 1>(v); // result r' in slot bitrev(r')
    const double2 t = v[1];
    v[1] = v[2];
    v[2] = t;
}
template <> __device__ __forceinline__ void dft<8>(double2 (&v)[8])
{
    dif<8, 1>(v);
    double2 t[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) t[i] = v[i];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = t[bitrev(i, 3)];
}
template <> __device__ __forceinline__ void dft<16>(double2 (&v)[16])
{
    dif<16, 1>(v);
    double2 t[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) t[i] = v[i];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = t[bitrev(i, 4)];
}
template <> __device__ __forceinline__ void dft<3>(double2 (&v)[3])
{
    constexpr double s = 0.86602540378443864676; // sin(2 pi / 3)
    const double2 t1 = cadd(v[1], v[2]), d = mul_mi(scal(s, csub(v[1], v[2])));
    const double2 m1 = axpy(-0.5, t1, v[0]);
    v[0] = cadd(v[0], t1);
    v[1] = cadd(m1, d);
    v[2] = csub(m1, d);
}
template <> __device__ __forceinline__ void dft<5>(double2 (&v)[5])
{
    constexpr double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410; // cos(2 pi/5), cos(4 pi/5)
    constexpr double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;  // sin(2 pi/5), sin(4 pi/5)
    const double2 a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]), b1 = csub(v[1], v[4]), b2 = csub(v[2], v[3]);
    const double2 e1 = axpy(c2, a2, axpy(c1, a1, v[0])), e2 = axpy(c1, a2, axpy(c2, a1, v[0]));
    const double2 d1 = mul_mi(axpy(s2, b2, scal(s1, b1))), d2 = mul_mi(axpy(-s1, b2, scal(s2, b1)));
    v[0] = cadd(v[0], cadd(a1, a2));
    v[1] = cadd(e1, d1);
    v[4] = csub(e1, d1);
    v[2] = cadd(e2, d2);
    v[3] = csub(e2, d2);
}
template <> __device__ __forceinline__ void dft<7>(double2 (&v)[7])
{
    constexpr double c1 = 0.62348980185873353053, c2 = -0.22252093395631440429, c3 = -0.90096886790241912624;
    constexpr double s1 = 0.78183148246802980871, s2 = 0.97492791218182360702, s3 = 0.43388373911755812048;
    const double2 a1 = cadd(v[1], v[6]), a2 = cadd(v[2], v[5]), a3 = cadd(v[3], v[4]);
    const double2 b1 = csub(v[1], v[6]), b2 = csub(v[2], v[5]), b3 = csub(v[3], v[4]);
    // X_m = v0 + sum_k cos(2 pi m k / 7) a_k - i sum_k sin(2 pi m k / 7) b_k
    const double2 e1 = axpy(c3, a3, axpy(c2, a2, axpy(c1, a1, v[0])));
    const double2 e2 = axpy(c1, a3, axpy(c3, a2, axpy(c2, a1, v[0])));   // m = 2: k = 1, 2, 3 -> angles 2, 4, 6 -> c2, c3, c1
    const double2 e3 = axpy(c2, a3, axpy(c1, a2, axpy(c3, a1, v[0])));   // m = 3: angles 3, 6, 9 = 2 -> c3, c1, c2
    const double2 d1 = mul_mi(axpy(s3, b3, axpy(s2, b2, scal(s1, b1))));
    const double2 d2 = mul_mi(axpy(-s1, b3, axpy(-s3, b2, scal(s2, b1)))); // sin(4) = -s3, sin(6) = -s1 (units of 2 pi / 7)
    const double2 d3 = mul_mi(axpy(s2, b3, axpy(-s1, b2, scal(s3, b1))));  // sin(6) = -s1, sin(9 = 2) = s2
    v[0] = cadd(v[0], cadd(a1, cadd(a2, a3)));
    v[1] = cadd(e1, d1); v[6] = csub(e1, d1);
    v[2] = cadd(e2, d2); v[5] = csub(e2, d2);
    v[3] = cadd(e3, d3); v[4] = csub(e3, d3);
}

// Composite radices.  Coprime factors (6, 10, 12, 14, 15): the prime-factor map, input
// n = (R2 n1 + R1 n2) mod R, output k with k = k1 (mod R1), k = k2 (mod R2), needs no twiddles
// between the two stages.  9 = 3 x 3: Cooley-Tukey with the constants w_9, w_9^2, w_9^4.
__host__ __device__ constexpr int crt_index(int R1, int R2, int k1, int k2)
{
    for (int k = 0; k < R1 * R2; ++k)
        if (k % R1 == k1 && k % R2 == k2) return k;
    return 0;
}
template <int R1, int R2> __device__ __forceinline__ void dft_pfa(double2 (&v)[R1 * R2])
{
    constexpr int R = R1 * R2;
    double2 a[R2][R1];
#pragma unroll
    for (int n2 = 0; n2 < R2; ++n2)
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) a[n2][n1] = v[(R2 * n1 + R1 * n2) % R];
#pragma unroll
    for (int n2 = 0; n2 < R2; ++n2) dft<R1>(a[n2]);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) {
        double2 b[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) b[n2] = a[n2][k1];
        dft<R2>(b);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) v[crt_index(R1, R2, k1, k2)] = b[k2];
    }
}
template <> __device__ __forceinline__ void dft<6>(double2 (&v)[6]) { dft_pfa<3, 2>(v); }
template <> __device__ __forceinline__ void dft<10>(double2 (&v)[10]) { dft_pfa<5, 2>(v); }
template <> __device__ __forceinline__ void dft<12>(double2 (&v)[12]) { dft_pfa<3, 4>(v); }
template <> __device__ __forceinline__ void dft<14>(double2 (&v)[14]) { dft_pfa<7, 2>(v); }
template <> __device__ __forceinline__ void dft<15>(double2 (&v)[15]) { dft_pfa<3, 5>(v); }
template <> __device__ __forceinline__ void dft<9>(double2 (&v)[9])
{
    // X[k1 + 3 k2] = sum_n2 w_9^{n2 k1} w_3^{n2 k2} sum_n1 x[3 n1 + n2] w_3^{n1 k1}
    constexpr double c1 = 0.766044443118978, s1 = 0.6427876096865393;    // cos, sin of 2 pi / 9
    constexpr double c2 = 0.17364817766693041, s2 = 0.984807753012208;   // of 4 pi / 9
    constexpr double c4 = -0.9396926207859084, s4 = 0.3420201433256687;  // of 8 pi / 9
    double2 a[3][3];
#pragma unroll
    for (int n2 = 0; n2 < 3; ++n2) {
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1) a[n2][n1] = v[3 * n1 + n2];
        dft<3>(a[n2]);
    }
    a[1][1] = cmul(a[1][1], make_double2(c1, -s1));
    a[1][2] = cmul(a[1][2], make_double2(c2, -s2));
    a[2][1] = cmul(a[2][1], make_double2(c2, -s2));
    a[2][2] = cmul(a[2][2], make_double2(c4, -s4));
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1) {
        double2 b[3] = {a[0][k1], a[1][k1], a[2][k1]};
        dft<3>(b);
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) v[k1 + 3 * k2] = b[k2];
    }
}

// butterflies per thread and pass: kE points or a little more (at most 21) up to radix 9, ONE
// butterfly of 10 ... 16 points above; the launch geometry sizes the CTA so that every pass fits
__host__ __device__ constexpr int bfly_per_thread(int R) { return R <= 9 ? (kE + R - 1) / R : 1; }

// Where a pass reads and writes: element pos of line ln sits at base[ln * sl + pos * sp].  A pass
// may read from global memory (the first one) or write to it (the last one): the lines then make
// no extra round trip through shared memory on their way in and out.  The imaginary part is
// negated on the way in where im < 0, the result multiplied by (re, im) on the way out (conjugation
// and scaling of the inverse transforms).
struct Side {
    double2 *base;
    int sl, sp;
    double re, im;
};

// One pass over `nlines` lines of complex length L.  tw[k * tws] = exp(-2 pi i k / L).
// lines_fastest: consecutive threads take the same butterfly of neighbouring lines (y columns).
template <int R>
__device__ __forceinline__ void pass(const Side in, const Side out, bool in_place, bool out_shared, int L, int Ns, int nlines,
                                     bool lines_fastest, const double2 *__restrict__ tw, int tws)
{
    constexpr int Q = bfly_per_thread(R);
    const int nb = L / R, W = nlines * nb, step = (L / (Ns * R)) * tws, kT = (int)blockDim.x;
    const int instr = nb * in.sp, outstr = Ns * out.sp;
    const bool conj_in = in.im < 0.0, scaled = out.re != 1.0 || out.im != 1.0;
    double2 v[Q][R];
    int obase[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        // work items past the end recompute item 0 and store nothing (no divergent definitions)
        const int w0 = (int)threadIdx.x + q * kT, w = (w0 < W) ? w0 : 0;
        const int ln = lines_fastest ? w % nlines : w / nb, j = lines_fastest ? w / nlines : w % nb;
        const int jm = j % Ns;
        const double2 *x = in.base + (ln * in.sl + j * in.sp);
        obase[q] = (w0 < W) ? ln * out.sl + ((j - jm) * R + jm) * out.sp : -1;
        // ONE twiddle look-up per butterfly, w = w_{Ns R}^{jm}; the powers w^r are products of at most
        // log2 R factors (ncu r02: with R - 1 scattered 16-byte look-ups per butterfly the kernels were
        // bound by the L1 / shared-memory data pipe at 17 % of the DRAM rate)
        double2 wp[R];
        wp[0] = make_double2(1.0, 0.0);
        if constexpr (R > 1) wp[1] = __ldg(&tw[jm * step]);
#pragma unroll
        for (int r = 2; r < R; ++r) {
            int hb = 1;
            while (hb * 2 <= r) hb *= 2;
            wp[r] = (r == hb) ? cmul(wp[hb / 2], wp[hb / 2]) : cmul(wp[hb], wp[r - hb]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double2 t = x[r * instr];
            if (conj_in) t.y = -t.y;
            if (r > 0) t = cmul(t, wp[r]);
            v[q][r] = t;
        }
        dft<R>(v[q]);
    }
    if (in_place) __syncthreads();
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        if (obase[q] >= 0) {
            double2 *y = out.base + obase[q];
#pragma unroll
            for (int r = 0; r < R; ++r) y[r * outstr] = scaled ? make_double2(v[q][r].x * out.re, v[q][r].y * out.im) : v[q][r];
        }
    }
    if (out_shared) __syncthreads();
}

// All passes of the lines of a CTA: the first reads `src`, the last writes `dst`, the ones between
// work in place in the shared-memory buffer `mid`.  src / dst may be `mid` itself.
__device__ __forceinline__ void all_passes(const Side src, const Side mid, const Side dst, int L, int nlines, bool lines_fastest,
                                           const double2 *__restrict__ tw, int tws, const Radices &rl)
{
    int Ns = 1;
    for (int i = 0; i < rl.n; ++i) {
        const Side in = (i == 0) ? src : mid, out = (i == rl.n - 1) ? dst : mid;
        const bool in_place = in.base == out.base, out_shared = out.base == mid.base;
        switch (rl.r[i]) {
#define PZ_PASS(R_) case R_: pass<R_>(in, out, in_place, out_shared, L, Ns, nlines, lines_fastest, tw, tws); break;
        PZ_PASS(2) PZ_PASS(3) PZ_PASS(4) PZ_PASS(5) PZ_PASS(6) PZ_PASS(7) PZ_PASS(8) PZ_PASS(9) PZ_PASS(10) PZ_PASS(12)
        PZ_PASS(14) PZ_PASS(15)
#undef PZ_PASS
        default: pass<16>(in, out, in_place, out_shared, L, Ns, nlines, lines_fastest, tw, tws); break;
        }
        Ns *= rl.r[i];
    }
}

// x lines: lpb lines of n = 2M reals per CTA.  twx[k] = exp(-2 pi i k / n).
template <bool INV>
__global__ void __launch_bounds__(kMaxT) gen_fft_x_kernel(double *__restrict__ p, const double2 *__restrict__ twx, int M, long long nlines, int lpb,
                                                          Radices rl, double scale)
{
    extern __shared__ double2 smem_gx[];
    const int kT = (int)blockDim.x;
    const long long l0 = (long long)blockIdx.x * lpb;
    const int nl = (int)((nlines - l0 < lpb) ? nlines - l0 : lpb);
    double2 *g = reinterpret_cast<double2 *>(p) + (size_t)l0 * M;
    const Side glob{g, M, 1, 1.0, 1.0}, mid{smem_gx, M, 1, 1.0, 1.0};
    const int H = M / 2 + 1;   // spectral indices k and M - k are handled together, k = 0 .. M/2
    if constexpr (INV) {
        // merge of the complex-to-real transform, conjugated (inverse through the forward passes):
        //   conj Z'_k = conj(s + i c),  s = X_k + conj X_{M-k},  c = conj(w_n^k) (X_k - conj X_{M-k}),
        // and, with w_n^{M-k} = -conj(w_n^k), Z'_{M-k} = conj(s) + i conj(c): both from one pair of
        // loads and one twiddle.  Staged through shared memory (formed on the way into the first
        // pass it was slower: 3.7 against 2.8 ms on 3456 x 3072 x 30).
        // four items per trip, their loads issued together (one item per trip left every trip
        // waiting on its own loads: ncu stall long_scoreboard 3.9 per issue)
        for (int q0 = threadIdx.x; q0 < nl * H; q0 += 4 * kT) {
            double2 xk[4], xp[4], w[4];
            int pos[4], kk[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int q = q0 + u * kT, qq = (q < nl * H) ? q : 0;
                const int ln = qq / H, k = qq - ln * H;
                pos[u] = ln * M;
                kk[u] = (q < nl * H) ? k : -1;
                xk[u] = g[(size_t)ln * M + k];
                xp[u] = g[(size_t)ln * M + (k ? M - k : 0)];
                w[u] = __ldg(&twx[k]);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int k = kk[u];
                if (k == 0) {
                    smem_gx[pos[u]] = make_double2(xk[u].x + xk[u].y, -(xk[u].x - xk[u].y));
                } else if (k > 0) {
                    const double2 xm = cconj(xp[u]);
                    const double2 sm = cadd(xk[u], xm), c = cmul_conj(csub(xk[u], xm), w[u]);
                    smem_gx[pos[u] + k] = make_double2(sm.x - c.y, -(sm.y + c.x));
                    if (2 * k != M) smem_gx[pos[u] + (M - k)] = make_double2(sm.x + c.y, sm.y - c.x);
                }
            }
        }
        __syncthreads();
        // every global read of the lines precedes this barrier: the last pass stores in place
        const Side dst{g, M, 1, scale, -scale};
        all_passes(mid, mid, dst, M, nl, false, twx, 2, rl);
    } else {
        all_passes(glob, mid, mid, M, nl, false, twx, 2, rl);
        // split: X_k = e + t, X_{M-k} = conj(e - t),  e = (Z_k + conj Z_{M-k}) / 2,
        //        t = -(i/2) w_n^k (Z_k - conj Z_{M-k})
        for (int q = threadIdx.x; q < nl * H; q += kT) {
            const int ln = q / H, k = q - ln * H;
            const double2 z = smem_gx[ln * M + k];
            if (k == 0) {
                g[(size_t)ln * M] = make_double2(z.x + z.y, z.x - z.y); // Re X_0, Re X_{n/2}
            } else {
                const double2 zm = cconj(smem_gx[ln * M + (M - k)]);
                const double2 ev = make_double2(0.5 * (z.x + zm.x), 0.5 * (z.y + zm.y));
                const double2 d = csub(z, zm);
                const double2 t = cmul(make_double2(0.5 * d.y, -0.5 * d.x), __ldg(&twx[k]));
                g[(size_t)ln * M + k] = cadd(ev, t);
                if (2 * k != M) g[(size_t)ln * M + (M - k)] = make_double2(ev.x - t.x, -(ev.y - t.y));
            }
        }
    }
}

// y columns: TC neighbouring packed pairs x all ny rows of one plane per CTA.  twy[k] = exp(-2 pi i k / ny).
// The first pass reads the rows from global memory, the last one stores them.
template <bool INV>
__global__ void __launch_bounds__(kMaxT) gen_fft_y_kernel(double *__restrict__ p, const double2 *__restrict__ twy, int nx, int ny, int tc, Radices rl)
{
    extern __shared__ double2 smem_gy[];
    double2 *gb = reinterpret_cast<double2 *>(p + (size_t)blockIdx.y * nx * ny) + (size_t)blockIdx.x * tc;
    const Side src{gb, 1, nx / 2, 1.0, INV ? -1.0 : 1.0}, dst{gb, 1, nx / 2, 1.0, INV ? -1.0 : 1.0}, mid{smem_gy, 1, tc, 1.0, 1.0};
    all_passes(src, mid, dst, ny, tc, true, twy, 1, rl);
}

// ---------------------------------------------------------------------------------------------
// Cosine / sine expansions ("Fourier / cosine / sine"; reading R17) for
// directions with zero-gradient (N) or zero-value (D) ends, through the same passes:
//   C_k = sum_i x_i cos(pi k (i + 1/2) / L)  =  (1/2) [w_k V_k + conj(w_k) V_{L-k}],  w_k = exp(-i pi k / (2L)),
//   V = FFT_L(v),  v_m = x_{2m},  v_{L-1-m} = x_{2m+1}                     (reordering of Makhoul)
// a complex-linear identity, so a complex column (two real sequences) transforms in one go;
//   S_k = sum_i x_i sin(pi (k+1) (i + 1/2) / L) = C_{L-1-k} of (-1)^i x_i.
// Inverse: V_0 = C_0, V_k = conj(w_k) (C_k - i C_{L-k}), v = IFFT_L(V) (unnormalised: L v).
// tw4[k] = exp(-i pi k / (2L)).
__device__ __forceinline__ double2 mul_i(double2 a) { return make_double2(-a.y, a.x); }

template <bool INV>
__global__ void __launch_bounds__(kMaxT) gen_r2r_y_kernel(double *__restrict__ p, const double2 *__restrict__ twy, const double2 *__restrict__ tw4, int nx, int L,
                                                          int tc, Radices rl, int dirichlet)
{
    extern __shared__ double2 smem_ry[];
    const int kT = (int)blockDim.x;
    const Side mid{smem_ry, 1, tc, 1.0, 1.0};
    double *base = p + (size_t)blockIdx.y * nx * L + 2 * (size_t)blockIdx.x * tc;
    auto at = [&](int row, int c) { return reinterpret_cast<double2 *>(base + (size_t)row * nx + 2 * c); };
    if constexpr (!INV) {
        for (int q = threadIdx.x; q < L * tc; q += kT) {
            const int row = q / tc, c = q - row * tc;
            double2 t = *at(row, c);
            if (dirichlet && (row & 1)) t = make_double2(-t.x, -t.y);
            const int pos = (row & 1) ? L - 1 - (row >> 1) : (row >> 1);
            smem_ry[pos * tc + c] = t;
        }
        __syncthreads();
        all_passes(mid, mid, mid, L, tc, true, twy, 1, rl);
        for (int q = threadIdx.x; q < (L / 2 + 1) * tc; q += kT) {
            const int k = q / tc, c = q - k * tc;
            const double2 vk = smem_ry[k * tc + c];
            if (k == 0) {
                *at(dirichlet ? L - 1 : 0, c) = vk;
            } else {
                const double2 vm = smem_ry[(L - k) * tc + c], w = __ldg(&tw4[k]);
                const double2 a = cmul(vk, w), b = cmul_conj(vm, w);
                const double2 ck = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y + b.y));
                const double2 cm = mul_i(make_double2(0.5 * (a.x - b.x), 0.5 * (a.y - b.y)));
                *at(dirichlet ? L - 1 - k : k, c) = ck;
                if (k != L - k) *at(dirichlet ? k - 1 : L - k, c) = cm;
            }
        }
    } else {
        for (int q = threadIdx.x; q < L * tc; q += kT) {
            const int k = q / tc, c = q - k * tc;
            smem_ry[q] = *at(dirichlet ? L - 1 - k : k, c);
        }
        __syncthreads();
        double2 va[(kE + 1) / 2 + 1], vb[(kE + 1) / 2 + 1];
#pragma unroll
        for (int e = 0; e < (kE + 1) / 2 + 1; ++e) {
            const int q = threadIdx.x + e * kT;
            if (q < (L / 2 + 1) * tc) {
                const int k = q / tc, c = q - k * tc;
                const double2 xk = smem_ry[k * tc + c];
                if (k == 0) {
                    va[e] = xk;
                } else {
                    const double2 xm = smem_ry[(L - k) * tc + c], w = __ldg(&tw4[k]);
                    // V_k = conj(w_k) (C_k - i C_{L-k}),  V_{L-k} = w_k (C_k + i C_{L-k})
                    va[e] = cmul_conj(make_double2(xk.x + xm.y, xk.y - xm.x), w);
                    vb[e] = cmul(make_double2(xk.x - xm.y, xk.y + xm.x), w);
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < (kE + 1) / 2 + 1; ++e) {
            const int q = threadIdx.x + e * kT;
            if (q < (L / 2 + 1) * tc) {
                const int k = q / tc, c = q - k * tc;
                smem_ry[k * tc + c] = cconj(va[e]);
                if (k != 0 && k != L - k) smem_ry[(L - k) * tc + c] = cconj(vb[e]);
            }
        }
        __syncthreads();
        all_passes(mid, mid, mid, L, tc, true, twy, 1, rl);
        for (int q = threadIdx.x; q < L * tc; q += kT) {
            const int row = q / tc, c = q - row * tc;
            const int pos = (row & 1) ? L - 1 - (row >> 1) : (row >> 1);
            double2 t = cconj(smem_ry[pos * tc + c]);
            if (dirichlet && (row & 1)) t = make_double2(-t.x, -t.y);
            *at(row, c) = t;
        }
    }
}

// The same expansions along x: lines of n = 2M REAL points.  The reordered line v is transformed
// as one complex transform of length M plus the real-to-complex split (as gen_fft_x_kernel), then
//   C_k = Re(w_k V_k),  C_{n-k} = -Im(w_k V_k)   (0 < k < M),  C_0 = V_0,  C_M = Re(w_M V_M);
// inverse: V_k = conj(w_k) (C_k - i C_{n-k}), complex-to-real merge, passes, un-reordering.
// Output / input: n real coefficients per line in natural order (sine: reversed, see above).
template <bool INV>
__global__ void __launch_bounds__(kMaxT) gen_r2r_x_kernel(double *__restrict__ p, const double2 *__restrict__ twx, const double2 *__restrict__ tw4, int M,
                                                          long long nlines, int lpb, Radices rl, double scale, int dirichlet)
{
    extern __shared__ double2 smem_rx[];
    const int kT = (int)blockDim.x;
    const Side mid{smem_rx, M, 1, 1.0, 1.0};
    double *sd = reinterpret_cast<double *>(smem_rx);
    const int n = 2 * M;
    const long long l0 = (long long)blockIdx.x * lpb;
    const int nl = (int)((nlines - l0 < lpb) ? nlines - l0 : lpb);
    double *g = p + (size_t)l0 * n;
    if constexpr (!INV) {
        for (int q = threadIdx.x; q < nl * n; q += kT) {
            const int ln = q / n, i = q - ln * n;
            double v = g[q];
            if (dirichlet && (i & 1)) v = -v;
            sd[ln * n + ((i & 1) ? n - 1 - (i >> 1) : (i >> 1))] = v;
        }
        __syncthreads();
        all_passes(mid, mid, mid, M, nl, false, twx, 2, rl);
        for (int q = threadIdx.x; q < nl * (M + 1); q += kT) {
            const int ln = q / (M + 1), k = q - ln * (M + 1);
            const double2 *z = smem_rx + (size_t)ln * M;
            double *o = g + (size_t)ln * n;
            auto put = [&](int coef, double val) { o[dirichlet ? n - 1 - coef : coef] = val; };
            if (k == 0) {
                put(0, z[0].x + z[0].y);
            } else if (k == M) {
                put(M, (z[0].x - z[0].y) * __ldg(&tw4[M]).x);
            } else {
                const double2 zk = z[k], zm = cconj(z[M - k]);
                const double2 ev = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y + zm.y));
                const double2 d = csub(zk, zm);
                const double2 vk = cadd(ev, cmul(make_double2(0.5 * d.y, -0.5 * d.x), __ldg(&twx[k])));
                const double2 t = cmul(vk, __ldg(&tw4[k]));
                put(k, t.x);
                put(n - k, -t.y);
            }
        }
    } else {
        for (int q = threadIdx.x; q < nl * n; q += kT) {
            const int ln = q / n, k = q - ln * n;
            sd[q] = g[(size_t)ln * n + (dirichlet ? n - 1 - k : k)];
        }
        __syncthreads();
        // half spectrum V_k (k = 0..M) of the real reordered line, merged into the complex line of length M
        double2 zr[kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int q = threadIdx.x + e * kT;
            if (q < nl * M) {
                const int ln = q / M, k = q - ln * M;
                const double *c = sd + (size_t)ln * n;
                auto V = [&](int kk) {   // kk in 1..M
                    const double2 w = __ldg(&tw4[kk]);
                    return cmul_conj(make_double2(c[kk], -c[n - kk]), w);
                };
                if (k == 0) {
                    const double v0 = c[0], vm = V(M).x;   // V_M is real
                    zr[e] = make_double2(v0 + vm, -(v0 - vm));
                } else {
                    const double2 xk = V(k), xm = cconj(V(M - k));
                    const double2 sm = cadd(xk, xm), cc = cmul_conj(csub(xk, xm), __ldg(&twx[k]));
                    zr[e] = make_double2(sm.x - cc.y, -(sm.y + cc.x));
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int q = threadIdx.x + e * kT;
            if (q < nl * M) smem_rx[q] = zr[e];
        }
        __syncthreads();
        all_passes(mid, mid, mid, M, nl, false, twx, 2, rl);
        for (int q = threadIdx.x; q < nl * n; q += kT) {
            const int ln = q / n, i = q - ln * n;
            const int pos = (i & 1) ? n - 1 - (i >> 1) : (i >> 1);
            double v = sd[ln * n + pos];
            if (pos & 1) v = -v;                       // imaginary parts come out conjugated
            if (dirichlet && (i & 1)) v = -v;
            g[q] = v * scale;
        }
    }
}

// Separation of the two real sequences held by EVERY packed pair after a complex transform along y
// (x expanded in cosines / sines: neighbouring columns are different real modes), as pair0_kernel
// of pz_fft_y.cu does for pair 0: rows (2r, 2r+1) hold (Re A_r, Re B_r), (Im A_r, Im B_r); rows
// 0, 1 hold r = 0, L/2.  One CTA per (pair, plane).
template <bool INV>
__global__ void __launch_bounds__(256) gen_allpairs_kernel(double *__restrict__ p, int nx, int L)
{
    extern __shared__ double2 smem_ap[];
    double *base = p + (size_t)blockIdx.y * nx * L + 2 * (size_t)blockIdx.x;
    auto at = [&](int row) { return reinterpret_cast<double2 *>(base + (size_t)row * nx); };
    for (int r = threadIdx.x; r < L; r += blockDim.x) smem_ap[r] = *at(r);
    __syncthreads();
    const int h = L / 2;
    for (int r = threadIdx.x; r <= h; r += blockDim.x) {
        if constexpr (!INV) {
            if (r == 0 || r == h) { *at(r == 0 ? 0 : 1) = smem_ap[r]; continue; }
            const double2 w = smem_ap[r], wm = cconj(smem_ap[L - r]);
            const double2 a = make_double2(0.5 * (w.x + wm.x), 0.5 * (w.y + wm.y));
            const double2 d = csub(w, wm);
            const double2 b = make_double2(0.5 * d.y, -0.5 * d.x);
            *at(2 * r) = make_double2(a.x, b.x);
            *at(2 * r + 1) = make_double2(a.y, b.y);
        } else {
            if (r == 0 || r == h) { *at(r) = smem_ap[r == 0 ? 0 : 1]; continue; }
            const double2 lo = smem_ap[2 * r], hi = smem_ap[2 * r + 1];
            *at(r) = make_double2(lo.x - hi.y, hi.x + lo.y);        // A_r + i B_r
            *at(L - r) = make_double2(lo.x + hi.y, lo.y - hi.x);    // conj(A_r) + i conj(B_r)
        }
    }
}

// Factorisation by a small cost model (shared-memory wavefronts per 32 points): 10 per pass (4 + 4
// for the reads and writes, 2 for the barriers) plus 4 per extra way of bank conflict of the FIRST
// pass, which writes with a stride of R elements (free of conflicts for odd R; later passes write
// runs of Ns consecutive elements).  Ties go to the most points per thread.  need_cap: a line (or
// tile) too long for 512 threads rules out the radices that keep fewer points per thread.
constexpr int kRadix[] = {16, 15, 14, 12, 10, 9, 8, 7, 6, 5, 4, 3, 2};
int points_per_thread(int R) { const int c = bfly_per_thread(R) * R; return c < kE ? c : kE; }

// bank-conflict ways of the first pass: 8 lanes of a quarter warp store 16-byte elements at
// (j R) sp + c, c < sp the line, j the butterfly
int first_pass_ways(int R, int sp)
{
    const int per = sp < 8 ? sp : 8;
    int hits[8] = {0}, ways = 1;
    for (int l = 0; l < 8; ++l) {
        const int c = l % per, j = l / per, unit = (j * R * sp + c) & 7;
        if (++hits[unit] > ways) ways = hits[unit];
    }
    return ways;
}

struct Search { int n, r[20], cost, cap, need_cap, sp; };
void search(int n, int start, int depth, int *cur, Search *best)
{
    if (n == 1) {
        int cap = kE, ways = 8;
        for (int i = 0; i < depth; ++i) {
            if (points_per_thread(cur[i]) < cap) cap = points_per_thread(cur[i]);
            if (first_pass_ways(cur[i], best->sp) < ways) ways = first_pass_ways(cur[i], best->sp);
        }
        const int cost = 10 * depth + 2 * (ways - 1);
        if (cost < best->cost || (cost == best->cost && cap > best->cap)) {
            best->n = depth;
            best->cost = cost;
            best->cap = cap;
            for (int i = 0; i < depth; ++i) best->r[i] = cur[i];
        }
        return;
    }
    if (10 * (depth + 1) > best->cost || depth >= 19) return;
    for (int i = start; i < (int)(sizeof(kRadix) / sizeof(kRadix[0])); ++i)
        if (n % kRadix[i] == 0 && points_per_thread(kRadix[i]) >= best->need_cap) {
            cur[depth] = kRadix[i];
            search(n / kRadix[i], i, depth + 1, cur, best);
        }
}

bool factor(int n, Radices *out, int need_cap = 1, int sp = 1)
{
    out->n = 0;
    if (n < 2 || need_cap > kE) return false;
    Search best;
    best.n = 0;
    best.cost = 1 << 30;
    best.cap = 0;
    best.need_cap = need_cap;
    best.sp = sp;
    int cur[20];
    search(n, 0, 0, cur, &best);
    if (best.n == 0) return false;
    // radices come out in descending order; the one with the fewest conflicts goes first
    int first = 0;
    for (int i = 1; i < best.n; ++i)
        if (first_pass_ways(best.r[i], sp) < first_pass_ways(best.r[first], sp)) first = i;
    const int f = best.r[first];
    for (int i = first; i > 0; --i) best.r[i] = best.r[i - 1];
    best.r[0] = f;
    out->n = best.n;
    for (int i = 0; i < best.n; ++i) out->r[i] = best.r[i];
    return true;
}

// threads a CTA needs for `pts` points: every pass must fit (one or a few butterflies per thread)
int threads_for(const Radices &rl, int pts)
{
    int t = (pts + kE - 1) / kE;
    for (int i = 0; i < rl.n; ++i) {
        const int R = rl.r[i], need = (pts / R + bfly_per_thread(R) - 1) / bfly_per_thread(R);
        if (need > t) t = need;
    }
    return (t + 31) / 32 * 32;
}

} // namespace

int fft_radices(int n, int min_points, int stride, int *radices, int cap)
{
    Radices r;
    if (!factor(n, &r, min_points < 1 ? 1 : min_points, stride < 1 ? 1 : stride)) return 0;
    for (int i = 0; i < r.n && i < cap; ++i) radices[i] = r.r[i];
    return r.n;
}

// lengths the mixed-radix kernels take: even, 7-smooth (nx / 2 resp. ny), a line within the
// 8192-point shared-memory buffer
bool generic_fft_x_ok(int nx)
{
    Radices r;
    const int M = nx / 2;
    return nx >= 8 && !(nx & 1) && M <= kPts && factor(M, &r, (M + kMaxT - 1) / kMaxT, 1) && threads_for(r, M) <= kMaxT;
}
bool generic_fft_y_ok(int ny)
{
    Radices r;
    return ny >= 8 && !(ny & 1) && ny <= kPts && factor(ny, &r, (ny + kMaxT - 1) / kMaxT, 1) && threads_for(r, ny) <= kMaxT;
}

// launch geometry of the x kernels: lines per CTA and threads per CTA, chosen for the most points
// in flight per SM (128 registers per thread: 512 threads per SM)
static int x_geometry(const pz_plan *pl, const Radices &rl, int M, long long nlines, int *lpb, int *kt)
{
    int best = 0, bl = 0;
    for (int l = 1; l <= 64 && l * M <= kPts; ++l) {
        const int pts = l * M, t = threads_for(rl, pts);
        if (t > kMaxT) continue;
        int ctas = kMaxT / t;
        const int by_smem = (227 * 1024) / (pts * (int)sizeof(double2) + 1024);
        if (by_smem < ctas) ctas = by_smem;
        if (ctas > 16) ctas = 16;
        // a lone CTA per SM cannot overlap its loads with another's passes
        const int value = ctas >= 2 ? ctas * pts : (ctas * pts * 5) / 8;
        if (value > best) { best = value; bl = l; }
    }
    if (!bl) { set_error("fft_x: nx = %d does not fit the %d-point buffer", 2 * M, kPts); return PZ_EUNSUPPORTED; }
    // keep the grid a few waves deep on small fields
    while (bl > 1 && (nlines + bl - 1) / bl < 4LL * pl->num_sms) bl /= 2;
    *lpb = bl;
    *kt = threads_for(rl, bl * M);
    return PZ_OK;
}

#define PZ_GEN_LAUNCH(KERNEL, GRID, SMEM, ...)                                                                 \
    do {                                                                                                        \
        int rc_;                                                                                                \
        if ((rc_ = smem_optin(pl, KERNEL<false>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc_;         \
        if ((rc_ = smem_optin(pl, KERNEL<true>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc_;          \
        if (inverse) KERNEL<true><<<GRID, kt, SMEM, st>>>(__VA_ARGS__);                                         \
        else KERNEL<false><<<GRID, kt, SMEM, st>>>(__VA_ARGS__);                                                \
        count_launch();                                                                                         \
        PZ_CUDA(cudaGetLastError());                                                                            \
    } while (0)

// radices + geometry of the x kernels (slot 0: Fourier, 2: cosine / sine), cached in the plan
static int x_setup(const pz_plan *pl, int slot, long long nlines, Radices *rl, int *lpb, int *kt)
{
    pz_plan::GenGeo &g = const_cast<pz_plan *>(pl)->gen_geo[slot];
    if (g.key != nlines) {
        const int M = pl->nx / 2;
        Radices r;
        if (!factor(M, &r, (M + kMaxT - 1) / kMaxT, 1)) {
            set_error("fft_x: nx / 2 = %d is not a product of 2, 3, 5, 7 that fits one CTA", M);
            return PZ_EUNSUPPORTED;
        }
        int l, t;
        const int rc = x_geometry(pl, r, M, nlines, &l, &t);
        if (rc != PZ_OK) return rc;
        g.n = r.n;
        for (int i = 0; i < r.n; ++i) g.r[i] = r.r[i];
        g.per_cta = l;
        g.threads = t;
        g.key = nlines;
    }
    rl->n = g.n;
    for (int i = 0; i < g.n; ++i) rl->r[i] = g.r[i];
    *lpb = g.per_cta;
    *kt = g.threads;
    return PZ_OK;
}

// radices + geometry of the y kernels (slot 1: Fourier, 3: cosine / sine): the widest rows (pairs
// per CTA) for which a factorisation fits 512 threads
static int y_setup(const pz_plan *pl, int slot, Radices *rl, int *tc, int *kt)
{
    pz_plan::GenGeo &g = const_cast<pz_plan *>(pl)->gen_geo[slot];
    if (g.key != 0) {
        const int L = pl->ny, npairs = pl->nx / 2;
        Radices r;
        int t = 8;
        for (;; t /= 2) {
            if (t == 0) { set_error("fft_y: ny = %d is not a product of 2, 3, 5, 7 that fits one CTA", L); return PZ_EUNSUPPORTED; }
            if (npairs % t != 0 || t * L > kPts) continue;
            if (factor(L, &r, (t * L + kMaxT - 1) / kMaxT, t) && threads_for(r, t * L) <= kMaxT) break;
        }
        g.n = r.n;
        for (int i = 0; i < r.n; ++i) g.r[i] = r.r[i];
        g.per_cta = t;
        g.threads = threads_for(r, t * L);
        g.key = 0;
    }
    rl->n = g.n;
    for (int i = 0; i < g.n; ++i) rl->r[i] = g.r[i];
    *tc = g.per_cta;
    *kt = g.threads;
    return PZ_OK;
}

int launch_fft_x_generic(const pz_plan *pl, double *p, long long nlines, bool inverse, cudaStream_t st)
{
    const int M = pl->nx / 2;
    Radices rl;
    int lpb, kt, rc;
    if ((rc = x_setup(pl, 0, nlines, &rl, &lpb, &kt)) != PZ_OK) return rc;
    const size_t smem = (size_t)lpb * M * sizeof(double2);
    const unsigned blocks = (unsigned)((nlines + lpb - 1) / lpb);
    const double scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    ProfScope prof(pl, inverse ? PZ_K_FFT_X_INV : PZ_K_FFT_X_FWD, st);
    PZ_GEN_LAUNCH(gen_fft_x_kernel, blocks, smem, p, pl->d_twx, M, nlines, lpb, rl, scale);
    return PZ_OK;
}

int launch_fft_y_generic(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st)
{
    const int L = pl->ny;
    Radices rl;
    int tc, kt, rc;
    if ((rc = y_setup(pl, 1, &rl, &tc, &kt)) != PZ_OK) return rc;
    const size_t smem = (size_t)tc * L * sizeof(double2);
    dim3 grid((unsigned)(pl->nx / 2 / tc), (unsigned)nk);
    ProfScope prof(pl, inverse ? PZ_K_FFT_Y_INV : PZ_K_FFT_Y_FWD, st);
    PZ_GEN_LAUNCH(gen_fft_y_kernel, grid, smem, p, pl->d_twy, pl->nx, L, tc, rl);
    return PZ_OK;
}

// ---- cosine / sine expansions (bcx / bcy = PZ_NEUMANN, PZ_DIRICHLET)
int launch_r2r_x(const pz_plan *pl, double *p, long long nlines, bool inverse, cudaStream_t st)
{
    const int M = pl->nx / 2;
    Radices rl;
    int lpb, kt, rc;
    if ((rc = x_setup(pl, 2, nlines, &rl, &lpb, &kt)) != PZ_OK) return rc;
    const size_t smem = (size_t)lpb * M * sizeof(double2);
    const unsigned blocks = (unsigned)((nlines + lpb - 1) / lpb);
    const double scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    const int dir = (pl->bcx == PZ_DIRICHLET) ? 1 : 0;
    ProfScope prof(pl, inverse ? PZ_K_FFT_X_INV : PZ_K_FFT_X_FWD, st);
    PZ_GEN_LAUNCH(gen_r2r_x_kernel, blocks, smem, p, pl->d_twx, pl->d_tw4x, M, nlines, lpb, rl, scale, dir);
    return PZ_OK;
}

int launch_r2r_y(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st)
{
    const int L = pl->ny;
    Radices rl;
    int tc, kt, rc;
    if ((rc = y_setup(pl, 3, &rl, &tc, &kt)) != PZ_OK) return rc;
    const size_t smem = (size_t)tc * L * sizeof(double2);
    const int dir = (pl->bcy == PZ_DIRICHLET) ? 1 : 0;
    dim3 grid((unsigned)(pl->nx / 2 / tc), (unsigned)nk);
    ProfScope prof(pl, inverse ? PZ_K_FFT_Y_INV : PZ_K_FFT_Y_FWD, st);
    PZ_GEN_LAUNCH(gen_r2r_y_kernel, grid, smem, p, pl->d_twy, pl->d_tw4y, pl->nx, L, tc, rl, dir);
    return PZ_OK;
}

// x in cosines / sines, y periodic: every pair of columns holds two real sequences
int launch_allpairs(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st)
{
    const size_t smem = (size_t)pl->ny * sizeof(double2);
    int rc;
    if ((rc = smem_optin(pl, gen_allpairs_kernel<false>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc;
    if ((rc = smem_optin(pl, gen_allpairs_kernel<true>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc;
    dim3 grid((unsigned)(pl->nx / 2), (unsigned)nk);
    ProfScope prof(pl, inverse ? PZ_K_PAIR0_INV : PZ_K_PAIR0_FWD, st);
    if (inverse) gen_allpairs_kernel<true><<<grid, 256, smem, st>>>(p, pl->nx, pl->ny);
    else gen_allpairs_kernel<false><<<grid, 256, smem, st>>>(p, pl->nx, pl->ny);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace pz
