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
constexpr int kPts = 512 * kE;   // largest buffer: 512 threads
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

// One in-place pass over `nlines` lines of complex length L in shared memory; element pos of line
// ln sits at s[ln * sl + pos * sp].  tw[k * tws] = exp(-2 pi i k / L).
template <int R, int kT>
__device__ __forceinline__ void pass(double2 *s, int L, int Ns, int nlines, int sl, int sp, const double2 *__restrict__ tw, int tws)
{
    constexpr int Q = (kE + R - 1) / R;
    const int nb = L / R, W = nlines * nb, step = (L / (Ns * R)) * tws;
    const int instr = nb * sp, outstr = Ns * sp;
    double2 v[Q][R];
    int obase[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        // work items past the end recompute item 0 and store nothing (no divergent definitions)
        const int w0 = (int)threadIdx.x + q * kT, w = (w0 < W) ? w0 : 0;
        // lines fastest when they are interleaved in memory (sl == 1), butterflies fastest otherwise
        const int ln = (sl == 1) ? w % nlines : w / nb, j = (sl == 1) ? w / nlines : w % nb;
        const int jm = j % Ns;
        const double2 *x = s + (ln * sl + j * sp);
        obase[q] = (w0 < W) ? ln * sl + ((j - jm) * R + jm) * sp : -1;
        const int tstep = jm * step;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double2 t = x[r * instr];
            if (r > 0) t = cmul(t, __ldg(&tw[r * tstep]));
            v[q][r] = t;
        }
        dft<R>(v[q]);
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        if (obase[q] >= 0) {
            double2 *y = s + obase[q];
#pragma unroll
            for (int r = 0; r < R; ++r) y[r * outstr] = v[q][r];
        }
    }
    __syncthreads();
}

template <int kT>
__device__ __forceinline__ void all_passes(double2 *s, int L, int nlines, int sl, int sp, const double2 *__restrict__ tw, int tws,
                                           const Radices &rl)
{
    int Ns = 1;
    for (int i = 0; i < rl.n; ++i) {
        switch (rl.r[i]) {
        case 2: pass<2, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        case 3: pass<3, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        case 4: pass<4, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        case 5: pass<5, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        case 7: pass<7, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        case 16: pass<16, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        default: pass<8, kT>(s, L, Ns, nlines, sl, sp, tw, tws); break;
        }
        Ns *= rl.r[i];
    }
}

// x lines: lpb lines of n = 2M reals per CTA.  twx[k] = exp(-2 pi i k / n).
template <bool INV, int kT>
__global__ void __launch_bounds__(kT, kT == 256 ? 2 : 1) gen_fft_x_kernel(double *__restrict__ p, const double2 *__restrict__ twx, int M, long long nlines,
                                                        int lpb, Radices rl, double scale)
{
    extern __shared__ double2 smem_gx[];
    const long long l0 = (long long)blockIdx.x * lpb;
    const int nl = (int)((nlines - l0 < lpb) ? nlines - l0 : lpb);
    double2 *g = reinterpret_cast<double2 *>(p) + (size_t)l0 * M;
    for (int q = threadIdx.x; q < nl * M; q += kT) {
        const int ln = q / M, k = q - ln * M;
        double2 z = g[q];
        if constexpr (INV) {
            // merge of the complex-to-real transform, conjugated (inverse through the forward passes)
            if (k == 0) {
                z = make_double2(z.x + z.y, -(z.x - z.y));
            } else {
                const double2 xm = cconj(g[(size_t)ln * M + (M - k)]);
                const double2 sm = cadd(z, xm), c = cmul_conj(csub(z, xm), __ldg(&twx[k]));
                z = make_double2(sm.x - c.y, -(sm.y + c.x));
            }
        }
        smem_gx[q] = z;
    }
    __syncthreads();
    all_passes<kT>(smem_gx, M, nl, M, 1, twx, 2, rl);
    for (int q = threadIdx.x; q < nl * M; q += kT) {
        const int ln = q / M, k = q - ln * M;
        const double2 z = smem_gx[q];
        double2 o;
        if constexpr (INV) {
            o = make_double2(z.x * scale, -z.y * scale);
        } else if (k == 0) {
            o = make_double2(z.x + z.y, z.x - z.y); // Re X_0, Re X_{n/2}
        } else {
            // split: X_k = (Z_k + conj Z_{M-k}) / 2 - (i/2) w_n^k (Z_k - conj Z_{M-k})
            const double2 zm = cconj(smem_gx[ln * M + (M - k)]);
            const double2 ev = make_double2(0.5 * (z.x + zm.x), 0.5 * (z.y + zm.y));
            const double2 d = csub(z, zm);
            o = cadd(ev, cmul(make_double2(0.5 * d.y, -0.5 * d.x), __ldg(&twx[k])));
        }
        g[q] = o;
    }
}

// y columns: TC neighbouring packed pairs x all ny rows of one plane per CTA.  twy[k] = exp(-2 pi i k / ny).
template <bool INV, int kT>
__global__ void __launch_bounds__(kT, kT == 256 ? 2 : 1) gen_fft_y_kernel(double *__restrict__ p, const double2 *__restrict__ twy, int nx, int ny, int tc,
                                                        Radices rl)
{
    extern __shared__ double2 smem_gy[];
    double *base = p + (size_t)blockIdx.y * nx * ny + 2 * (size_t)blockIdx.x * tc;
    for (int q = threadIdx.x; q < ny * tc; q += kT) {
        const int row = q / tc, c = q - row * tc;
        const double2 t = *reinterpret_cast<const double2 *>(base + (size_t)row * nx + 2 * c);
        smem_gy[q] = INV ? cconj(t) : t;
    }
    __syncthreads();
    all_passes<kT>(smem_gy, ny, tc, 1, tc, twy, 1, rl);
    for (int q = threadIdx.x; q < ny * tc; q += kT) {
        const int row = q / tc, c = q - row * tc;
        const double2 t = smem_gy[q];
        *reinterpret_cast<double2 *>(base + (size_t)row * nx + 2 * c) = INV ? cconj(t) : t;
    }
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

template <bool INV, int kT>
__global__ void __launch_bounds__(kT, kT == 256 ? 2 : 1) gen_r2r_y_kernel(double *__restrict__ p, const double2 *__restrict__ twy, const double2 *__restrict__ tw4,
                                                        int nx, int L, int tc, Radices rl, int dirichlet)
{
    extern __shared__ double2 smem_ry[];
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
        all_passes<kT>(smem_ry, L, tc, 1, tc, twy, 1, rl);
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
        all_passes<kT>(smem_ry, L, tc, 1, tc, twy, 1, rl);
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
template <bool INV, int kT>
__global__ void __launch_bounds__(kT, kT == 256 ? 2 : 1) gen_r2r_x_kernel(double *__restrict__ p, const double2 *__restrict__ twx, const double2 *__restrict__ tw4,
                                                        int M, long long nlines, int lpb, Radices rl, double scale, int dirichlet)
{
    extern __shared__ double2 smem_rx[];
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
        all_passes<kT>(smem_rx, M, nl, M, 1, twx, 2, rl);
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
        all_passes<kT>(smem_rx, M, nl, M, 1, twx, 2, rl);
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

bool factor(int n, Radices *out)
{
    out->n = 0;
    // odd radices first: their strided writes of the first pass are free of bank conflicts
    for (int f : {7, 5, 3})
        while (n % f == 0) { out->r[out->n++] = f; n /= f; }
    while (n % 16 == 0) { out->r[out->n++] = 16; n /= 16; }
    while (n % 8 == 0) { out->r[out->n++] = 8; n /= 8; }
    if (n % 4 == 0) { out->r[out->n++] = 4; n /= 4; }
    if (n % 2 == 0) { out->r[out->n++] = 2; n /= 2; }
    return n == 1 && out->n <= 20;
}

} // namespace

// lengths the mixed-radix kernels take: even, 7-smooth (nx / 2 resp. ny), a line within the
// 8192-point shared-memory buffer
bool generic_fft_x_ok(int nx)
{
    Radices r;
    return nx >= 8 && !(nx & 1) && nx / 2 <= kPts && factor(nx / 2, &r);
}
bool generic_fft_y_ok(int ny)
{
    Radices r;
    return ny >= 8 && !(ny & 1) && ny <= kPts && factor(ny, &r);
}

// launch geometry of the x kernels: lines per CTA and threads per CTA
static void x_geometry(const pz_plan *pl, int M, long long nlines, int *lpb, int *kt)
{
    *kt = (M <= 256 * kE) ? 256 : 512;
    int l = (*kt * kE) / M;
    if (l > 64) l = 64;
    // keep the grid a few waves deep on small fields
    while (l > 1 && (nlines + l - 1) / l < 4LL * pl->num_sms) l /= 2;
    *lpb = l;
}

// pairs per CTA and threads per CTA of the y kernels: rows as wide as the buffer allows (<= 128 bytes)
static int y_geometry(const pz_plan *pl, int L, int *tc, int *kt)
{
    const int npairs = pl->nx / 2;
    int t = 8;
    while (t > 1 && (npairs % t != 0 || t * L > kPts)) t /= 2;
    if (t * L > kPts) { set_error("fft_y: ny = %d exceeds the %d-point buffer", L, kPts); return PZ_EUNSUPPORTED; }
    *tc = t;
    *kt = (t * L <= 256 * kE) ? 256 : 512;
    return PZ_OK;
}

#define PZ_GEN_LAUNCH(KERNEL, GRID, SMEM, ...)                                                                    \
    do {                                                                                                           \
        int rc_;                                                                                                   \
        if (kt == 256) {                                                                                           \
            if ((rc_ = smem_optin(pl, KERNEL<false, 256>, (size_t)256 * kE * sizeof(double2))) != PZ_OK) return rc_; \
            if ((rc_ = smem_optin(pl, KERNEL<true, 256>, (size_t)256 * kE * sizeof(double2))) != PZ_OK) return rc_;  \
            if (inverse) KERNEL<true, 256><<<GRID, 256, SMEM, st>>>(__VA_ARGS__);                                  \
            else KERNEL<false, 256><<<GRID, 256, SMEM, st>>>(__VA_ARGS__);                                         \
        } else {                                                                                                   \
            if ((rc_ = smem_optin(pl, KERNEL<false, 512>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc_;   \
            if ((rc_ = smem_optin(pl, KERNEL<true, 512>, (size_t)kPts * sizeof(double2))) != PZ_OK) return rc_;    \
            if (inverse) KERNEL<true, 512><<<GRID, 512, SMEM, st>>>(__VA_ARGS__);                                  \
            else KERNEL<false, 512><<<GRID, 512, SMEM, st>>>(__VA_ARGS__);                                         \
        }                                                                                                          \
        count_launch();                                                                                            \
        PZ_CUDA(cudaGetLastError());                                                                               \
    } while (0)

int launch_fft_x_generic(const pz_plan *pl, double *p, long long nlines, bool inverse, cudaStream_t st)
{
    const int M = pl->nx / 2;
    Radices rl;
    if (!factor(M, &rl)) { set_error("fft_x: nx / 2 = %d has a prime factor above 7", M); return PZ_EUNSUPPORTED; }
    int lpb, kt;
    x_geometry(pl, M, nlines, &lpb, &kt);
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
    if (!factor(L, &rl)) { set_error("fft_y: ny = %d has a prime factor above 7", L); return PZ_EUNSUPPORTED; }
    int tc, kt;
    const int rc = y_geometry(pl, L, &tc, &kt);
    if (rc != PZ_OK) return rc;
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
    if (!factor(M, &rl)) { set_error("r2r_x: nx / 2 = %d has a prime factor above 7", M); return PZ_EUNSUPPORTED; }
    int lpb, kt;
    x_geometry(pl, M, nlines, &lpb, &kt);
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
    if (!factor(L, &rl)) { set_error("r2r_y: ny = %d has a prime factor above 7", L); return PZ_EUNSUPPORTED; }
    int tc, kt;
    const int rc = y_geometry(pl, L, &tc, &kt);
    if (rc != PZ_OK) return rc;
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
