// pz_zsolve_pair.cuh -- the per-warp cyclic-reduction solve of one complex column pair (step a3),
// shared by the two z-solve kernels (pz_zsolve_cr.cu: manual staging; pz_zsolve_tma.cu: TMA
// pipeline).  See pz_zsolve_cr.cu for the algorithm and pz_zsolve.cu for the
// M-matrix form that keeps the elimination free of cancellation.
#pragma once
#include <cuda_runtime.h>

namespace pz {

constexpr int kLanes = 32; // sub-domains per column = lanes of the warp that owns it

// 1/x to ~1 ulp: hardware seed r0 (relative error e0 <= ~2^-20: rcp.approx.ftz.f64 reads only the
// upper 32 bits of x) and one cubic step r0 (1 + e + e^2), e = 1 - x r0, which leaves e0^3 < 2^-59.
// x is a positive, normal pivot.
__device__ __forceinline__ double fast_rcp(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}

__device__ __forceinline__ double shfl_up(double v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ double shfl_down(double v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }

// One column pair, one sub-domain per lane.  d(i) is a reference to row i of this lane's
// sub-domain inside the tile (a double2: Re, Im of the pair).  al/ga: this lane's alpha_i, gamma_i (sub-/super-diagonal
// magnitudes, zero on padding rows and at the walls) in shared memory.  MASK bit 0 / 1: which
// component (x / y of the double2) is solved and written back.
//
// Sweeps (Algorithm 1 re-ordered so that only the pivot reciprocals are thread-private):
//   A  rows M-2..1, read only: UL elimination -> this sub-domain's row 0 in terms of
//      (x_{M-1} of the previous lane, x_0, x_{M-1})
//   B  rows 1..M-1, read only: LU elimination -> row M-1 in terms of (x_0, x_{M-1}, next x_0);
//      keeps rb_i = 1/pivot_i in registers.  A and B run interleaved (two independent chains).
//   reduced system across lanes (warp shuffles, parallel cyclic reduction)
//   C  rows 1..M-2 forward: g_i = (r_i + alpha_i g_{i-1}) rb_i with g_0 := x_0  (overwrites the tile)
//   D  rows M-2..1 backward: x_i = g_i + gamma_i rb_i x_{i+1}
// FULL: nz == 32 M and the column is not the pinned one: no padding rows, no row tests.
// HELM: the fully implicit Helmholtz system of Eq. (8), in the same M-matrix form:
//   -a A_k x_{k-1} + (a A_k + a C_k + ex0_k + a sigma) x_k - a C_k x_{k+1} = +d_k,
// al/ga hold a A_k / a C_k, ex0_k = 1 + a W_k (Dirichlet wall term), sigma is passed pre-scaled.
// OPEN: the rows of ONE z-slab of a distributed solve once the neighbouring
//   slabs' boundary values are known: the couplings of the first and last row to the rows outside
//   are on the right-hand side (bprev = A_first phi_prev, bnext = C_last phi_next, added to rows
//   0 and nz-1 of the slab), al / ga hold 0 there and ex0_k the diagonal excess they leave behind.
template <int M, int MASK, bool pin, bool FULL = false, bool HELM = false, bool OPEN = false, class Acc>
__device__ __forceinline__ void solve_pair(const Acc d, const double *al, const double *ga, double sigma,
                                           int k0, int nz, const double *__restrict__ dzf, double inv_lz,
                                           const double *ex0 = nullptr, double2 bprev = make_double2(0.0, 0.0),
                                           double2 bnext = make_double2(0.0, 0.0))
{
    static_assert(!(HELM && (pin || FULL)), "the Helmholtz system has no pinned column and takes the general path");
    static_assert(!(OPEN && (pin || FULL || HELM)), "a slab takes the general path");
    // row coefficients: real rows have excess sigma, padding rows (k >= nz) are x = 0,
    // the pinned row (gauge of the singular column) likewise.
    static_assert(!(FULL && pin), "the pinned column takes the general path");
    auto eps_of = [&](int i) {
        if constexpr (FULL) return sigma;
        else if constexpr (HELM || OPEN) return (k0 + i < nz) ? ex0[i] + sigma : 1.0;
        else return (k0 + i < nz && !(pin && k0 + i == nz - 1)) ? sigma : 1.0;
    };
    auto alpha_of = [&](int i) { return (pin && k0 + i == nz - 1) ? 0.0 : al[i]; };
    auto rhs_of = [&](int i) {
        const double2 v = d(i);
        if constexpr (FULL) {
            return make_double2(-v.x, -v.y);
        } else {
            const bool live = (k0 + i < nz) && !(pin && k0 + i == nz - 1);
            if constexpr (HELM) {
                return live ? v : make_double2(0.0, 0.0);
            } else if constexpr (OPEN) {
                double2 r = live ? make_double2(-v.x, -v.y) : make_double2(0.0, 0.0);
                if (k0 + i == 0) { r.x += bprev.x; r.y += bprev.y; }
                if (k0 + i == nz - 1) { r.x += bnext.x; r.y += bnext.y; }
                return r;
            } else {
                return live ? make_double2(-v.x, -v.y) : make_double2(0.0, 0.0);
            }
        }
    };

    // ---- sweeps A (UL, descending) and B (LU, ascending), interleaved
    double rb[M];
    double chat = ga[M - 2], eps2 = eps_of(M - 2);
    double2 rp2 = rhs_of(M - 2);
    double rb2 = fast_rcp(alpha_of(M - 2) + chat + eps2);
    double ahat = alpha_of(1), eps = eps_of(1);
    double2 rp = rhs_of(1);
    rb[1] = fast_rcp(ahat + ga[1] + eps);
#pragma unroll
    for (int t = 0; t < M - 2; ++t) {
        {   // A: row i = M-3-t (for t < M-3)
            const int i = M - 3 - t;
            if (i >= 1) {
                const double nn = ga[i] * rb2;
                const double2 r = rhs_of(i);
                chat = nn * chat;
                eps2 = fma(nn, eps2, eps_of(i));
                rp2.x = fma(nn, rp2.x, r.x);
                rp2.y = fma(nn, rp2.y, r.y);
                rb2 = fast_rcp(alpha_of(i) + chat + eps2);
            }
        }
        {   // B: row i = 2+t
            const int i = 2 + t;
            const double mm = alpha_of(i) * rb[i - 1];
            const double2 r = rhs_of(i);
            ahat = mm * ahat;
            eps = fma(mm, eps, eps_of(i));
            rp.x = fma(mm, rp.x, r.x);
            rp.y = fma(mm, rp.y, r.y);
            rb[i] = fast_rcp(ahat + ga[i] + eps);
        }
    }
    // normalised row 0:  -a0 X_{s-1} + x_0 - c0 X_s = r0, excess e0
    double a0, c0, e0;
    double2 r0;
    {
        const double nn = ga[0] * rb2;
        const double2 r = rhs_of(0);
        a0 = alpha_of(0);
        c0 = nn * chat;
        e0 = fma(nn, eps2, eps_of(0));
        r0.x = fma(nn, rp2.x, r.x);
        r0.y = fma(nn, rp2.y, r.y);
        const double rbn = fast_rcp(a0 + c0 + e0);
        a0 *= rbn; c0 *= rbn; e0 *= rbn; r0.x *= rbn; r0.y *= rbn;
    }
    // normalised last row:  -a x_0 + X_s - c (next lane's x_0) = r, excess e
    double a = ahat * rb[M - 1], c = ga[M - 1] * rb[M - 1], e = eps * rb[M - 1];
    double2 r = make_double2(rp.x * rb[M - 1], rp.y * rb[M - 1]);

    // ---- reduced system: first eliminate the x_0 unknowns (local row 0 and the next lane's)
    {
        const double c0n = shfl_down(c0, 1), e0n = shfl_down(e0, 1);
        const double r0nx = shfl_down(r0.x, 1), r0ny = shfl_down(r0.y, 1);
        const double k1 = a, k2 = c; // c = 0 on the last lane (wall or padding)
        a = k1 * a0;
        c = k2 * c0n;
        e = fma(k1, e0, fma(k2, e0n, e));
        r.x = fma(k1, r0.x, fma(k2, r0nx, r.x));
        r.y = fma(k1, r0.y, fma(k2, r0ny, r.y));
        const double rbn = fast_rcp(a + c + e);
        a *= rbn; c *= rbn; e *= rbn; r.x *= rbn; r.y *= rbn;
    }
    // ---- parallel cyclic reduction across the 32 lanes (unknown X_s = last row of lane s)
#pragma unroll
    for (int h = 1; h < kLanes; h *= 2) {
        const double am = shfl_up(a, h), em = shfl_up(e, h), rmx = shfl_up(r.x, h), rmy = shfl_up(r.y, h);
        const double cp = shfl_down(c, h), ep = shfl_down(e, h), rpx = shfl_down(r.x, h), rpy = shfl_down(r.y, h);
        // a == 0 whenever lane-h < 0 and c == 0 whenever lane+h > 31, so out-of-range partners
        // (whose shuffled values are the lane's own, finite) contribute nothing.
        const double k1 = a, k2 = c;
        a = k1 * am;
        c = k2 * cp;
        e = fma(k1, em, fma(k2, ep, e));
        r.x = fma(k1, rmx, fma(k2, rpx, r.x));
        r.y = fma(k1, rmy, fma(k2, rpy, r.y));
        const double rbn = fast_rcp(a + c + e);
        a *= rbn; c *= rbn; e *= rbn; r.x *= rbn; r.y *= rbn;
    }
    // r = X_s.  x_0 of this lane from its normalised row 0:  x_0 = r0 + a0 X_{s-1} + c0 X_s
    const double xpx = shfl_up(r.x, 1), xpy = shfl_up(r.y, 1); // lane 0: a0 = 0
    const double2 x0 = make_double2(fma(a0, xpx, fma(c0, r.x, r0.x)), fma(a0, xpy, fma(c0, r.y, r0.y)));

    double2 wsum = make_double2(0.0, 0.0);
    auto put = [&](int i, double2 val) {
        double2 t = val;
        if (MASK != 3) {
            t = d(i);
            if (MASK & 1) t.x = val.x;
            if (MASK & 2) t.y = val.y;
        }
        d(i) = t;
    };
    auto acc = [&](int i, double2 val) {
        if (pin && k0 + i < nz) wsum.x = fma(dzf[k0 + i], val.x, wsum.x);
    };

    // ---- sweep C: forward substitution of the right-hand side with x_0 known
    // (rows 1..M-2; unmasked components of the tile stay untouched)
    double2 gprev = x0;
#pragma unroll
    for (int i = 1; i <= M - 2; ++i) {
        const double2 rr = rhs_of(i);
        const double av = alpha_of(i);
        gprev.x = fma(av, gprev.x, rr.x) * rb[i];
        gprev.y = fma(av, gprev.y, rr.y) * rb[i];
        put(i, gprev);
    }
    // ---- sweep D: back substitution
    double2 x = r;
    put(M - 1, x);
    acc(M - 1, x);
#pragma unroll
    for (int i = M - 2; i >= 1; --i) {
        const double2 gi = d(i);
        const double w = ga[i] * rb[i];
        x.x = fma(w, x.x, gi.x);
        x.y = fma(w, x.y, gi.y);
        put(i, x);
        acc(i, x);
    }
    put(0, x0);
    acc(0, x0);

    if constexpr (pin) {
        // zero volume mean of the (0,0) mode: subtract sum_k dzf_k phi_k / sum_k dzf_k
        double s = wsum.x;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        s *= inv_lz;
#pragma unroll
        for (int i = 0; i < M; ++i)
            if (k0 + i < nz) d(i).x -= s;
    }
}

// Slab-local reduction of one column pair (or of its coefficient right-hand sides), one
// sub-domain of M rows per lane: sweeps A / B of solve_pair with NC right-hand-side components,
// the lane-boundary system by warp-shuffle PCR, then the first (F) and last (L) value of the
// slab's solution.  rhs(i, out): the NC components of row i of this lane (0 on padding rows).
template <int M, int NC, class Rhs>
__device__ __forceinline__ void reduce_pair(const double *al, const double *ga, const double *ex, double sigma, int k0,
                                            int nk, Rhs rhs, double (&F)[NC], double (&L)[NC])
{
    auto eps_of = [&](int i) { return (k0 + i < nk) ? ex[i] + sigma : 1.0; };
    const int lane = threadIdx.x & 31;
    double rp2[NC], rp[NC], t[NC], rcap[NC];
    double chat = ga[M - 2], eps2 = eps_of(M - 2);
    rhs(M - 2, rp2);
    double rb2 = fast_rcp(al[M - 2] + chat + eps2);
    double ahat = al[1], eps = eps_of(1);
    rhs(1, rp);
    double rbp = fast_rcp(ahat + ga[1] + eps);
    double acap = 0.0;
#pragma unroll
    for (int c = 0; c < NC; ++c) rcap[c] = 0.0;
    auto capture = [&](int i) {
        if (k0 + i == nk - 1) {
            acap = ahat * rbp;
#pragma unroll
            for (int c = 0; c < NC; ++c) rcap[c] = rp[c] * rbp;
        }
    };
    capture(1);
#pragma unroll
    for (int s = 0; s < M - 2; ++s) {
        {   // A: row i = M-3-s
            const int i = M - 3 - s;
            if (i >= 1) {
                const double nn = ga[i] * rb2;
                rhs(i, t);
                chat = nn * chat;
                eps2 = fma(nn, eps2, eps_of(i));
#pragma unroll
                for (int c = 0; c < NC; ++c) rp2[c] = fma(nn, rp2[c], t[c]);
                rb2 = fast_rcp(al[i] + chat + eps2);
            }
        }
        {   // B: row i = 2+s
            const int i = 2 + s;
            const double mm = al[i] * rbp;
            rhs(i, t);
            ahat = mm * ahat;
            eps = fma(mm, eps, eps_of(i));
#pragma unroll
            for (int c = 0; c < NC; ++c) rp[c] = fma(mm, rp[c], t[c]);
            rbp = fast_rcp(ahat + ga[i] + eps);
            capture(i);
        }
    }
    // normalised row 0:  -a0 X_{s-1} + x_0 - c0 X_s = r0, excess e0
    double a0, c0, e0, r0[NC];
    {
        const double nn = ga[0] * rb2;
        rhs(0, t);
        a0 = al[0];
        c0 = nn * chat;
        e0 = fma(nn, eps2, eps_of(0));
        const double rbn = fast_rcp(a0 + c0 + e0);
#pragma unroll
        for (int c = 0; c < NC; ++c) r0[c] = fma(nn, rp2[c], t[c]) * rbn;
        a0 *= rbn; c0 *= rbn; e0 *= rbn;
    }
    // normalised last row:  -a x_0 + X_s - c (next lane's x_0) = r, excess e
    double a = ahat * rbp, c = ga[M - 1] * rbp, e = eps * rbp, r[NC];
#pragma unroll
    for (int q = 0; q < NC; ++q) r[q] = rp[q] * rbp;
    // eliminate the x_0 unknowns (local row 0 and the next lane's)
    {
        const double c0n = shfl_down(c0, 1), e0n = shfl_down(e0, 1);
        const double k1 = a, k2 = c;
#pragma unroll
        for (int q = 0; q < NC; ++q) r[q] = fma(k1, r0[q], fma(k2, shfl_down(r0[q], 1), r[q]));
        a = k1 * a0;
        c = k2 * c0n;
        e = fma(k1, e0, fma(k2, e0n, e));
        const double rbn = fast_rcp(a + c + e);
        a *= rbn; c *= rbn; e *= rbn;
#pragma unroll
        for (int q = 0; q < NC; ++q) r[q] *= rbn;
    }
#pragma unroll
    for (int h = 1; h < kLanes; h *= 2) {
        const double am = shfl_up(a, h), em = shfl_up(e, h);
        const double cp = shfl_down(c, h), ep = shfl_down(e, h);
        const double k1 = a, k2 = c;
#pragma unroll
        for (int q = 0; q < NC; ++q) r[q] = fma(k1, shfl_up(r[q], h), fma(k2, shfl_down(r[q], h), r[q]));
        a = k1 * am;
        c = k2 * cp;
        e = fma(k1, em, fma(k2, ep, e));
        const double rbn = fast_rcp(a + c + e);
        a *= rbn; c *= rbn; e *= rbn;
#pragma unroll
        for (int q = 0; q < NC; ++q) r[q] *= rbn;
    }
    // r = X_s (last row of lane s); x_0 = r0 + a0 X_{s-1} + c0 X_s (lane 0: a0 = 0)
    const int sL = (nk - 1) / M, iL = (nk - 1) - sL * M;
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        const double x0 = fma(a0, shfl_up(r[q], 1), fma(c0, r[q], r0[q]));
        // last real row: x_0 of its lane if it is the lane's row 0, else (sweep B, row iL) rcap + acap x_0
        const double lv = (iL == 0) ? x0 : fma(acap, x0, rcap[q]);
        F[q] = __shfl_sync(0xffffffffu, x0, 0);
        L[q] = __shfl_sync(0xffffffffu, lv, sL);
    }
    (void)lane;
}

} // namespace pz
