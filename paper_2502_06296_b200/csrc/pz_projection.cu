// pz_projection.cu -- the steps either side of the Poisson solve: the
// right-hand side of Eq. (4), D u* / (gamma dt), and the correction of Eqs. (5)-(6),
// u -= gamma dt G Phi, p += Phi, on the staggered grid of PAPER.md:49.
//
// Index convention (reading R15): arrays are [k][j][i]; u on the x-face between cells i
// and i+1, v on the y-face between j and j+1 (both periodic), w on the z-face zf[k+1] (the bottom
// wall face carries w = 0 and is not stored, w[nz-1] is the top wall face), p and Phi at centres:
//   (D u)_ijk = (u_i - u_{i-1})/dx + (v_j - v_{j-1})/dy + (w_k - w_{k-1})/dzf_k
//   (G Phi)^x_i = (Phi_{i+1} - Phi_i)/dx, ^y likewise, ^z_k = (Phi_{k+1} - Phi_k)/dzc_k (0 at k = nz-1)
// so that D G is exactly the operator L_h of poisson_solve and the corrected velocity is
// divergence free to rounding.
//
// Both kernels are pure streaming stencils: one thread per pair of x-neighbours (16-byte accesses),
// the x / y / z neighbours come from L1 / L2.  Algorithmic bytes per point: 32 (three velocity
// reads, one write) and 72 (Phi, u, v, w, p read; u, v, w, p written).
#include "pz_internal.h"

namespace pz {

namespace {

__device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void st2(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }

__global__ void __launch_bounds__(256)
    divergence_rhs_kernel(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                          double *__restrict__ out, const double *__restrict__ dzf, int nx, int ny, int nz, double rdx,
                          double rdy, double scale)
{
    const size_t plane = (size_t)nx * ny, npairs = plane * nz / 2;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < npairs; q += (size_t)gridDim.x * blockDim.x) {
        const size_t c = 2 * q;
        const int i = (int)(c % nx);
        const size_t row = c / nx;
        const int j = (int)(row % ny), k = (int)(row / ny);
        const double2 uc = ld2(u + c), vc = ld2(v + c), wc = ld2(w + c);
        const double um = u[c - i + (i == 0 ? nx - 1 : i - 1)];
        const double2 vm = ld2(v + (j == 0 ? c + (size_t)(ny - 1) * nx : c - nx));
        double2 wm = make_double2(0.0, 0.0);
        if (k > 0) wm = ld2(w + c - plane);
        const double rdz = 1.0 / dzf[k];
        double2 d;
        d.x = ((uc.x - um) * rdx + (vc.x - vm.x) * rdy + (wc.x - wm.x) * rdz) * scale;
        d.y = ((uc.y - uc.x) * rdx + (vc.y - vm.y) * rdy + (wc.y - wm.y) * rdz) * scale;
        st2(out + c, d);
    }
}

__global__ void __launch_bounds__(256)
    project_kernel(double *__restrict__ u, double *__restrict__ v, double *__restrict__ w, double *__restrict__ p,
                   const double *__restrict__ phi, const double *__restrict__ zc, int nx, int ny, int nz, double gdx,
                   double gdy, double gdt)
{
    const size_t plane = (size_t)nx * ny, npairs = plane * nz / 2;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < npairs; q += (size_t)gridDim.x * blockDim.x) {
        const size_t c = 2 * q;
        const int i = (int)(c % nx);
        const size_t row = c / nx;
        const int j = (int)(row % ny), k = (int)(row / ny);
        const double2 f = ld2(phi + c);
        const double fxp = phi[c - i + (i + 2 == nx ? 0 : i + 2)];   // Phi_{i+2} for the second point
        const double2 fyp = ld2(phi + (j + 1 == ny ? c - (size_t)(ny - 1) * nx : c + nx));
        double2 uu = ld2(u + c), vv = ld2(v + c), pp = ld2(p + c);
        uu.x -= gdx * (f.y - f.x);
        uu.y -= gdx * (fxp - f.y);
        vv.x -= gdy * (fyp.x - f.x);
        vv.y -= gdy * (fyp.y - f.y);
        pp.x += f.x;
        pp.y += f.y;
        st2(u + c, uu);
        st2(v + c, vv);
        st2(p + c, pp);
        if (k + 1 < nz) {
            const double2 fzp = ld2(phi + c + plane);
            const double gz = gdt / (zc[k + 1] - zc[k]);
            double2 ww = ld2(w + c);
            ww.x -= gz * (fzp.x - f.x);
            ww.y -= gz * (fzp.y - f.y);
            st2(w + c, ww);
        }
    }
}

// Right-hand side of Eq. (11): r = u** - a L_z u^k, in place in u**, with
// (L_z q)_k = A_k (q_{k-1} - q_k) + C_k (q_{k+1} - q_k) - W_k q_k (Dirichlet walls, reading R7).
// Streaming z stencil: 24 algorithmic bytes per point (u**, u^k read; r written).
// Each thread owns one pair of x-neighbours and marches over kZChunk rows with u^k in a rolling
// window, so every value of u^k is read once (plus two halo rows per chunk).
constexpr int kZChunk = 32;

__global__ void __launch_bounds__(256)
    helmholtz_z_rhs_kernel(double *__restrict__ u2, const double *__restrict__ uk, const double *__restrict__ A,
                           const double *__restrict__ C, int nx, int ny, int nz, double a, double w0, double w1)
{
    const size_t plane = (size_t)nx * ny, ppairs = plane / 2;
    const size_t pr = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pr >= ppairs) return;
    const int kb = blockIdx.y * kZChunk, ke = min(kb + kZChunk, nz);
    const size_t c0 = 2 * pr;
    double2 qm = make_double2(0.0, 0.0), qc = ld2(uk + (size_t)kb * plane + c0);
    if (kb > 0) qm = ld2(uk + (size_t)(kb - 1) * plane + c0);
    for (int k = kb; k < ke; ++k) {
        const size_t c = (size_t)k * plane + c0;
        double2 qn = make_double2(0.0, 0.0);
        if (k + 1 < nz) qn = ld2(uk + c + plane);
        double2 lz = make_double2(0.0, 0.0);
        if (k > 0) {
            const double ak = A[k];
            lz.x += ak * (qm.x - qc.x);
            lz.y += ak * (qm.y - qc.y);
        }
        if (k + 1 < nz) {
            const double ck = C[k];
            lz.x += ck * (qn.x - qc.x);
            lz.y += ck * (qn.y - qc.y);
        }
        const double wk = (k == 0 ? w0 : 0.0) + (k == nz - 1 ? w1 : 0.0);
        lz.x -= wk * qc.x;
        lz.y -= wk * qc.y;
        double2 r = ld2(u2 + c);
        r.x -= a * lz.x;
        r.y -= a * lz.y;
        st2(u2 + c, r);
        qm = qc;
        qc = qn;
    }
}

int grid_for(const pz_plan *pl)
{
    const size_t npairs = pl->n / 2;
    size_t blocks = (npairs + 255) / 256;
    const size_t cap = (size_t)pl->num_sms * 16;
    return (int)(blocks < cap ? blocks : cap);
}

} // namespace

int launch_divergence_rhs(pz_plan *pl, const double *u, const double *v, const double *w, double *out, double inv_gdt,
                          cudaStream_t st)
{
    const double dx = pl->lx / pl->nx, dy = pl->ly / pl->ny;
    ProfScope prof(pl, PZ_K_DIV_RHS, st);
    divergence_rhs_kernel<<<grid_for(pl), 256, 0, st>>>(u, v, w, out, pl->d_dzf, pl->nx, pl->ny, pl->nz, 1.0 / dx, 1.0 / dy,
                                                        inv_gdt);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

int launch_helmholtz_z_rhs(pz_plan *pl, double *u2, const double *uk, double a, cudaStream_t st)
{
    ProfScope prof(pl, PZ_K_HELM_RHS, st);
    const size_t ppairs = (size_t)pl->nx * pl->ny / 2;
    const dim3 grid((unsigned)((ppairs + 255) / 256), (unsigned)((pl->nz + kZChunk - 1) / kZChunk));
    helmholtz_z_rhs_kernel<<<grid, 256, 0, st>>>(u2, uk, pl->d_A, pl->d_C, pl->nx, pl->ny, pl->nz, a, pl->wall_w0,
                                                         pl->wall_w1);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

int launch_project(pz_plan *pl, double *u, double *v, double *w, double *p, const double *phi, double gdt, cudaStream_t st)
{
    const double dx = pl->lx / pl->nx, dy = pl->ly / pl->ny;
    ProfScope prof(pl, PZ_K_PROJECT, st);
    project_kernel<<<grid_for(pl), 256, 0, st>>>(u, v, w, p, phi, pl->d_zc, pl->nx, pl->ny, pl->nz, gdt / dx, gdt / dy, gdt);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace pz
