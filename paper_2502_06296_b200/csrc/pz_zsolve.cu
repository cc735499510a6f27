// pz_zsolve.cu -- step a3 of the hot path: one real tridiagonal solve along z per spectral
// column (Eq. 12; steps 4-6 of PAPER.md:127-129):
//     A_k phi_{k-1} + (-(A_k+C_k) + lambda) phi_k + C_k phi_{k+1} = d_k,   lambda = lambda_x + lambda_y.
// Real and imaginary parts are separate real systems with the same matrix.
//
// Numerics (reading R5).  Every row is kept in M-matrix form
//     -alpha x_{k-1} + (alpha + gamma + eps) x_k - gamma x_{k+1} = r,   alpha, gamma, eps >= 0,
// with the excess eps (= sigma = -lambda at the start) carried explicitly.  Elimination then
// only ever ADDS non-negative numbers (eps' = eps + m eps_prev), so the near-singular low modes
// on strongly stretched grids are solved to ~1e-14 instead of ~1e-11 (forming -(A+C)+lambda in
// double and subtracting loses 4-5 digits).
//
// Variant 0 (this file, reference variant): one thread per column, serial Thomas sweeps through
// global memory ("each i,j index is assigned to a thread, which serially performs
// operations along the third domain direction"), forward result and C_k/p_k staged in HBM.
// Variant 1 (pz_zsolve_cr.cu): chunked cyclic reduction in shared memory (Algorithm 1).
#include "pz_internal.h"
#include "pz_zsolve_pair.cuh"

namespace pz {

int launch_zsolve_cr(pz_plan *pl, double *p, cudaStream_t st, double helm_a);
int launch_zsolve_tma(pz_plan *pl, double *p, cudaStream_t st, double helm_a);

namespace {

__global__ void __launch_bounds__(128)
    zsolve_thomas_kernel(double *__restrict__ p, double *__restrict__ work, const double *__restrict__ A,
                         const double *__restrict__ C, const double *__restrict__ dzf,
                         const double *__restrict__ lamx, const double *__restrict__ lamy_nat,
                         const double *__restrict__ lamy_pk, int nx, int ny, int nz, double inv_lz, double pw0,
                         double pw1, int zflags, double ha)
{
    // ha >= 0: the fully implicit Helmholtz systems of Eq. (8), the same recurrence on
    //   -a A x_{k-1} + (a A + a C + (1 + a sigma) + a W_k) x_k - a C x_{k+1} = +d
    // (pw0, pw1 are then the Dirichlet wall terms W of the velocity, no singular column)
    const bool helm = ha >= 0.0;
    const double sc = helm ? ha : 1.0, rs = helm ? -1.0 : 1.0;
    pw0 *= sc;
    pw1 *= sc;
    const size_t plane = (size_t)nx * ny;
    const size_t col = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= plane) return;
    const int i = (int)(col % nx), j = (int)(col / nx);
    const double sig = -(lamx[i] + (i < 2 ? lamy_pk[j] : lamy_nat[j]));
    const double sigma = helm ? 1.0 + ha * sig : sig;
    const bool singular = (i == 0 && j == 0) && (zflags & 2) && !helm;

    // forward: p_k = C_k + e_k, e_k = sigma + A_k e_{k-1}/p_{k-1}; g_k = (-d_k + A_k g_{k-1})/p_k
    double e = sigma + pw0;   // Dirichlet wall: extra diagonal term of the first row
    double pk = sc * C[0] + e;
    double rp = 1.0 / pk;
    double g = -rs * p[col] * rp;
    p[col] = g;
    work[col] = sc * C[0] * rp;
    for (int k = 1; k < nz; ++k) {
        const double a = sc * A[k], c = sc * C[k];
        const double d = rs * p[(size_t)k * plane + col];
        e = fma(a * e, rp, sigma) + (k == nz - 1 ? pw1 : 0.0);
        pk = c + e;
        if (singular && k == nz - 1) {
            // gauge: the last equation of the singular (0,0) system is replaced by phi = 0
            g = 0.0;
            rp = 0.0;
        } else {
            rp = 1.0 / pk;
            g = fma(a, g, -d) * rp;
        }
        p[(size_t)k * plane + col] = g;
        work[(size_t)k * plane + col] = c * rp;
    }
    // backward: phi_k = g_k + (C_k/p_k) phi_{k+1}
    double x = g;
    for (int k = nz - 2; k >= 0; --k) {
        x = fma(work[(size_t)k * plane + col], x, p[(size_t)k * plane + col]);
        p[(size_t)k * plane + col] = x;
    }
    if (singular) {
        double s = 0.0;
        for (int k = 0; k < nz; ++k) s = fma(dzf[k], p[(size_t)k * plane + col], s);
        s *= inv_lz;
        for (int k = 0; k < nz; ++k) p[(size_t)k * plane + col] -= s;
    }
}

// Variant 4 (nz <= 64, e.g. the 30 planes per GPU of the paper's weak-scaling grid):
// one thread per column, the whole column in registers -- one coalesced read and one write per
// point, the same pivot recurrence as above.  Rows past nz are identity rows.

template <int kCap>   // rows held per thread: nz rounded up to 8, 16, 24, 32, 48 or 64
__global__ void __launch_bounds__(128, (kCap > 32) ? 3 : (kCap > 16) ? 4 : 6)
    zsolve_small_kernel(double *__restrict__ p, const double *__restrict__ A, const double *__restrict__ C,
                        const double *__restrict__ dzf, const double *__restrict__ lamx, const double *__restrict__ lamy_nat,
                        const double *__restrict__ lamy_pk, int nx, int ny, int nz, double inv_lz, double pw0, double pw1,
                        int zflags)
{
    // The column goes through shared memory ([row][thread]: conflict-free) by asynchronous copies:
    // all its loads are in flight at once and hold no registers (ncu r02: with plain loads ptxas
    // scheduled one load per step of the recurrence and every step waited a DRAM latency), several
    // CTAs per SM are in different phases, so loads, recurrence and stores overlap.
    extern __shared__ double smem_small[];
    double (*sg)[128] = reinterpret_cast<double (*)[128]>(smem_small);
    double *sA = smem_small + kCap * 128, *sC = sA + kCap, *sD = sC + kCap;
    const size_t plane = (size_t)nx * ny;
    const size_t col0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = col0 < plane;
    const size_t col = active ? col0 : 0;
#pragma unroll
    for (int k = 0; k < kCap; ++k) {
        if (k < nz) {
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&sg[k][threadIdx.x]);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(p + (size_t)k * plane + col) : "memory");
        }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    if (threadIdx.x < kCap) {
        const int k = threadIdx.x;
        sA[k] = (k < nz && k > 0) ? A[k] : 0.0;
        sC[k] = (k < nz) ? C[k] : 0.0;
        sD[k] = (k < nz) ? dzf[k] : 0.0;
    }
    const int i = (int)(col % nx), j = (int)(col / nx);
    const double sigma = -(lamx[i] + (i < 2 ? lamy_pk[j] : lamy_nat[j]));
    const bool singular = (i == 0 && j == 0) && (zflags & 2);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();   // sA, sC, sD
    double cw[kCap];
    double e = 0.0, rp = 0.0, gp = 0.0;
#pragma unroll
    for (int k = 0; k < kCap; ++k) {
        const bool live = k < nz;
        const double a = sA[k], c = sC[k];
        e = fma(a * e, rp, sigma) + (k == 0 ? pw0 : 0.0) + (k == nz - 1 ? pw1 : 0.0);
        const bool gauge = singular && k == nz - 1;   // last equation of the singular column replaced by phi = 0
        const double pk = (live && !gauge) ? c + e : 1.0;
        rp = fast_rcp(pk);
        gp = (live && !gauge) ? fma(a, gp, -sg[k][threadIdx.x]) * rp : 0.0;
        if (!live || gauge) rp = 0.0;
        sg[k][threadIdx.x] = gp;
        cw[k] = c * rp;
    }
    double x = 0.0, s = 0.0;
#pragma unroll
    for (int k = kCap - 1; k >= 0; --k) {
        x = fma(cw[k], x, sg[k][threadIdx.x]);
        sg[k][threadIdx.x] = x;
        s = fma(sD[k], x, s);
    }
    const double shift = singular ? s * inv_lz : 0.0;
#pragma unroll
    for (int k = 0; k < kCap; ++k)
        if (k < nz && active) p[(size_t)k * plane + col] = sg[k][threadIdx.x] - shift;
}

} // namespace

int launch_zsolve(pz_plan *pl, double *p, cudaStream_t st, double helm_a)
{
    if (pl->opt.zsolve_variant == 4 && helm_a < 0.0) {
        const size_t plane = (size_t)pl->nx * pl->ny;
        ProfScope prof(pl, PZ_K_Z_SOLVE, st);
        const unsigned blocks = (unsigned)((plane + 127) / 128);
#define PZ_SMALL(CAP)                                                                                                       \
    do {                                                                                                                    \
        const size_t smem = (size_t)(CAP) * (128 + 3) * sizeof(double);                                                     \
        const int rc = smem_optin(pl, zsolve_small_kernel<CAP>, smem);                                                      \
        if (rc != PZ_OK) return rc;                                                                                         \
        zsolve_small_kernel<CAP><<<blocks, 128, smem, st>>>(p, pl->d_A, pl->d_C, pl->d_dzf, pl->d_lamx, pl->d_lamy_nat,      \
                                                            pl->d_lamy_pk, pl->nx, pl->ny, pl->nz, pl->inv_lz, pl->pw0,     \
                                                            pl->pw1, pl->zflags());                                         \
    } while (0)
        if (pl->nz <= 8) PZ_SMALL(8);
        else if (pl->nz <= 16) PZ_SMALL(16);
        else if (pl->nz <= 24) PZ_SMALL(24);
        else if (pl->nz <= 32) PZ_SMALL(32);
        else if (pl->nz <= 48) PZ_SMALL(48);
        else PZ_SMALL(64);
#undef PZ_SMALL
        count_launch();
        PZ_CUDA(cudaGetLastError());
        return PZ_OK;
    }
    if (pl->opt.zsolve_variant == 3 && helm_a < 0.0) return launch_zsolve_islab(pl, p, st);
    if (pl->opt.zsolve_variant == 1 || pl->opt.zsolve_variant == 4) return launch_zsolve_cr(pl, p, st, helm_a);
    if (pl->opt.zsolve_variant == 2) return launch_zsolve_tma(pl, p, st, helm_a);
    // helm_a >= 0 above 1024 planes: the thread-per-column sweep takes the Helmholtz systems too
    if (!pl->d_zwork) {
        cudaError_t e = cudaMalloc(&pl->d_zwork, pl->n * sizeof(double));
        if (e != cudaSuccess) {
            set_error("z-solve variant 0 workspace (%zu bytes): %s", pl->n * sizeof(double), cudaGetErrorString(e));
            return PZ_ENOMEM;
        }
    }
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)((plane + 127) / 128);
    ProfScope prof(pl, PZ_K_Z_SOLVE, st);
    zsolve_thomas_kernel<<<blocks, 128, 0, st>>>(p, pl->d_zwork, pl->d_A, pl->d_C, pl->d_dzf, pl->d_lamx,
                                                  pl->d_lamy_nat, pl->d_lamy_pk, pl->nx, pl->ny, pl->nz, pl->inv_lz,
                                                  helm_a >= 0.0 ? pl->wall_w0 : pl->pw0, helm_a >= 0.0 ? pl->wall_w1 : pl->pw1,
                                                  pl->zflags(), helm_a);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}

} // namespace pz

// -------------------------------------------------------------------------------------------------
// poisson_zsolve_noalloc (include/pz.h): the sweep above with its workspace in a file-scope device
// array instead of pl->d_zwork, for callers that may not allocate.  In host code `g_noalloc_work` is
// only a stand-in for the device symbol -- a kernel given it would fault (or, where the GPU can
// reach host memory, quietly use the wrong memory) --, so its device address is looked up once per
// device, with that device current, and that pointer goes to the kernel.
namespace pz {
namespace {

static __device__ __align__(256) double g_noalloc_work[PZ_NOALLOC_MAX_POINTS];

constexpr int kMaxDevices = 64;
double *g_noalloc_ptr[kMaxDevices];   // device address of g_noalloc_work on each device (nullptr: not yet looked up)

int noalloc_workspace(int device, double **out)
{
    if (device < 0 || device >= kMaxDevices) { set_error("poisson_zsolve_noalloc: device %d out of range", device); return PZ_EUNSUPPORTED; }
    double *ptr = __atomic_load_n(&g_noalloc_ptr[device], __ATOMIC_ACQUIRE);
    if (!ptr) {
        // the same address whoever gets here first: a race between two threads is benign
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_noalloc_work);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_work)");
        if (!ptr) { set_error("poisson_zsolve_noalloc: the workspace symbol has no device address"); return PZ_ECUDA; }
        __atomic_store_n(&g_noalloc_ptr[device], ptr, __ATOMIC_RELEASE);
    }
    *out = ptr;
    return PZ_OK;
}

} // namespace
} // namespace pz

extern "C" int poisson_zsolve_noalloc(pz_plan *pl, double *p, void *stream)
{
    using namespace pz;
    if (!pl || !p) { set_error("poisson_zsolve_noalloc: NULL argument"); return PZ_EINVAL; }
    if (((uintptr_t)p & 7) != 0) { set_error("poisson_zsolve_noalloc: p must be 8-byte aligned"); return PZ_EINVAL; }
    if (pl->slab_G > 0 && !pl->slab_internal) { set_error("poisson_zsolve_noalloc: a z-slab plan holds part of every column"); return PZ_EINVAL; }
    if (pl->n > (size_t)PZ_NOALLOC_MAX_POINTS) {
        set_error("poisson_zsolve_noalloc: %zu points exceed the static workspace of %lld (PZ_NOALLOC_MAX_POINTS); use poisson_solve", pl->n,
                  (long long)PZ_NOALLOC_MAX_POINTS);
        return PZ_EUNSUPPORTED;
    }
    int dev = -1;
    PZ_CUDA(cudaGetDevice(&dev));
    if (dev != pl->device) { set_error("poisson_zsolve_noalloc: the plan lives on device %d, device %d is current", pl->device, dev); return PZ_EINVAL; }
    double *work = nullptr;
    const int rc = noalloc_workspace(dev, &work);
    if (rc != PZ_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t plane = (size_t)pl->nx * pl->ny;
    const unsigned blocks = (unsigned)((plane + 127) / 128);
    zsolve_thomas_kernel<<<blocks, 128, 0, st>>>(p, work, pl->d_A, pl->d_C, pl->d_dzf, pl->d_lamx, pl->d_lamy_nat, pl->d_lamy_pk, pl->nx,
                                                  pl->ny, pl->nz, pl->inv_lz, pl->pw0, pl->pw1, pl->zflags(), -1.0);
    count_launch();
    PZ_CUDA(cudaGetLastError());
    return PZ_OK;
}
