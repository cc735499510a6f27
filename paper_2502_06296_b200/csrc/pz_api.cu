// pz_api.cu -- the C ABI of include/pz.h: plan / pre-processing (step a0), solve orchestration,
// options, error reporting.  Host code only; kernels live in the other translation units.
#include "pz_internal.h"

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

namespace pz {

static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches{0};

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char *what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return PZ_ECUDA;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int ensure_smem_optin(pz_plan *pl, const void *kernel, int bytes)
{
    for (const void *k : pl->smem_optin)
        if (k == kernel) return PZ_OK;
    PZ_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    pl->smem_optin.push_back(kernel);
    return PZ_OK;
}

static cudaEvent_t prof_event(pz_plan *pl)
{
    cudaEvent_t e = nullptr;
    if (!pl->prof_pool.empty()) { e = pl->prof_pool.back(); pl->prof_pool.pop_back(); return e; }
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
}

ProfScope::ProfScope(const pz_plan *plan, int cls, cudaStream_t stream) : pl(const_cast<pz_plan *>(plan)), st(stream)
{
    if (!pl->prof_on) return;
    cudaEvent_t a = prof_event(pl), b = prof_event(pl);
    if (!a || !b) return;
    cudaEventRecord(a, st);
    pl->prof_recs.push_back({cls, a, b});
    stop = b;
}
ProfScope::~ProfScope()
{
    if (stop) cudaEventRecord(stop, st);
}

namespace {



typedef long double ld;
const ld kPi = 3.141592653589793238462643383279502884L;

// lambda_q = -4 sin^2(pi q / n) / delta^2, folded to q <= n/2 (R1, R6)
// eigenvalue q of the second difference with zero-gradient (half = 0) or zero-value (half = 1) ends,
// -4 sin^2(pi (q + half) / (2 n)) / delta^2 (reading R17)
double lambda_r2r(int q, int n, double length, int dirichlet)
{
    const ld delta = (ld)length / (ld)n;
    const ld s = sinl(kPi * (ld)(q + (dirichlet ? 1 : 0)) / (ld)(2 * (long long)n));
    return (double)(-(ld)4 * s * s / (delta * delta));
}

double lambda(int q, int n, double length)
{
    if (q > n - q) q = n - q;
    const ld delta = (ld)length / (ld)n;
    const ld s = sinl(kPi * (ld)q / (ld)n);
    return (double)(-(ld)4 * s * s / (delta * delta));
}

// exp(-2 pi i k / n) with the argument folded into the first octant
void twiddle(int k, int n, double *re, double *im)
{
    // angle = 2 pi k / n, k in [0, n); use symmetries about multiples of pi/4 where n is a multiple of 8
    const int e = (n % 8 == 0) ? n / 8 : 0;
    int oct = (e > 0) ? k / e : 0;
    int rem = (e > 0) ? k % e : 0;
    ld c, s;
    if (e == 0) {
        c = cosl(2 * kPi * (ld)k / (ld)n);
        s = sinl(2 * kPi * (ld)k / (ld)n);
    } else {
        // theta = (oct*e + rem) * 2 pi / n = oct*pi/4 + rem*2pi/n
        ld base_c, base_s;
        const bool odd = oct & 1;
        const ld th = odd ? (ld)(e - rem) * 2 * kPi / (ld)n : (ld)rem * 2 * kPi / (ld)n; // in [0, pi/4]
        const ld ct = cosl(th), st = sinl(th);
        // angle within the quadrant: odd octant -> pi/2 - th
        if (odd) { base_c = st; base_s = ct; } else { base_c = ct; base_s = st; }
        switch (oct / 2) { // quadrant rotation
        case 0: c = base_c; s = base_s; break;
        case 1: c = -base_s; s = base_c; break;
        case 2: c = -base_c; s = -base_s; break;
        default: c = base_s; s = -base_c; break;
        }
    }
    *re = (double)c;
    *im = (double)(-s);
}

int ensure_zwork(pz_plan *pl)
{
    if (pl->d_zwork) return PZ_OK;
    cudaError_t e = cudaMalloc(&pl->d_zwork, pl->n * sizeof(double));
    if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("z-solve variant 0 workspace (%zu bytes): %s", pl->n * sizeof(double), cudaGetErrorString(e));
        return PZ_ENOMEM;
    }
    return PZ_OK;
}

int slab_planes(const pz_plan *pl)
{
    if (pl->opt.slab_planes > 0) return pl->opt.slab_planes < pl->nz ? pl->opt.slab_planes : pl->nz;
    // auto: one launch per transform direction over the whole field.  (Slabs of planes that stay
    // inside the 126 MB L2 between the x and y transforms save HBM traffic but, as separate small
    // launches, lose more to launch tails than they save: profiles/r01a.)
    size_t sp = (size_t)pl->nz;
    return (int)sp;
}

bool fused_sizes(const pz_plan *pl)
{
    const int nx = pl->nx, ny = pl->ny;
    return (nx == 256 || nx == 512 || nx == 1024 || nx == 2048) && (ny == 256 || ny == 512 || ny == 1024);
}

bool use_fused(const pz_plan *pl)
{
    if (pl->opt.slab_planes > 0 || pl->opt.fft_fused == 0 || !fused_sizes(pl) || pl->bcx || pl->bcy) return false;
    if (pl->opt.fft_fused == 1) return true;
    // auto: the fused kernel hands a plane from the x to the y transform through L2 (16 instead of
    // 32 DRAM bytes per point, ncu r02), which needs the few planes in flight to stay L2-resident
    // (planes of 16 MB: at most three planes ahead, one plane of prefetch, launch_xy).  Against the
    // separate kernels, per solve: 512^3 1.63 / 1.90 ms, 1024 x 1024 x 256 3.51 / 4.24 ms,
    // 2048 x 512 x 512 7.4 / 7.9 ms, 2048 x 256 x 1024 9.1 / 9.4 ms, 2048 x 1024 x 512 15.5 / 18.2 ms
    // (ncu: 17.6 / 21.8 GB of DRAM traffic per direction against 34.4).  A field of L2 size is served
    // from L2 by the separate kernels anyway (256^3: 0.30 against 0.32 ms).
    return pl->n * sizeof(double) >= ((size_t)512 << 20);
}

int forward_xy(pz_plan *pl, double *p, cudaStream_t st)
{
    if (use_fused(pl)) return launch_fft_xy_fwd(pl, p, st);
    const int sp = slab_planes(pl);
    for (int k0 = 0; k0 < pl->nz; k0 += sp) {
        const int nk = (k0 + sp <= pl->nz) ? sp : pl->nz - k0;
        int rc = launch_fft_x(pl, p, k0, nk, false, st);
        if (rc) return rc;
        rc = launch_fft_y(pl, p, k0, nk, false, st);
        if (rc) return rc;
        rc = launch_pair0(pl, p, k0, nk, false, st);
        if (rc) return rc;
    }
    return PZ_OK;
}

int inverse_xy(pz_plan *pl, double *p, cudaStream_t st)
{
    if (use_fused(pl)) return launch_fft_xy_inv(pl, p, st);
    const int sp = slab_planes(pl);
    for (int k0 = 0; k0 < pl->nz; k0 += sp) {
        const int nk = (k0 + sp <= pl->nz) ? sp : pl->nz - k0;
        int rc = launch_pair0(pl, p, k0, nk, true, st);
        if (rc) return rc;
        rc = launch_fft_y(pl, p, k0, nk, true, st);
        if (rc) return rc;
        rc = launch_fft_x(pl, p, k0, nk, true, st);
        if (rc) return rc;
    }
    return PZ_OK;
}

} // namespace
} // namespace pz

using namespace pz;

extern "C" {

const char *pz_last_error(void) { return g_err; }
long long pz_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
int pz_version(void) { return 200; }
int pz_fft_radices(int n, int min_points, int stride, int *radices, int cap)
{
    if (!radices || cap < 0) return 0;
    return pz::fft_radices(n, min_points, stride, radices, cap);
}

static int slab_state_create(pz_plan *pl, int n_slabs, const int *kbounds, bool internal);

// kb0 / nk: the planes [kb0, kb0 + nk) this plan transforms and owns (the whole grid for an ordinary plan)
static int plan_create(pz_plan **out, int nx, int ny, int nz, double lx, double ly, const double *zc, const double *zf,
                       int bc, int kb0, int nk)
{
    g_err[0] = 0;
    if (!out) { set_error("poisson_plan_create: out is NULL"); return PZ_EINVAL; }
    *out = nullptr;
    if (!zc || !zf) { set_error("poisson_plan_create: zc/zf is NULL"); return PZ_EINVAL; }
    if (nx <= 0 || ny <= 0 || nz <= 0) { set_error("poisson_plan_create: non-positive size %d x %d x %d", nx, ny, nz); return PZ_EINVAL; }
    if (!(lx > 0.0) || !(ly > 0.0) || !std::isfinite(lx) || !std::isfinite(ly)) { set_error("poisson_plan_create: lx, ly must be positive and finite"); return PZ_EINVAL; }
    const int bcx = bc & 3, bcy = (bc >> 2) & 3, bcz = (bc >> 4) & 3;
    if (bc < 0 || bc >= 64 || bcx == 3 || bcy == 3) { set_error("poisson_plan_create: unsupported bc %d", bc); return PZ_EUNSUPPORTED; }
    if (bc != 0 && nk != nz) { set_error("poisson_slab_plan_create: z-slab plans need bc = 0 (got %d)", bc); return PZ_EUNSUPPORTED; }
    if (!((bcx == PZ_PERIODIC && fast_fft_len(nx)) || generic_fft_x_ok(nx)) || !((bcy == PZ_PERIODIC && bcx == PZ_PERIODIC && fast_fft_len(ny)) || generic_fft_y_ok(ny)) ||
        ((long long)nx * ny) % 16 != 0) {
        set_error("poisson_plan_create: nx, ny must be even with nx / 2 and ny products of 2, 3, 5, 7 (nx <= 16384, ny <= 8192) and "
                  "nx ny a multiple of 16 (got %d, %d)", nx, ny);
        return PZ_EUNSUPPORTED;
    }
    if (nz < 4) { set_error("poisson_plan_create: nz must be >= 4 (got %d)", nz); return PZ_EUNSUPPORTED; }
    for (int k = 0; k < nz; ++k) {
        if (!(zf[k + 1] > zf[k]) || !std::isfinite(zf[k]) || !std::isfinite(zf[k + 1])) { set_error("poisson_plan_create: zf not strictly increasing at k = %d", k); return PZ_EINVAL; }
        if (!(zc[k] > zf[k] && zc[k] < zf[k + 1])) { set_error("poisson_plan_create: zc[%d] outside its cell", k); return PZ_EINVAL; }
    }

    int dev_count = 0;
    cudaError_t ce = cudaGetDeviceCount(&dev_count);
    if (ce != cudaSuccess || dev_count == 0) {
        cudaGetLastError();
        set_error("poisson_plan_create: no CUDA device (%s); there is no CPU fallback", cudaGetErrorString(ce));
        return PZ_ECUDA;
    }

    pz_plan *pl = new (std::nothrow) pz_plan();
    if (!pl) { set_error("poisson_plan_create: out of host memory"); return PZ_ENOMEM; }
    pl->nx = nx; pl->ny = ny; pl->nz = nk; pl->nz_glob = nz; pl->lx = lx; pl->ly = ly;
    pl->n = (size_t)nx * ny * nk;
    (void)kb0;
    int rc = PZ_OK;
    auto fail = [&](int code) { poisson_plan_destroy(pl); return code; };
    if (cudaGetDevice(&pl->device) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaGetDevice"));
    cudaDeviceGetAttribute(&pl->num_sms, cudaDevAttrMultiProcessorCount, pl->device);

    // z-metric tables in double, exactly as the definition states them (one division each)
    pl->zc.assign(zc, zc + nz);
    pl->zf.assign(zf, zf + nz + 1);
    pl->dzf.resize(nz); pl->dzc.resize(nz > 1 ? nz - 1 : 0); pl->A.resize(nz); pl->C.resize(nz);
    double lz = 0.0;
    for (int k = 0; k < nz; ++k) { pl->dzf[k] = zf[k + 1] - zf[k]; lz += pl->dzf[k]; }
    for (int k = 0; k + 1 < nz; ++k) pl->dzc[k] = zc[k + 1] - zc[k];
    for (int k = 0; k < nz; ++k) {
        pl->A[k] = (k >= 1) ? 1.0 / (pl->dzf[k] * pl->dzc[k - 1]) : 0.0;
        pl->C[k] = (k + 1 < nz) ? 1.0 / (pl->dzf[k] * pl->dzc[k]) : 0.0;
    }
    pl->inv_lz = 1.0 / lz;
    pl->wall_w0 = 2.0 / (pl->dzf[0] * (2.0 * (zc[0] - zf[0])));
    pl->wall_w1 = 2.0 / (pl->dzf[nz - 1] * (2.0 * (zf[nz] - zc[nz - 1])));
    pl->bcx = bcx; pl->bcy = bcy; pl->bcz = bcz;
    pl->pw0 = (bcz == PZ_Z_DD || bcz == PZ_Z_DN) ? pl->wall_w0 : 0.0;
    pl->pw1 = (bcz == PZ_Z_DD || bcz == PZ_Z_ND) ? pl->wall_w1 : 0.0;
    pl->singular00 = (bcx != PZ_DIRICHLET && bcy != PZ_DIRICHLET && bcz == PZ_Z_NN);

    // one device allocation for all tables
    const size_t ndbl = 4 * (size_t)nz + (size_t)nx + 2 * (size_t)ny + 4 * (size_t)nx + 4 * (size_t)ny + 14;
    std::vector<double> host(ndbl, 0.0);
    size_t off = 0;
    auto take = [&](size_t cnt) { size_t o = off; off += (cnt + 1) & ~(size_t)1; return o; }; // keep 16-B alignment
    const size_t oA = take(nz), oC = take(nz), oD = take(nz), oZc = take(nz), oLx = take(nx), oLyn = take(ny), oLyp = take(ny);
    const size_t oTx = take(2 * (size_t)nx), oTy = take(2 * (size_t)ny), oQx = take(2 * (size_t)nx), oQy = take(2 * (size_t)ny);
    for (int k = 0; k < nz; ++k) { host[oA + k] = pl->A[k]; host[oC + k] = pl->C[k]; host[oD + k] = pl->dzf[k]; host[oZc + k] = zc[k]; }
    // modified wavenumbers re-ordered for the packed layout
    // (cosine / sine expansions: one real coefficient per index, natural order)
    for (int i = 0; i < nx; ++i)
        host[oLx + i] = (bcx == PZ_PERIODIC) ? lambda(i == 0 ? 0 : (i == 1 ? nx / 2 : i / 2), nx, lx) : lambda_r2r(i, nx, lx, bcx == PZ_DIRICHLET);
    for (int j = 0; j < ny; ++j) {
        host[oLyn + j] = (bcy == PZ_PERIODIC) ? lambda(j, ny, ly) : lambda_r2r(j, ny, ly, bcy == PZ_DIRICHLET);
        host[oLyp + j] = (bcy == PZ_PERIODIC) ? lambda(j == 0 ? 0 : (j == 1 ? ny / 2 : j / 2), ny, ly) : host[oLyn + j];
        // x in cosines / sines, y periodic: EVERY column is a real sequence whose spectrum along y is packed
        if (bcx != PZ_PERIODIC && bcy == PZ_PERIODIC) host[oLyn + j] = host[oLyp + j];
    }
    for (int k = 0; k < nx; ++k) twiddle(k, nx, &host[oTx + 2 * k], &host[oTx + 2 * k + 1]);
    for (int k = 0; k < ny; ++k) twiddle(k, ny, &host[oTy + 2 * k], &host[oTy + 2 * k + 1]);
    // exp(-i pi k / (2 n)) = the 4n-th roots of unity, for the cosine / sine expansions
    for (int k = 0; k < nx; ++k) { host[oQx + 2 * k] = (double)cosl(kPi * (ld)k / (ld)(2 * nx)); host[oQx + 2 * k + 1] = (double)-sinl(kPi * (ld)k / (ld)(2 * nx)); }
    for (int k = 0; k < ny; ++k) { host[oQy + 2 * k] = (double)cosl(kPi * (ld)k / (ld)(2 * ny)); host[oQy + 2 * k + 1] = (double)-sinl(kPi * (ld)k / (ld)(2 * ny)); }

    ce = cudaMalloc(&pl->tables, off * sizeof(double));
    if (ce != cudaSuccess) { cudaGetLastError(); set_error("plan tables: %s", cudaGetErrorString(ce)); return fail(PZ_ENOMEM); }
    ce = cudaMemcpy(pl->tables, host.data(), off * sizeof(double), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) return fail(cuda_fail(ce, "cudaMemcpy(tables)"));
    pl->d_A = pl->tables + oA; pl->d_C = pl->tables + oC; pl->d_dzf = pl->tables + oD; pl->d_zc = pl->tables + oZc;
    pl->d_lamx = pl->tables + oLx; pl->d_lamy_nat = pl->tables + oLyn; pl->d_lamy_pk = pl->tables + oLyp;
    pl->d_twx = reinterpret_cast<double2 *>(pl->tables + oTx);
    pl->d_twy = reinterpret_cast<double2 *>(pl->tables + oTy);
    pl->d_tw4x = reinterpret_cast<double2 *>(pl->tables + oQx);
    pl->d_tw4y = reinterpret_cast<double2 *>(pl->tables + oQy);

    ce = cudaStreamCreateWithFlags(&pl->upload_stream, cudaStreamNonBlocking);
    if (ce != cudaSuccess) return fail(cuda_fail(ce, "cudaStreamCreate"));
    ce = cudaMalloc(&pl->d_xyctr, 2 * (size_t)(nk + 64) * sizeof(int));
    if (ce != cudaSuccess) { cudaGetLastError(); set_error("plan counters: %s", cudaGetErrorString(ce)); return fail(PZ_ENOMEM); }
    // measured at 512 x 512 x nz: variant 2 wins from nz = 256 up to 1024, variant 1 below
    pl->opt.zsolve_variant = (nz <= 64) ? 4 : (nz <= 128) ? 1 : (nz <= 1024) ? 2 : 0;
    // (cutting columns of 1024 planes or fewer was measured slower than the whole-column pipeline:
    // 2.06 against 1.74 ms at 512 x 512 x 1024)
    if (nk == nz && nz > 1024 && nz <= 16 * 512 && bc == 0) {
        // whole columns longer than the pipeline's tile: the plan's own cut in z (pz_zslab.cu), slabs of
        // at most 512 planes (16 rows per lane: three pipeline stages fit shared memory)
        // full slabs of 512 planes (no padding rows in their tiles) and one remainder of at least 3
        int G = (nz + 511) / 512;
        std::vector<int> kb(G + 1, 0);
        for (int g = 0; g < G; ++g) kb[g + 1] = (g + 1 < G) ? 512 * (g + 1) : nz;
        if (nz - kb[G - 1] < 3) kb[G - 1] -= 3;
        if (slab_state_create(pl, G, kb.data(), true) == PZ_OK) {
            pl->opt.zsolve_variant = 3;
        } else {
            // not enough memory for the coefficient planes: the thread-per-column sweep needs one field of workspace
            cudaGetLastError();
            if (pl->d_slab_kb) { cudaFree(pl->d_slab_kb); pl->d_slab_kb = nullptr; }
            if (pl->slab_coef) { cudaFree(pl->slab_coef); pl->slab_coef = nullptr; }
            if (pl->slab_phi) { cudaFree(pl->slab_phi); pl->slab_phi = nullptr; }
            if (pl->islab_ball) { cudaFree(pl->islab_ball); pl->islab_ball = nullptr; }
            pl->slab_G = 0; pl->slab_internal = false;
        }
    }
    if (nk == nz && pl->opt.zsolve_variant == 0 && (rc = ensure_zwork(pl)) != PZ_OK) return fail(rc);
    *out = pl;
    return PZ_OK;
}

int poisson_plan_create(pz_plan **out, int nx, int ny, int nz, double lx, double ly, const double *zc,
                        const double *zf, int bc)
{
    return plan_create(out, nx, ny, nz, lx, ly, zc, zf, bc, 0, nz);
}

// Device state of a cut in z (coefficient planes of every slab, this slab's phi_prev / phi_next):
// shared by the distributed plans and by the internal cut of a single-GPU plan with nz > 1024.
static int slab_state_create(pz_plan *pl, int n_slabs, const int *kbounds, bool internal)
{
    const size_t plane = (size_t)pl->nx * pl->ny;
    int nkmax = 0;
    for (int j = 0; j < n_slabs; ++j)
        if (kbounds[j + 1] - kbounds[j] > nkmax) nkmax = kbounds[j + 1] - kbounds[j];
    pl->slab_G = n_slabs;
    pl->slab_kb.assign(kbounds, kbounds + n_slabs + 1);
    pl->slab_bstride = 2 * plane + (size_t)((nkmax + 1) & ~1);
    pl->slab_internal = internal;
    cudaError_t ce;
    if ((ce = cudaMalloc(&pl->d_slab_kb, (n_slabs + 1) * sizeof(int))) != cudaSuccess ||
        (ce = cudaMalloc(&pl->slab_coef, (size_t)n_slabs * 6 * plane * sizeof(double))) != cudaSuccess ||
        (ce = cudaMalloc(&pl->slab_phi, 2 * plane * sizeof(double))) != cudaSuccess ||
        (internal && (ce = cudaMalloc(&pl->islab_ball, (size_t)n_slabs * pl->slab_bstride * sizeof(double))) != cudaSuccess)) {
        cudaGetLastError();
        set_error("z-slab state: %s", cudaGetErrorString(ce));
        return PZ_ENOMEM;
    }
    if ((ce = cudaMemcpy(pl->d_slab_kb, kbounds, (n_slabs + 1) * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(ce, "cudaMemcpy(kbounds)");
    // every rank computes the interface coefficients of ALL slabs itself: no collective
    int rc;
    if ((rc = launch_slab_coefficients(pl, nullptr)) != PZ_OK) return rc;
    if ((ce = cudaDeviceSynchronize()) != cudaSuccess) return cuda_fail(ce, "slab coefficients");
    return PZ_OK;
}

int poisson_slab_plan_create(pz_plan **out, int nx, int ny, int nz, double lx, double ly, const double *zc,
                             const double *zf, int bc, int n_slabs, int slab, const int *kbounds)
{
    if (out) *out = nullptr;
    if (!kbounds || n_slabs < 1 || n_slabs > 16 || slab < 0 || slab >= n_slabs) {
        set_error("poisson_slab_plan_create: need 1 <= n_slabs <= 16, 0 <= slab < n_slabs and the plane bounds");
        return PZ_EINVAL;
    }
    if (kbounds[0] != 0 || kbounds[n_slabs] != nz) { set_error("poisson_slab_plan_create: kbounds must run from 0 to nz"); return PZ_EINVAL; }
    if (nz > 16384) { set_error("poisson_slab_plan_create: at most 16384 planes in all (got %d)", nz); return PZ_EUNSUPPORTED; }
    int nkmax = 0;
    for (int j = 0; j < n_slabs; ++j) {
        const int nk = kbounds[j + 1] - kbounds[j];
        // Algorithms 1 and 2 need three rows per sub-domain (reading R9)
        if (nk < 3 || nk > 1024) { set_error("poisson_slab_plan_create: slab %d has %d planes (3..1024 supported)", j, nk); return PZ_EUNSUPPORTED; }
        if (nk > nkmax) nkmax = nk;
    }
    pz_plan *pl = nullptr;
    int rc = plan_create(&pl, nx, ny, nz, lx, ly, zc, zf, bc, kbounds[slab], kbounds[slab + 1] - kbounds[slab]);
    if (rc != PZ_OK) return rc;
    auto fail = [&](int code) { poisson_plan_destroy(pl); return code; };
    pl->slab_g = slab;
    if ((rc = slab_state_create(pl, n_slabs, kbounds, false)) != PZ_OK) return fail(rc);
    *out = pl;
    return PZ_OK;
}

long long poisson_slab_boundary_doubles(const pz_plan *pl)
{
    return (pl && pl->slab_G > 0 && !pl->slab_internal) ? (long long)pl->slab_bstride : 0;
}

int poisson_solve_reduce(pz_plan *pl, double *p, double *boundary_out, void *stream)
{
    if (!pl || !p || !boundary_out) { set_error("poisson_solve_reduce: NULL argument"); return PZ_EINVAL; }
    if (pl->slab_G < 1 || pl->slab_internal) { set_error("poisson_solve_reduce: the plan is not a slab plan"); return PZ_EINVAL; }
    if ((((uintptr_t)p | (uintptr_t)boundary_out) & 15) != 0) { set_error("poisson_solve_reduce: buffers must be 16-byte aligned"); return PZ_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
    if ((rc = forward_xy(pl, p, st)) != PZ_OK) return rc;
    BoutSet one;
    one.n = 1;
    one.p[0] = boundary_out;
    return launch_slab_reduce(pl, p, one, st);
}

int poisson_solve_reduce_push(pz_plan *pl, double *p, double *const *boundary_all_of_rank, long long *const *flags_of_rank,
                              long long epoch, void *stream)
{
    if (!pl || !p || !boundary_all_of_rank || !flags_of_rank) { set_error("poisson_solve_reduce_push: NULL argument"); return PZ_EINVAL; }
    if (pl->slab_G < 1 || pl->slab_internal) { set_error("poisson_solve_reduce_push: the plan is not a slab plan"); return PZ_EINVAL; }
    BoutSet all;
    all.n = pl->slab_G;
    for (int r = 0; r < pl->slab_G; ++r) {
        if (!boundary_all_of_rank[r] || !flags_of_rank[r] || ((uintptr_t)boundary_all_of_rank[r] & 15) != 0) {
            set_error("poisson_solve_reduce_push: buffer of rank %d is NULL or not 16-byte aligned", r);
            return PZ_EINVAL;
        }
        all.p[r] = boundary_all_of_rank[r] + (size_t)pl->slab_g * pl->slab_bstride; // this rank's slot in rank r's gathered buffer
    }
    if (((uintptr_t)p & 15) != 0) { set_error("poisson_solve_reduce_push: p must be 16-byte aligned"); return PZ_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
    if ((rc = forward_xy(pl, p, st)) != PZ_OK) return rc;
    if ((rc = launch_slab_reduce(pl, p, all, st)) != PZ_OK) return rc;
    return launch_slab_signal(pl, flags_of_rank, pl->slab_G, pl->slab_g, epoch, st);
}

int poisson_solve_finish_wait(pz_plan *pl, double *p, const double *boundary_all, const long long *flags, long long epoch,
                              void *stream)
{
    if (!pl || !flags) { set_error("poisson_solve_finish_wait: NULL argument"); return PZ_EINVAL; }
    if (pl->slab_G < 1 || pl->slab_internal) { set_error("poisson_solve_finish_wait: the plan is not a slab plan"); return PZ_EINVAL; }
    const int rc = launch_slab_wait(pl, flags, pl->slab_G, epoch, (cudaStream_t)stream);
    if (rc != PZ_OK) return rc;
    return poisson_solve_finish(pl, p, boundary_all, stream);
}

int poisson_solve_finish(pz_plan *pl, double *p, const double *boundary_all, void *stream)
{
    if (!pl || !p || !boundary_all) { set_error("poisson_solve_finish: NULL argument"); return PZ_EINVAL; }
    if (pl->slab_G < 1 || pl->slab_internal) { set_error("poisson_solve_finish: the plan is not a slab plan"); return PZ_EINVAL; }
    if ((((uintptr_t)p | (uintptr_t)boundary_all) & 15) != 0) { set_error("poisson_solve_finish: buffers must be 16-byte aligned"); return PZ_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if ((rc = launch_slab_finish(pl, p, boundary_all, st)) != PZ_OK) return rc;
    if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
    return inverse_xy(pl, p, st);
}

int poisson_plan_destroy(pz_plan *pl)
{
    if (!pl) return PZ_OK;
    cudaDeviceSynchronize();
    if (pl->tables) cudaFree(pl->tables);
    if (pl->d_zwork) cudaFree(pl->d_zwork);
    if (pl->d_host_stage) cudaFree(pl->d_host_stage);
    if (pl->d_xyctr) cudaFree(pl->d_xyctr);
    if (pl->d_slab_kb) cudaFree(pl->d_slab_kb);
    if (pl->slab_coef) cudaFree(pl->slab_coef);
    if (pl->slab_phi) cudaFree(pl->slab_phi);
    if (pl->islab_ball) cudaFree(pl->islab_ball);
    for (int b = 0; b < 3; ++b)
        if (pl->d_batch_stage[b]) cudaFree(pl->d_batch_stage[b]);
    if (pl->h2d_stream) cudaStreamDestroy(pl->h2d_stream);
    if (pl->d2h_stream) cudaStreamDestroy(pl->d2h_stream);
    for (auto e : pl->batch_events) cudaEventDestroy(e);
    for (auto &t : pl->helm) {
        if (t.dev) cudaFree(t.dev);
        if (t.host) cudaFreeHost(t.host);
        if (t.uploaded) cudaEventDestroy(t.uploaded);
        if (t.last_use) cudaEventDestroy(t.last_use);
    }
    if (pl->upload_stream) cudaStreamDestroy(pl->upload_stream);
    for (auto &r : pl->prof_recs) { cudaEventDestroy(r.start); cudaEventDestroy(r.stop); }
    for (auto e : pl->prof_pool) cudaEventDestroy(e);
    cudaGetLastError();
    delete pl;
    return PZ_OK;
}

int pz_poisson_stage(pz_plan *pl, double *p, int stage, void *stream)
{
    if (!pl || !p) { set_error("pz_poisson_stage: NULL argument"); return PZ_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    switch (stage) {
    case PZ_STAGE_FFT_X_FWD: return launch_fft_x(pl, p, 0, pl->nz, false, st);
    case PZ_STAGE_FFT_Y_FWD:
        if ((rc = launch_fft_y(pl, p, 0, pl->nz, false, st)) != PZ_OK) return rc;
        return launch_pair0(pl, p, 0, pl->nz, false, st);
    case PZ_STAGE_Z_SOLVE: return launch_zsolve(pl, p, st);
    case PZ_STAGE_FFT_Y_INV:
        if ((rc = launch_pair0(pl, p, 0, pl->nz, true, st)) != PZ_OK) return rc;
        return launch_fft_y(pl, p, 0, pl->nz, true, st);
    case PZ_STAGE_FFT_X_INV: return launch_fft_x(pl, p, 0, pl->nz, true, st);
    case PZ_STAGE_FFT_XY_FWD:
    case PZ_STAGE_FFT_XY_INV:
        if (!fused_sizes(pl)) { set_error("pz_poisson_stage: the fused x/y kernel needs nx in {256, 512, 1024, 2048}, ny in {256, 512, 1024}"); return PZ_EUNSUPPORTED; }
        PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
        return stage == PZ_STAGE_FFT_XY_FWD ? launch_fft_xy_fwd(pl, p, st) : launch_fft_xy_inv(pl, p, st);
    default: set_error("pz_poisson_stage: unknown stage %d", stage); return PZ_EINVAL;
    }
}

int poisson_solve(pz_plan *pl, double *p, void *stream)
{
    if (!pl || !p) { set_error("poisson_solve: NULL argument"); return PZ_EINVAL; }
    if (pl->slab_G > 0 && !pl->slab_internal) { set_error("poisson_solve: a slab plan solves through poisson_solve_reduce / poisson_solve_finish"); return PZ_EINVAL; }
    if (((uintptr_t)p & 15) != 0) { set_error("poisson_solve: p must be 16-byte aligned"); return PZ_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
    if ((rc = forward_xy(pl, p, st)) != PZ_OK) return rc;
    if ((rc = launch_zsolve(pl, p, st)) != PZ_OK) return rc;
    return inverse_xy(pl, p, st);
}

static bool misaligned(const void *q) { return ((uintptr_t)q & 15) != 0; }

int pz_divergence_rhs(pz_plan *pl, const double *u, const double *v, const double *w, double *rhs, double inv_gdt, void *stream)
{
    if (!pl || !u || !v || !w || !rhs) { set_error("pz_divergence_rhs: NULL argument"); return PZ_EINVAL; }
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(rhs)) { set_error("pz_divergence_rhs: fields must be 16-byte aligned"); return PZ_EINVAL; }
    if (!std::isfinite(inv_gdt)) { set_error("pz_divergence_rhs: 1/(gamma dt) must be finite"); return PZ_EINVAL; }
    if (pl->bcx || pl->bcy || pl->bcz) { set_error("pz_divergence_rhs: needs a plan with bc = 0"); return PZ_EUNSUPPORTED; }
    return launch_divergence_rhs(pl, u, v, w, rhs, inv_gdt, (cudaStream_t)stream);
}

int pz_project(pz_plan *pl, double *u, double *v, double *w, double *p, const double *phi, double gdt, void *stream)
{
    if (!pl || !u || !v || !w || !p || !phi) { set_error("pz_project: NULL argument"); return PZ_EINVAL; }
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(p) || misaligned(phi)) { set_error("pz_project: fields must be 16-byte aligned"); return PZ_EINVAL; }
    if (!std::isfinite(gdt)) { set_error("pz_project: gamma dt must be finite"); return PZ_EINVAL; }
    if (pl->bcx || pl->bcy || pl->bcz) { set_error("pz_project: needs a plan with bc = 0"); return PZ_EUNSUPPORTED; }
    return launch_project(pl, u, v, w, p, phi, gdt, (cudaStream_t)stream);
}

int pz_pressure_correction(pz_plan *pl, double *u, double *v, double *w, double *p, double *work, double gdt, void *stream)
{
    if (!(gdt > 0.0) || !std::isfinite(gdt)) { set_error("pz_pressure_correction: gamma dt must be positive and finite"); return PZ_EINVAL; }
    int rc;
    if (pl && u && v && w && work && pl->opt.div_fused != 0 && pl->opt.slab_planes == 0 && fast_fft_len(pl->nx) && !pl->bcx && !pl->bcy && !pl->bcz &&
        !misaligned(u) && !misaligned(v) && !misaligned(w) && !misaligned(work)) {
        // Eq. (4)'s right-hand side is formed inside the forward x transform: it never touches HBM
        cudaStream_t st = (cudaStream_t)stream;
        DivSrc ds;
        ds.u = u; ds.v = v; ds.w = w; ds.dzf = pl->d_dzf;
        ds.rdx = 1.0 / (pl->lx / pl->nx); ds.rdy = 1.0 / (pl->ly / pl->ny); ds.scale = 1.0 / gdt; ds.ny = pl->ny;
        if ((rc = launch_fft_x(pl, work, 0, pl->nz, false, st, &ds)) != PZ_OK) return rc;
        if ((rc = launch_fft_y(pl, work, 0, pl->nz, false, st)) != PZ_OK) return rc;
        if ((rc = launch_pair0(pl, work, 0, pl->nz, false, st)) != PZ_OK) return rc;
        if ((rc = launch_zsolve(pl, work, st)) != PZ_OK) return rc;
        if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
        if ((rc = inverse_xy(pl, work, st)) != PZ_OK) return rc;
        return pz_project(pl, u, v, w, p, work, gdt, stream);
    }
    if ((rc = pz_divergence_rhs(pl, u, v, w, work, 1.0 / gdt, stream)) != PZ_OK) return rc;
    if ((rc = poisson_solve(pl, work, stream)) != PZ_OK) return rc;
    return pz_project(pl, u, v, w, p, work, gdt, stream);
}

int helmholtz_z_rhs(pz_plan *pl, double *ustar2, const double *uk, void *stream)
{
    if (!pl || !ustar2 || !uk) { set_error("helmholtz_z_rhs: NULL argument"); return PZ_EINVAL; }
    if (misaligned(ustar2) || misaligned(uk)) { set_error("helmholtz_z_rhs: fields must be 16-byte aligned"); return PZ_EINVAL; }
    if (pl->helm_cur < 0) { set_error("helmholtz_z_rhs: call helmholtz_z_setup first"); return PZ_ENOTSETUP; }
    return launch_helmholtz_z_rhs(pl, ustar2, uk, pl->helm_a, (cudaStream_t)stream);
}

int helmholtz_z_step(pz_plan *pl, double *ustar2, const double *uk, void *stream)
{
    if (pl && ustar2 && uk && !misaligned(ustar2) && !misaligned(uk) && pl->helm_cur >= 0) {
        const int fused = launch_helmholtz_step(pl, ustar2, uk, (cudaStream_t)stream);
        if (fused != PZ_EUNSUPPORTED) return fused;
    }
    const int rc = helmholtz_z_rhs(pl, ustar2, uk, stream);
    if (rc != PZ_OK) return rc;
    return helmholtz_z_solve(pl, ustar2, stream);
}

int helmholtz3d_setup(pz_plan *pl, double a)
{
    if (!pl) { set_error("helmholtz3d_setup: plan is NULL"); return PZ_EINVAL; }
    if (!(a >= 0.0) || !std::isfinite(a)) { set_error("helmholtz3d_setup: a must be finite and >= 0"); return PZ_EINVAL; }
    pl->h3_a = a; // the coefficient tables are scaled inside the kernel: nothing to upload
    return PZ_OK;
}

int helmholtz3d_solve(pz_plan *pl, double *u, void *stream)
{
    if (!pl || !u) { set_error("helmholtz3d_solve: NULL argument"); return PZ_EINVAL; }
    if (((uintptr_t)u & 15) != 0) { set_error("helmholtz3d_solve: u must be 16-byte aligned"); return PZ_EINVAL; }
    if (pl->h3_a < 0.0) { set_error("helmholtz3d_solve: call helmholtz3d_setup first"); return PZ_ENOTSETUP; }
    if (pl->bcx || pl->bcy || pl->bcz) { set_error("helmholtz3d_solve: needs a plan with bc = 0"); return PZ_EUNSUPPORTED; }
    if (pl->slab_G > 0 && !pl->slab_internal) { set_error("helmholtz3d_solve: not available on a z-slab plan"); return PZ_EUNSUPPORTED; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (use_fused(pl)) PZ_CUDA(cudaMemsetAsync(pl->d_xyctr, 0, 2 * (size_t)(pl->nz + 64) * sizeof(int), st));
    if ((rc = forward_xy(pl, u, st)) != PZ_OK) return rc;
    if ((rc = launch_zsolve(pl, u, st, pl->h3_a)) != PZ_OK) return rc;
    return inverse_xy(pl, u, st);
}

int helmholtz_z_setup(pz_plan *pl, double a)
{
    if (!pl) { set_error("helmholtz_z_setup: plan is NULL"); return PZ_EINVAL; }
    if (!(a >= 0.0) || !std::isfinite(a)) { set_error("helmholtz_z_setup: a must be finite and >= 0"); return PZ_EINVAL; }
    if (pl->slab_G > 0 && !pl->slab_internal) { set_error("helmholtz_z_setup: not available on a z-slab plan (columns are cut; shard Helmholtz solves in y)"); return PZ_EUNSUPPORTED; }
    return helmholtz_build_tables(pl, a);
}

int helmholtz_w_setup(pz_plan *pl, double a)
{
    if (!pl) { set_error("helmholtz_w_setup: plan is NULL"); return PZ_EINVAL; }
    if (!(a >= 0.0) || !std::isfinite(a)) { set_error("helmholtz_w_setup: a must be finite and >= 0"); return PZ_EINVAL; }
    if (pl->slab_G > 0 && !pl->slab_internal) { set_error("helmholtz_w_setup: not available on a z-slab plan (columns are cut; shard Helmholtz solves in y)"); return PZ_EUNSUPPORTED; }
    return helmholtz_build_tables(pl, a, 1);
}

int helmholtz_w_solve(pz_plan *pl, double *w, void *stream)
{
    if (!pl || !w) { set_error("helmholtz_w_solve: NULL argument"); return PZ_EINVAL; }
    if (pl->helm_w_cur < 0) { set_error("helmholtz_w_solve: call helmholtz_w_setup first"); return PZ_ENOTSETUP; }
    double *one[1] = {w};
    return launch_helmholtz_n(pl, one, 1, (cudaStream_t)stream, 1);
}

int helmholtz_z_solve(pz_plan *pl, double *u, void *stream)
{
    if (!pl || !u) { set_error("helmholtz_z_solve: NULL argument"); return PZ_EINVAL; }
    if (pl->helm_cur < 0) { set_error("helmholtz_z_solve: call helmholtz_z_setup first"); return PZ_ENOTSETUP; }
    double *one[1] = {u};
    return launch_helmholtz_n(pl, one, 1, (cudaStream_t)stream);
}

int helmholtz_z_solve_n(pz_plan *pl, double *const *u, int n, void *stream)
{
    if (!pl || !u || n < 0) { set_error("helmholtz_z_solve_n: bad argument"); return PZ_EINVAL; }
    if (pl->helm_cur < 0) { set_error("helmholtz_z_solve_n: call helmholtz_z_setup first"); return PZ_ENOTSETUP; }
    for (int c = 0; c < n; ++c)
        if (!u[c]) { set_error("helmholtz_z_solve_n: field %d is NULL", c); return PZ_EINVAL; }
    return launch_helmholtz_n(pl, u, n, (cudaStream_t)stream);
}

static int ensure_host_stage(pz_plan *pl)
{
    if (pl->d_host_stage) return PZ_OK;
    cudaError_t e = cudaMalloc(&pl->d_host_stage, pl->n * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); set_error("host staging field: %s", cudaGetErrorString(e)); return PZ_ENOMEM; }
    return PZ_OK;
}

int poisson_solve_host(pz_plan *pl, double *p_host, void *stream)
{
    if (!pl || !p_host) { set_error("poisson_solve_host: NULL argument"); return PZ_EINVAL; }
    int rc = ensure_host_stage(pl);
    if (rc != PZ_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    PZ_CUDA(cudaMemcpyAsync(pl->d_host_stage, p_host, pl->n * sizeof(double), cudaMemcpyHostToDevice, st));
    if ((rc = poisson_solve(pl, pl->d_host_stage, stream)) != PZ_OK) return rc;
    PZ_CUDA(cudaMemcpyAsync(p_host, pl->d_host_stage, pl->n * sizeof(double), cudaMemcpyDeviceToHost, st));
    return PZ_OK;
}

int helmholtz_z_solve_host(pz_plan *pl, double *u_host, void *stream)
{
    if (!pl || !u_host) { set_error("helmholtz_z_solve_host: NULL argument"); return PZ_EINVAL; }
    if (pl->helm_cur < 0) { set_error("helmholtz_z_solve_host: call helmholtz_z_setup first"); return PZ_ENOTSETUP; }
    int rc = ensure_host_stage(pl);
    if (rc != PZ_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    PZ_CUDA(cudaMemcpyAsync(pl->d_host_stage, u_host, pl->n * sizeof(double), cudaMemcpyHostToDevice, st));
    if ((rc = helmholtz_z_solve(pl, pl->d_host_stage, stream)) != PZ_OK) return rc;
    PZ_CUDA(cudaMemcpyAsync(u_host, pl->d_host_stage, pl->n * sizeof(double), cudaMemcpyDeviceToHost, st));
    return PZ_OK;
}

int pz_solve_host_batch(pz_plan *pl, double *p_host, double *const *u_host, int n_u, void *stream)
{
    if (!pl || n_u < 0 || (n_u > 0 && !u_host)) { set_error("pz_solve_host_batch: bad argument"); return PZ_EINVAL; }
    for (int c = 0; c < n_u; ++c)
        if (!u_host[c]) { set_error("pz_solve_host_batch: field %d is NULL", c); return PZ_EINVAL; }
    if (n_u > 0 && pl->helm_cur < 0) { set_error("pz_solve_host_batch: call helmholtz_z_setup first"); return PZ_ENOTSETUP; }
    const int nf = (p_host ? 1 : 0) + n_u;
    if (nf == 0) return PZ_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = pl->n * sizeof(double);
    for (int b = 0; b < 3 && b < nf; ++b)
        if (!pl->d_batch_stage[b]) {
            cudaError_t e = cudaMalloc(&pl->d_batch_stage[b], bytes);
            if (e != cudaSuccess) { cudaGetLastError(); set_error("batch staging field: %s", cudaGetErrorString(e)); return PZ_ENOMEM; }
        }
    if (!pl->h2d_stream) PZ_CUDA(cudaStreamCreateWithFlags(&pl->h2d_stream, cudaStreamNonBlocking));
    if (!pl->d2h_stream) PZ_CUDA(cudaStreamCreateWithFlags(&pl->d2h_stream, cudaStreamNonBlocking));
    // events: [0] start, then per field (uploaded, solved, downloaded)
    while ((int)pl->batch_events.size() < 1 + 3 * nf) {
        cudaEvent_t e = nullptr;
        PZ_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        pl->batch_events.push_back(e);
    }
    auto ev = [&](int f, int which) { return pl->batch_events[1 + 3 * f + which]; };
    PZ_CUDA(cudaEventRecord(pl->batch_events[0], st));
    PZ_CUDA(cudaStreamWaitEvent(pl->h2d_stream, pl->batch_events[0], 0));
    for (int f = 0; f < nf; ++f) {
        const bool is_p = (p_host && f == 0);
        double *host = is_p ? p_host : u_host[f - (p_host ? 1 : 0)];
        double *dev = pl->d_batch_stage[f % 3];
        if (f >= 3) PZ_CUDA(cudaStreamWaitEvent(pl->h2d_stream, ev(f - 3, 2), 0)); // staging field free again
        PZ_CUDA(cudaMemcpyAsync(dev, host, bytes, cudaMemcpyHostToDevice, pl->h2d_stream));
        PZ_CUDA(cudaEventRecord(ev(f, 0), pl->h2d_stream));
        PZ_CUDA(cudaStreamWaitEvent(st, ev(f, 0), 0));
        const int rc = is_p ? poisson_solve(pl, dev, stream) : helmholtz_z_solve(pl, dev, stream);
        if (rc != PZ_OK) return rc;
        PZ_CUDA(cudaEventRecord(ev(f, 1), st));
        PZ_CUDA(cudaStreamWaitEvent(pl->d2h_stream, ev(f, 1), 0));
        PZ_CUDA(cudaMemcpyAsync(host, dev, bytes, cudaMemcpyDeviceToHost, pl->d2h_stream));
        PZ_CUDA(cudaEventRecord(ev(f, 2), pl->d2h_stream));
    }
    PZ_CUDA(cudaStreamWaitEvent(st, ev(nf - 1, 2), 0)); // downloads are in order on one stream
    return PZ_OK;
}

int pz_profile_enable(pz_plan *pl, int on)
{
    if (!pl) { set_error("pz_profile_enable: plan is NULL"); return PZ_EINVAL; }
    if (on) {
        for (auto &r : pl->prof_recs) { pl->prof_pool.push_back(r.start); pl->prof_pool.push_back(r.stop); }
        pl->prof_recs.clear();
    }
    pl->prof_on = (on != 0);
    return PZ_OK;
}

int pz_profile_read(pz_plan *pl, int cls, double *total_ms, long long *launches)
{
    if (!pl || !total_ms || !launches || cls < 0 || cls >= PZ_K_COUNT) { set_error("pz_profile_read: bad argument"); return PZ_EINVAL; }
    double sum = 0.0;
    long long cnt = 0;
    for (auto &r : pl->prof_recs) {
        if (r.cls != cls) continue;
        PZ_CUDA(cudaEventSynchronize(r.stop));
        float ms = 0.f;
        PZ_CUDA(cudaEventElapsedTime(&ms, r.start, r.stop));
        sum += ms;
        ++cnt;
    }
    *total_ms = sum;
    *launches = cnt;
    return PZ_OK;
}

static int *option_slot(pz_plan *pl, const char *key)
{
    if (!std::strcmp(key, "zsolve_variant")) return &pl->opt.zsolve_variant;
    if (!std::strcmp(key, "zsolve_stages")) return &pl->opt.zsolve_stages;
    if (kProbes && !std::strcmp(key, "zsolve_probe")) return &pl->opt.zsolve_probe;
    if (!std::strcmp(key, "slab_planes")) return &pl->opt.slab_planes;
    if (!std::strcmp(key, "fft_fused")) return &pl->opt.fft_fused;
    if (!std::strcmp(key, "xy_lag")) return &pl->opt.xy_lag;
    if (!std::strcmp(key, "xy_bps")) return &pl->opt.xy_bps;
    if (!std::strcmp(key, "xy_prefetch")) return &pl->opt.xy_prefetch;
    if (!std::strcmp(key, "xy_xshare")) return &pl->opt.xy_xshare;
    if (!std::strcmp(key, "xy_group")) return &pl->opt.xy_group;
    if (!std::strcmp(key, "helm_variant")) return &pl->opt.helm_variant;
    if (kProbes && !std::strcmp(key, "helm_probe")) return &pl->opt.helm_probe;
    if (!std::strcmp(key, "helm_cluster")) return &pl->opt.helm_cluster;
    if (!std::strcmp(key, "helm_box_rows")) return &pl->opt.helm_box_rows;
    if (!std::strcmp(key, "helm_l2promo")) return &pl->opt.helm_l2promo;
    if (!std::strcmp(key, "helm_tx")) return &pl->opt.helm_tx;
    if (!std::strcmp(key, "helm_m")) return &pl->opt.helm_m;
    if (!std::strcmp(key, "helm_zsplit")) return &pl->opt.helm_zsplit;
    if (!std::strcmp(key, "fft_y_tc")) return &pl->opt.fft_y_tc;
    if (!std::strcmp(key, "div_fused")) return &pl->opt.div_fused;
    if (!std::strcmp(key, "step_fused")) return &pl->opt.step_fused;
    if (!std::strcmp(key, "fft_y_p0")) return &pl->opt.fft_y_p0;
    if (!std::strcmp(key, "fft_x_lpb")) return &pl->opt.fft_x_lpb;
    return nullptr;
}

int pz_set_option(pz_plan *pl, const char *key, int value)
{
    if (!pl || !key) { set_error("pz_set_option: NULL argument"); return PZ_EINVAL; }
    int *slot = option_slot(pl, key);
    if (!slot) { set_error("pz_set_option: unknown key '%s'", key); return PZ_EUNSUPPORTED; }
    if (slot == &pl->opt.zsolve_variant) {
        if (value < 0 || value > 4) { set_error("zsolve_variant must be 0 ... 4"); return PZ_EUNSUPPORTED; }
        if (value == 4 && pl->nz > 64) { set_error("zsolve_variant 4 supports nz <= 64"); return PZ_EUNSUPPORTED; }
        if ((value == 1 || value == 2) && pl->nz > 1024) { set_error("zsolve_variant %d supports nz <= 1024", value); return PZ_EUNSUPPORTED; }
        if (value == 3 && !pl->slab_internal) { set_error("zsolve_variant 3 is the plan's own z cut (nz > 1024)"); return PZ_EUNSUPPORTED; }
        if (value == 0) { const int rc = ensure_zwork(pl); if (rc != PZ_OK) return rc; }
    } else if (value < 0) {
        set_error("pz_set_option: '%s' must be >= 0", key);
        return PZ_EUNSUPPORTED;
    }
    *slot = value;
    if (slot == &pl->opt.helm_tx || slot == &pl->opt.helm_m || slot == &pl->opt.helm_variant || slot == &pl->opt.helm_zsplit) {
        // geometry changed: rebuild the tables
        int rc = PZ_OK;
        if (pl->helm_cur >= 0) rc = helmholtz_build_tables(pl, pl->helm_a, 0);
        if (rc == PZ_OK && pl->helm_w_cur >= 0) rc = helmholtz_build_tables(pl, pl->helm_w_a, 1);
        return rc;
    }
    return PZ_OK;
}

int pz_get_option(const pz_plan *pl, const char *key, int *value)
{
    if (!pl || !key || !value) { set_error("pz_get_option: NULL argument"); return PZ_EINVAL; }
    int *slot = option_slot(const_cast<pz_plan *>(pl), key);
    if (!slot) {
        if (!std::strcmp(key, "helm_m_actual")) { *value = pl->helm_m; return PZ_OK; }
        if (!std::strcmp(key, "helm_variant_actual")) { *value = pl->helm_variant; return PZ_OK; }
        if (!std::strcmp(key, "helm_tx_actual")) { *value = pl->helm_tx; return PZ_OK; }
        if (!std::strcmp(key, "helm_p_actual")) { *value = pl->helm_P; return PZ_OK; }
        if (!std::strcmp(key, "helm_zsplit_actual")) { *value = pl->helm_zs; return PZ_OK; }
        if (!std::strcmp(key, "slab_planes_actual")) { *value = slab_planes(pl); return PZ_OK; }
        set_error("pz_get_option: unknown key '%s'", key);
        return PZ_EUNSUPPORTED;
    }
    *value = *slot;
    return PZ_OK;
}

} // extern "C"
