// pz_internal.h -- plan object and launch declarations shared by the translation units of
// libpz_b200.so.  Not installed; the public boundary is include/pz.h.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/pz.h"

namespace pz {

// Helmholtz pre-processing tables of Algorithm 2, one set per buffer.
// Rows are padded to nzp = P*m with identity rows so that every sub-domain has m rows.
struct HelmTables {
    double *dev = nullptr;      // one allocation: [fA | bC | rb | ra | rc] (5*nzp) + reduced PCR tables
    size_t bytes = 0;
    cudaEvent_t uploaded = nullptr;   // recorded on the upload stream after the H2D copy
    cudaEvent_t last_use = nullptr;   // recorded on the caller's stream after each solve
    double *host = nullptr;           // pinned staging of this set's upload
    size_t host_bytes = 0;
    bool used = false;
    bool upload_seen = false;         // host has observed the upload's completion: solves need no ordering
    bool captured = false;            // a CUDA graph holds this set's address: never rewritten or freed before destroy
};

struct Options {
    int zsolve_variant = 0;   // 3 = nz > 1024: the plan's own z-slabs through variant 2 (pz_zslab.cu)
                              // 0 = thread-per-column Thomas through global memory (2 sweeps)
                              // 1 = chunked cyclic reduction in shared memory
                              // 2 = the same solve inside a TMA load / solve / TMA store pipeline
    int zsolve_probe = 0;     // diagnostic (variant 2): 2 = no arithmetic (results are wrong)
    int zsolve_stages = 0;    // variant 2: shared-memory stages (0 = as many as fit, at most 3)
    int fft_fused = -1;       // -1 = auto (use_fused, pz_api.cu); 0 = separate kernels; 1 = fused x/y kernel
                              // (nx, ny in {256, 512, 1024, 2048})
    int xy_lag = 0;           // fused kernel: planes by which the first phase runs ahead (0 = auto)
    int xy_bps = 0;           // fused kernel: resident CTAs per SM (0 = as many as fit)
    int xy_xshare = 0;        // fused kernel: sixteenths of the SMs that prefer the first phase (0 = auto)
    int xy_group = 0;         // fused kernel: SMs per role group (0 = auto)
    int xy_prefetch = 0;      // fused kernel: planes by which first-phase inputs are prefetched into L2 (0 = auto)
    int slab_planes = 0;      // 0 = auto: z-planes per L2-resident slab for the fused x/y FFT passes
    int helm_variant = -1;    // -1 = auto; 1 = persistent TMA-fed pipeline (nz <= 1024); 0 = register tile, direct loads
    int helm_box_rows = 0;    // diagnostic (variant 1): rows per TMA box (0 = 256)
    int helm_l2promo = 1;     // diagnostic (variant 1): tensor-map L2 promotion 0 none, 1 128 B, 2 256 B, 3 64 B
    int helm_cluster = 0;     // variant 1: CTAs per cluster walking neighbouring tiles in step (0 = auto)
    int helm_probe = 0;       // diagnostic (variant 1): 1 = no stores, 2 = no arithmetic (results are wrong)
    int helm_tx = 0;          // 0 = auto: columns per CTA in the Helmholtz kernel (variant 0)
    int helm_m = 0;           // 0 = auto: rows per sub-domain in the Helmholtz kernel
    int helm_zsplit = 0;      // 0 = auto: 1 = whole columns per CTA, 2 = column cut over the two CTAs of a cluster
    int fft_y_p0 = 1;         // 1 = pair-0 conversion inside the y-FFT kernel, 0 = separate small kernel
    int step_fused = 1;       // helmholtz_z_step: 1 = right-hand side of Eq. (11) formed inside the solve kernel
    int div_fused = 1;        // pz_pressure_correction: 1 = divergence formed inside the forward x transform
    int fft_y_tc = 0;         // 0 = auto: complex column pairs per CTA in the y FFT
    int fft_x_lpb = 0;        // 0 = auto: lines per CTA in the x FFT
};

} // namespace pz

struct pz_plan {
    int nx = 0, ny = 0, nz = 0;
    double lx = 0, ly = 0;
    int device = 0;
    int num_sms = 0;
    size_t n = 0;

    // host copies
    std::vector<double> zc, zf, dzf, dzc, A, C;

    // device tables (one allocation, freed as `tables`)
    double *tables = nullptr;
    double *d_A = nullptr, *d_C = nullptr, *d_dzf = nullptr, *d_zc = nullptr;   // nz each
    double *d_lamx = nullptr;        // nx: lambda_x per real column i in packed order
    double *d_lamy_nat = nullptr;    // ny: lambda_y, natural order (complex pairs i >= 2)
    double *d_lamy_pk = nullptr;     // ny: lambda_y, packed order (columns i = 0, 1)
    double2 *d_twx = nullptr;        // nx: exp(-2 pi i k / nx)
    double2 *d_twy = nullptr;        // ny: exp(-2 pi i k / ny)
    double2 *d_tw4x = nullptr;       // nx: exp(-i pi k / (2 nx)), cosine / sine expansions
    double2 *d_tw4y = nullptr;       // ny: exp(-i pi k / (2 ny))
    double inv_lz = 0;               // 1 / sum dzf
    double wall_w0 = 0, wall_w1 = 0; // Dirichlet wall terms W_0, W_{nz-1} of the Helmholtz operators
    double h3_a = -1.0;              // helmholtz3d_setup: a of the fully implicit Helmholtz solve
    int bcx = 0, bcy = 0, bcz = 0;   // pz_bc_dir, pz_bc_dir, pz_bc_z of the Poisson solve
    double pw0 = 0, pw1 = 0;         // Poisson: Dirichlet wall terms of the first / last z row (0 = Neumann)
    bool singular00 = true;          // the (0,0) column is singular (no Dirichlet end anywhere) and is pinned
    int zflags() const { return ((pw0 != 0.0 || pw1 != 0.0) ? 1 : 0) | (singular00 ? 2 : 0); }

    // optional workspaces (allocated on first use)
    double *d_zwork = nullptr;       // variant-0 z solve: N doubles
    double *d_host_stage = nullptr;  // *_host calls: N doubles
    // pz_solve_host_batch: staging fields, copy streams, events (created on first use)
    double *d_batch_stage[3] = {nullptr, nullptr, nullptr};
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    std::vector<cudaEvent_t> batch_events;
    int *d_xyctr = nullptr;          // fused x/y kernels: 2 x (64 + nz) ticket / per-plane counters
    int xy_bps[2] = {0, 0};          // fused x/y kernels: resident CTAs per SM (forward, inverse), 0 = not yet queried

    // Helmholtz
    double helm_a = -1.0;
    int helm_m = 0, helm_P = 0, helm_tx = 0, helm_levels = 0;
    int helm_variant = 0;            // variant the current tables were built for
    int helm_zs = 1;                 // variant 1: chunks the column is cut into (CTAs of a cluster), helm_P = sub-domains per chunk
    int helm_bps = 0;                // variant 1: resident CTAs per SM
    int helm_cn_P = 0, helm_cn_levels = 0; // whole-column tables for the one-kernel step of Eq. (11) (0 = none)
    size_t helm_cn_off = 0;          // their offset (doubles) in a table set
    size_t helm_cstride = 0;         // doubles of one chunk's table block
    int helm_nclusters[3] = {0, 0, 0}; // variant 1: resident clusters of 2 / 4 / 8 CTAs (0 = not yet queried)
    std::vector<pz::HelmTables> helm; // table sets: the current one, one being uploaded, and any a captured graph reads
    int helm_cur = -1;               // current set of the cell-centred operator (u, v)
    int helm_w_cur = -1;             // current set of the face-centred operator (w), helmholtz_w_setup
    double helm_w_a = -1.0;
    cudaStream_t upload_stream = nullptr;

    // z-slab of a distributed Poisson solve (poisson_slab_plan_create): nz above is the slab's own
    // number of planes; the z tables (d_A, d_C, d_dzf, d_zc) cover the global grid
    int slab_G = 0, slab_g = 0, nz_glob = 0;
    std::vector<int> slab_kb;        // G + 1 plane bounds
    int *d_slab_kb = nullptr;
    double *slab_coef = nullptr;     // [G][6][nx ny] interface coefficients of every slab
    double *slab_phi = nullptr;      // [2][nx ny] phi_prev, phi_next of this rank's slab
    size_t slab_bstride = 0;         // doubles per rank in the gathered boundary buffer
    bool slab_internal = false;      // the cut is the plan's own (one GPU, nz > 1024): poisson_solve runs all slabs
    double *islab_ball = nullptr;    // internal cut: the boundary buffers of all slabs

    // mixed-radix transforms (pz_fft_generic.cu): radices and launch geometry, worked out once per
    // (kernel family, number of lines); [x, y, cosine / sine x, cosine / sine y]
    struct GenGeo { long long key = -1; int n = 0, r[20] = {0}, per_cta = 0, threads = 0; };
    GenGeo gen_geo[4];

    // z-solve variant 2: launch geometry per (sub-domain rows M, HELM), queried once per plan (= per device)
    struct ZtGeo { int blocks = 0, stages = 0; };
    ZtGeo zt[4][4];   // [M][whole columns, HELM, slab reduce, slab finish]

    // tensor maps of the column-tile kernels, keyed by (field pointer, geometry): a solve that sees the
    // same field again encodes nothing
    struct MapEntry { const void *ptr; size_t ncols; int nz, tx, box_rows, l2promo, swz; CUtensorMap map; };
    std::vector<MapEntry> maps;
    size_t maps_next = 0;

    // kernels whose dynamic shared-memory limit has been raised on THIS plan's device (function
    // attributes are per device: no process-wide statics)
    std::vector<const void *> smem_optin;

    pz::Options opt;

    // optional per-launch event timing (pz_profile_enable)
    bool prof_on = false;
    struct ProfRec { int cls; cudaEvent_t start, stop; };
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_pool;
};

namespace pz {

// Timing-only diagnostics that skip arithmetic or stores (results are WRONG): compiled in only with
// -DPZ_PROBES (python -m paper_2502_06296_b200.build --probes); the shipped library has none.
#ifdef PZ_PROBES
constexpr bool kProbes = true;
#else
constexpr bool kProbes = false;
#endif

void set_error(const char *fmt, ...);
int cuda_fail(cudaError_t e, const char *what);
void count_launch(int n = 1);

#define PZ_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return ::pz::cuda_fail(e__, #call);                                \
    } while (0)

// Brackets one kernel launch with events when profiling is on.
struct ProfScope {
    pz_plan *pl; cudaStream_t st; cudaEvent_t stop = nullptr;
    ProfScope(const pz_plan *plan, int cls, cudaStream_t stream);
    ~ProfScope();
};

// kernels (each returns a pz_status)
// velocity source of the fused divergence (forward x transform, pz_fft_x.cu)
struct DivSrc {
    const double *u = nullptr, *v = nullptr, *w = nullptr, *dzf = nullptr;
    double rdx = 0, rdy = 0, scale = 0;
    int ny = 0;
};
int launch_fft_x(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st, const DivSrc *div = nullptr);
int launch_fft_y(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st);
int launch_pair0(const pz_plan *pl, double *p, int k0, int nk, bool inverse, cudaStream_t st);
int launch_zsolve(pz_plan *pl, double *p, cudaStream_t st, double helm_a = -1.0); // helm_a >= 0: Eq. (8) systems
int launch_divergence_rhs(pz_plan *pl, const double *u, const double *v, const double *w, double *out, double inv_gdt,
                          cudaStream_t st);
int launch_helmholtz_z_rhs(pz_plan *pl, double *u2, const double *uk, double a, cudaStream_t st);
int launch_project(pz_plan *pl, double *u, double *v, double *w, double *p, const double *phi, double gdt, cudaStream_t st);
// mixed-radix (2, 3, 5, 7) transforms for lengths the power-of-two kernels do not take (pz_fft_generic.cu)
int fft_radices(int n, int min_points, int stride, int *radices, int cap);
bool generic_fft_x_ok(int nx);
bool generic_fft_y_ok(int ny);
inline bool fast_fft_len(int n) { return n >= 8 && n <= 4096 && (n & (n - 1)) == 0; }
int launch_fft_x_generic(const pz_plan *pl, double *p, long long nlines, bool inverse, cudaStream_t st);
int launch_fft_y_generic(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st);
int launch_r2r_x(const pz_plan *pl, double *p, long long nlines, bool inverse, cudaStream_t st);
int launch_r2r_y(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st);
int launch_allpairs(const pz_plan *pl, double *p, int nk, bool inverse, cudaStream_t st);
int launch_fft_xy_fwd(pz_plan *pl, double *p, cudaStream_t st);
int launch_fft_xy_inv(pz_plan *pl, double *p, cudaStream_t st);
// where a slab's boundary block goes: one buffer (all-gather by the caller) or the slot of this
// rank in the gathered buffer of EVERY rank (peer memory over NVLink: the reduction kernel's own
// stores are the exchange)
struct BoutSet { double *p[16]; int n = 0; };
int launch_zslab_tma(pz_plan *pl, double *p, int kb, int nk, const BoutSet *bout, const double *phi_prev, const double *phi_next,
                     cudaStream_t st);
int launch_slab_coefficients(pz_plan *pl, cudaStream_t st);
int launch_slab_reduce(pz_plan *pl, double *p, const BoutSet &bout, cudaStream_t st);
int launch_slab_signal(pz_plan *pl, long long *const *flags, int n, int slot, long long epoch, cudaStream_t st);
int launch_slab_wait(pz_plan *pl, const long long *flags, int n, long long epoch, cudaStream_t st);
int launch_zsolve_islab(pz_plan *pl, double *p, cudaStream_t st);
int launch_slab_finish(pz_plan *pl, double *p, const double *ball, cudaStream_t st);
int launch_helmholtz_n(pz_plan *pl, double *const *u, int n, cudaStream_t st, int kind = 0); // kind 1: face-centred w
int launch_helmholtz_tma(pz_plan *pl, double *const *u, int n, const double *tab, cudaStream_t st);
int helmholtz_tma_prepare(pz_plan *pl);
int launch_helmholtz_tma_cn(pz_plan *pl, double *u2, const double *uk, const double *tab, cudaStream_t st);
int launch_helmholtz_step(pz_plan *pl, double *u2, const double *uk, cudaStream_t st);
int helmholtz_build_tables(pz_plan *pl, double a, int kind = 0);
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (plan, kernel)
int ensure_smem_optin(pz_plan *pl, const void *kernel, int bytes);
template <class K> int smem_optin(const pz_plan *pl, K kernel, size_t bytes)
{
    return ensure_smem_optin(const_cast<pz_plan *>(pl), reinterpret_cast<const void *>(kernel), (int)bytes);
}
// encode_column_tile_map (pz_tma.cuh) through the plan's small cache (at most 16 maps, round robin)
int cached_column_map(pz_plan *pl, const CUtensorMap **out, const double *field, size_t ncols, int nz, int tx, int box_rows,
                      int l2promo, bool swizzle128);

} // namespace pz
