// afid_plan.cu -- host side of the C ABI in include/afid.h: plan construction (metrics,
// tridiagonal coefficients, modified wavenumbers, twiddle tables), validation, and the
// launch sequence of one projection.  No CPU fallback and no library FFT: an unsupported
// size is an error.
#include "../../include/afid.h"
#include "afid_kernels.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace afid;

namespace {

thread_local std::string g_err;
thread_local int g_err_code = 0;

int fail(int code, const std::string& msg)
{
    g_err = msg;
    g_err_code = code;
    return code;
}

// ---- FFT length table: complex length -> radix plan and threads per line ------------------
//      X(N, R0, R1, R2, R3, TPL)
#define AFID_FFT_SIZES(X)       \
    X(8, 8, 1, 1, 1, 1)         \
    X(16, 16, 1, 1, 1, 1)       \
    X(24, 8, 3, 1, 1, 3)        \
    X(32, 8, 4, 1, 1, 4)        \
    X(48, 16, 3, 1, 1, 4)       \
    X(64, 8, 8, 1, 1, 8)        \
    X(96, 16, 6, 1, 1, 8)       \
    X(128, 16, 8, 1, 1, 8)      \
    X(192, 16, 12, 1, 1, 16)    \
    X(256, 16, 16, 1, 1, 16)    \
    X(384, 8, 8, 6, 1, 48)      \
    X(512, 8, 8, 8, 1, 64)      \
    X(768, 16, 16, 3, 1, 48)    \
    X(1024, 16, 8, 8, 1, 64)    \
    X(1536, 16, 16, 6, 1, 96)   \
    X(2048, 16, 16, 8, 1, 128)  \
    X(3072, 16, 16, 12, 1, 192) \
    X(4096, 16, 16, 16, 1, 256) \
    X(40, 8, 5, 1, 1, 5)        \
    X(80, 16, 5, 1, 1, 5)       \
    X(160, 8, 4, 5, 1, 20)      \
    X(320, 8, 8, 5, 1, 40)      \
    X(640, 16, 8, 5, 1, 40)     \
    X(1280, 16, 16, 5, 1, 80)   \
    X(2560, 16, 16, 2, 5, 160)  \
    X(72, 12, 6, 1, 1, 6)       \
    X(144, 12, 12, 1, 1, 12)    \
    X(216, 6, 6, 6, 1, 36)      \
    X(288, 12, 12, 2, 1, 24)    \
    X(432, 12, 6, 6, 1, 36)     \
    X(576, 12, 12, 4, 1, 48)    \
    X(648, 12, 6, 3, 3, 54)     \
    X(864, 12, 12, 6, 1, 72)    \
    X(1152, 12, 12, 8, 1, 96)   \
    X(1296, 12, 12, 3, 3, 108)  \
    X(1728, 12, 12, 12, 1, 144) \
    X(2304, 16, 12, 12, 1, 144) \
    X(2592, 12, 12, 6, 3, 216)  \
    X(3456, 12, 12, 12, 2, 288)

// z-direction lines (K1, K5; complex length nz/2): plans with <= 12 elements per thread where
// it matters, so that twice as many warps are resident while the loads are in flight
#define AFID_FFT_SIZES_Z(X)     \
    X(8, 8, 1, 1, 1, 1)         \
    X(16, 16, 1, 1, 1, 1)       \
    X(24, 8, 3, 1, 1, 3)        \
    X(32, 8, 4, 1, 1, 4)        \
    X(48, 16, 3, 1, 1, 4)       \
    X(64, 8, 8, 1, 1, 8)        \
    X(96, 16, 6, 1, 1, 8)       \
    X(128, 16, 8, 1, 1, 8)      \
    X(192, 16, 12, 1, 1, 16)    \
    X(256, 16, 16, 1, 1, 16)    \
    X(384, 8, 8, 6, 1, 48)      \
    X(512, 8, 8, 8, 1, 64)      \
    X(768, 16, 16, 3, 1, 48)    \
    X(1024, 8, 16, 8, 1, 128)   \
    X(40, 8, 5, 1, 1, 5)        \
    X(80, 16, 5, 1, 1, 5)       \
    X(160, 8, 4, 5, 1, 20)      \
    X(320, 8, 8, 5, 1, 40)      \
    X(640, 16, 8, 5, 1, 40)     \
    X(1280, 16, 16, 5, 1, 80)   \
    X(1536, 16, 16, 6, 1, 96)   \
    X(12, 12, 1, 1, 1, 1)       \
    X(18, 6, 3, 1, 1, 3)        \
    X(36, 6, 6, 1, 1, 6)        \
    X(54, 6, 3, 3, 1, 9)        \
    X(72, 12, 6, 1, 1, 6)       \
    X(108, 12, 3, 3, 1, 9)      \
    X(144, 12, 12, 1, 1, 12)    \
    X(162, 6, 3, 3, 3, 27)      \
    X(216, 6, 6, 6, 1, 36)      \
    X(288, 12, 12, 2, 1, 24)    \
    X(324, 6, 6, 3, 3, 54)      \
    X(432, 12, 6, 6, 1, 36)     \
    X(576, 12, 12, 4, 1, 48)    \
    X(648, 12, 6, 3, 3, 54)     \
    X(864, 12, 12, 6, 1, 72)    \
    X(1152, 12, 12, 8, 1, 96)   \
    X(1296, 12, 12, 3, 3, 108)

constexpr int K1_NL = 4; // lines per CTA in K1 (two CTAs fill one 128-byte row of B)
// lines per CTA in K2 / K4: 2 (256-byte gather segments), 1 for the longest lines (two 256-thread CTAs per SM
// instead of one 512-thread CTA)
template <class PL> constexpr int ky_nl() { return tpl8<PL>() >= 256 ? 1 : 2; }

struct LaunchCfg {
    const void* fn;
    int threads;
    size_t smem;
    int ctas_per_sm; // CTAs per SM the shared-memory carveout is sized for (the rest stays L1)
    int nl;          // lines per CTA (K2 / K4)
};

template <class PL> LaunchCfg cfg_k1()
{
    return {(const void*)k_div_r2c<PL, K1_NL>, K1_NL * PL::TPL, (size_t)K1_NL * PL::LS * sizeof(cplx), 3};
}
template <class PL> LaunchCfg cfg_k2()
{
    return {(const void*)k_fft_y<PL, ky_nl<PL>()>, ky_nl<PL>() * tpl8<PL>(), (size_t)ky_nl<PL>() * PL::LS * sizeof(cplx), 3, ky_nl<PL>()};
}
template <class PL> LaunchCfg cfg_k4()
{
    return {(const void*)k_ifft_y<PL, ky_nl<PL>()>, ky_nl<PL>() * tpl8<PL>(), (size_t)ky_nl<PL>() * PL::LS * sizeof(cplx), 3, ky_nl<PL>()};
}
// K5: all 8 lines of a tile in one round where that leaves >= 128 registers per thread, else two rounds of 4;
// two tile buffers (TMA prefetch of the next tile) where they fit the 227 KB of an SM
template <class PL> constexpr int k5_lpr() { return (8 * PL::TPL <= 512) ? 8 : 4; }
// bytes of K5's staged twiddle table (nz/2 + 1 complex, rounded up to 128 bytes)
template <class PL> constexpr size_t k5_tw_bytes() { return ((size_t)(PL::N + 1) * sizeof(cplx) + 127) / 128 * 128; }
template <class PL> constexpr size_t k5_tile_bytes() { return (size_t)k5_smem_rows<PL>() * 8 * sizeof(cplx); }
template <class PL> constexpr int k5_nbuf() { return (2 * k5_tile_bytes<PL>() + 2048 <= 227 * 1024) ? 2 : 1; }
template <class PL> constexpr bool k5_stw() { return k5_nbuf<PL>() * k5_tile_bytes<PL>() + k5_tw_bytes<PL>() + 2048 <= 227 * 1024; }
template <class PL> LaunchCfg cfg_k5()
{
    // .nl = CTAs per SM the launch is sized for
    return {(const void*)k_c2r_z<PL, k5_lpr<PL>(), k5_nbuf<PL>(), k5_stw<PL>()>, k5_lpr<PL>() * PL::TPL,
            k5_nbuf<PL>() * k5_tile_bytes<PL>() + (k5_stw<PL>() ? k5_tw_bytes<PL>() : 0) + 1024, 1, 1};
}

bool lookup_fft_y(int n, LaunchCfg* k2, LaunchCfg* k4)
{
    switch (n) {
#define X(N, R0, R1, R2, R3, TPL)                   \
    case N: {                                       \
        typedef FftPlan<R0, R1, R2, R3, TPL> PL;    \
        if (k2) *k2 = cfg_k2<PL>();                 \
        if (k4) *k4 = cfg_k4<PL>();                 \
        return true;                                \
    }
        AFID_FFT_SIZES(X)
#undef X
    default:
        return false;
    }
}
bool lookup_fft_z(int n, LaunchCfg* k1, LaunchCfg* k5)
{
    switch (n) {
#define X(N, R0, R1, R2, R3, TPL)                   \
    case N: {                                       \
        typedef FftPlan<R0, R1, R2, R3, TPL> PL;    \
        if (k1) *k1 = cfg_k1<PL>();                 \
        if (k5) *k5 = cfg_k5<PL>();                 \
        return true;                                \
    }
        AFID_FFT_SIZES_Z(X)
#undef X
    default:
        return false;
    }
}

constexpr int MAX_NX = 2048;

// K3 instantiation, block size and shared memory for nx rows
LaunchCfg select_k3(int nx, int* kw_out, int* m_out)
{
    LaunchCfg c{};
    int M, kw = 8;
    if (nx < 64) { M = 4; c.fn = (nx % 4 == 0) ? (const void*)k_solve_x<4, true, 8, 128> : (const void*)k_solve_x<4, false, 8, 128>; }
    else {
        M = 16;
        // 8-wide tiles if two of them fit an SM, else 4-wide ones (two CTAs per SM: one gathers while the other computes)
        const size_t smem8 = (size_t)k3_tile_rows(nx) * 8 * sizeof(cplx) + (size_t)10 * ((nx + 15) / 16) * 8 * sizeof(double)
                             + (size_t)k3_coef_slots(nx, 16) * sizeof(double2) + 128;
        if (2 * (smem8 + 1024) > 228 * 1024) kw = 4;
        const bool ex = (nx % 16 == 0);
        if (kw == 8) c.fn = ex ? (const void*)k_solve_x<16, true, 8, 512> : (const void*)k_solve_x<16, false, 8, 512>;
        else if (nx <= 1024) c.fn = ex ? (const void*)k_solve_x<16, true, 4, 256> : (const void*)k_solve_x<16, false, 4, 256>;
        else if (nx <= 1536) c.fn = ex ? (const void*)k_solve_x<16, true, 4, 384> : (const void*)k_solve_x<16, false, 4, 384>;
        else c.fn = ex ? (const void*)k_solve_x<16, true, 4, 512> : (const void*)k_solve_x<16, false, 4, 512>;
    }
    const int pch = (nx + M - 1) / M;
    c.threads = kw * pch;
    c.smem = (size_t)k3_tile_rows(nx) * kw * sizeof(cplx) + (size_t)10 * pch * kw * sizeof(double)
             + (size_t)k3_coef_slots(nx, M) * sizeof(double2) + 128;
    c.ctas_per_sm = 4;
    c.nl = 0;
    *kw_out = kw;
    *m_out = M;
    return c;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup (no link-time
// dependency on libcuda, so the library still loads on a machine without a driver)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// 3-D fp64 tensor map over a complex array [d2][d1][d0/2 complex]; box = (b0 doubles, b1, b2)
bool make_map3(CUtensorMap* m, void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t b0, uint32_t b1, uint32_t b2,
               CUtensorMapSwizzle swz)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {d0 * 8, d0 * d1 * 8};
    cuuint32_t box[3] = {b0, b1, b2};
    cuuint32_t es[3] = {1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

} // namespace

// the auxiliary streams / events of the plane-pipelined sweeps (afid_plan_set_pipeline)
constexpr int PIPE_STREAMS = 3;
constexpr int PIPE_EVENTS = 8;   // per kind; >= the largest rotation depth + 1

constexpr int MAX_RANKS = 64;   // sharded plans

struct afid_plan {
    int nx, ny, nz, nzh;   // nx = planes of THIS plan's x-slab (= the whole grid for an unsharded plan)
    int device;        // the device the plan was created on (its work arrays and tensor maps live there)
    // sharded plans: the global grid has gnx planes; this rank owns the x-slab [bx[rank], bx[rank+1]) for the
    // divergence, the transforms and the correction, and the modes kz in [bk[rank], bk[rank+1]) for the x-solves
    int gnx, rank, nranks;
    int bx[MAX_RANKS + 1], bk[MAX_RANKS + 1];
    DevParams dp;      // slab kernels (K1, K2, K4, K5, K6): nx = slab planes, metric tables offset to the slab
    DevParams dps;     // x-solve (K3): nx = gnx, nzh = this rank's kz count, lamz offset to its first kz
    void* tables;      // one device allocation holding all tables
    size_t tables_bytes;
    cplx* ws[2];       // work arrays, nx*nzh*ny complex each
    size_t ws_bytes;
    LaunchCfg k1, k2, k4, k5, k3;
    bool accumulate;   // p += phi instead of p = phi (afid_plan_set_accumulate)
    int* cfl_sync;     // afid_project_cfl: ticket counter + one "corrected" flag per K6 item (device)
    size_t cfl_sync_bytes;
    int cfl_ctas;      // resident CTAs of k_correct_cfl<K6_U, 1>
    int cfl_ctas2;     // ... of the <2, 2> variant (hint bit 32)
    int k3_kw;         // systems per K3 CTA (8 or 4)
    alignas(64) CUtensorMap mapC;   // K3's gather of C = ws[1] viewed as [nzh][nx][2 ny] doubles
    alignas(64) CUtensorMap mapD;   // K5's gather of D = ws[1], same view, 128-byte swizzle
    int n_sm;
    // plane-pipelined sweeps (afid_plan_set_pipeline): batches of pipe_batch planes, intermediates B and D in
    // a rotating buffer of pipe_rot batches that stays in L2
    int pipe_batch, pipe_rot;
    cudaStream_t aux[PIPE_STREAMS];
    cudaEvent_t ev_fork, ev_join[PIPE_STREAMS], ev_a[PIPE_EVENTS], ev_b[PIPE_EVENTS];
    bool pipe_ready;
    // optional per-kernel timing (afid_plan_enable_timing): NK+1 events around the NK kernels
    bool timing;
    cudaEvent_t ev[7];
    bool ev_valid;
};

static const char* const KERNEL_NAMES[6] = {"k_div_r2c", "k_fft_y", "k_solve_x", "k_ifft_y", "k_c2r_z", "k_correct"};
// pipelined: the kernels of a sweep overlap, so only the three sweeps can be timed
static const char* const SWEEP_NAMES[3] = {"sweep_forward", "k_solve_x", "sweep_inverse"};
static bool pipelined(const afid_plan* pl) { return pl->pipe_batch > 0; }

#define AFID_EXPORT __attribute__((visibility("default")))

extern "C" {

AFID_EXPORT const char* afid_version(void) { return "afid-project-b200 0.2 (sm_100a, fp64)"; }
AFID_EXPORT const char* afid_last_error(void) { return g_err.c_str(); }
AFID_EXPORT int afid_last_error_code(void) { return g_err_code; }
AFID_EXPORT int afid_max_nx(void) { return MAX_NX; }
AFID_EXPORT int afid_fft_length_supported(int n) { return lookup_fft_y(n, nullptr, nullptr) ? 1 : 0; }
AFID_EXPORT int afid_fft_half_length_supported(int n) { return lookup_fft_z(n, nullptr, nullptr) ? 1 : 0; }

} // extern "C"

// One kernel instantiation serves many grid sizes (and several live plans), so the dynamic shared-memory
// limit of a function is raised to the device maximum once and never lowered; the carveout is a hint only.
static int set_smem_attr(const LaunchCfg& c, size_t optin_max)
{
    {
        const size_t per_sm = 228 * 1024;
        size_t want = (size_t)c.ctas_per_sm * (c.smem + 1024);
        if (want > per_sm) want = per_sm;
        const int pct = (int)((want * 100 + per_sm - 1) / per_sm);
        cudaFuncSetAttribute(c.fn, cudaFuncAttributePreferredSharedMemoryCarveout, pct);
    }
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, c.fn);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaFuncGetAttributes: ") + cudaGetErrorString(e));
    if (c.smem + fa.sharedSizeBytes > optin_max) return fail(AFID_ERR_UNSUPPORTED_SIZE, "tile does not fit shared memory");
    e = cudaFuncSetAttribute(c.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(optin_max - fa.sharedSizeBytes));
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
    return AFID_OK;
}

static void destroy_pipeline(afid_plan* pl)
{
    if (!pl->pipe_ready) return;
    cudaEventDestroy(pl->ev_fork);
    for (int k = 0; k < PIPE_STREAMS; ++k) {
        cudaStreamDestroy(pl->aux[k]);
        cudaEventDestroy(pl->ev_join[k]);
    }
    for (int k = 0; k < PIPE_EVENTS; ++k) {
        cudaEventDestroy(pl->ev_a[k]);
        cudaEventDestroy(pl->ev_b[k]);
    }
    pl->pipe_ready = false;
}

// free whatever a partially built plan holds (the struct is zero-initialised; cudaFree(nullptr) is a no-op)
static void discard_plan(afid_plan* pl)
{
    destroy_pipeline(pl);
    cudaFree(pl->ws[0]);
    cudaFree(pl->ws[1]);
    cudaFree(pl->tables);
    cudaFree(pl->cfl_sync);
    delete pl;
}

extern "C" {

} // extern "C"

// balanced contiguous partition of n items over R parts: part r = [n r / R, n (r+1) / R)
static int part_bound(int n, int R, int r) { return (int)((long long)n * r / R); }

// nx = GLOBAL number of planes; the plan built is rank `rank` of `nranks` (1 rank: the whole problem)
static afid_plan* create_impl(int nx, int ny, int nz, const double* xc, double Ly, double Lz, int rank, int nranks)
{
    g_err.clear();
    g_err_code = 0;
    if (!xc) { fail(AFID_ERR_NULL, "xc is NULL"); return nullptr; }
    if (nx < 2 || nx > MAX_NX) { fail(AFID_ERR_UNSUPPORTED_SIZE, "nx must be in [2, afid_max_nx()]"); return nullptr; }
    if (ny < 8 || nz < 16 || (nz & 1)) { fail(AFID_ERR_UNSUPPORTED_SIZE, "ny >= 8 and even nz >= 16 required"); return nullptr; }
    if (!(Ly > 0.0) || !(Lz > 0.0) || !std::isfinite(Ly) || !std::isfinite(Lz)) { fail(AFID_ERR_GRID, "Ly, Lz must be finite and > 0"); return nullptr; }
    for (int i = 0; i <= nx; ++i)
        if (!std::isfinite(xc[i]) || (i > 0 && !(xc[i] > xc[i - 1]))) { fail(AFID_ERR_GRID, "xc must be finite and strictly increasing"); return nullptr; }
    const int nh = nz / 2;
    if (nranks < 1 || nranks > MAX_RANKS || rank < 0 || rank >= nranks) { fail(AFID_ERR_UNSUPPORTED_SIZE, "rank / nranks out of range (nranks <= 64)"); return nullptr; }
    if (nranks > nx || nranks > nh + 1) { fail(AFID_ERR_UNSUPPORTED_SIZE, "more ranks than x-planes or kz modes"); return nullptr; }
    afid_plan* pl = new (std::nothrow) afid_plan();
    if (!pl) { fail(AFID_ERR_NOMEM, "host allocation failed"); return nullptr; }
    std::memset(pl, 0, sizeof(*pl));
    if (!lookup_fft_y(ny, &pl->k2, &pl->k4)) { delete pl; fail(AFID_ERR_UNSUPPORTED_SIZE, "ny is not a supported FFT length"); return nullptr; }
    if (!lookup_fft_z(nh, &pl->k1, &pl->k5)) { delete pl; fail(AFID_ERR_UNSUPPORTED_SIZE, "nz/2 is not a supported FFT length"); return nullptr; }
    pl->gnx = nx; pl->rank = rank; pl->nranks = nranks;
    for (int r = 0; r <= nranks; ++r) { pl->bx[r] = part_bound(nx, nranks, r); pl->bk[r] = part_bound(nh + 1, nranks, r); }
    const int xs = pl->bx[rank], nxl = pl->bx[rank + 1] - xs, ks = pl->bk[rank], nkz = pl->bk[rank + 1] - ks;
    pl->nx = nxl; pl->ny = ny; pl->nz = nz; pl->nzh = nh + 1;

    // ---- K3 configuration
    int k3_m = 0;
    pl->k3 = select_k3(nx, &pl->k3_kw, &k3_m);

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        delete pl; fail(AFID_ERR_CUDA, "no CUDA device"); return nullptr;
    }
    if (prop.major != 10) { delete pl; fail(AFID_ERR_CUDA, "this library is built for sm_100a (B200) only"); return nullptr; }
    pl->device = dev;
    pl->n_sm = prop.multiProcessorCount;
    for (const LaunchCfg* c : {&pl->k1, &pl->k2, &pl->k3, &pl->k4, &pl->k5}) {
        if (c->smem > prop.sharedMemPerBlockOptin) { delete pl; fail(AFID_ERR_UNSUPPORTED_SIZE, "tile does not fit shared memory"); return nullptr; }
        if (set_smem_attr(*c, prop.sharedMemPerBlockOptin) != AFID_OK) { delete pl; return nullptr; }
    }

    {   // K5 is persistent: as many CTAs as are resident at once
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pl->k5.fn, pl->k5.threads, pl->k5.smem) != cudaSuccess || occ < 1) {
            cudaGetLastError(); delete pl; fail(AFID_ERR_CUDA, "k_c2r_z does not fit an SM"); return nullptr;
        }
        pl->k5.nl = occ;
    }

    // ---- host tables (long double, rounded once to fp64)
    typedef long double ld;
    std::vector<double> dx(nx), dc(nx + 1, 0.0), rdx(nx), rdc(nx + 1, 0.0), ca(nx, 0.0), cc(nx, 0.0), lamy(ny), lamz(nh + 1);
    // metrics: one fp64 subtraction of the inputs each (R1/R4)
    for (int i = 0; i < nx; ++i) dx[i] = xc[i + 1] - xc[i];
    for (int i = 1; i < nx; ++i) dc[i] = (xc[i + 1] - xc[i - 1]) / 2.0;
    ld vol = 0.0L;
    for (int i = 0; i < nx; ++i) {
        rdx[i] = (double)(1.0L / (ld)dx[i]);
        vol += (ld)dx[i];
        if (i >= 1) { rdc[i] = (double)(1.0L / (ld)dc[i]); ca[i] = (double)(1.0L / ((ld)dx[i] * (ld)dc[i])); }
        if (i <= nx - 2) cc[i] = (double)(1.0L / ((ld)dx[i] * (ld)dc[i + 1]));
    }
    const ld pi = acosl(-1.0L);
    const double dy = Ly / ny, dz = Lz / nz;
    // modified wavenumbers 2(1-cos(2 pi k/n))/Delta^2 = 4 sin^2(pi k/n)/Delta^2
    for (int k = 0; k < ny; ++k) { ld s = sinl(pi * (ld)k / (ld)ny); lamy[k] = (double)(4.0L * s * s / ((ld)dy * (ld)dy)); }
    for (int k = 0; k <= nh; ++k) { ld s = sinl(pi * (ld)k / (ld)nz); lamz[k] = (double)(4.0L * s * s / ((ld)dz * (ld)dz)); }
    std::vector<double> twy(2 * (size_t)ny), twzh(2 * (size_t)nh), twz(2 * (size_t)(nh + 1));
    auto fill_tw = [&](std::vector<double>& t, int count, int n) {
        for (int k = 0; k < count; ++k) {
            const ld ang = 2.0L * pi * (ld)k / (ld)n;
            t[2 * k] = (double)cosl(ang);
            t[2 * k + 1] = (double)(-sinl(ang));
        }
    };
    fill_tw(twy, ny, ny);
    fill_tw(twzh, nh, nh);
    fill_tw(twz, nh + 1, nz);
    // K3's coefficient table {a_i, c_i} in the kernel's shared-memory layout (one bulk copy per CTA)
    std::vector<double> acp(2 * (size_t)k3_coef_slots(nx, k3_m), 0.0);
    {
        const int sk = (pl->k3_kw == 4) ? K3_SKEW : 0, pch = (nx + k3_m - 1) / k3_m;
        for (int q = 0; q < pch; ++q)
            for (int i = k3_chunk_start(q, k3_m, sk, nx, pch); i < k3_chunk_start(q + 1, k3_m, sk, nx, pch); ++i) {
                const size_t slot = (size_t)q * (k3_m + 1) + (i - k3_chunk_start(q, k3_m, sk, nx, pch));
                acp[2 * slot] = ca[i];
                acp[2 * slot + 1] = cc[i];
            }
    }

    // ---- one device allocation for all tables (each sub-table 256-byte aligned)
    struct Item { const void* src; size_t bytes; size_t off; };
    std::vector<Item> items = {
        {rdx.data(), rdx.size() * 8, 0}, {rdc.data(), rdc.size() * 8, 0}, {dx.data(), dx.size() * 8, 0},
        {ca.data(), ca.size() * 8, 0},   {cc.data(), cc.size() * 8, 0},   {lamy.data(), lamy.size() * 8, 0},
        {lamz.data(), lamz.size() * 8, 0}, {twy.data(), twy.size() * 8, 0}, {twzh.data(), twzh.size() * 8, 0},
        {twz.data(), twz.size() * 8, 0}, {acp.data(), acp.size() * 8, 0}};
    size_t off = 0;
    for (auto& it : items) { it.off = off; off += (it.bytes + 255) / 256 * 256; }
    pl->tables_bytes = off;
    if (cudaMalloc(&pl->tables, off) != cudaSuccess) { cudaGetLastError(); discard_plan(pl); fail(AFID_ERR_NOMEM, "cudaMalloc(tables) failed"); return nullptr; }
    for (auto& it : items)
        if (cudaMemcpy((char*)pl->tables + it.off, it.src, it.bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
            discard_plan(pl); fail(AFID_ERR_CUDA, "cudaMemcpy(tables) failed"); return nullptr;
        }
    {   // a work array holds the slab's half spectrum (nxl planes x all kz) or this rank's modes (all planes x nkz)
        const size_t a = (size_t)nxl * pl->nzh, b = (size_t)nx * nkz;
        pl->ws_bytes = (a > b ? a : b) * ny * sizeof(cplx);
    }
    for (int b = 0; b < 2; ++b)
        if (cudaMalloc((void**)&pl->ws[b], pl->ws_bytes) != cudaSuccess) {
            cudaGetLastError();
            discard_plan(pl); fail(AFID_ERR_NOMEM, "cudaMalloc(work arrays) failed"); return nullptr;
        }
    {   // afid_project_cfl: flags and the persistent grid of the fused correction + CFL kernel
        pl->cfl_sync_bytes = (1 + (size_t)nxl * (ny / K6_JL)) * sizeof(int);
        if (cudaMalloc((void**)&pl->cfl_sync, pl->cfl_sync_bytes) != cudaSuccess) {
            cudaGetLastError();
            discard_plan(pl); fail(AFID_ERR_NOMEM, "cudaMalloc(cfl flags) failed"); return nullptr;
        }
        int occ = 0, occ2 = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)k_correct_cfl<K6_U, 1>, K6_JL * K6_TX, 0) != cudaSuccess || occ < 1 ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, (const void*)k_correct_cfl<2, 2>, K6_JL * K6_TX, 0) != cudaSuccess || occ2 < 1) {
            cudaGetLastError();
            discard_plan(pl); fail(AFID_ERR_CUDA, "k_correct_cfl does not fit an SM"); return nullptr;
        }
        pl->cfl_ctas = occ * pl->n_sm;
        pl->cfl_ctas2 = occ2 * pl->n_sm;
    }
    if (!make_map3(&pl->mapC, pl->ws[1], 2 * (uint64_t)ny, (uint64_t)nx, (uint64_t)nkz, 2 * (uint32_t)pl->k3_kw, (uint32_t)k3_box_rows(nx), 1,
                   CU_TENSOR_MAP_SWIZZLE_NONE)) {
        discard_plan(pl);
        fail(AFID_ERR_CUDA, "cuTensorMapEncodeTiled failed"); return nullptr;
    }
    if (!make_map3(&pl->mapD, pl->ws[1], 2 * (uint64_t)ny, (uint64_t)pl->nzh, (uint64_t)nxl, 16, (uint32_t)k5_box_rows(nh), 1,
                   CU_TENSOR_MAP_SWIZZLE_128B)) {
        discard_plan(pl);
        fail(AFID_ERR_CUDA, "cuTensorMapEncodeTiled failed"); return nullptr;
    }
    char* tb = (char*)pl->tables;
    DevParams& d = pl->dp;
    d.nx = nx; d.ny = ny; d.nz = nz; d.nzh = nh + 1;
    d.rdy = (double)(1.0L / (ld)dy);
    d.rdz = (double)(1.0L / (ld)dz);
    d.spec_scale = (double)(-1.0L / ((ld)ny * (ld)nz));
    d.rdx = (const double*)(tb + items[0].off);
    d.rdc = (const double*)(tb + items[1].off);
    d.dxw = (const double*)(tb + items[2].off);
    d.ca = (const double*)(tb + items[3].off);
    d.cc = (const double*)(tb + items[4].off);
    d.lamy = (const double*)(tb + items[5].off);
    d.lamz = (const double*)(tb + items[6].off);
    d.tw_y = (const cplx*)(tb + items[7].off);
    d.tw_zh = (const cplx*)(tb + items[8].off);
    d.tw_z = (const cplx*)(tb + items[9].off);
    d.acp = (const double2*)(tb + items[10].off);
    d.inv_vol = (double)(1.0L / vol);
    d.hints = 0;
    d.has_mean = (ks == 0) ? 1 : 0;
    d.k3_prefetch = 0;
    {   // K3 prefetch distance = the CTAs resident at once
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pl->k3.fn, pl->k3.threads, pl->k3.smem) == cudaSuccess && occ >= 1) d.k3_prefetch = occ * pl->n_sm;
        else cudaGetLastError();
    }
    pl->dps = d;                 // x-solve: all planes, this rank's kz
    pl->dps.nzh = nkz;
    pl->dps.lamz = d.lamz + ks;
    d.nx = nxl;                  // slab kernels: this rank's planes, all kz
    d.rdx += xs;
    d.rdc += xs;
    d.dxw += xs;
    return pl;
}

extern "C" {

AFID_EXPORT afid_plan* afid_plan_create(int nx, int ny, int nz, const double* xc, double Ly, double Lz)
{
    return create_impl(nx, ny, nz, xc, Ly, Lz, 0, 1);
}

AFID_EXPORT int afid_plan_destroy(afid_plan* pl)
{
    if (!pl) return AFID_OK;
    if (pl->timing)
        for (int k = 0; k < 7; ++k) cudaEventDestroy(pl->ev[k]);
    discard_plan(pl);
    return AFID_OK;
}

AFID_EXPORT size_t afid_plan_workspace_bytes(const afid_plan* pl) { return pl ? 2 * pl->ws_bytes + pl->tables_bytes : 0; }

AFID_EXPORT int afid_plan_num_launches(const afid_plan* pl)
{
    if (!pl) return 0;
    if (!pipelined(pl)) return 6;
    const int nb = (pl->nx + pl->pipe_batch - 1) / pl->pipe_batch;
    return 5 * nb + 1;
}

AFID_EXPORT int afid_plan_set_l2_hints(afid_plan* pl, int mask)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    if (mask < 0 || mask > 63) return fail(AFID_ERR_UNSUPPORTED_SIZE, "hint mask must be in [0, 63]");
    pl->dp.hints = mask;
    return AFID_OK;
}

AFID_EXPORT int afid_plan_set_pipeline(afid_plan* pl, int planes_per_batch, int rotation)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    if (planes_per_batch <= 0) { pl->pipe_batch = 0; pl->pipe_rot = 0; return AFID_OK; }
    if (rotation < 2 || rotation >= PIPE_EVENTS) return fail(AFID_ERR_UNSUPPORTED_SIZE, "rotation must be in [2, 7]");
    if ((planes_per_batch % pl->k4.nl) != 0) return fail(AFID_ERR_UNSUPPORTED_SIZE, "planes_per_batch must be a multiple of the planes one inverse-transform CTA handles");
    if ((size_t)planes_per_batch * rotation > (size_t)pl->nx) return fail(AFID_ERR_UNSUPPORTED_SIZE, "planes_per_batch * rotation exceeds nx");
    if (!pl->pipe_ready) {
        bool ok = cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming) == cudaSuccess;
        for (int k = 0; k < PIPE_STREAMS && ok; ++k)
            ok = cudaStreamCreateWithFlags(&pl->aux[k], cudaStreamNonBlocking) == cudaSuccess && cudaEventCreateWithFlags(&pl->ev_join[k], cudaEventDisableTiming) == cudaSuccess;
        for (int k = 0; k < PIPE_EVENTS && ok; ++k)
            ok = cudaEventCreateWithFlags(&pl->ev_a[k], cudaEventDisableTiming) == cudaSuccess && cudaEventCreateWithFlags(&pl->ev_b[k], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) return fail(AFID_ERR_CUDA, "stream / event creation failed");
        pl->pipe_ready = true;
    }
    pl->pipe_batch = planes_per_batch;
    pl->pipe_rot = rotation;
    return AFID_OK;
}

} // extern "C"

static int launch(const LaunchCfg& c, unsigned grid, cudaStream_t st, void** args, const char* name)
{
    cudaError_t e = cudaLaunchKernel(c.fn, dim3(grid), dim3(c.threads), args, c.smem, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string(name) + ": " + cudaGetErrorString(e));
    return AFID_OK;
}

static int check_ptr(const void* p, const char* name)
{
    if (!p) return fail(AFID_ERR_NULL, std::string(name) + " is NULL");
    if (((size_t)p & 15) != 0) return fail(AFID_ERR_ALIGN, std::string(name) + " is not 16-byte aligned");
    return AFID_OK;
}

// the plan's work arrays, tables and tensor maps live on the device it was created on
static int check_device(const afid_plan* pl)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(AFID_ERR_CUDA, "cudaGetDevice failed");
    if (dev != pl->device) return fail(AFID_ERR_CUDA, "the current device is not the device the plan was created on");
    return AFID_OK;
}

static int record(cudaEvent_t ev, cudaStream_t st)
{
    cudaError_t e = cudaEventRecord(ev, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaEventRecord: ") + cudaGetErrorString(e));
    return AFID_OK;
}
static int wait_on(cudaStream_t st, cudaEvent_t ev)
{
    cudaError_t e = cudaStreamWaitEvent(st, ev, 0);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaStreamWaitEvent: ") + cudaGetErrorString(e));
    return AFID_OK;
}

static int launch_k1(afid_plan* pl, const double* u, const double* v, const double* w, cplx* B, int i_base, int np, int bmod, cudaStream_t st)
{
    void* args[] = {&pl->dp, (void*)&u, (void*)&v, (void*)&w, (void*)&B, &i_base, &np, &bmod};
    return launch(pl->k1, (unsigned)(np * (pl->ny / K1_NL)), st, args, "k_div_r2c");
}
static int launch_k2(afid_plan* pl, const cplx* B, cplx* C, int i_base, int np, int bmod, cudaStream_t st)
{
    const int ngrp2 = (pl->nzh + pl->k2.nl - 1) / pl->k2.nl;
    void* args[] = {&pl->dp, (void*)&B, (void*)&C, &i_base, &bmod};
    return launch(pl->k2, (unsigned)(np * ngrp2), st, args, "k_fft_y");
}
static int launch_k4(afid_plan* pl, const cplx* T, cplx* D, int i_base, int np, int dmod, cudaStream_t st)
{
    void* args[] = {&pl->dp, (void*)&T, (void*)&D, &i_base, &np, &dmod};
    return launch(pl->k4, (unsigned)(pl->nzh * ((np + pl->k4.nl - 1) / pl->k4.nl)), st, args, "k_ifft_y");
}
static int launch_k5(afid_plan* pl, double* phi, int i_base, int np, int dmod, cudaStream_t st)
{
    void* args[] = {&pl->dp, (void*)&pl->mapD, (void*)&phi, &i_base, &np, &dmod};
    const long long ntile = (long long)np * (pl->ny / 8), resident = (long long)pl->n_sm * pl->k5.nl;   // persistent CTAs
    return launch(pl->k5, (unsigned)(ntile < resident ? ntile : resident), st, args, "k_c2r_z");
}
static int launch_correct(afid_plan* pl, double* u, double* v, double* w, double* p, int i_base, int np, cudaStream_t st, double* pacc,
                          const double* p_halo = nullptr)
{
    void* args[] = {&pl->dp, (void*)&p, (void*)&u, (void*)&v, (void*)&w, &i_base, &np, (void*)&pacc, (void*)&p_halo};
    cudaError_t e = cudaLaunchKernel((const void*)k_correct, dim3((unsigned)(np * (pl->ny / K6_JL))), dim3(K6_TX, K6_JL), args, 0, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("k_correct: ") + cudaGetErrorString(e));
    return AFID_OK;
}

// the fused correction + CFL maximum (afid_project_cfl): zero the ticket / flags, floor into *cfl, one persistent launch
static int launch_correct_cfl(afid_plan* pl, double* u, double* v, double* w, double* p, cudaStream_t st, double* pacc, double* cfl)
{
    cudaError_t e = cudaMemsetAsync(pl->cfl_sync, 0, pl->cfl_sync_bytes, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e));
    k_cfl_init<<<1, 1, 0, st>>>(cfl);
    const long long nitems = (long long)pl->nx * (pl->ny / K6_JL);
    const bool v2 = (pl->dp.hints & 32) != 0;
    const int ctas = v2 ? pl->cfl_ctas2 : pl->cfl_ctas;
    const int grid = (int)(nitems < ctas ? nitems : ctas);
    int lag = grid + 16;
    int* sync = pl->cfl_sync;
    void* args[] = {&pl->dp, (void*)&p, (void*)&u, (void*)&v, (void*)&w, (void*)&pacc, (void*)&cfl, (void*)&sync, &lag};
    e = cudaLaunchKernel(v2 ? (const void*)k_correct_cfl<2, 2> : (const void*)k_correct_cfl<K6_U, 1>, dim3((unsigned)grid), dim3(K6_TX, K6_JL), args, 0, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("k_correct_cfl: ") + cudaGetErrorString(e));
    return AFID_OK;
}

// fork the auxiliary streams off `st` / join them back (both capturable in a CUDA graph)
static int pipe_fork(afid_plan* pl, cudaStream_t st, int ns)
{
    int rc;
    if ((rc = record(pl->ev_fork, st))) return rc;
    for (int k = 0; k < ns; ++k)
        if ((rc = wait_on(pl->aux[k], pl->ev_fork))) return rc;
    return AFID_OK;
}
static int pipe_join(afid_plan* pl, cudaStream_t st, int ns)
{
    int rc;
    for (int k = 0; k < ns; ++k)
        if ((rc = record(pl->ev_join[k], pl->aux[k])) || (rc = wait_on(st, pl->ev_join[k]))) return rc;
    return AFID_OK;
}

// K1 + K2: u,v,w -> C layout spectrum in `outC`
static int run_forward(afid_plan* pl, const double* u, const double* v, const double* w, cplx* wsB, cplx* outC, cudaStream_t st,
                       cudaEvent_t ev_mid)
{
    int rc;
    if (!pipelined(pl)) {
        if ((rc = launch_k1(pl, u, v, w, wsB, 0, pl->nx, pl->nx, st))) return rc;
        if (ev_mid && (rc = record(ev_mid, st))) return rc;
        return launch_k2(pl, wsB, outC, 0, pl->nx, pl->nx, st);
    }
    // plane-pipelined: K1 of batch b (stream 0) overlaps K2 of batch b-1 (stream 1); B is a rotating buffer of
    // `rot` batches (the first planes of the work array), so that it is produced and consumed inside L2
    const int nb = pl->pipe_batch, rot = pl->pipe_rot, bmod = nb * rot;
    if ((rc = pipe_fork(pl, st, 2))) return rc;
    int b = 0;
    for (int i_base = 0; i_base < pl->nx; i_base += nb, ++b) {
        const int np = (pl->nx - i_base < nb) ? pl->nx - i_base : nb;
        if (b >= rot && (rc = wait_on(pl->aux[0], pl->ev_b[(b - rot) % PIPE_EVENTS]))) return rc;   // slot consumed
        if ((rc = launch_k1(pl, u, v, w, wsB, i_base, np, bmod, pl->aux[0]))) return rc;
        if ((rc = record(pl->ev_a[b % PIPE_EVENTS], pl->aux[0])) || (rc = wait_on(pl->aux[1], pl->ev_a[b % PIPE_EVENTS]))) return rc;
        if ((rc = launch_k2(pl, wsB, outC, i_base, np, bmod, pl->aux[1]))) return rc;
        if ((rc = record(pl->ev_b[b % PIPE_EVENTS], pl->aux[1]))) return rc;
    }
    return pipe_join(pl, st, 2);
}

// K3: C (always ws[1]: the tensor map is bound to it) -> T
static int run_solve(afid_plan* pl, cplx* outT, cudaStream_t st)
{
    void* args[] = {&pl->dps, (void*)&pl->mapC, (void*)&outT};
    return launch(pl->k3, (unsigned)(pl->dps.nzh * (pl->ny / pl->k3_kw)), st, args, "k_solve_x");
}

// K4 + K5 + K6: T -> D -> p, u, v, w
static int run_inverse(afid_plan* pl, const cplx* T, cplx* D, double* u, double* v, double* w, double* p, cudaStream_t st,
                       cudaEvent_t ev_a, cudaEvent_t ev_b, double* cfl = nullptr)
{
    int rc;
    // accumulate mode: phi goes to the (now dead) T work array, K6 corrects from it and adds it to p
    double* phi = pl->accumulate ? reinterpret_cast<double*>(pl->ws[0]) : p;
    double* pacc = pl->accumulate ? p : nullptr;
    if (!pipelined(pl) || pl->accumulate) {   // (accumulate: phi overwrites T plane by plane, which the pipelined K4 still reads)
        if ((rc = launch_k4(pl, T, D, 0, pl->nx, pl->nx, st))) return rc;
        if (ev_a && (rc = record(ev_a, st))) return rc;
        if ((rc = launch_k5(pl, phi, 0, pl->nx, pl->nx, st))) return rc;
        if (ev_b && (rc = record(ev_b, st))) return rc;
        if (cfl) return launch_correct_cfl(pl, u, v, w, phi, st, pacc, cfl);
        return launch_correct(pl, u, v, w, phi, 0, pl->nx, st, pacc);
    }
    if (cfl) return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_project_cfl: not available with plane-pipelined sweeps");
    // plane-pipelined: K4 of batch b (stream 0), K5 of batch b-1 (stream 1) and K6 of batch b-2 (stream 2)
    // overlap; D is a rotating buffer of `rot` batches, p is read back by K6 right after K5 wrote it
    const int nb = pl->pipe_batch, rot = pl->pipe_rot, dmod = nb * rot;
    if ((rc = pipe_fork(pl, st, 3))) return rc;
    int b = 0;
    for (int i_base = 0; i_base < pl->nx; i_base += nb, ++b) {
        const int np = (pl->nx - i_base < nb) ? pl->nx - i_base : nb;
        if (b >= rot && (rc = wait_on(pl->aux[0], pl->ev_b[(b - rot) % PIPE_EVENTS]))) return rc;   // slot consumed
        if ((rc = launch_k4(pl, T, D, i_base, np, dmod, pl->aux[0]))) return rc;
        if ((rc = record(pl->ev_a[b % PIPE_EVENTS], pl->aux[0])) || (rc = wait_on(pl->aux[1], pl->ev_a[b % PIPE_EVENTS]))) return rc;
        if ((rc = launch_k5(pl, phi, i_base, np, dmod, pl->aux[1]))) return rc;
        // K6 of this batch also needs plane i_base-1 of phi: written by K5 of batch b-1, earlier on stream 1
        if ((rc = record(pl->ev_b[b % PIPE_EVENTS], pl->aux[1])) || (rc = wait_on(pl->aux[2], pl->ev_b[b % PIPE_EVENTS]))) return rc;
        if ((rc = launch_correct(pl, u, v, w, phi, i_base, np, pl->aux[2], pacc))) return rc;
    }
    return pipe_join(pl, st, 3);
}

extern "C" {

static int project_impl(afid_plan* pl, double* u, double* v, double* w, double* p, double* cfl, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(u, "u")) || (rc = check_ptr(v, "v")) || (rc = check_ptr(w, "w")) || (rc = check_ptr(p, "p"))) return rc;
    if ((rc = check_device(pl))) return rc;
    if (pl->nranks != 1) return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_project on a sharded plan: use the afid_shard_* stages");
    cudaStream_t st = (cudaStream_t)stream;
    const bool tm = pl->timing;
    cplx* wsB = pl->ws[0];
    cplx* wsC = pl->ws[1];
    if (tm && (rc = record(pl->ev[0], st))) return rc;
    if ((rc = run_forward(pl, u, v, w, wsB, wsC, st, tm ? pl->ev[1] : nullptr))) return rc;   // B in ws0, C in ws1
    if (tm && (rc = record(pl->ev[2], st))) return rc;
    if ((rc = run_solve(pl, pl->ws[0], st))) return rc;             // T in ws0
    if (tm && (rc = record(pl->ev[3], st))) return rc;
    if ((rc = run_inverse(pl, pl->ws[0], pl->ws[1], u, v, w, p, st, tm ? pl->ev[4] : nullptr, tm ? pl->ev[5] : nullptr, cfl))) return rc;
    if (tm) {
        if ((rc = record(pl->ev[6], st))) return rc;
        pl->ev_valid = true;
    }
    return AFID_OK;
}

AFID_EXPORT int afid_project(afid_plan* pl, double* u, double* v, double* w, double* p, void* stream)
{
    return project_impl(pl, u, v, w, p, nullptr, stream);
}

AFID_EXPORT int afid_project_cfl(afid_plan* pl, double* u, double* v, double* w, double* p, double* cfl, void* stream)
{
    if (!cfl) return fail(AFID_ERR_NULL, "cfl is NULL");
    if (((size_t)cfl & 7) != 0) return fail(AFID_ERR_ALIGN, "cfl is not 8-byte aligned");
    return project_impl(pl, u, v, w, p, cfl, stream);
}

// ---- the projection sharded over ranks (one process per GPU) -----------------------------------
// Two exchanges per projection instead of the paper's six all-to-alls: x-slabs for the
// divergence, both transforms and the correction, a kz partition for the x-solves.  C and T are kz-major, so the
// blocks that travel are contiguous on the sending side of exchange 1 and on the receiving side of exchange 2;
// the other two sides are one strided device copy per peer (the re-layouts below).
AFID_EXPORT afid_plan* afid_shard_plan_create(int nx, int ny, int nz, const double* xc, double Ly, double Lz, int rank, int nranks)
{
    return create_impl(nx, ny, nz, xc, Ly, Lz, rank, nranks);
}

AFID_EXPORT int afid_shard_bounds(int n, int nranks, int rank, int* lo, int* hi)
{
    if (nranks < 1 || rank < 0 || rank >= nranks || n < nranks || !lo || !hi) return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_shard_bounds: bad arguments");
    *lo = part_bound(n, nranks, rank);
    *hi = part_bound(n, nranks, rank + 1);
    return AFID_OK;
}

// Host arithmetic only (no device, no plan): what rank `rank` sends to / receives from every peer in exchange
// `phase` (1: forward spectrum C, slabs -> kz partition; 2: solved spectrum T, kz partition -> slabs), in complex
// elements (16 bytes), as offsets into the send / receive buffers of afid_shard_buffers.
AFID_EXPORT int afid_shard_layout(int nx, int ny, int nz, int nranks, int rank, int phase, long long* send_count, long long* send_off,
                                  long long* recv_count, long long* recv_off)
{
    if (nranks < 1 || nranks > MAX_RANKS || rank < 0 || rank >= nranks || nx < nranks || nz / 2 + 1 < nranks || (phase != 1 && phase != 2) ||
        !send_count || !send_off || !recv_count || !recv_off)
        return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_shard_layout: bad arguments");
    const int nzh = nz / 2 + 1;
    auto bx = [&](int r) { return (long long)part_bound(nx, nranks, r); };
    auto bk = [&](int r) { return (long long)part_bound(nzh, nranks, r); };
    const long long nxl = bx(rank + 1) - bx(rank), nkz = bk(rank + 1) - bk(rank);
    for (int r = 0; r < nranks; ++r) {
        const long long nxr = bx(r + 1) - bx(r), nkr = bk(r + 1) - bk(r);
        if (phase == 1) {   // send C_loc[kz of r][my planes][ky]; receive [my kz][planes of r][ky]
            send_count[r] = nkr * nxl * ny;  send_off[r] = bk(r) * nxl * ny;
            recv_count[r] = nkz * nxr * ny;  recv_off[r] = nkz * bx(r) * ny;
        } else {            // send [my kz][kyt][planes of r][8]; receive T_loc[kz of r][kyt][my planes][8]
            send_count[r] = nkz * nxr * ny;  send_off[r] = nkz * bx(r) * ny;
            recv_count[r] = nkr * nxl * ny;  recv_off[r] = bk(r) * nxl * ny;
        }
    }
    return AFID_OK;
}

// device pointers of the buffers exchange `phase` sends from / receives into (both are the plan's work arrays)
AFID_EXPORT int afid_shard_buffers(afid_plan* pl, int phase, void** send, void** recv)
{
    if (!pl || !send || !recv) return fail(AFID_ERR_NULL, "plan, send or recv is NULL");
    if (phase != 1 && phase != 2) return fail(AFID_ERR_UNSUPPORTED_SIZE, "phase must be 1 or 2");
    *send = pl->ws[1];
    *recv = pl->ws[0];
    return AFID_OK;
}

AFID_EXPORT int afid_shard_info(const afid_plan* pl, int* rank, int* nranks, int* xs, int* xe, int* ks, int* ke)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    if (rank) *rank = pl->rank;
    if (nranks) *nranks = pl->nranks;
    if (xs) *xs = pl->bx[pl->rank];
    if (xe) *xe = pl->bx[pl->rank + 1];
    if (ks) *ks = pl->bk[pl->rank];
    if (ke) *ke = pl->bk[pl->rank + 1];
    return AFID_OK;
}

// stage 1: divergence + forward transforms of this rank's slab; the send buffer of exchange 1 is ready afterwards
AFID_EXPORT int afid_shard_forward(afid_plan* pl, const double* u, const double* v, const double* w, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(u, "u")) || (rc = check_ptr(v, "v")) || (rc = check_ptr(w, "w"))) return rc;
    if ((rc = check_device(pl))) return rc;
    return run_forward(pl, u, v, w, pl->ws[0], pl->ws[1], (cudaStream_t)stream, nullptr);
}

static int copy2d(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width, size_t height, cudaStream_t st)
{
    cudaError_t e = cudaMemcpy2DAsync(dst, dpitch, src, spitch, width, height, cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("cudaMemcpy2DAsync: ") + cudaGetErrorString(e));
    return AFID_OK;
}

// stage 2 (after exchange 1): received blocks -> C[kz][i][ky] over all planes, x-solves, T -> per-peer send blocks
AFID_EXPORT int afid_shard_solve(afid_plan* pl, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_device(pl))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ny = pl->ny, gnx = pl->gnx, nkz = pl->dps.nzh, E = sizeof(cplx);
    {   // block of peer r: [nkz][planes of r][ny] -> rows bx[r].. of every kz  (one rank: a plain copy, the exchange still runs)
        for (int r = 0; r < pl->nranks; ++r) {
            const size_t x0 = pl->bx[r], nxr = pl->bx[r + 1] - pl->bx[r];
            if ((rc = copy2d(pl->ws[1] + x0 * ny, gnx * ny * E, pl->ws[0] + nkz * x0 * ny, nxr * ny * E, nxr * ny * E, nkz, st))) return rc;
        }
    }
    if ((rc = run_solve(pl, pl->ws[0], st))) return rc;
    {   // T[kz][kyt][i][8] -> block of peer r: [nkz][kyt][planes of r][8]
        const size_t rows = nkz * (ny / 8);
        for (int r = 0; r < pl->nranks; ++r) {
            const size_t x0 = pl->bx[r], nxr = pl->bx[r + 1] - pl->bx[r];
            if ((rc = copy2d(pl->ws[1] + nkz * x0 * ny, nxr * 8 * E, pl->ws[0] + x0 * 8, gnx * 8 * E, nxr * 8 * E, rows, st))) return rc;
        }
    }
    return AFID_OK;
}

// stage 3 (after exchange 2): inverse transforms of this rank's slab, phi -> p
AFID_EXPORT int afid_shard_inverse(afid_plan* pl, double* p, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(p, "p"))) return rc;
    if ((rc = check_device(pl))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = launch_k4(pl, pl->ws[0], pl->ws[1], 0, pl->nx, pl->nx, st))) return rc;
    return launch_k5(pl, p, 0, pl->nx, pl->nx, st);
}

// stage 4 (after the halo exchange of phi): correction of this rank's slab.  p_halo = the last plane of phi of the
// rank below (ny*nz doubles, device), NULL on rank 0 (plane 0 is the wall).
AFID_EXPORT int afid_shard_correct(afid_plan* pl, double* u, double* v, double* w, double* p, const double* p_halo, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(u, "u")) || (rc = check_ptr(v, "v")) || (rc = check_ptr(w, "w")) || (rc = check_ptr(p, "p"))) return rc;
    if (pl->rank > 0 && (rc = check_ptr(p_halo, "p_halo"))) return rc;
    if ((rc = check_device(pl))) return rc;
    return launch_correct(pl, u, v, w, p, 0, pl->nx, (cudaStream_t)stream, nullptr, pl->rank > 0 ? p_halo : nullptr);
}

AFID_EXPORT int afid_max_cfl(afid_plan* pl, const double* u, const double* v, const double* w, double* cfl, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(u, "u")) || (rc = check_ptr(v, "v")) || (rc = check_ptr(w, "w"))) return rc;
    if (!cfl) return fail(AFID_ERR_NULL, "cfl is NULL");
    if (((size_t)cfl & 7) != 0) return fail(AFID_ERR_ALIGN, "cfl is not 8-byte aligned");
    if ((rc = check_device(pl))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    k_cfl_init<<<1, 1, 0, st>>>(cfl);
    void* args[] = {&pl->dp, (void*)&u, (void*)&v, (void*)&w, (void*)&cfl};
    cudaError_t e = cudaLaunchKernel((const void*)k_max_cfl, dim3((unsigned)(pl->nx * (pl->ny / K6_JL))), dim3(K6_TX, K6_JL), args, 0, st);
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("k_max_cfl: ") + cudaGetErrorString(e));
    return AFID_OK;
}

// Host arithmetic only (no device, no plan): the schedule of afid_project_cfl's fused launch, for tests.
// Item `item` of the correction order = lines 4 jg .. 4 jg + 3 of plane i; its reduce step owns the lines
// [line_lo, line_hi] (plus `extra_line` >= 0 for the last group) and waits for the items deps[0..4] (-1 = none).
AFID_EXPORT int afid_cfl_schedule(int nx, int ny, int item, int* i, int* jg, int* line_lo, int* line_hi, int* extra_line, int* deps)
{
    if (nx < 1 || ny < K6_JL || (ny % K6_JL) != 0 || !i || !jg || !line_lo || !line_hi || !extra_line || !deps)
        return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_cfl_schedule: bad arguments");
    const int ngrp = ny / K6_JL;
    if (item < 0 || item >= nx * ngrp) return fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_cfl_schedule: item out of range");
    k6_item_to_ij(item, nx, ngrp, *i, *jg);
    *line_lo = (*jg == 0) ? 0 : *jg * K6_JL - 1;
    *line_hi = *jg * K6_JL + K6_JL - 2;
    *extra_line = (*jg == ngrp - 1) ? ny - 1 : -1;
    for (int d = 0; d < 5; ++d) {   // the rule of k_correct_cfl's threads 0..4
        const int di = (d & 1) ? *i + 1 : *i;
        const int dg = (d == 4) ? 0 : ((d & 2) ? *jg - 1 : *jg);
        const bool need = (di < nx) && (dg >= 0) && (d < 4 || (*jg == ngrp - 1 && di == *i));
        deps[d] = need ? k6_ij_to_item(di, dg, nx, ngrp) : -1;
    }
    return AFID_OK;
}

AFID_EXPORT int afid_plan_set_accumulate(afid_plan* pl, int on)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    pl->accumulate = on != 0;
    return AFID_OK;
}

// ---- batched real tridiagonal solves in x on a field (implicit wall-normal step) ----------
struct afid_xsolve {
    afid_plan* pl;
    DevParams dp;
    LaunchCfg k;
    XsTables xt;       // device tables of the row-only quantities (k_xsolve_field)
    void* tables;      // one device allocation holding them
    double* map_for;   // the field pointer `map` was encoded for (re-encoded only when it changes)
    alignas(64) CUtensorMap map;
};

AFID_EXPORT afid_xsolve* afid_xsolve_create(afid_plan* pl, const double* a_in, const double* c_in, const double* lam)
{
    g_err.clear();
    g_err_code = 0;
    if (!pl || !a_in || !c_in || !lam) { fail(AFID_ERR_NULL, "plan, a, c or lam is NULL"); return nullptr; }
    if (pl->nranks != 1) { fail(AFID_ERR_UNSUPPORTED_SIZE, "afid_xsolve_create needs an unsharded plan (the columns span all x)"); return nullptr; }
    const int nx = pl->nx;
    for (int i = 0; i < nx; ++i)
        if (!(a_in[i] >= 0.0) || !(c_in[i] >= 0.0) || !(lam[i] > 0.0) || !std::isfinite(a_in[i]) || !std::isfinite(c_in[i]) || !std::isfinite(lam[i])) {
            fail(AFID_ERR_GRID, "afid_xsolve_create needs finite a_i >= 0, c_i >= 0, lam_i > 0 (an M-matrix)");
            return nullptr;
        }
    afid_xsolve* h = new (std::nothrow) afid_xsolve();
    if (!h) { fail(AFID_ERR_NOMEM, "host allocation failed"); return nullptr; }
    h->pl = pl;
    h->dp = pl->dp;
    const int M = (nx < 64) ? 4 : (nx <= 1024 ? 16 : 32);
    const int KW = (nx <= 1024) ? 8 : 4;   // 128-byte rows wherever the tile fits shared memory
    const int PCH = (nx + M - 1) / M;
    if (KW == 4) h->k.fn = (M == 4) ? (const void*)k_xsolve_field<4, 4> : (M == 16 ? (const void*)k_xsolve_field<16, 4> : (const void*)k_xsolve_field<32, 4>);
    else h->k.fn = (M == 4) ? (const void*)k_xsolve_field<4, 8> : (const void*)k_xsolve_field<16, 8>;
    h->k.threads = PCH * KW;
    h->k.smem = (size_t)k3_tile_rows(nx) * KW * sizeof(cplx) + (size_t)2 * PCH * KW * sizeof(cplx) + 128;
    h->k.ctas_per_sm = 3;
    h->k.nl = KW;   // (complex lanes per tile)
    {
        cudaDeviceProp prop;
        if (cudaGetDeviceProperties(&prop, pl->device) != cudaSuccess) { delete h; fail(AFID_ERR_CUDA, "cudaGetDeviceProperties failed"); return nullptr; }
        if (h->k.smem > prop.sharedMemPerBlockOptin) { delete h; fail(AFID_ERR_UNSUPPORTED_SIZE, "tile does not fit shared memory"); return nullptr; }
        if (set_smem_attr(h->k, prop.sharedMemPerBlockOptin) != AFID_OK) { delete h; return nullptr; }
    }

    // ---- the row-only quantities of the partitioned solve, in long double (same algebra as k_solve_x)
    typedef long double ld;
    std::vector<ld> a(nx), c(nx);
    for (int i = 0; i < nx; ++i) { a[i] = (i == 0) ? 0.0L : (ld)a_in[i]; c[i] = (i == nx - 1) ? 0.0L : (ld)c_in[i]; }
    std::vector<double> UP(2 * (size_t)nx, 0.0), DN(2 * (size_t)nx, 0.0), GH(2 * (size_t)nx, 0.0), CH(2 * (size_t)PCH, 0.0), RE(PCH, 0.0);
    std::vector<ld> A(PCH, 0.0L), C(PCH, 0.0L), L(PCH, 0.0L), hup(PCH, 1.0L), tup(PCH, 0.0L);
    for (int q = 0; q < PCH; ++q) {
        const int i0 = q * M, i1 = std::min(i0 + M, nx) - 1;
        ld hh = 1.0L, tt = 0.0L;
        for (int i = i1 - 1; i >= i0; --i) {                    // upward
            const ld nh = c[i] * hh, nt = (ld)lam[i] + c[i] * tt, rr = 1.0L / (a[i] + (nh + nt));
            hh = nh * rr; tt = nt * rr;
            UP[2 * i] = (double)(c[i] * rr); UP[2 * i + 1] = (double)rr;
        }
        hup[q] = hh; tup[q] = tt;
        hh = 1.0L; tt = 0.0L;
        for (int i = i0; i < i1; ++i) {                         // downward
            const ld nh = a[i] * hh, nt = (ld)lam[i] + a[i] * tt, rr = 1.0L / (c[i] + (nh + nt));
            hh = nh * rr; tt = nt * rr;
            DN[2 * i] = (double)(a[i] * rr); DN[2 * i + 1] = (double)rr;
            GH[2 * i] = (double)(c[i] * rr); GH[2 * i + 1] = (double)hh;
        }
        const ld ab = a[i1], cb = (q > 0) ? c[i0 - 1] : 0.0L;
        CH[2 * q] = (double)ab; CH[2 * q + 1] = (double)cb;
        A[q] = ab * hh;
        L[q] = (ld)lam[i1] + ab * tt;
    }
    for (int q = 0; q + 1 < PCH; ++q) {                          // the next chunk's upward relation enters row q
        const ld cb = c[(q + 1) * M - 1];
        C[q] = cb * hup[q + 1];
        L[q] += cb * tup[q + 1];
    }
    int nlev = 0;
    for (int d = 1; d < PCH; d <<= 1) ++nlev;
    std::vector<double> PC(2 * (size_t)std::max(nlev, 1) * PCH, 0.0);
    {
        int lev = 0;
        for (int d = 1; d < PCH; d <<= 1, ++lev) {
            std::vector<ld> A2(PCH, 0.0L), C2(PCH, 0.0L), L2(L);
            for (int q = 0; q < PCH; ++q) {
                ld al = 0.0L, ga = 0.0L;
                if (q - d >= 0) { const int m = q - d; al = A[q] / (A[m] + C[m] + L[m]); A2[q] = al * A[m]; L2[q] += al * L[m]; }
                if (q + d < PCH) { const int m = q + d; ga = C[q] / (A[m] + C[m] + L[m]); C2[q] = ga * C[m]; L2[q] += ga * L[m]; }
                PC[2 * ((size_t)lev * PCH + q)] = (double)al;
                PC[2 * ((size_t)lev * PCH + q) + 1] = (double)ga;
            }
            A = A2; C = C2; L = L2;
        }
    }
    for (int q = 0; q < PCH; ++q) RE[q] = (double)(1.0L / (A[q] + C[q] + L[q]));

    struct Item { const void* src; size_t bytes; size_t off; };
    std::vector<Item> items = {{UP.data(), UP.size() * 8, 0}, {DN.data(), DN.size() * 8, 0}, {GH.data(), GH.size() * 8, 0},
                               {CH.data(), CH.size() * 8, 0}, {RE.data(), RE.size() * 8, 0}, {PC.data(), PC.size() * 8, 0}};
    size_t off = 0;
    for (auto& it : items) { it.off = off; off += (it.bytes + 255) / 256 * 256; }
    if (cudaMalloc(&h->tables, off) != cudaSuccess) { cudaGetLastError(); delete h; fail(AFID_ERR_NOMEM, "cudaMalloc(xsolve tables) failed"); return nullptr; }
    for (auto& it : items)
        if (cudaMemcpy((char*)h->tables + it.off, it.src, it.bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaFree(h->tables); delete h; fail(AFID_ERR_CUDA, "cudaMemcpy(xsolve tables) failed"); return nullptr;
        }
    char* tb = (char*)h->tables;
    h->xt.UP = (const double2*)(tb + items[0].off);
    h->xt.DN = (const double2*)(tb + items[1].off);
    h->xt.GH = (const double2*)(tb + items[2].off);
    h->xt.CH = (const double2*)(tb + items[3].off);
    h->xt.RE = (const double*)(tb + items[4].off);
    h->xt.PC = (const double2*)(tb + items[5].off);
    h->xt.nlev = nlev;
    return h;
}

AFID_EXPORT int afid_xsolve_apply(afid_xsolve* h, double* f, void* stream)
{
    if (!h) return fail(AFID_ERR_NULL, "xsolve handle is NULL");
    int rc;
    if ((rc = check_ptr(f, "f"))) return rc;
    const afid_plan* pl = h->pl;
    if ((rc = check_device(pl))) return rc;
    if (h->map_for != f) {
        if (!make_map3(&h->map, f, (uint64_t)pl->nz, (uint64_t)pl->ny, (uint64_t)pl->nx, 2 * (uint32_t)h->k.nl, 1, (uint32_t)k3_box_rows(pl->nx),
                       CU_TENSOR_MAP_SWIZZLE_NONE))
            return fail(AFID_ERR_CUDA, "cuTensorMapEncodeTiled failed");
        h->map_for = f;
    }
    cplx* fc = reinterpret_cast<cplx*>(f);
    void* args[] = {&h->dp, &h->xt, (void*)&h->map, (void*)&fc};
    return launch(h->k, (unsigned)(pl->ny * ((pl->nz / 2) / h->k.nl)), (cudaStream_t)stream, args, "k_xsolve_field");
}

AFID_EXPORT int afid_xsolve_destroy(afid_xsolve* h)
{
    if (!h) return AFID_OK;
    cudaFree(h->tables);
    delete h;
    return AFID_OK;
}

AFID_EXPORT int afid_plan_enable_timing(afid_plan* pl, int on)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    if (on && !pl->timing) {
        for (int k = 0; k < 7; ++k)
            if (cudaEventCreate(&pl->ev[k]) != cudaSuccess) return fail(AFID_ERR_CUDA, "cudaEventCreate failed");
        pl->timing = true;
        pl->ev_valid = false;
    } else if (!on && pl->timing) {
        for (int k = 0; k < 7; ++k) cudaEventDestroy(pl->ev[k]);
        pl->timing = false;
        pl->ev_valid = false;
    }
    return AFID_OK;
}

AFID_EXPORT int afid_plan_kernel_times(afid_plan* pl, float* ms, int n)
{
    if (!pl || !ms) return fail(AFID_ERR_NULL, "plan or ms is NULL");
    if (!pl->timing || !pl->ev_valid) return fail(AFID_ERR_CUDA, "timing not enabled or no projection recorded");
    if (cudaEventSynchronize(pl->ev[6]) != cudaSuccess) return fail(AFID_ERR_CUDA, "cudaEventSynchronize failed");
    if (pipelined(pl)) {   // the kernels of a sweep overlap: forward sweep, x-solve, inverse sweep
        const int a[3] = {0, 2, 3}, b[3] = {2, 3, 6};
        for (int k = 0; k < 3 && k < n; ++k)
            if (cudaEventElapsedTime(&ms[k], pl->ev[a[k]], pl->ev[b[k]]) != cudaSuccess) return fail(AFID_ERR_CUDA, "cudaEventElapsedTime failed");
        return AFID_OK;
    }
    for (int k = 0; k < 6 && k < n; ++k)
        if (cudaEventElapsedTime(&ms[k], pl->ev[k], pl->ev[k + 1]) != cudaSuccess) return fail(AFID_ERR_CUDA, "cudaEventElapsedTime failed");
    return AFID_OK;
}

AFID_EXPORT int afid_plan_num_timed(const afid_plan* pl) { return pl ? (pipelined(pl) ? 3 : 6) : 0; }

AFID_EXPORT const char* afid_plan_kernel_name(const afid_plan* pl, int k)
{
    if (pl && pipelined(pl)) return (k >= 0 && k < 3) ? SWEEP_NAMES[k] : "";
    return (k >= 0 && k < 6) ? KERNEL_NAMES[k] : "";
}

} // extern "C"

// The taps speak [i][kz][ky]; the work array C is [kz][i][ky]: small re-layout kernels (not on the hot path).
__global__ void k_tap_C_to_api(DevParams P, const cplx* __restrict__ C, cplx* __restrict__ A, int to_api)
{
    const size_t n = (size_t)P.nx * P.nzh * P.ny;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const int ky = (int)(t % P.ny);
        const size_t r = t / P.ny;
        const int kz = (int)(r % P.nzh), i = (int)(r / P.nzh);       // t indexes the API layout
        const size_t c = ((size_t)kz * P.nx + i) * P.ny + ky;
        if (to_api) A[t] = C[c];
        else const_cast<cplx*>(C)[c] = A[t];
    }
}
__global__ void k_tap_T_to_api(DevParams P, const cplx* __restrict__ T, cplx* __restrict__ A)
{
    const size_t n = (size_t)P.nx * P.nzh * P.ny;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const int ky = (int)(t % P.ny);
        const size_t r = t / P.ny;
        const int kz = (int)(r % P.nzh), i = (int)(r / P.nzh);
        A[t] = T[(((size_t)kz * (P.ny / 8) + ky / 8) * P.nx + i) * 8 + (ky & 7)];
    }
}

extern "C" {

AFID_EXPORT int afid_stage_forward(afid_plan* pl, const double* u, const double* v, const double* w, double* spec, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(u, "u")) || (rc = check_ptr(v, "v")) || (rc = check_ptr(w, "w")) || (rc = check_ptr(spec, "spec"))) return rc;
    if (pl->nranks != 1) return fail(AFID_ERR_UNSUPPORTED_SIZE, "stage taps need an unsharded plan");
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = run_forward(pl, u, v, w, pl->ws[0], pl->ws[1], st, nullptr))) return rc;
    k_tap_C_to_api<<<pl->n_sm * 8, 256, 0, st>>>(pl->dp, pl->ws[1], (cplx*)spec, 1);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("k_tap_C_to_api: ") + cudaGetErrorString(e));
    return AFID_OK;
}

AFID_EXPORT int afid_stage_solve(afid_plan* pl, double* spec, void* stream)
{
    if (!pl) return fail(AFID_ERR_NULL, "plan is NULL");
    int rc;
    if ((rc = check_ptr(spec, "spec"))) return rc;
    if (pl->nranks != 1) return fail(AFID_ERR_UNSUPPORTED_SIZE, "stage taps need an unsharded plan");
    cudaStream_t st = (cudaStream_t)stream;
    k_tap_C_to_api<<<pl->n_sm * 8, 256, 0, st>>>(pl->dp, pl->ws[1], (cplx*)spec, 0);
    if ((rc = run_solve(pl, pl->ws[0], st))) return rc;
    k_tap_T_to_api<<<pl->n_sm * 8, 256, 0, st>>>(pl->dp, pl->ws[0], (cplx*)spec);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(AFID_ERR_CUDA, std::string("k_tap: ") + cudaGetErrorString(e));
    return AFID_OK;
}

} // extern "C"
