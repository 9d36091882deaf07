// C-ABI implementation of include/purify_op.h (sm_100a).  Host logic only: validation, create-time
// binning, launches.  Every arithmetic step of the path runs in the kernels of kernels.cuh,
// degrid.cuh, grid.cuh; the FFT stage is cuFFT (allowed by the north star, timed separately).
// There is no CPU fallback: without a CUDA device every entry point returns PURIFY_ERR_NO_DEVICE.
#include "../../include/purify_op.h"

#include <cub/cub.cuh>
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <vector>

#include "batched.cuh"
#include "degrid.cuh"
#include "grid.cuh"
#include "kb_host.hpp"
#include "kernels.cuh"
#include "ubench.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int status, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return status;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? PURIFY_ERR_ALLOC : PURIFY_ERR_CUDA,     \
                        "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)
#define CKFFT(call)                                                                                \
    do {                                                                                           \
        cufftResult r_ = (call);                                                                   \
        if (r_ != CUFFT_SUCCESS)                                                                   \
            return fail(PURIFY_ERR_CUFFT, "%s failed: cufftResult %d (%s:%d)", #call, (int)r_, __FILE__, __LINE__); \
    } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int grid_for(long long work, int threads, int cap = 148 * 16) {
    long long b = (work + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > cap) b = cap;
    return (int)b;
}

// degree of the per-tap polynomial per (dtype, J): kb_host.hpp fit errors
// (degree 6 at J = 6 was tried: 1.6 % faster, rel-L2 2.5e-5 - outside the 1e-5 tolerance)
constexpr int deg_c64(int J) { return J == 4 ? 8 : 7; }
constexpr int deg_c128(int J) { return J == 4 ? 17 : (J == 6 ? 16 : 15); }

}  // namespace

namespace pkerr {
int set(int status, const char* fmt, ...) {          // the detail string is shared with wavelet.cu (same library)
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return status;
}
}  // namespace pkerr

struct purify_op {
    int n = 0, K = 0, J = 0, dtype = 0, mode = 0, table_R = 0, chunk = 4096, time_stages = 0;
    long long M = 0;
    int ntx = 0, n_tiles = 0, n_items = 0, n_tiles_nonempty = 0;
    long long max_tile_count = 0;
    int poly_degree = 0;
    double poly_err = 0;
    long long device_bytes = 0;
    // device memory (owned)
    void* grid = nullptr;     // K*K complex, internal layout
    void* uv_s = nullptr;     // native-order (u, v)
    void* w_s = nullptr;      // native-order weights
    unsigned* perm = nullptr; // native -> caller
    unsigned* inv_perm = nullptr; // caller -> native (batched layout)
    // routed permutation (kernels.cuh), index arrays built at create when M >= ROUTED_MIN
    unsigned short* loc_a = nullptr;   // pass A: rank of every native slot inside its block (NONE16: padding)
    unsigned* dst_a = nullptr;         //         A-order position of every sorted rank
    unsigned short* loc_b = nullptr;   // pass B: rank of every A-order element inside its block
    unsigned* dst_b = nullptr;         //         mid position of every sorted rank
    unsigned short* loc_idx = nullptr; // pass C: position of every mid element inside its caller tile
    void* perm_ws = nullptr;           // intermediate vectors (M complex from native, 2 M complex to native), lazily allocated
    size_t perm_ws_bytes = 0;
    pk::Item* items = nullptr;
    void* corr = nullptr;     // s[n]
    void* table = nullptr;
    int table_len = 0;
    void* y_ws = nullptr;     // M_native complex (purify_normal / host paths), lazily allocated
    void* x_ws = nullptr;     // n*n complex staging for host paths
    void* y_ws2 = nullptr;    // caller-order staging for host paths / z of the unfused ADMM step
    size_t y_ws_bytes = 0, x_ws_bytes = 0, y_ws2_bytes = 0, scal_ws_bytes = 0;
    double* scal_ws = nullptr; // one fp64 scalar (norms)
    bool admm_unfused = false; // opts.admm_unfused: purify_admm_fidelity_step uses separate norm / update kernels
    cufftHandle plan = 0;
    bool plan_ok = false;
    CUtensorMap tmap;
    pk::KbCoef<float> coef32;
    pk::KbCoef<double> coef64;
    cudaEvent_t ev[2 * PURIFY_STAGE_COUNT];
    bool ev_ok = false;
    bool stage_ran[PURIFY_STAGE_COUNT];
    int launches = 0;
    // complex64 batched ("cell-stationary") layout, batched.cuh
    bool batched = false;
    long long M_native = 0;       // slots (batched) or M (sorted layout)
    int n_bands = 0, n_bands_nonempty = 0;
    unsigned n_batches = 0;
    uint2* x_bhdr = nullptr;
    unsigned* x_blane = nullptr;
    pk::XItem* x_items = nullptr;
    unsigned* x_counter = nullptr;
    CUtensorMap tmap_x;
    std::map<const void*, int> x_ctas;   // persistent grid size per kernel instantiation (occupancy query done once)
    // purify_normal replayed from a CUDA graph (captured on an internal stream, launched on the caller's)
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t normal_exec = nullptr;
    const void* normal_in = nullptr;
    void* normal_out = nullptr;
    int normal_launches = 0;
    bool graph_stale = false, graph_failed = false, normal_warm = false;
    // f3: side stream on which the caller's all-reduce of the image bands is enqueued, and the events that chain it
    cudaStream_t comm_stream = nullptr;
    std::vector<cudaEvent_t> band_ev;
    cudaEvent_t comm_done = nullptr;
};

namespace {

size_t csize(const purify_op* op) { return op->dtype == PURIFY_C64 ? 8 : 16; }
size_t rsize(const purify_op* op) { return op->dtype == PURIFY_C64 ? 4 : 8; }

int dev_alloc(purify_op* op, void** p, size_t bytes) {
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        *p = nullptr;
        cudaGetLastError();
        return fail(PURIFY_ERR_ALLOC, "cudaMalloc(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
    }
    op->device_bytes += (long long)bytes;
    return PURIFY_OK;
}

struct StageTimer {
    purify_op* op; int stage; cudaStream_t st;
    StageTimer(purify_op* o, int s, cudaStream_t t) : op(o), stage(s), st(t) {
        if (op->time_stages && op->ev_ok) { cudaEventRecord(op->ev[2 * stage], st); op->stage_ran[stage] = true; }
    }
    ~StageTimer() { if (op->time_stages && op->ev_ok) cudaEventRecord(op->ev[2 * stage + 1], st); }
};

template <typename R> pk::OpParams<R> make_params(const purify_op* op, bool caller_order) {
    pk::OpParams<R> p;
    p.grid = (typename pk::Cplx<R>::type*)op->grid;
    p.K = op->K; p.Kh = op->K / 2;
    p.kmask = (op->K & (op->K - 1)) == 0 ? op->K - 1 : 0;
    p.items = op->items;
    p.uv = (const typename pk::Cplx<R>::type*)op->uv_s;
    p.w = (const R*)op->w_s;
    p.perm = caller_order ? op->perm : nullptr;
    if (sizeof(R) == 4) memcpy(&p.coef, &op->coef32, sizeof(p.coef)); else memcpy(&p.coef, &op->coef64, sizeof(p.coef));
    p.table = (const R*)op->table;
    p.table_R = (R)op->table_R;
    p.table_len = op->table_len;
    return p;
}

// ------------------------------------------------------------------------------- launches
template <typename R, int J, int DEG> int launch_degrid_t(purify_op* op, void* y, bool caller_order, cudaStream_t st) {
    typedef typename pk::Cplx<R>::type C;
    if (op->n_items == 0) return PURIFY_OK;
    constexpr int BOX = pk::DegridCfg<J>::BOX;
    const size_t smem = sizeof(C) * BOX * BOX + 16;
    pk::OpParams<R> p = make_params<R>(op, caller_order);
    if (op->mode == PURIFY_KERNEL_ANALYTIC) {
        auto kern = pk::degrid_kernel<R, J, DEG, 0>;
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<op->n_items, pk::DegridCfg<J>::THREADS, smem, st>>>(op->tmap, p, (C*)y);
    } else {
        auto kern = pk::degrid_kernel<R, J, DEG, 1>;
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<op->n_items, pk::DegridCfg<J>::THREADS, smem, st>>>(op->tmap, p, (C*)y);
    }
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

template <typename R, int J, int DEG> int launch_grid_t(purify_op* op, const void* y, bool caller_order, cudaStream_t st) {
    typedef typename pk::Cplx<R>::type C;
    if (op->n_items == 0) return PURIFY_OK;
    const size_t smem = pk::grid_smem_bytes<R, J>();
    pk::OpParams<R> p = make_params<R>(op, caller_order);
    if (op->mode == PURIFY_KERNEL_ANALYTIC) {
        auto kern = pk::grid_kernel<R, J, DEG, 0>;
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<op->n_items, pk::GridCfg<J>::THREADS, smem, st>>>(p, (const C*)y);
    } else {
        auto kern = pk::grid_kernel<R, J, DEG, 1>;
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<op->n_items, pk::GridCfg<J>::THREADS, smem, st>>>(p, (const C*)y);
    }
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

template <typename F> pk::XParamsT<F> make_xparams(const purify_op* op) {
    typedef typename pk::Cplx<F>::type F2;
    pk::XParamsT<F> p;
    p.grid = (F2*)op->grid;
    p.K = op->K; p.Kh = op->K / 2;
    p.kmask = (op->K & (op->K - 1)) == 0 ? op->K - 1 : 0;
    p.items = op->x_items;
    p.n_items = op->n_items;
    p.counter = op->x_counter;
    p.bhdr = op->x_bhdr;
    p.blane = op->x_blane;
    p.rec = (const F*)op->uv_s;
    if (sizeof(F) == 4) memcpy(&p.coef, &op->coef32, sizeof(p.coef)); else memcpy(&p.coef, &op->coef64, sizeof(p.coef));
    p.table = (const F*)op->table;
    p.table_R = (F)op->table_R;
    p.table_len = op->table_len;
    p.s_in = nullptr; p.yobs = nullptr; p.s_out = nullptr; p.norm2 = op->scal_ws; p.eps = 0.0; p.varrho = 0.0;
    return p;
}

// persistent grid: as many CTAs as fit on the device at once (capped by the number of items).  The occupancy query
// and the shared-memory attribute are done once per handle and kernel instantiation, not per launch.
template <typename Kern> int x_grid_size(purify_op* op, Kern kern, int threads, size_t smem, int warps, int* out) {
    const void* key = (const void*)kern;
    auto hit = op->x_ctas.find(key);
    if (hit != op->x_ctas.end()) { *out = hit->second; return PURIFY_OK; }
    int dev = 0, sms = 0, per_sm = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
    if (per_sm < 1) per_sm = 1;
    int g = sms * per_sm;
    const int need = (op->n_items + warps - 1) / warps;
    if (g > need) g = need;
    if (g < 1) g = 1;
    op->x_ctas[key] = g;
    *out = g;
    return PURIFY_OK;
}

// ring geometry (iterations per chunk, stages) of the two complex64 kernels (batched.cuh "ring")
constexpr int X_CH_DEGRID = 16, X_S_DEGRID = 2, X_CH_GRID = 6, X_S_GRID = 2;
// TABLE mode.  A table of up to 64 KB (R J/2 + 2 floats; 32 KB at R = 4096, J = 4) is copied into shared memory by
// every CTA (MODE 2, 8 warps per CTA): 32 lanes looking up unrelated entries cost ~3.5 shared-memory wavefronts per
// lookup, against many more L1 tag look-ups when the table sits in global memory.  Larger tables (the paper's
// R = 2e5) stay in global memory (MODE 1) with small rings, so that L1 keeps as much of the table as it can
// (measured at config 5 before MODE 2 existed: grid 26.8 ms with a (4, 2) ring - table evicted from L1 - and
// 4.4 ms with (3, 2)).
constexpr int X_CH_DEGRID_T = 4, X_S_DEGRID_T = 2, X_CH_GRID_T = 3, X_S_GRID_T = 2;
constexpr size_t X_TABLE_SMEM_MAX = 64 * 1024;

struct AdmmArgs { const void* y_obs; void* s; double eps, varrho; };

template <typename F, int J, int DEG, int MODE, int CH, int S, int FUSE = 0>
int launch_degrid_x_m(purify_op* op, void* y, size_t extra_smem, cudaStream_t st, const AdmmArgs* aa = nullptr) {
    typedef typename pk::Cplx<F>::type F2;
    constexpr int NW = pk::x_warps(MODE);
    const size_t smem = pk::XSmem<F, J, CH, S, FUSE ? 2 : 0, NW>::TOTAL + extra_smem;
    pk::XParamsT<F> p = make_xparams<F>(op);
    if (aa) { p.s_in = (const F2*)aa->s; p.yobs = (const F2*)aa->y_obs; p.s_out = (F2*)aa->s; p.eps = aa->eps; p.varrho = aa->varrho; }
    int g = 0, rc;
    auto kern = pk::degrid_x_kernel<F, J, DEG, MODE, CH, S, FUSE>;
    if ((rc = x_grid_size(op, kern, NW * 32, smem, NW, &g))) return rc;
    p.n_warps = g * NW;
    kern<<<g, NW * 32, smem, st>>>(op->tmap_x, p, (F2*)y);
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

template <typename F, int J, int DEG, int MODE, int CH, int S, int FUSE = 0>
int launch_grid_x_m(purify_op* op, const void* y, size_t extra_smem, cudaStream_t st, const AdmmArgs* aa = nullptr) {
    typedef typename pk::Cplx<F>::type F2;
    constexpr int NW = pk::x_warps(MODE);
    const size_t smem = pk::XSmem<F, J, CH, S, FUSE ? 3 : 1, NW>::TOTAL + extra_smem;
    pk::XParamsT<F> p = make_xparams<F>(op);
    if (aa) { p.s_in = (const F2*)aa->s; p.yobs = (const F2*)aa->y_obs; p.s_out = (F2*)aa->s; p.eps = aa->eps; p.varrho = aa->varrho; }
    int g = 0, rc;
    auto kern = pk::grid_x_kernel<F, J, DEG, MODE, CH, S, FUSE>;
    if ((rc = x_grid_size(op, kern, NW * 32, smem, NW, &g))) return rc;
    p.n_warps = g * NW;
    kern<<<g, NW * 32, smem, st>>>(op->tmap_x, p, (const F2*)y);
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

template <int J, int DEG> int launch_degrid_x_t(purify_op* op, void* y, cudaStream_t st) {
    if (op->n_items == 0) return PURIFY_OK;
    const size_t tb = sizeof(float) * (size_t)op->table_len;
    if (op->mode != PURIFY_KERNEL_TABLE) return launch_degrid_x_m<float, J, DEG, 0, X_CH_DEGRID, X_S_DEGRID>(op, y, 0, st);
    if (tb <= X_TABLE_SMEM_MAX) return launch_degrid_x_m<float, J, DEG, 2, X_CH_DEGRID_T, X_S_DEGRID_T>(op, y, tb, st);
    return launch_degrid_x_m<float, J, DEG, 1, X_CH_DEGRID_T, X_S_DEGRID_T>(op, y, 0, st);
}

template <int J, int DEG> int launch_grid_x_t(purify_op* op, const void* y, cudaStream_t st) {
    if (op->n_items == 0) return PURIFY_OK;
    const size_t tb = sizeof(float) * (size_t)op->table_len;
    if (op->mode != PURIFY_KERNEL_TABLE) return launch_grid_x_m<float, J, DEG, 0, X_CH_GRID, X_S_GRID>(op, y, 0, st);
    if (tb <= X_TABLE_SMEM_MAX) return launch_grid_x_m<float, J, DEG, 2, X_CH_GRID_T, X_S_GRID_T>(op, y, tb, st);
    return launch_grid_x_m<float, J, DEG, 1, X_CH_GRID_T, X_S_GRID_T>(op, y, 0, st);
}

// complex128 in the batched layout (J = 4, 6; J = 8 does not fit the register file and keeps the tile-sorted kernels):
// same kernels instantiated for double - component-wise fp64 arithmetic, one visibility per trip, table in global memory
constexpr int X_CH_DEGRID_D = 8, X_S_DEGRID_D = 2, X_CH_GRID_D = 4, X_S_GRID_D = 2;

template <int J, int DEG> int launch_degrid_x_d(purify_op* op, void* y, cudaStream_t st) {
    if (op->n_items == 0) return PURIFY_OK;
    if (op->mode != PURIFY_KERNEL_TABLE) return launch_degrid_x_m<double, J, DEG, 0, X_CH_DEGRID_D, X_S_DEGRID_D>(op, y, 0, st);
    return launch_degrid_x_m<double, J, DEG, 1, X_CH_DEGRID_D, X_S_DEGRID_D>(op, y, 0, st);
}

template <int J, int DEG> int launch_grid_x_d(purify_op* op, const void* y, cudaStream_t st) {
    if (op->n_items == 0) return PURIFY_OK;
    if (op->mode != PURIFY_KERNEL_TABLE) return launch_grid_x_m<double, J, DEG, 0, X_CH_GRID_D, X_S_GRID_D>(op, y, 0, st);
    return launch_grid_x_m<double, J, DEG, 1, X_CH_GRID_D, X_S_GRID_D>(op, y, 0, st);
}

// f1, fused (complex64 batched layout, ANALYTIC weights): ring geometries that keep the occupancy of the plain kernels
constexpr int X_CH_DEGRID_F = 6, X_S_DEGRID_F = 2, X_CH_GRID_F = 3, X_S_GRID_F = 2;

int launch_degrid_fused(purify_op* op, void* v, const AdmmArgs& aa, cudaStream_t st) {
    StageTimer t(op, PURIFY_STAGE_DEGRID, st);
    if (op->n_items == 0) return PURIFY_OK;
    switch (op->J) {
        case 4: return launch_degrid_x_m<float, 4, deg_c64(4), 0, X_CH_DEGRID_F, X_S_DEGRID_F, 1>(op, v, 0, st, &aa);
        case 6: return launch_degrid_x_m<float, 6, deg_c64(6), 0, X_CH_DEGRID_F, X_S_DEGRID_F, 1>(op, v, 0, st, &aa);
        default: return launch_degrid_x_m<float, 8, deg_c64(8), 0, X_CH_DEGRID_F, X_S_DEGRID_F, 1>(op, v, 0, st, &aa);
    }
}

int launch_grid_fused(purify_op* op, const void* v, const AdmmArgs& aa, cudaStream_t st) {
    {
        StageTimer tz(op, PURIFY_STAGE_ZERO, st);
        CK(cudaMemsetAsync(op->grid, 0, csize(op) * (size_t)op->K * op->K, st));
    }
    StageTimer t(op, PURIFY_STAGE_GRID, st);
    if (op->n_items == 0) return PURIFY_OK;
    switch (op->J) {
        case 4: return launch_grid_x_m<float, 4, deg_c64(4), 0, X_CH_GRID_F, X_S_GRID_F, 1>(op, v, 0, st, &aa);
        case 6: return launch_grid_x_m<float, 6, deg_c64(6), 0, X_CH_GRID_F, X_S_GRID_F, 1>(op, v, 0, st, &aa);
        default: return launch_grid_x_m<float, 8, deg_c64(8), 0, X_CH_GRID_F, X_S_GRID_F, 1>(op, v, 0, st, &aa);
    }
}

int launch_degrid(purify_op* op, void* y, bool caller_order, cudaStream_t st) {
    StageTimer t(op, PURIFY_STAGE_DEGRID, st);
    if (op->batched && op->dtype == PURIFY_C128)
        return op->J == 4 ? launch_degrid_x_d<4, deg_c128(4)>(op, y, st) : launch_degrid_x_d<6, deg_c128(6)>(op, y, st);
    if (op->batched) {
        switch (op->J) {
            case 4: return launch_degrid_x_t<4, deg_c64(4)>(op, y, st);
            case 6: return launch_degrid_x_t<6, deg_c64(6)>(op, y, st);
            default: return launch_degrid_x_t<8, deg_c64(8)>(op, y, st);
        }
    }
    // the tile-sorted kernels below serve complex128 with J = 8 (its J x J patch does not fit the register file)
    switch (op->J) {
        case 4: return launch_degrid_t<double, 4, deg_c128(4)>(op, y, caller_order, st);
        case 6: return launch_degrid_t<double, 6, deg_c128(6)>(op, y, caller_order, st);
        default: return launch_degrid_t<double, 8, deg_c128(8)>(op, y, caller_order, st);
    }
}

int launch_grid(purify_op* op, const void* y, bool caller_order, cudaStream_t st) {
    {
        StageTimer tz(op, PURIFY_STAGE_ZERO, st);
        CK(cudaMemsetAsync(op->grid, 0, csize(op) * (size_t)op->K * op->K, st));
    }
    StageTimer t(op, PURIFY_STAGE_GRID, st);
    if (op->batched && op->dtype == PURIFY_C128)
        return op->J == 4 ? launch_grid_x_d<4, deg_c128(4)>(op, y, st) : launch_grid_x_d<6, deg_c128(6)>(op, y, st);
    if (op->batched) {
        switch (op->J) {
            case 4: return launch_grid_x_t<4, deg_c64(4)>(op, y, st);
            case 6: return launch_grid_x_t<6, deg_c64(6)>(op, y, st);
            default: return launch_grid_x_t<8, deg_c64(8)>(op, y, st);
        }
    }
    switch (op->J) {
        case 4: return launch_grid_t<double, 4, deg_c128(4)>(op, y, caller_order, st);
        case 6: return launch_grid_t<double, 6, deg_c128(6)>(op, y, caller_order, st);
        default: return launch_grid_t<double, 8, deg_c128(8)>(op, y, caller_order, st);
    }
}

int launch_pad(purify_op* op, const void* x, cudaStream_t st) {
    StageTimer t(op, PURIFY_STAGE_PAD, st);
    const long long vecs = (long long)op->K * op->K * (long long)csize(op) / 16;
    if (op->dtype == PURIFY_C64)
        pk::pad_kernel<float><<<grid_for(vecs, 256, 148 * 32), 256, 0, st>>>((const float2*)x, (const float*)op->corr,
                                                                             (float2*)op->grid, op->n, op->K);
    else
        pk::pad_kernel<double><<<grid_for(vecs, 256, 148 * 32), 256, 0, st>>>((const double2*)x, (const double*)op->corr,
                                                                              (double2*)op->grid, op->n, op->K);
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

int launch_crop(purify_op* op, void* x, cudaStream_t st, int row0 = 0, int row1 = -1, bool timed = true) {
    if (row1 < 0) row1 = op->n;
    if (timed && op->time_stages && op->ev_ok) { cudaEventRecord(op->ev[2 * PURIFY_STAGE_CROP], st); op->stage_ran[PURIFY_STAGE_CROP] = true; }
    const long long tot = (long long)(row1 - row0) * op->n;
    if (tot > 0) {
        if (op->dtype == PURIFY_C64)
            pk::crop_kernel<float><<<grid_for(tot, 256, 148 * 32), 256, 0, st>>>((const float2*)op->grid, (const float*)op->corr,
                                                                                 (float2*)x, op->n, op->K, row0, row1);
        else
            pk::crop_kernel<double><<<grid_for(tot, 256, 148 * 32), 256, 0, st>>>((const double2*)op->grid, (const double*)op->corr,
                                                                                  (double2*)x, op->n, op->K, row0, row1);
        op->launches++;
    }
    if (timed && op->time_stages && op->ev_ok) cudaEventRecord(op->ev[2 * PURIFY_STAGE_CROP + 1], st);
    CK(cudaGetLastError());
    return PURIFY_OK;
}

int launch_fft(purify_op* op, int dir, cudaStream_t st) {
    StageTimer t(op, dir == CUFFT_FORWARD ? PURIFY_STAGE_FFT : PURIFY_STAGE_IFFT, st);
    CKFFT(cufftSetStream(op->plan, st));
    if (op->dtype == PURIFY_C64)
        CKFFT(cufftExecC2C(op->plan, (cufftComplex*)op->grid, (cufftComplex*)op->grid, dir));
    else
        CKFFT(cufftExecZ2Z(op->plan, (cufftDoubleComplex*)op->grid, (cufftDoubleComplex*)op->grid, dir));
    return PURIFY_OK;
}

int ensure_ws(purify_op* op, void** p, size_t* have, size_t bytes);

// below this many visibilities the permutation is L2-resident and one gather is cheaper than three passes
constexpr long long ROUTED_MIN = 1ll << 24;   // (measured: 1e7 elements 0.065 ms by one gather against 0.125 ms routed; 1e8: 2.16 against 1.07 ms)
// block size of the routing passes: 2^13 complex64 / 2^12 complex128 elements = 64 KB of shared memory
inline int route_bs(const purify_op* op) { return op->dtype == PURIFY_C64 ? 13 : 12; }

template <typename C, int BS>
int launch_permute_routed(purify_op* op, const C* in, C* out, int to_native, cudaStream_t st) {
    const long long M = op->M, S = op->M_native;
    const unsigned n_tiles = (unsigned)((M + pk::PERM_TILE - 1) / pk::PERM_TILE);
    const unsigned blocks_a = (unsigned)((S + (1ll << BS) - 1) >> BS), blocks_b = (unsigned)((M + (1ll << BS) - 1) >> BS);
    const size_t smem_r = sizeof(C) << BS, smem_t = sizeof(C) * pk::PERM_TILE;
    static bool attr_done = false;
    if (!attr_done) {
        CK(cudaFuncSetAttribute(pk::route_kernel<C, BS, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r));
        CK(cudaFuncSetAttribute(pk::route_kernel<C, BS, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r));
        CK(cudaFuncSetAttribute(pk::tile_permute_kernel<C, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t));
        CK(cudaFuncSetAttribute(pk::tile_permute_kernel<C, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t));
        attr_done = true;
    }
    int rc = ensure_ws(op, &op->perm_ws, &op->perm_ws_bytes, sizeof(C) * (size_t)M * (to_native ? 2 : 1));
    if (rc) return rc;
    C* w0 = (C*)op->perm_ws;
    C* w1 = w0 + M;
    if (!to_native) {              // native -> A order -> mid (in the caller's buffer) -> caller order (in place)
        pk::route_kernel<C, BS, 0><<<blocks_a, pk::PERM_THREADS, smem_r, st>>>(in, w0, op->loc_a, op->dst_a, S);
        pk::route_kernel<C, BS, 0><<<blocks_b, pk::PERM_THREADS, smem_r, st>>>(w0, out, op->loc_b, op->dst_b, M);
        pk::tile_permute_kernel<C, 0><<<n_tiles, pk::PERM_THREADS, smem_t, st>>>(out, out, op->loc_idx, M);
    } else {                       // caller order -> mid -> A order -> native (padding slots: 0)
        pk::tile_permute_kernel<C, 1><<<n_tiles, pk::PERM_THREADS, smem_t, st>>>(in, w0, op->loc_idx, M);
        pk::route_kernel<C, BS, 1><<<blocks_b, pk::PERM_THREADS, smem_r, st>>>(w0, w1, op->loc_b, op->dst_b, M);
        pk::route_kernel<C, BS, 1><<<blocks_a, pk::PERM_THREADS, smem_r, st>>>(w1, out, op->loc_a, op->dst_a, S);
    }
    op->launches += 3;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

int launch_permute(purify_op* op, const void* in, void* out, int to_native, cudaStream_t st) {
    StageTimer t(op, PURIFY_STAGE_PERMUTE, st);
    if (op->M_native == 0) return PURIFY_OK;
    if (op->loc_a && op->M > 0)
        return op->dtype == PURIFY_C64 ? launch_permute_routed<float2, 13>(op, (const float2*)in, (float2*)out, to_native, st)
                                       : launch_permute_routed<double2, 12>(op, (const double2*)in, (double2*)out, to_native, st);
    if (!to_native && op->inv_perm) {
        if (op->M > 0 && op->dtype == PURIFY_C64)
            pk::gather_from_native_kernel<float2><<<grid_for(op->M, 256, 148 * 32), 256, 0, st>>>((const float2*)in, (float2*)out, op->inv_perm, op->M);
        else if (op->M > 0)
            pk::gather_from_native_kernel<double2><<<grid_for(op->M, 256, 148 * 32), 256, 0, st>>>((const double2*)in, (double2*)out, op->inv_perm, op->M);
        op->launches++;
        CK(cudaGetLastError());
        return PURIFY_OK;
    }
    if (op->dtype == PURIFY_C64)
        pk::permute_kernel<float2><<<grid_for(op->M_native, 256, 148 * 32), 256, 0, st>>>((const float2*)in, (float2*)out, op->perm, op->M_native, to_native);
    else
        pk::permute_kernel<double2><<<grid_for(op->M_native, 256, 148 * 32), 256, 0, st>>>((const double2*)in, (double2*)out, op->perm, op->M_native, to_native);
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

// lazily allocated workspace of at least `bytes` (grown when a later call needs more: the pointer may change)
int ensure_ws(purify_op* op, void** p, size_t* have, size_t bytes) {
    if (*p && *have >= bytes) return PURIFY_OK;
    if (*p) {
        cudaError_t e = cudaDeviceSynchronize();      // work enqueued on the old buffer must finish before it is freed
        if (e != cudaSuccess) return fail(PURIFY_ERR_CUDA, "synchronise before workspace growth failed: %s", cudaGetErrorString(e));
        cudaFree(*p);
        op->device_bytes -= (long long)*have;
        *p = nullptr; *have = 0;
        op->graph_stale = true;                       // a captured graph may hold the old pointer
    }
    int rc = dev_alloc(op, p, bytes);
    if (rc == PURIFY_OK) *have = bytes ? bytes : 16;
    return rc;
}
#define WS_Y(op, bytes) ensure_ws(op, &(op)->y_ws, &(op)->y_ws_bytes, bytes)
#define WS_Y2(op, bytes) ensure_ws(op, &(op)->y_ws2, &(op)->y_ws2_bytes, bytes)
#define WS_X(op, bytes) ensure_ws(op, &(op)->x_ws, &(op)->x_ws_bytes, bytes)
#define WS_SCAL(op) ensure_ws(op, (void**)&(op)->scal_ws, &(op)->scal_ws_bytes, sizeof(double))

void begin_call(purify_op* op) {
    op->launches = 0;
    for (int i = 0; i < PURIFY_STAGE_COUNT; ++i) op->stage_ran[i] = false;
}

int check_device() {
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev <= 0) {
        cudaGetLastError();
        return fail(PURIFY_ERR_NO_DEVICE, "no CUDA device available (%s); this library has no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    return PURIFY_OK;
}

}  // namespace

// =============================================================================== create
namespace {

template <typename R>
int build_bins(purify_op* op, const void* uv_dev, const void* w_dev, cudaStream_t st) {
    typedef typename pk::Cplx<R>::type C;
    const long long M = op->M;
    const int K = op->K;
    const int kmask = (K & (K - 1)) == 0 ? K - 1 : 0;
    op->ntx = (K + pk::TILE - 1) / pk::TILE;
    op->n_tiles = op->ntx * op->ntx;

    int rc;
    if ((rc = dev_alloc(op, &op->uv_s, sizeof(C) * (size_t)M))) return rc;
    if ((rc = dev_alloc(op, &op->w_s, sizeof(R) * (size_t)M))) return rc;
    if ((rc = dev_alloc(op, (void**)&op->perm, sizeof(unsigned) * (size_t)M))) return rc;

    // temporaries (freed before return)
    unsigned *keys = nullptr, *keys2 = nullptr, *idx = nullptr;
    int *bad = nullptr, *tile_start = nullptr, *n_chunks = nullptr, *chunk_off = nullptr;
    void* cub_tmp = nullptr;
    auto cleanup = [&]() {
        cudaFree(keys); cudaFree(keys2); cudaFree(idx); cudaFree(bad);
        cudaFree(tile_start); cudaFree(n_chunks); cudaFree(chunk_off); cudaFree(cub_tmp);
    };
#define CKC(call)                                                                                       \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            cleanup();                                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? PURIFY_ERR_ALLOC : PURIFY_ERR_CUDA,          \
                        "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);    \
        }                                                                                               \
    } while (0)

    const size_t Mz = M > 0 ? (size_t)M : 1;
    CKC(cudaMalloc(&keys, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&keys2, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&idx, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&bad, sizeof(int)));
    CKC(cudaMalloc(&tile_start, sizeof(int) * (size_t)(op->n_tiles + 1)));
    CKC(cudaMalloc(&n_chunks, sizeof(int) * (size_t)(op->n_tiles + 1)));
    CKC(cudaMalloc(&chunk_off, sizeof(int) * (size_t)(op->n_tiles + 1)));
    CKC(cudaMemsetAsync(bad, 0, sizeof(int), st));
    CKC(cudaMemsetAsync(n_chunks, 0, sizeof(int) * (size_t)(op->n_tiles + 1), st));

    if (M > 0) {
        pk::key_kernel<R><<<grid_for(M, 256), 256, 0, st>>>((const C*)uv_dev, M, K, kmask, op->ntx, keys, idx, bad);
        CKC(cudaGetLastError());
        int h_bad = 0;
        CKC(cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        CKC(cudaStreamSynchronize(st));
        if (h_bad) {
            cleanup();
            return fail(PURIFY_ERR_UV_NONFINITE, "uv contains NaN, Inf or |coordinate| >= 2^30");
        }
        // device radix sort on (tile, cell) id; only the significant key bits are sorted
        int bits = 1;
        while (bits < 32 && (1ull << bits) < (unsigned long long)op->n_tiles * pk::TILE * pk::TILE) ++bits;
        size_t tmp_bytes = 0;
        CKC(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, idx, op->perm, (int)M, 0, bits, st));
        CKC(cudaMalloc(&cub_tmp, tmp_bytes ? tmp_bytes : 16));
        CKC(cub::DeviceRadixSort::SortPairs(cub_tmp, tmp_bytes, keys, keys2, idx, op->perm, (int)M, 0, bits, st));
        pk::gather_kernel<R><<<grid_for(M, 256), 256, 0, st>>>((const C*)uv_dev, (const R*)w_dev, op->perm, M,
                                                                (C*)op->uv_s, (R*)op->w_s);
        CKC(cudaGetLastError());
    }
    pk::tile_start_kernel<<<(op->n_tiles + 1 + 255) / 256, 256, 0, st>>>(keys2, M, op->n_tiles, tile_start);
    CKC(cudaGetLastError());
    pk::tile_chunks_kernel<<<(op->n_tiles + 255) / 256, 256, 0, st>>>(tile_start, op->n_tiles, op->chunk, n_chunks);
    CKC(cudaGetLastError());
    {
        size_t tmp2 = 0;
        void* t2 = nullptr;
        CKC(cub::DeviceScan::ExclusiveSum(nullptr, tmp2, n_chunks, chunk_off, op->n_tiles + 1, st));
        CKC(cudaMalloc(&t2, tmp2 ? tmp2 : 16));
        cudaError_t e2 = cub::DeviceScan::ExclusiveSum(t2, tmp2, n_chunks, chunk_off, op->n_tiles + 1, st);
        cudaError_t e3 = cudaStreamSynchronize(st);
        cudaFree(t2);
        CKC(e2);
        CKC(e3);
    }
    CKC(cudaMemcpy(&op->n_items, chunk_off + op->n_tiles, sizeof(int), cudaMemcpyDeviceToHost));
    // tile statistics (host side; n_tiles is small)
    {
        std::vector<int> ts((size_t)op->n_tiles + 1);
        CKC(cudaMemcpy(ts.data(), tile_start, sizeof(int) * ts.size(), cudaMemcpyDeviceToHost));
        op->n_tiles_nonempty = 0;
        op->max_tile_count = 0;
        for (int t = 0; t < op->n_tiles; ++t) {
            const int c = ts[t + 1] - ts[t];
            if (c > 0) op->n_tiles_nonempty++;
            if (c > op->max_tile_count) op->max_tile_count = c;
        }
    }
    {
        void* items = nullptr;
        cudaError_t e = cudaMalloc(&items, sizeof(pk::Item) * (size_t)(op->n_items > 0 ? op->n_items : 1));
        if (e != cudaSuccess) { cleanup(); cudaGetLastError(); return fail(PURIFY_ERR_ALLOC, "cudaMalloc(items) failed"); }
        op->items = (pk::Item*)items;
        op->device_bytes += (long long)sizeof(pk::Item) * (op->n_items > 0 ? op->n_items : 1);
    }
    if (op->n_items > 0) {
        pk::fill_items_kernel<<<(op->n_tiles + 255) / 256, 256, 0, st>>>(tile_start, chunk_off, op->n_tiles, op->ntx,
                                                                         op->chunk, op->items);
        CKC(cudaGetLastError());
    }
    CKC(cudaStreamSynchronize(st));
    cleanup();
#undef CKC
    return PURIFY_OK;
}

// a0 for complex64: the batched layout of batched.cuh (device radix sort on band/cell id, per-band
// batch construction, slot fill).
template <typename F>
int build_bins_x(purify_op* op, const void* uv_dev, const void* w_dev, cudaStream_t st) {
    typedef typename pk::Cplx<F>::type F2;
    const long long M = op->M;
    const int K = op->K;
    const int nbx = (K + pk::XBW - 1) / pk::XBW, nby = (K + pk::XBH - 1) / pk::XBH;
    const int n_bands = nbx * nby;
    op->n_bands = n_bands;
    op->ntx = nbx;
    op->n_tiles = n_bands;
    op->batched = true;

    unsigned *keys = nullptr, *keys2 = nullptr, *idx = nullptr, *perm0 = nullptr, *band_start = nullptr;
    unsigned *a_nb = nullptr, *a_it = nullptr, *a_items = nullptr, *o_nb = nullptr, *o_it = nullptr, *o_items = nullptr;
    unsigned *lsrc = nullptr, *nonempty = nullptr;
    pk::BandTotals* totals = nullptr;
    int* bad = nullptr;
    void *cub_tmp = nullptr, *scan_tmp = nullptr;
    auto cleanup = [&]() {
        cudaFree(keys); cudaFree(keys2); cudaFree(idx); cudaFree(perm0); cudaFree(band_start); cudaFree(a_nb);
        cudaFree(a_it); cudaFree(a_items); cudaFree(o_nb); cudaFree(o_it); cudaFree(o_items); cudaFree(lsrc);
        cudaFree(nonempty); cudaFree(totals); cudaFree(bad); cudaFree(cub_tmp); cudaFree(scan_tmp);
    };
#define CKC(call)                                                                                       \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            cleanup();                                                                                  \
            cudaGetLastError();                                                                         \
            return fail(e_ == cudaErrorMemoryAllocation ? PURIFY_ERR_ALLOC : PURIFY_ERR_CUDA,          \
                        "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);    \
        }                                                                                               \
    } while (0)
    const size_t Mz = M > 0 ? (size_t)M : 1, nb1 = (size_t)n_bands + 1;
    CKC(cudaMalloc(&keys, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&keys2, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&idx, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&perm0, sizeof(unsigned) * Mz));
    CKC(cudaMalloc(&band_start, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&totals, sizeof(pk::BandTotals) * nb1));
    CKC(cudaMalloc(&a_nb, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&a_it, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&a_items, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&o_nb, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&o_it, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&o_items, sizeof(unsigned) * nb1));
    CKC(cudaMalloc(&nonempty, sizeof(unsigned)));
    CKC(cudaMalloc(&bad, sizeof(int)));
    CKC(cudaMemsetAsync(bad, 0, sizeof(int), st));
    CKC(cudaMemsetAsync(nonempty, 0, sizeof(unsigned), st));

    if (M > 0) {
        pk::xkey_kernel<F><<<grid_for(M, 256), 256, 0, st>>>((const F2*)uv_dev, M, K, nbx, keys, idx, bad);
        CKC(cudaGetLastError());
        int h_bad = 0;
        CKC(cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        CKC(cudaStreamSynchronize(st));
        if (h_bad) {
            cleanup();
            return fail(PURIFY_ERR_UV_NONFINITE, "uv contains NaN, Inf or |coordinate| >= 2^30");
        }
        int bits = 1;
        while (bits < 32 && (1ull << bits) < (unsigned long long)n_bands * pk::XCELLS) ++bits;
        size_t tmp_bytes = 0;
        CKC(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, idx, perm0, (int)M, 0, bits, st));
        CKC(cudaMalloc(&cub_tmp, tmp_bytes ? tmp_bytes : 16));
        CKC(cub::DeviceRadixSort::SortPairs(cub_tmp, tmp_bytes, keys, keys2, idx, perm0, (int)M, 0, bits, st));
    }
    pk::band_start_kernel<<<(n_bands + 1 + 255) / 256, 256, 0, st>>>(keys2, M, n_bands, band_start);
    CKC(cudaGetLastError());
    pk::band_build_kernel<1><<<n_bands, pk::XCELLS, 0, st>>>(keys2, band_start, nbx, pk::XBW + op->J, totals, nullptr, nullptr, nullptr,
                                                             nullptr, nullptr, nullptr, nullptr);
    CKC(cudaGetLastError());
    pk::split_totals_kernel<<<(n_bands + 1 + 255) / 256, 256, 0, st>>>(totals, n_bands, a_nb, a_it, a_items, nonempty);
    CKC(cudaGetLastError());
    {
        size_t tmp2 = 0;
        CKC(cub::DeviceScan::ExclusiveSum(nullptr, tmp2, a_nb, o_nb, n_bands + 1, st));
        CKC(cudaMalloc(&scan_tmp, tmp2 ? tmp2 : 16));
        CKC(cub::DeviceScan::ExclusiveSum(scan_tmp, tmp2, a_nb, o_nb, n_bands + 1, st));
        CKC(cub::DeviceScan::ExclusiveSum(scan_tmp, tmp2, a_it, o_it, n_bands + 1, st));
        CKC(cub::DeviceScan::ExclusiveSum(scan_tmp, tmp2, a_items, o_items, n_bands + 1, st));
    }
    unsigned h_tot[4] = {0, 0, 0, 0};
    CKC(cudaMemcpyAsync(&h_tot[0], o_nb + n_bands, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CKC(cudaMemcpyAsync(&h_tot[1], o_it + n_bands, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CKC(cudaMemcpyAsync(&h_tot[2], o_items + n_bands, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CKC(cudaMemcpyAsync(&h_tot[3], nonempty, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CKC(cudaStreamSynchronize(st));
    op->n_batches = h_tot[0];
    op->M_native = (long long)h_tot[1] * 32;
    op->n_items = (int)h_tot[2];
    op->n_bands_nonempty = (int)h_tot[3];
    op->n_tiles_nonempty = (int)h_tot[3];
    int rc;
    const size_t S = op->M_native > 0 ? (size_t)op->M_native : 1, NBz = op->n_batches > 0 ? op->n_batches : 1;
    // per-iteration records (uv[32] | w[32]); uv_s holds them, w_s is unused in this layout
    if ((rc = dev_alloc(op, &op->uv_s, (size_t)pk::REC_FLOATS * sizeof(F) * (S / 32 + 1)))) { cleanup(); return rc; }
    if ((rc = dev_alloc(op, (void**)&op->perm, sizeof(unsigned) * S))) { cleanup(); return rc; }
    if ((rc = dev_alloc(op, (void**)&op->x_bhdr, sizeof(uint2) * NBz))) { cleanup(); return rc; }
    if ((rc = dev_alloc(op, (void**)&op->x_blane, sizeof(unsigned) * 32 * NBz))) { cleanup(); return rc; }
    if ((rc = dev_alloc(op, (void**)&op->x_items, sizeof(pk::XItem) * (size_t)(op->n_items > 0 ? op->n_items : 1)))) { cleanup(); return rc; }
    if ((rc = dev_alloc(op, (void**)&op->x_counter, 2 * sizeof(unsigned)))) { cleanup(); return rc; }
    CKC(cudaMemsetAsync(op->x_counter, 0, 2 * sizeof(unsigned), st));     // the kernels leave the queue at 0 (batched.cuh x_queue_finish)
    CKC(cudaMalloc(&lsrc, sizeof(unsigned) * 32 * NBz));
    if (op->n_batches > 0) {
        pk::band_build_kernel<2><<<n_bands, pk::XCELLS, 0, st>>>(keys2, band_start, nbx, pk::XBW + op->J, nullptr, o_nb, o_it, o_items,
                                                                 op->x_bhdr, op->x_blane, lsrc, op->x_items);
        CKC(cudaGetLastError());
        pk::item_iters_kernel<<<(op->n_items + 255) / 256, 256, 0, st>>>(op->x_items, op->n_items, op->x_bhdr);
        CKC(cudaGetLastError());
        // Few items per persistent warp (< 16): longest items first, so that the tail of a launch consists of short items
        // (config 3: -9 %).  With many items per warp the band order is kept: it is friendlier to L2 / DRAM pages
        // (config 4 and 5 lose 1-3 % when reordered).  Stable sort: band order inside one length class.
        if (op->n_items < 16 * 148 * 16) {
            const int ni = op->n_items;
            unsigned *ik = nullptr, *ik2 = nullptr, *ii = nullptr, *ii2 = nullptr;
            pk::XItem* sorted = nullptr;
            void* tmp = nullptr;
            size_t tb = 0;
            auto free5 = [&]() { cudaFree(ik); cudaFree(ik2); cudaFree(ii); cudaFree(ii2); cudaFree(tmp); };
            cudaError_t e = cudaMalloc(&ik, sizeof(unsigned) * ni);
            if (e == cudaSuccess) e = cudaMalloc(&ik2, sizeof(unsigned) * ni);
            if (e == cudaSuccess) e = cudaMalloc(&ii, sizeof(unsigned) * ni);
            if (e == cudaSuccess) e = cudaMalloc(&ii2, sizeof(unsigned) * ni);
            if (e == cudaSuccess) e = cudaMalloc((void**)&sorted, sizeof(pk::XItem) * ni);
            if (e == cudaSuccess) e = cub::DeviceRadixSort::SortPairs(nullptr, tb, ik, ik2, ii, ii2, ni, 0, 16, st);
            if (e == cudaSuccess) e = cudaMalloc(&tmp, tb ? tb : 16);
            if (e == cudaSuccess) {
                pk::item_key_kernel<<<(ni + 255) / 256, 256, 0, st>>>(op->x_items, ni, ik, ii);
                e = cub::DeviceRadixSort::SortPairs(tmp, tb, ik, ik2, ii, ii2, ni, 0, 16, st);
            }
            if (e == cudaSuccess) {
                pk::item_gather_kernel<<<(ni + 255) / 256, 256, 0, st>>>(op->x_items, ii2, ni, sorted);
                e = cudaStreamSynchronize(st);
            }
            if (e == cudaSuccess) { cudaFree(op->x_items); op->x_items = sorted; sorted = nullptr; }
            cudaFree(sorted);
            free5();
            CKC(e);
        }
        pk::slot_fill_kernel<F><<<grid_for((long long)op->n_batches * 32, 256), 256, 0, st>>>(
            op->x_bhdr, op->x_blane, lsrc, op->n_batches, perm0, (const F2*)uv_dev, (const F*)w_dev, K,
            op->perm, (F*)op->uv_s);
        CKC(cudaGetLastError());
    }
    if (M >= ROUTED_MIN) {
        // index arrays of the routed permutation (kernels.cuh): four stable radix sorts over the slots
        const long long S = op->M_native;
        const int bs = route_bs(op);
        const unsigned n_tiles = (unsigned)((M + pk::PERM_TILE - 1) / pk::PERM_TILE);
        int cs = pk::PERM_TILE_SHIFT + 3;                 // coarse bucket = 2^cs caller indices: at most 256 buckets, at least 8 tiles
        while (((M - 1) >> cs) >= 256) ++cs;
        const int kb = cs - pk::PERM_TILE_SHIFT + 1;
        auto nbits = [](unsigned long long v) { int b = 1; while ((1ull << b) <= v) ++b; return b; };
        unsigned *tk = nullptr, *tk2 = nullptr, *tv = nullptr, *tv2 = nullptr, *apos = nullptr, *slot_a = nullptr, *q = nullptr;
        void* tmp2 = nullptr;
        size_t tmp2_bytes = 0;
        auto free_t = [&]() { cudaFree(tk); cudaFree(tk2); cudaFree(tv); cudaFree(tv2); cudaFree(apos); cudaFree(slot_a); cudaFree(q); cudaFree(tmp2); };
        cudaError_t e = cudaMalloc(&tk, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&tk2, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&tv, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&tv2, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&apos, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&q, sizeof(unsigned) * S);
        if (e == cudaSuccess) e = cudaMalloc(&slot_a, sizeof(unsigned) * (size_t)M);
        if (e == cudaSuccess) e = cub::DeviceRadixSort::SortPairs(nullptr, tmp2_bytes, tk, tk2, tv, tv2, (int)S, 0, 32, st);
        if (e == cudaSuccess) e = cudaMalloc(&tmp2, tmp2_bytes ? tmp2_bytes : 16);
        if (e != cudaSuccess) { cudaGetLastError(); free_t(); cleanup(); return fail(PURIFY_ERR_ALLOC, "routed permutation: temporaries: %s", cudaGetErrorString(e)); }
        if ((rc = dev_alloc(op, (void**)&op->loc_a, sizeof(unsigned short) * (size_t)S)) ||
            (rc = dev_alloc(op, (void**)&op->dst_a, sizeof(unsigned) * (size_t)S)) ||
            (rc = dev_alloc(op, (void**)&op->loc_b, sizeof(unsigned short) * (size_t)M)) ||
            (rc = dev_alloc(op, (void**)&op->dst_b, sizeof(unsigned) * (size_t)M)) ||
            (rc = dev_alloc(op, (void**)&op->loc_idx, sizeof(unsigned short) * (size_t)M))) { free_t(); cleanup(); return rc; }
        const int g1 = grid_for(S, 256), gm = grid_for(M, 256);
        // (1) mid order: by caller tile; q[slot] = mid position, loc_idx = position inside the tile
        pk::tile_key_kernel<<<g1, 256, 0, st>>>(op->perm, S, n_tiles, tk, tv);
        e = cub::DeviceRadixSort::SortPairs(tmp2, tmp2_bytes, tk, tk2, tv, tv2, (int)S, 0, nbits(n_tiles), st);
        if (e == cudaSuccess) {
            pk::mid_fill_kernel<<<gm, 256, 0, st>>>(tv2, op->perm, M, q, op->loc_idx);
            // (2) A order: by coarse bucket; apos[slot] = A position, slot_a[k] = slot of A element k
            pk::coarse_key_kernel<<<g1, 256, 0, st>>>(op->perm, S, cs, bs, 0, tk, tv);
            e = cub::DeviceRadixSort::SortPairs(tmp2, tmp2_bytes, tk, tk2, tv, tv2, (int)S, 0, 9, st);
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(slot_a, tv2, sizeof(unsigned) * (size_t)M, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) {
            pk::a_pos_kernel<<<gm, 256, 0, st>>>(slot_a, M, apos);
            // (3) pass A: order inside every native block by bucket
            pk::coarse_key_kernel<<<g1, 256, 0, st>>>(op->perm, S, cs, bs, 1, tk, tv);
            e = cub::DeviceRadixSort::SortPairs(tmp2, tmp2_bytes, tk, tk2, tv, tv2, (int)S, 0, 9 + nbits((unsigned long long)((S - 1) >> bs)), st);
        }
        if (e == cudaSuccess) {
            pk::pass_a_fill_kernel<<<g1, 256, 0, st>>>(tv2, op->perm, apos, S, bs, op->loc_a, op->dst_a);
            // (4) pass B: order inside every A block by tile
            pk::pass_b_key_kernel<<<gm, 256, 0, st>>>(slot_a, op->perm, M, cs, bs, kb, tk, tv);
            e = cub::DeviceRadixSort::SortPairs(tmp2, tmp2_bytes, tk, tk2, tv, tv2, (int)M, 0, kb + nbits((unsigned long long)((M - 1) >> bs)), st);
        }
        if (e == cudaSuccess) {
            pk::pass_b_fill_kernel<<<gm, 256, 0, st>>>(tv2, slot_a, q, M, bs, op->loc_b, op->dst_b);
            e = cudaStreamSynchronize(st);
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        free_t();
        CKC(e);
    } else if (M > 0) {
        if ((rc = dev_alloc(op, (void**)&op->inv_perm, sizeof(unsigned) * (size_t)M))) { cleanup(); return rc; }
        pk::invert_perm_kernel<<<grid_for(op->M_native, 256), 256, 0, st>>>(op->perm, op->M_native, op->inv_perm);
        CKC(cudaGetLastError());
    }
    CKC(cudaStreamSynchronize(st));
    // statistics: fullest band
    {
        std::vector<unsigned> bsv(nb1);
        CKC(cudaMemcpy(bsv.data(), band_start, sizeof(unsigned) * nb1, cudaMemcpyDeviceToHost));
        op->max_tile_count = 0;
        for (int b = 0; b < n_bands; ++b) {
            const long long c = (long long)bsv[b + 1] - (long long)bsv[b];
            if (c > op->max_tile_count) op->max_tile_count = c;
        }
    }
    cleanup();
#undef CKC
    return PURIFY_OK;
}

template <typename R>
int build_tables(purify_op* op, cudaStream_t st) {
    int rc;
    // gridding correction s[n]
    std::vector<double> s;
    kbhost::correction(op->n, op->J, s);
    std::vector<R> sr(s.begin(), s.end());
    if ((rc = dev_alloc(op, &op->corr, sizeof(R) * (size_t)op->n))) return rc;
    CK(cudaMemcpyAsync(op->corr, sr.data(), sizeof(R) * (size_t)op->n, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    // kernel polynomial
    kbhost::PolyFit fit;
    const int deg = sizeof(R) == 4 ? deg_c64(op->J) : deg_c128(op->J);
    kbhost::fit_poly(op->J, deg, fit);
    op->poly_degree = deg;
    op->poly_err = fit.max_abs_err;
    for (int j = 0; j < 4; ++j)
        for (int m = 0; m < 9; ++m) {
            op->coef32.e[j][m] = (float)fit.e[j][m]; op->coef32.o[j][m] = (float)fit.o[j][m];
            op->coef64.e[j][m] = fit.e[j][m];        op->coef64.o[j][m] = fit.o[j][m];
        }
    // pre-sampled table
    if (op->mode == PURIFY_KERNEL_TABLE) {
        std::vector<double> T;
        kbhost::table(op->J, op->table_R, T);
        std::vector<R> Tr(T.begin(), T.end());
        op->table_len = (int)Tr.size();
        if ((rc = dev_alloc(op, &op->table, sizeof(R) * Tr.size()))) return rc;
        CK(cudaMemcpyAsync(op->table, Tr.data(), sizeof(R) * Tr.size(), cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    return PURIFY_OK;
}

int build_tmap(purify_op* op) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess)
        return fail(PURIFY_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    const int BOX = pk::TILE + op->J;
    const bool f32 = op->dtype == PURIFY_C64;
    if (op->batched) {
        const cuuint64_t dims[2] = {(cuuint64_t)2 * op->K, (cuuint64_t)op->K};
        const cuuint64_t strides[1] = {(cuuint64_t)op->K * csize(op)};
        const cuuint32_t box[2] = {(cuuint32_t)(2 * (pk::XBW + op->J)), (cuuint32_t)(pk::XBH + op->J - 1)};
        const cuuint32_t estr[2] = {1, 1};
        if (box[0] > (cuuint32_t)2 * op->K || box[1] > (cuuint32_t)op->K) {       // grid smaller than one box: no interior band
            memset(&op->tmap_x, 0, sizeof(op->tmap_x));
            return PURIFY_OK;
        }
        CUresult r = ((EncodeTiledFn)fn)(&op->tmap_x, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, op->grid, dims, strides, box, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(PURIFY_ERR_CUDA, "cuTensorMapEncodeTiled (band box) failed: CUresult %d", (int)r);
        return PURIFY_OK;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)2 * op->K, (cuuint64_t)op->K};            // inner extent in reals
    const cuuint64_t strides[1] = {(cuuint64_t)op->K * csize(op)};                     // row pitch, bytes
    const cuuint32_t box[2] = {(cuuint32_t)(2 * BOX), (cuuint32_t)BOX};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)fn)(&op->tmap, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64,
                                     2, op->grid, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(PURIFY_ERR_CUDA, "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
    return PURIFY_OK;
}

int create_impl(purify_op** out, int n, int oversample, int J, long long M, const void* uv, const void* w,
                bool host_inputs, int dtype, const purify_opts* opts, void* stream) {
    if (!out) return fail(PURIFY_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (n <= 0 || (n & 1)) return fail(PURIFY_ERR_INVALID_ARG, "n must be positive and even (got %d)", n);
    if (n > 16384) return fail(PURIFY_ERR_INVALID_ARG, "n too large (got %d, max 16384)", n);
    if (oversample != 2) return fail(PURIFY_ERR_UNSUPPORTED, "only oversample = 2 is supported (got %d)", oversample);
    if (J != 4 && J != 6 && J != 8) return fail(PURIFY_ERR_INVALID_ARG, "J must be 4, 6 or 8 (got %d)", J);
    if (M < 0 || M >= (1ll << 31)) return fail(PURIFY_ERR_INVALID_ARG, "M must be in [0, 2^31) (got %lld)", M);
    if (M > 0 && !uv) return fail(PURIFY_ERR_INVALID_ARG, "uv is NULL");
    if (dtype != PURIFY_C64 && dtype != PURIFY_C128) return fail(PURIFY_ERR_UNSUPPORTED, "unknown dtype %d", dtype);
    int mode = PURIFY_KERNEL_ANALYTIC, R = 4096, chunk = 4096, time_stages = 0;
    bool admm_unfused = false;
    if (opts) {
        mode = opts->kernel_mode;
        if (opts->table_samples_per_unit) R = opts->table_samples_per_unit;
        if (opts->chunk) chunk = opts->chunk;
        time_stages = opts->time_stages;
        admm_unfused = opts->admm_unfused != 0;
        if (opts->reserved[0] || opts->reserved[1]) return fail(PURIFY_ERR_INVALID_ARG, "purify_opts.reserved must be 0");
    }
    if (mode != PURIFY_KERNEL_ANALYTIC && mode != PURIFY_KERNEL_TABLE)
        return fail(PURIFY_ERR_UNSUPPORTED, "unknown kernel mode %d", mode);
    if (R < 1 || (long long)R * J / 2 + 2 > (1ll << 30)) return fail(PURIFY_ERR_INVALID_ARG, "bad table density %d", R);
    if (chunk < 32 || chunk > (1 << 24)) return fail(PURIFY_ERR_INVALID_ARG, "chunk must be in [32, 2^24] (got %d)", chunk);
    int rc = check_device();
    if (rc) return rc;

    purify_op* op = new (std::nothrow) purify_op();
    if (!op) return fail(PURIFY_ERR_ALLOC, "host allocation failed");
    op->n = n; op->K = 2 * n; op->J = J; op->M = M; op->dtype = dtype; op->mode = mode; op->table_R = R;
    op->chunk = chunk; op->time_stages = time_stages; op->admm_unfused = admm_unfused;
    cudaStream_t st = (cudaStream_t)stream;

    void *uv_tmp = nullptr, *w_tmp = nullptr;
    auto bail = [&](int code) { cudaFree(uv_tmp); cudaFree(w_tmp); purify_op_destroy(op); return code; };

    const void *uv_dev = uv, *w_dev = w;
    if (host_inputs && M > 0) {
        const size_t ub = csize(op) * (size_t)M, wb = rsize(op) * (size_t)M;
        if (cudaMalloc(&uv_tmp, ub) != cudaSuccess) { cudaGetLastError(); return bail(fail(PURIFY_ERR_ALLOC, "cudaMalloc(uv) failed")); }
        if (cudaMemcpyAsync(uv_tmp, uv, ub, cudaMemcpyHostToDevice, st) != cudaSuccess) return bail(fail(PURIFY_ERR_CUDA, "H2D copy of uv failed"));
        uv_dev = uv_tmp;
        if (w) {
            if (cudaMalloc(&w_tmp, wb) != cudaSuccess) { cudaGetLastError(); return bail(fail(PURIFY_ERR_ALLOC, "cudaMalloc(w) failed")); }
            if (cudaMemcpyAsync(w_tmp, w, wb, cudaMemcpyHostToDevice, st) != cudaSuccess) return bail(fail(PURIFY_ERR_CUDA, "H2D copy of w failed"));
            w_dev = w_tmp;
        }
    }

    rc = dev_alloc(op, &op->grid, csize(op) * (size_t)op->K * op->K);
    if (rc) return bail(rc);
    if (dtype == PURIFY_C64) {
        rc = build_bins_x<float>(op, uv_dev, w_dev, st);
    } else if (J <= 6 && !(opts && opts->force_tile_sorted)) {
        rc = build_bins_x<double>(op, uv_dev, w_dev, st);
    } else {
        rc = build_bins<double>(op, uv_dev, w_dev, st);
        op->M_native = M;
    }
    if (rc) return bail(rc);
    rc = dtype == PURIFY_C64 ? build_tables<float>(op, st) : build_tables<double>(op, st);
    if (rc) return bail(rc);
    rc = build_tmap(op);
    if (rc) return bail(rc);
    {
        cufftResult r = cufftPlan2d(&op->plan, op->K, op->K, dtype == PURIFY_C64 ? CUFFT_C2C : CUFFT_Z2Z);
        if (r != CUFFT_SUCCESS) return bail(fail(r == CUFFT_ALLOC_FAILED ? PURIFY_ERR_ALLOC : PURIFY_ERR_CUFFT,
                                                 "cufftPlan2d(%d x %d) failed: cufftResult %d", op->K, op->K, (int)r));
        op->plan_ok = true;
        size_t ws = 0;
        if (cufftGetSize(op->plan, &ws) == CUFFT_SUCCESS) op->device_bytes += (long long)ws;
    }
    for (int i = 0; i < 2 * PURIFY_STAGE_COUNT; ++i) {
        if (cudaEventCreate(&op->ev[i]) != cudaSuccess) return bail(fail(PURIFY_ERR_CUDA, "cudaEventCreate failed"));
    }
    op->ev_ok = true;
    begin_call(op);
    if (cudaStreamSynchronize(st) != cudaSuccess) return bail(fail(PURIFY_ERR_CUDA, "stream synchronise failed in create"));
    cudaFree(uv_tmp);
    cudaFree(w_tmp);
    *out = op;
    return PURIFY_OK;
}

}  // namespace

// =============================================================================== C ABI
#define NEED_OP(op)                                                                 \
    do {                                                                            \
        if (!(op)) return fail(PURIFY_ERR_INVALID_ARG, "op is NULL");               \
    } while (0)
#define NEED_PTR(p, name)                                                           \
    do {                                                                            \
        if (!(p)) return fail(PURIFY_ERR_INVALID_ARG, name " is NULL");             \
    } while (0)
#define RUN(expr)                 \
    do {                          \
        int rc_ = (expr);         \
        if (rc_) return rc_;      \
    } while (0)

extern "C" {

int purify_op_create(purify_op** out, int n, int oversample, int J, long long M, const void* uv_dev,
                     const void* w_dev, int dtype, const purify_opts* opts, void* cuda_stream) {
    return create_impl(out, n, oversample, J, M, uv_dev, w_dev, false, dtype, opts, cuda_stream);
}

int purify_op_create_host(purify_op** out, int n, int oversample, int J, long long M, const void* uv_host,
                          const void* w_host, int dtype, const purify_opts* opts, void* cuda_stream) {
    return create_impl(out, n, oversample, J, M, uv_host, w_host, true, dtype, opts, cuda_stream);
}

int purify_op_destroy(purify_op* op) {
    if (!op) return PURIFY_OK;
    cudaFree(op->grid); cudaFree(op->uv_s); cudaFree(op->w_s); cudaFree(op->perm); cudaFree(op->inv_perm); cudaFree(op->loc_a); cudaFree(op->dst_a); cudaFree(op->loc_b); cudaFree(op->dst_b); cudaFree(op->loc_idx); cudaFree(op->perm_ws); cudaFree(op->scal_ws); cudaFree(op->items);
    cudaFree(op->corr); cudaFree(op->table); cudaFree(op->y_ws); cudaFree(op->x_ws); cudaFree(op->y_ws2);
    cudaFree(op->x_bhdr); cudaFree(op->x_blane); cudaFree(op->x_items); cudaFree(op->x_counter);
    for (cudaEvent_t e : op->band_ev) cudaEventDestroy(e);
    if (op->comm_done) cudaEventDestroy(op->comm_done);
    if (op->comm_stream) cudaStreamDestroy(op->comm_stream);
    if (op->normal_exec) cudaGraphExecDestroy(op->normal_exec);
    if (op->cap_stream) cudaStreamDestroy(op->cap_stream);
    if (op->plan_ok) cufftDestroy(op->plan);
    if (op->ev_ok) for (int i = 0; i < 2 * PURIFY_STAGE_COUNT; ++i) cudaEventDestroy(op->ev[i]);
    cudaGetLastError();
    delete op;
    return PURIFY_OK;
}

int purify_op_info(const purify_op* op, purify_info* info) {
    NEED_OP(op);
    NEED_PTR(info, "info");
    info->n = op->n; info->K = op->K; info->J = op->J; info->dtype = op->dtype; info->kernel_mode = op->mode;
    info->table_samples_per_unit = op->table_R; info->M = op->M; info->tile = pk::TILE; info->n_tiles = op->n_tiles;
    info->n_tiles_nonempty = op->n_tiles_nonempty; info->n_items = op->n_items; info->poly_degree = op->poly_degree;
    info->poly_max_abs_err = op->poly_err; info->device_bytes = op->device_bytes; info->max_tile_count = op->max_tile_count;
    info->M_native = op->M_native; info->n_batches = (long long)op->n_batches; info->layout = op->batched ? 1 : 0;
    if (op->batched) { info->tile = pk::XBW; info->tile_h = pk::XBH; } else { info->tile_h = pk::TILE; }
    return PURIFY_OK;
}

int purify_op_permutation(const purify_op* op, const unsigned** perm_dev) {
    NEED_OP(op);
    NEED_PTR(perm_dev, "perm_dev");
    *perm_dev = op->perm;
    return PURIFY_OK;
}

// The complex64 (batched) kernels work in native order only; caller order is one extra permutation
// pass through the handle's native-order workspace (faster than scattering from inside the kernel).
static int degrid_impl(purify_op* op, const void* x, void* y, bool caller_order, cudaStream_t st) {
    RUN(launch_pad(op, x, st));
    RUN(launch_fft(op, CUFFT_FORWARD, st));
    if (op->batched && caller_order) {
        RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
        RUN(launch_degrid(op, op->y_ws, false, st));
        return launch_permute(op, op->y_ws, y, 0, st);
    }
    RUN(launch_degrid(op, y, caller_order, st));
    return PURIFY_OK;
}

static int grid_impl(purify_op* op, const void* y, void* x, bool caller_order, cudaStream_t st) {
    if (op->batched && caller_order) {
        RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
        RUN(launch_permute(op, y, op->y_ws, 1, st));
        y = op->y_ws;
        caller_order = false;
    }
    RUN(launch_grid(op, y, caller_order, st));
    RUN(launch_fft(op, CUFFT_INVERSE, st));
    RUN(launch_crop(op, x, st));
    return PURIFY_OK;
}

int purify_degrid(purify_op* op, const void* x_dev, void* y_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); if (op->M > 0) NEED_PTR(y_dev, "y");
    begin_call(op);
    return degrid_impl(op, x_dev, y_dev, true, (cudaStream_t)cuda_stream);
}

int purify_degrid_native(purify_op* op, const void* x_dev, void* y_native_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); if (op->M > 0) NEED_PTR(y_native_dev, "y");
    begin_call(op);
    return degrid_impl(op, x_dev, y_native_dev, false, (cudaStream_t)cuda_stream);
}

int purify_grid(purify_op* op, const void* y_dev, void* x_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); if (op->M > 0) NEED_PTR(y_dev, "y");
    begin_call(op);
    return grid_impl(op, y_dev, x_dev, true, (cudaStream_t)cuda_stream);
}

int purify_grid_native(purify_op* op, const void* y_native_dev, void* x_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); if (op->M > 0) NEED_PTR(y_native_dev, "y");
    if (op->batched && ((uintptr_t)y_native_dev & 15u))       // the kernel streams y with 16-byte-aligned bulk copies
        return fail(PURIFY_ERR_INVALID_ARG, "y_native must be 16-byte aligned for the batched layout");
    begin_call(op);
    return grid_impl(op, y_native_dev, x_dev, false, (cudaStream_t)cuda_stream);
}

// The step of an ADMM iteration / power iteration.  Its seven launches (S+Z, F, W G, memset, G^dagger W^dagger,
// F^dagger, Z^dagger S^dagger) are captured ONCE per (x_in, x_out) pair into a CUDA graph - on an internal stream,
// because the caller's may be the legacy default stream, which cannot capture - and replayed on the caller's stream.
// Stage timing needs events between the launches: with it switched on the launches are issued one by one.
static int normal_eager(purify_op* op, const void* x_in, void* x_out, cudaStream_t st) {
    RUN(degrid_impl(op, x_in, op->y_ws, false, st));
    RUN(grid_impl(op, op->y_ws, x_out, false, st));
    return PURIFY_OK;
}

int purify_normal(purify_op* op, const void* x_in_dev, void* x_out_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_in_dev, "x_in"); NEED_PTR(x_out_dev, "x_out");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
    if (op->time_stages || op->graph_failed) return normal_eager(op, x_in_dev, x_out_dev, st);
    if (!op->normal_exec || op->graph_stale || op->normal_in != x_in_dev || op->normal_out != x_out_dev) {
        if (op->normal_exec) { cudaGraphExecDestroy(op->normal_exec); op->normal_exec = nullptr; }
        if (!op->cap_stream && cudaStreamCreateWithFlags(&op->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError(); op->cap_stream = nullptr; op->graph_failed = true;
            return normal_eager(op, x_in_dev, x_out_dev, st);
        }
        // first use of every kernel instantiation outside the capture (occupancy queries, attributes, lazy module load)
        if (!op->normal_warm || op->graph_stale) {
            RUN(normal_eager(op, x_in_dev, x_out_dev, st));
            op->normal_warm = true; op->graph_stale = false;
            return PURIFY_OK;                           // (this call is done; the next one captures)
        }
        cudaGraph_t g = nullptr;
        bool ok = cudaStreamBeginCapture(op->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        int rc = PURIFY_OK;
        if (ok) {
            const int l0 = op->launches;
            rc = normal_eager(op, x_in_dev, x_out_dev, op->cap_stream);
            op->normal_launches = op->launches - l0;
            op->launches = l0;
            ok = cudaStreamEndCapture(op->cap_stream, &g) == cudaSuccess && rc == PURIFY_OK && g;
        }
        if (ok) ok = cudaGraphInstantiate(&op->normal_exec, g, 0) == cudaSuccess;
        if (g) cudaGraphDestroy(g);
        cufftSetStream(op->plan, st);
        if (!ok) {                                      // no graph on this system: issue the launches one by one from now on
            cudaGetLastError();
            op->normal_exec = nullptr; op->graph_failed = true;
            return normal_eager(op, x_in_dev, x_out_dev, st);
        }
        op->normal_in = x_in_dev; op->normal_out = x_out_dev;
    }
    CK(cudaGraphLaunch(op->normal_exec, st));
    op->launches += op->normal_launches;
    return PURIFY_OK;
}

// ---- f3: the distributed-image operator (Eq. 37-38; Algorithm 2).  Every rank
// holds its own visibilities and a replica of x; Phi needs no exchange; Phi^dagger ends with the sum over ranks of
// the n x n images.  The exchange itself is the caller's (NCCL, MPI, ...): the library hands the image to
// `allreduce` in `bands` horizontal bands as they leave the crop kernel - band k is being reduced on the handle's side
// stream while band k + 1 is cropped on the caller's stream - and makes the caller's stream wait for the last one.
static int grid_dist_tail(purify_op* op, void* x, int bands, purify_allreduce_fn allreduce, void* user, cudaStream_t st) {
    if (bands < 1) bands = 1;
    if (bands > op->n) bands = op->n;
    if (!allreduce) return launch_crop(op, x, st);
    if (!op->comm_stream) CK(cudaStreamCreateWithFlags(&op->comm_stream, cudaStreamNonBlocking));
    if (!op->comm_done) CK(cudaEventCreateWithFlags(&op->comm_done, cudaEventDisableTiming));
    while ((int)op->band_ev.size() < bands) {
        cudaEvent_t e;
        CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        op->band_ev.push_back(e);
    }
    const size_t row_bytes = csize(op) * (size_t)op->n;
    if (op->time_stages && op->ev_ok) { cudaEventRecord(op->ev[2 * PURIFY_STAGE_CROP], st); op->stage_ran[PURIFY_STAGE_CROP] = true; }
    for (int k = 0; k < bands; ++k) {
        const int r0 = (int)((long long)op->n * k / bands), r1 = (int)((long long)op->n * (k + 1) / bands);
        RUN(launch_crop(op, x, st, r0, r1, false));
        CK(cudaEventRecord(op->band_ev[k], st));
        CK(cudaStreamWaitEvent(op->comm_stream, op->band_ev[k], 0));
        const int rc = allreduce(user, (char*)x + row_bytes * (size_t)r0, (long long)(r1 - r0) * op->n * 2,
                                 op->dtype == PURIFY_C128, (void*)op->comm_stream);
        if (rc != 0) return fail(PURIFY_ERR_CUDA, "the all-reduce callback failed on band %d (returned %d)", k, rc);
    }
    CK(cudaEventRecord(op->comm_done, op->comm_stream));
    CK(cudaStreamWaitEvent(st, op->comm_done, 0));
    if (op->time_stages && op->ev_ok) cudaEventRecord(op->ev[2 * PURIFY_STAGE_CROP + 1], st);      // crop + exchange
    return PURIFY_OK;
}

int purify_grid_dist(purify_op* op, const void* y_native_dev, void* x_dev, int bands, purify_allreduce_fn allreduce,
                     void* user, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); if (op->M > 0) NEED_PTR(y_native_dev, "y");
    if (op->batched && ((uintptr_t)y_native_dev & 15u))
        return fail(PURIFY_ERR_INVALID_ARG, "y_native must be 16-byte aligned for the batched layout");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RUN(launch_grid(op, y_native_dev, false, st));
    RUN(launch_fft(op, CUFFT_INVERSE, st));
    return grid_dist_tail(op, x_dev, bands, allreduce, user, st);
}

int purify_normal_dist(purify_op* op, const void* x_in_dev, void* x_out_dev, int bands, purify_allreduce_fn allreduce,
                       void* user, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_in_dev, "x_in"); NEED_PTR(x_out_dev, "x_out");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
    RUN(degrid_impl(op, x_in_dev, op->y_ws, false, st));
    RUN(launch_grid(op, op->y_ws, false, st));
    RUN(launch_fft(op, CUFFT_INVERSE, st));
    return grid_dist_tail(op, x_out_dev, bands, allreduce, user, st);
}

int purify_permute_to_native(purify_op* op, const void* y_caller_dev, void* y_native_dev, void* cuda_stream) {
    NEED_OP(op); if (op->M > 0) { NEED_PTR(y_caller_dev, "y_caller"); NEED_PTR(y_native_dev, "y_native"); }
    begin_call(op);
    return launch_permute(op, y_caller_dev, y_native_dev, 1, (cudaStream_t)cuda_stream);
}

int purify_permute_from_native(purify_op* op, const void* y_native_dev, void* y_caller_dev, void* cuda_stream) {
    NEED_OP(op); if (op->M > 0) { NEED_PTR(y_caller_dev, "y_caller"); NEED_PTR(y_native_dev, "y_native"); }
    begin_call(op);
    return launch_permute(op, y_native_dev, y_caller_dev, 0, (cudaStream_t)cuda_stream);
}

// ---- host-buffer entry points (end-to-end path: H2D + operator + D2H inside the call)
int purify_degrid_host(purify_op* op, const void* x_host, void* y_host, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_host, "x"); if (op->M > 0) NEED_PTR(y_host, "y");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t xb = csize(op) * (size_t)op->n * op->n, yb = csize(op) * (size_t)op->M;
    RUN(WS_X(op, xb));
    RUN(WS_Y2(op, yb));
    CK(cudaMemcpyAsync(op->x_ws, x_host, xb, cudaMemcpyHostToDevice, st));
    RUN(degrid_impl(op, op->x_ws, op->y_ws2, true, st));
    if (yb) CK(cudaMemcpyAsync(y_host, op->y_ws2, yb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return PURIFY_OK;
}

int purify_grid_host(purify_op* op, const void* y_host, void* x_host, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_host, "x"); if (op->M > 0) NEED_PTR(y_host, "y");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t xb = csize(op) * (size_t)op->n * op->n, yb = csize(op) * (size_t)op->M;
    RUN(WS_X(op, xb));
    RUN(WS_Y2(op, yb));
    if (yb) CK(cudaMemcpyAsync(op->y_ws2, y_host, yb, cudaMemcpyHostToDevice, st));
    RUN(grid_impl(op, op->y_ws2, op->x_ws, true, st));
    CK(cudaMemcpyAsync(x_host, op->x_ws, xb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return PURIFY_OK;
}

int purify_normal_host(purify_op* op, const void* x_in_host, void* x_out_host, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_in_host, "x_in"); NEED_PTR(x_out_host, "x_out");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t xb = csize(op) * (size_t)op->n * op->n;
    RUN(WS_X(op, xb));
    RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
    CK(cudaMemcpyAsync(op->x_ws, x_in_host, xb, cudaMemcpyHostToDevice, st));
    RUN(degrid_impl(op, op->x_ws, op->y_ws, false, st));
    RUN(grid_impl(op, op->y_ws, op->x_ws, false, st));
    CK(cudaMemcpyAsync(x_out_host, op->x_ws, xb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return PURIFY_OK;
}

// ---- f2: operator norm by the power method
int purify_op_norm(purify_op* op, const void* x0_dev, int max_iter, double rel_tol, double* lambda_out, int* iters_out,
                   void* cuda_stream) {
    NEED_OP(op); NEED_PTR(lambda_out, "lambda_out");
    if (max_iter < 1) return fail(PURIFY_ERR_INVALID_ARG, "max_iter must be >= 1 (got %d)", max_iter);
    if (!(rel_tol >= 0.0)) return fail(PURIFY_ERR_INVALID_ARG, "rel_tol must be >= 0");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long N = (long long)op->n * op->n;
    const size_t xb = csize(op) * (size_t)N;
    RUN(WS_X(op, xb));
    RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
    RUN(WS_SCAL(op));
    const bool f32 = op->dtype == PURIFY_C64;
    auto norm2 = [&](const void* v, double* host) -> int {
        CK(cudaMemsetAsync(op->scal_ws, 0, sizeof(double), st));
        if (f32) pk::norm2_kernel<float><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((const float2*)v, N, op->scal_ws);
        else pk::norm2_kernel<double><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((const double2*)v, N, op->scal_ws);
        op->launches++;
        CK(cudaGetLastError());
        if (host) { CK(cudaMemcpyAsync(host, op->scal_ws, sizeof(double), cudaMemcpyDeviceToHost, st)); CK(cudaStreamSynchronize(st)); }
        return PURIFY_OK;
    };
    auto normalise = [&]() -> int {                    // x_ws <- x_ws / sqrt(scal_ws)
        if (f32) pk::normalise_kernel<float><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((const float2*)op->x_ws, (float2*)op->x_ws, N, op->scal_ws);
        else pk::normalise_kernel<double><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((const double2*)op->x_ws, (double2*)op->x_ws, N, op->scal_ws);
        op->launches++;
        CK(cudaGetLastError());
        return PURIFY_OK;
    };
    // start vector: the caller's, or all ones
    if (x0_dev) {
        CK(cudaMemcpyAsync(op->x_ws, x0_dev, xb, cudaMemcpyDeviceToDevice, st));
    } else {
        if (f32) pk::fill_ones_kernel<float><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((float2*)op->x_ws, N);
        else pk::fill_ones_kernel<double><<<grid_for(N, 256, 148 * 8), 256, 0, st>>>((double2*)op->x_ws, N);
        op->launches++;
        CK(cudaGetLastError());
    }
    double lambda = 0.0, prev = 0.0, n2 = 0.0;
    int it = 0;
    RUN(norm2(op->x_ws, &n2));
    if (!(n2 > 0.0)) return fail(PURIFY_ERR_INVALID_ARG, "power method: the start vector is zero or not finite");
    for (it = 1; it <= max_iter; ++it) {
        RUN(normalise());                               // ||x|| = 1
        RUN(degrid_impl(op, op->x_ws, op->y_ws, false, st));
        RUN(grid_impl(op, op->y_ws, op->x_ws, false, st));       // x <- Phi^dagger Phi x
        // the host only needs lambda_k for the stopping rule (or after the last iteration): no sync otherwise
        const bool need = rel_tol > 0.0 || it == max_iter;
        RUN(norm2(op->x_ws, need ? &n2 : nullptr));
        if (!need) continue;
        prev = lambda;
        lambda = sqrt(n2);                              // ||Phi^dagger Phi x|| with ||x|| = 1 -> largest eigenvalue
        if (!(lambda > 0.0) || (it > 1 && fabs(lambda - prev) <= rel_tol * lambda)) break;
    }
    if (it > max_iter) it = max_iter;
    *lambda_out = lambda;
    if (iters_out) *iters_out = it;
    return PURIFY_OK;
}

// ---- f1: data-fidelity half of one ADMM iteration (Algorithm 1 lines 3-6), native-order vectors
int purify_admm_fidelity_step(purify_op* op, const void* x_dev, const void* y_native_dev, void* s_native_dev, double epsilon,
                              double varrho, void* g_dev, double* resid_norm_out, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); NEED_PTR(g_dev, "g");
    if (op->M > 0) { NEED_PTR(y_native_dev, "y_native"); NEED_PTR(s_native_dev, "s_native"); }
    if (!(epsilon >= 0.0)) return fail(PURIFY_ERR_INVALID_ARG, "epsilon must be >= 0");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long Mn = op->M_native;
    RUN(WS_Y(op, csize(op) * (size_t)Mn));
    RUN(WS_SCAL(op));
    if (op->batched && op->dtype == PURIFY_C64 && op->mode == PURIFY_KERNEL_ANALYTIC && !op->admm_unfused) {
        // fused form: the norm is accumulated inside the degridding kernel, r / s_new / z are formed slot by slot inside
        // the gridding kernel (z is never stored); two passes over the M-sized vectors less than the unfused form below
        if (((uintptr_t)y_native_dev & 15u) || ((uintptr_t)s_native_dev & 15u))
            return fail(PURIFY_ERR_INVALID_ARG, "y_native and s_native must be 16-byte aligned for the complex64 layout");
        const AdmmArgs aa = {y_native_dev, s_native_dev, epsilon, varrho};
        CK(cudaMemsetAsync(op->scal_ws, 0, sizeof(double), st));
        RUN(launch_pad(op, x_dev, st));
        RUN(launch_fft(op, CUFFT_FORWARD, st));
        RUN(launch_degrid_fused(op, op->y_ws, aa, st));
        RUN(launch_grid_fused(op, op->y_ws, aa, st));
        RUN(launch_fft(op, CUFFT_INVERSE, st));
        RUN(launch_crop(op, g_dev, st));
        if (resid_norm_out) {
            double n2 = 0.0;
            CK(cudaMemcpyAsync(&n2, op->scal_ws, sizeof(double), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            *resid_norm_out = sqrt(n2);
        }
        return PURIFY_OK;
    }
    RUN(WS_Y2(op, csize(op) * (size_t)(Mn > op->M ? Mn : op->M)));      // z = v - r + s_new, M_native entries
    const unsigned* pm = op->batched ? op->perm : nullptr;     // padding mask (batched layout only)
    // line 3: v = Phi x
    RUN(degrid_impl(op, x_dev, op->y_ws, false, st));
    // line 4: ||v + s - y||^2 (fp64 accumulation)
    CK(cudaMemsetAsync(op->scal_ws, 0, sizeof(double), st));
    if (Mn > 0) {
        if (op->dtype == PURIFY_C64)
            pk::admm_norm2_kernel<float><<<grid_for(Mn, 256, 148 * 8), 256, 0, st>>>((const float2*)op->y_ws, (const float2*)s_native_dev,
                                                                                    (const float2*)y_native_dev, pm, Mn, op->scal_ws);
        else
            pk::admm_norm2_kernel<double><<<grid_for(Mn, 256, 148 * 8), 256, 0, st>>>((const double2*)op->y_ws, (const double2*)s_native_dev,
                                                                                     (const double2*)y_native_dev, pm, Mn, op->scal_ws);
        op->launches++;
        CK(cudaGetLastError());
        // lines 4-6: r, s <- s + varrho (v - r), z = v - r + s
        if (op->dtype == PURIFY_C64)
            pk::admm_update_kernel<float><<<grid_for(Mn, 256, 148 * 16), 256, 0, st>>>((const float2*)op->y_ws, (float2*)s_native_dev,
                                                                                      (const float2*)y_native_dev, pm, Mn, op->scal_ws,
                                                                                      epsilon, varrho, (float2*)op->y_ws2);
        else
            pk::admm_update_kernel<double><<<grid_for(Mn, 256, 148 * 16), 256, 0, st>>>((const double2*)op->y_ws, (double2*)s_native_dev,
                                                                                       (const double2*)y_native_dev, pm, Mn, op->scal_ws,
                                                                                       epsilon, varrho, (double2*)op->y_ws2);
        op->launches++;
        CK(cudaGetLastError());
    }
    // line 6: g = Phi^dagger (v - r + s)
    RUN(grid_impl(op, op->y_ws2, g_dev, false, st));
    if (resid_norm_out) {
        double n2 = 0.0;
        CK(cudaMemcpyAsync(&n2, op->scal_ws, sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        *resid_norm_out = sqrt(n2);
    }
    return PURIFY_OK;
}

// ---- single stages in the mathematical layout (tests)
static int relayout(purify_op* op, const void* in, void* out, cudaStream_t st) {
    const long long tot = (long long)op->K * op->K;
    if (op->dtype == PURIFY_C64)
        pk::relayout_kernel<float><<<grid_for(tot, 256, 148 * 32), 256, 0, st>>>((const float2*)in, (float2*)out, op->K, 1);
    else
        pk::relayout_kernel<double><<<grid_for(tot, 256, 148 * 32), 256, 0, st>>>((const double2*)in, (double2*)out, op->K, 1);
    op->launches++;
    CK(cudaGetLastError());
    return PURIFY_OK;
}

int purify_stage_fourier_grid(purify_op* op, const void* x_dev, void* B_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(x_dev, "x"); NEED_PTR(B_dev, "B");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RUN(launch_pad(op, x_dev, st));
    RUN(launch_fft(op, CUFFT_FORWARD, st));
    return relayout(op, op->grid, B_dev, st);
}

int purify_stage_gridded(purify_op* op, const void* y_dev, void* B_dev, void* cuda_stream) {
    NEED_OP(op); NEED_PTR(B_dev, "B"); if (op->M > 0) NEED_PTR(y_dev, "y");
    begin_call(op);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (op->batched) {
        RUN(WS_Y(op, csize(op) * (size_t)op->M_native));
        RUN(launch_permute(op, y_dev, op->y_ws, 1, st));
        RUN(launch_grid(op, op->y_ws, false, st));
    } else {
        RUN(launch_grid(op, y_dev, true, st));
    }
    return relayout(op, op->grid, B_dev, st);
}

int purify_stage_times_ms(const purify_op* op, float out[PURIFY_STAGE_COUNT]) {
    NEED_OP(op); NEED_PTR(out, "out");
    for (int i = 0; i < PURIFY_STAGE_COUNT; ++i) out[i] = 0.f;
    if (!op->time_stages || !op->ev_ok) return fail(PURIFY_ERR_INVALID_ARG, "handle was created without opts.time_stages");
    CK(cudaDeviceSynchronize());
    for (int i = 0; i < PURIFY_STAGE_COUNT; ++i)
        if (op->stage_ran[i]) CK(cudaEventElapsedTime(&out[i], op->ev[2 * i], op->ev[2 * i + 1]));
    return PURIFY_OK;
}

int purify_op_set_time_stages(purify_op* op, int enable) {
    NEED_OP(op);
    op->time_stages = enable != 0;
    return PURIFY_OK;
}

int purify_last_launch_count(const purify_op* op) { return op ? op->launches : 0; }

// ---- issue-rate probe of the packed fp32 instruction forms (csrc/ubench.cuh)
int purify_ubench_fma(int form, int warps_per_sm, double* cycles_per_instr_out, double* sm_ghz_out) {
    NEED_PTR(cycles_per_instr_out, "cycles_per_instr_out");
    if (form < 0 || form > 4) return fail(PURIFY_ERR_INVALID_ARG, "form must be in [0, 4] (got %d)", form);
    if (warps_per_sm < 4 || warps_per_sm > 32 || (warps_per_sm & 3)) return fail(PURIFY_ERR_INVALID_ARG, "warps_per_sm must be 4, 8, ..., 32");
    RUN(check_device());
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* out = nullptr; long long* cyc = nullptr;
    CK(cudaMalloc(&out, sizeof(float) * (size_t)sms * 1024));
    if (cudaMalloc(&cyc, sizeof(long long) * (size_t)sms) != cudaSuccess) { cudaFree(out); cudaGetLastError(); return fail(PURIFY_ERR_ALLOC, "cudaMalloc failed"); }
    const int iters = 4000, threads = warps_per_sm * 32;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto launch = [&](int n) {
        switch (form) {
            case 0: pk::ubench_fma_kernel<0><<<sms, threads>>>(out, cyc, n, 1.0001f, 0.3f); break;
            case 1: pk::ubench_fma_kernel<1><<<sms, threads>>>(out, cyc, n, 1.0001f, 0.3f); break;
            case 2: pk::ubench_fma_kernel<2><<<sms, threads>>>(out, cyc, n, 1.0001f, 0.3f); break;
            case 3: pk::ubench_fma_kernel<3><<<sms, threads>>>(out, cyc, n, 1.0001f, 0.3f); break;
            default: pk::ubench_fma_kernel<4><<<sms, threads>>>(out, cyc, n, 1.0001f, 0.3f); break;
        }
    };
    launch(10);
    cudaEventRecord(e0);
    launch(iters);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    std::vector<long long> h((size_t)sms);
    if (e == cudaSuccess) e = cudaMemcpy(h.data(), cyc, sizeof(long long) * (size_t)sms, cudaMemcpyDeviceToHost);
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out); cudaFree(cyc);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(PURIFY_ERR_CUDA, "ubench failed: %s", cudaGetErrorString(e)); }
    double c = 0;
    for (int i = 0; i < sms; ++i) c += (double)h[i];
    c /= sms;
    // instructions per SM sub-partition: every warp issues iters x REP x NA instructions (form 0: two scalar FFMA each)
    const double per_smsp = (double)iters * pk::UB_REP * pk::UB_NA * (form == 0 ? 2.0 : 1.0) * (warps_per_sm / 4.0);
    *cycles_per_instr_out = c / per_smsp;
    if (sm_ghz_out) *sm_ghz_out = ms > 0.f ? c / (ms * 1e6) : 0.0;
    return PURIFY_OK;
}

const char* purify_strerror(int status) {
    switch (status) {
        case PURIFY_OK: return "ok";
        case PURIFY_ERR_INVALID_ARG: return "invalid argument";
        case PURIFY_ERR_UNSUPPORTED: return "unsupported configuration";
        case PURIFY_ERR_UV_NONFINITE: return "non-finite or out-of-range (u, v) coordinate";
        case PURIFY_ERR_ALLOC: return "allocation failed";
        case PURIFY_ERR_CUDA: return "CUDA error";
        case PURIFY_ERR_CUFFT: return "cuFFT error";
        case PURIFY_ERR_NO_DEVICE: return "no CUDA device (no CPU fallback)";
        default: return "unknown status";
    }
}

const char* purify_last_error(void) { return g_err; }
int purify_version(void) { return 100; }

}  // extern "C"
