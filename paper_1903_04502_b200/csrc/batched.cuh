// complex64 hot path: the "cell-stationary" batched layout and its create-time construction (a0).
//
// Why (profiles/r1a_summary.md): with one thread per visibility both W G and its adjoint are bound
// by the fp32 pipe / issue rate, not by HBM (235 lane-instructions per visibility at J = 6), and the
// adjoint additionally pays shared-memory read-modify-writes per visibility.  Here a THREAD OWNS A
// GRID CELL for a run of visibilities: degridding keeps the cell's J x J patch of the Fourier grid
// in registers, gridding keeps the J x J accumulators in registers, and the inner loop over the
// run's visibilities touches no grid data in shared memory at all.  The 2J^2 complex x real MACs
// and the paired Horner chains of the kernel weights are issued as packed fp32 (FFMA2, sm_100).
//
// Layout (built once at create):
//   band   32 x 16 cells of the oversampled grid (internal DC-centred layout); one WARP works on one
//          band at a time with a private (16+J-1) x (32+J) shared-memory box.
//   unit   up to UNIT_CAP (128) visibilities of ONE cell.  A cell with c visibilities gives floor(c/CAP)
//          full units and one remainder unit.
//   batch  32 consecutive units of the band's unit sequence, one per lane, processed in lockstep for
//          n_iter = (count of the batch's first unit) iterations.  The sequence is: the full units in
//          layer-major order (layer j = the j-th full unit of every cell that has one, cells
//          ascending), then the remainder units by descending count - so counts never increase along
//          the sequence, the counts inside a batch are nearly equal (padding a few per cent), and two
//          units of the same cell can only meet in a batch that straddles a layer boundary (flagged:
//          the adjoint then flushes with shared-memory atomics instead of plain read-modify-writes).
//   slots  visibility data in "native order": slot = 32*(iter0 + i) + lane for iteration i of a
//          batch.  Slots past a unit's count are padding: perm = 0xFFFFFFFF, w = 0, uv = the unit's
//          first visibility, y_native = 0.  The per-slot inputs are stored as one record per
//          ITERATION: 32 x (u, v) then 32 x w = 384 bytes, so a chunk of iterations is ONE bulk copy.
//   item   a run of batches of one band with about ITEM_ITERS (64) iterations: the unit of dynamic
//          scheduling (persistent warps pull items from an atomic counter); its slots are contiguous.
//
// Kernels: degrid_x_kernel (a3) and grid_x_kernel (a4), templated on the taps J, the polynomial
// degree, the weight MODE (0 analytic polynomial, 1 table in global memory, 2 table in shared memory), the ring
// geometry (CH iterations per chunk, S stages) and FUSE (1: the ADMM data-fidelity step of Algorithm 1 lines 3-6 is
// folded in - residual norm in a3; projection, dual update and residual in a4).
#pragma once
#include "kernels.cuh"

namespace pk {

constexpr int XBW = 32, XBH = 16, XCELLS = XBW * XBH;   // band geometry
constexpr int UNIT_CAP = 128;                           // visibilities per unit
constexpr int ITEM_ITERS = 64;                          // iterations per item
constexpr unsigned PERM_PAD = 0xFFFFFFFFu;
constexpr int REC_FLOATS = 96, REC_BYTES = 384;         // per-iteration record: uv[32] | w[32]
// visibilities per inner-loop trip (statement-interleaved dependency graphs): degridding gains from 2 (0.73 ->
// 0.69 ms at config 4, 160 registers, 3 CTAs / SM); gridding loses (its flush phases want the 4th CTA)
constexpr int XVD = 2, XVG6 = 1, XVG4 = 1;

template <int J> struct XCfg {
    static constexpr int XOFF = (J / 2 - 1) & 1;        // makes the box's first column even (TMA: 16-byte aligned)
    static constexpr int BOXW = XBW + J;                // columns (even)
    static constexpr int BOXH = XBH + J - 1;            // rows
    static constexpr int REGION_BYTES = ((BOXW * BOXH * 8 + 127) / 128) * 128;
    static constexpr int WARPS = 4;
    static constexpr int THREADS = WARPS * 32;
};

struct XItem {
    int x0, y0;          // band origin, internal layout
    int begin, end;      // batch range
    unsigned iter0;      // first iteration (slot / 32) of the item: its slots are one contiguous stream
    unsigned iters;      // number of iterations (sum of n_iter over the item's batches)
    int pad0, pad1;
};

template <typename F> struct XParamsT {
    typedef typename Cplx<F>::type F2;
    F2* grid;                 // K*K, internal layout
    int K, Kh, kmask;
    const XItem* items;
    int n_items;
    unsigned* counter;            // [0] dynamic item queue, [1] warps finished: the last warp to leave zeroes both
    int n_warps;                  // persistent warps of this launch
    const uint2* bhdr;            // per batch: x = first iteration, y = n_iter | flags << 16 (bit 0: a cell may occur twice)
    const unsigned* blane;        // per batch 32 lane words: cell (ly << 5 | lx) | count << 16
    const F* rec;             // per-iteration records (REC_FLOATS floats each)
    KbCoef<F> coef;
    const F* table;
    F table_R;
    int table_len;
    // f1 (fused ADMM data-fidelity step): dual variable s (in / out), measurements y, ||v + s - y||^2, radius, step
    const F2* s_in;
    const F2* yobs;
    F2* s_out;
    double* norm2;
    double eps, varrho;
};
typedef XParamsT<float> XParams;

// ---------------------------------------------------------------------------------------------
// a0.1: reduce (u, v) to the principal period, key = band * 512 + cell (band-major).
template <typename F>
__global__ void xkey_kernel(const typename Cplx<F>::type* __restrict__ uv, long long M, int K, int nbx,
                            unsigned* __restrict__ keys, unsigned* __restrict__ idx, int* __restrict__ bad) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const typename Cplx<F>::type c = uv[k];
        unsigned key = 0;
        if (!(fabs(c.x) < (F)1073741824.0) || !(fabs(c.y) < (F)1073741824.0)) {
            atomicOr(bad, 1);
        } else {
            const long long fx = (long long)floor_r(c.x) + K / 2, fy = (long long)floor_r(c.y) + K / 2;
            long long gx = fx % K, gy = fy % K;
            if (gx < 0) gx += K;
            if (gy < 0) gy += K;
            const unsigned band = (unsigned)(gy / XBH) * nbx + (unsigned)(gx / XBW);
            key = band * XCELLS + (unsigned)(gy % XBH) * XBW + (unsigned)(gx % XBW);
        }
        keys[k] = key;
        idx[k] = (unsigned)k;
    }
}

// principal-period coordinate: u - m K with m = floor((floor(u) + K/2) / K); exact (double arithmetic,
// the result is a multiple of ulp(u) of small magnitude, hence representable).
template <typename F> __device__ __forceinline__ F x_reduce(F u, int K) {
    const long long f = (long long)floor_r(u) + K / 2;
    long long m = f / K;
    if (f % K < 0) --m;
    return (F)((double)u - (double)m * (double)K);
}

__global__ void band_start_kernel(const unsigned* __restrict__ keys, long long M, int n_bands, unsigned* __restrict__ band_start) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > n_bands) return;
    const unsigned long long target = (unsigned long long)t * XCELLS;
    long long lo = 0, hi = M;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if ((unsigned long long)keys[mid] < target) lo = mid + 1; else hi = mid;
    }
    band_start[t] = (unsigned)lo;
}

// ---------------------------------------------------------------------------------------------
// a0.2 / a0.3: per-band batch construction.  One CTA of 512 threads per band, thread t <-> cell t
// (ly = t >> 5, lx = t & 31).  PASS 1 counts batches / iterations / items, PASS 2 (after the
// exclusive scans over bands) writes batch headers, lane words, unit sources and items.
struct BandTotals { unsigned nb, iters, items; };

template <int PASS>
__global__ void __launch_bounds__(XCELLS)
band_build_kernel(const unsigned* __restrict__ keys, const unsigned* __restrict__ band_start, int nbx, int boxw,
                  BandTotals* __restrict__ totals,                      // PASS 1 out
                  const unsigned* __restrict__ nb_off, const unsigned* __restrict__ iter_off,
                  const unsigned* __restrict__ item_off,                // PASS 2 in (exclusive scans)
                  uint2* __restrict__ bhdr, unsigned* __restrict__ blane, unsigned* __restrict__ lsrc,
                  XItem* __restrict__ items) {
    __shared__ unsigned s_rem[XCELLS], s_remsorted[XCELLS], s_scan[XCELLS], s_ni[XCELLS];
    __shared__ unsigned s_w[XCELLS / 32];
    __shared__ unsigned s_F, s_Rn, s_maxfull, s_carry, s_lastni, s_icarry;

    const int band = blockIdx.x;
    const unsigned bs = band_start[band], be = band_start[band + 1];
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
    if (bs == be) {
        if (PASS == 1 && t == 0) { totals[band].nb = 0; totals[band].iters = 0; totals[band].items = 0; }
        return;
    }
    if (t == 0) { s_F = 0; s_Rn = 0; s_maxfull = 0; s_carry = 0; s_lastni = 0; s_icarry = 0; }
    // --- this cell's visibilities: [start, start + cnt) of the sorted order
    unsigned start, cnt;
    {
        const unsigned k0 = (unsigned)band * XCELLS + (unsigned)t;
        unsigned lo = bs, hi = be;
        while (lo < hi) { const unsigned mid = lo + ((hi - lo) >> 1); if (keys[mid] < k0) lo = mid + 1; else hi = mid; }
        unsigned lo2 = lo, hi2 = be;
        while (lo2 < hi2) { const unsigned mid = lo2 + ((hi2 - lo2) >> 1); if (keys[mid] <= k0) lo2 = mid + 1; else hi2 = mid; }
        start = lo;
        cnt = lo2 - lo;
    }
    const unsigned myfull = cnt / UNIT_CAP, myrem = cnt % UNIT_CAP;
    s_rem[t] = myrem;
    __syncthreads();
    if (myfull) { atomicAdd(&s_F, myfull); atomicMax(&s_maxfull, myfull); }
    if (myrem) atomicAdd(&s_Rn, 1u);
    // rank of the remainder unit: descending count (zeros sort last).  Units of EQUAL count are ordered so that 32
    // consecutive ones spread over the 16 shared-memory bank classes: by their index among the cells of the same count
    // and class first, then by class, then by cell.  (Which equal-count unit lands in which batch costs no padding.)
    const unsigned mycls = (((unsigned)t >> 5) * (unsigned)boxw + ((unsigned)t & 31u)) & 15u;
    unsigned ric = 0;
    for (int q = 0; q < t; ++q) {
        const unsigned cq = (((unsigned)q >> 5) * (unsigned)boxw + ((unsigned)q & 31u)) & 15u;
        ric += (s_rem[q] == myrem && cq == mycls) ? 1u : 0u;
    }
    const unsigned mykey = ((unsigned)(UNIT_CAP - myrem) << 19) | (ric << 13) | (mycls << 9) | (unsigned)t;
    s_scan[t] = mykey;                                   // (s_scan is free until the batch scan below)
    __syncthreads();
    unsigned rank = 0;
    for (int q = 0; q < XCELLS; ++q) rank += s_scan[q] < mykey ? 1u : 0u;
    __syncthreads();
    s_remsorted[rank] = myrem;
    __syncthreads();
    const unsigned F = s_F, Rn = s_Rn, maxfull = s_maxfull;
    const unsigned Q = F + Rn, NB = (Q + 31) >> 5;
    // n_iter of batch b = count of its first unit (counts never increase along the sequence)
    auto batch_iters = [&](unsigned b) -> unsigned { return 32u * b < F ? (unsigned)UNIT_CAP : s_remsorted[32u * b - F]; };

    const unsigned nb0 = PASS == 2 ? nb_off[band] : 0, it0 = PASS == 2 ? iter_off[band] : 0,
                   item0 = PASS == 2 ? item_off[band] : 0;
    const int x0 = (band % nbx) * XBW, y0 = (band / nbx) * XBH;

    // --- batches: n_iter, prefix of iterations, item boundaries (chunks of 512 batches).  A batch opens a new
    // item when the iterations before it cross a multiple of ITEM_ITERS; items are numbered by a scan of these flags.
    auto block_scan = [&](unsigned v) -> unsigned {          // inclusive scan over the CTA's 512 threads
        s_scan[t] = v;
        __syncthreads();
        for (int off = 1; off < XCELLS; off <<= 1) {
            const unsigned u = t >= off ? s_scan[t - off] : 0;
            __syncthreads();
            s_scan[t] += u;
            __syncthreads();
        }
        const unsigned r = s_scan[t];
        __syncthreads();
        return r;
    };
    unsigned total_iters = 0;
    for (unsigned base = 0; base < NB; base += XCELLS) {
        const unsigned b = base + t;
        const unsigned ni = b < NB ? batch_iters(b) : 0u;
        s_ni[t] = ni;
        const unsigned incl = block_scan(ni) + s_carry, excl = incl - ni;
        const unsigned ni_prev = t > 0 ? s_ni[t - 1] : s_lastni;
        const bool first = b < NB && (b == 0 || excl / ITEM_ITERS != (excl - ni_prev) / ITEM_ITERS);
        const unsigned fincl = block_scan(first ? 1u : 0u) + s_icarry;
        if (PASS == 2 && b < NB) {
            const unsigned item = fincl - 1;
            bhdr[nb0 + b] = make_uint2(it0 + excl, ni);                 // flags are OR-ed in below
            if (first) {
                items[item0 + item].x0 = x0;
                items[item0 + item].y0 = y0;
                items[item0 + item].begin = (int)(nb0 + b);
                items[item0 + item].iter0 = it0 + excl;
                if (item > 0) items[item0 + item - 1].end = (int)(nb0 + b);
            }
            if (b == NB - 1) items[item0 + item].end = (int)(nb0 + NB);
        }
        __syncthreads();
        if (t == XCELLS - 1) { s_carry = incl; s_lastni = ni; s_icarry = fincl; }
        __syncthreads();
        total_iters = s_carry;
    }
    if constexpr (PASS == 1) {
        if (t == 0) {
            totals[band].nb = NB;
            totals[band].iters = total_iters;
            totals[band].items = s_icarry;
        }
        return;
    } else {
    // ---------------- PASS 2: lane words (idle default first), then every thread emits its cell's units
    for (unsigned i = t; i < NB * 32; i += XCELLS) { blane[(size_t)nb0 * 32 + i] = 0; lsrc[(size_t)nb0 * 32 + i] = 0; }
    __syncthreads();
    auto emit = [&](unsigned g, unsigned count, unsigned src) {
        blane[(size_t)nb0 * 32 + g] = (unsigned)t | (count << 16);
        lsrc[(size_t)nb0 * 32 + g] = src;
    };
    // full units, layer by layer: layer j holds the cells with more than j full units, cells ascending
    unsigned G = 0;                                       // units before layer j
    for (unsigned j = 0; j < maxfull; ++j) {
        const bool in = myfull > j;
        const unsigned bal = __ballot_sync(0xffffffffu, in);
        if (lane == 0) s_w[warp] = __popc(bal);
        __syncthreads();
        unsigned pre = 0, N = 0;
        for (int q = 0; q < XCELLS / 32; ++q) { const unsigned c = s_w[q]; if (q < warp) pre += c; N += c; }
        if (in) {
            const unsigned g = G + pre + __popc(bal & ((1u << lane) - 1u));
            emit(g, UNIT_CAP, start + j * UNIT_CAP);
            // the batch leaves this layer => it may hold one cell twice
            const unsigned b0 = g & ~31u;
            if (b0 < G || min(b0 + 32u, Q) > G + N) atomicOr(&bhdr[nb0 + (g >> 5)].y, 1u << 16);
        }
        G += N;
        __syncthreads();
    }
    if (myrem) {
        const unsigned g = F + rank;
        emit(g, myrem, start + myfull * UNIT_CAP);
        if ((g & ~31u) < F) atomicOr(&bhdr[nb0 + (g >> 5)].y, 1u << 16);
    }
    // ---- bank-aware lane assignment.  Which lane of a batch runs which unit is free; the 16 lanes of
    // a half-warp access the box together with 8-byte words, and two of them collide when their
    // cells fall into the same class (ly * boxw + lx) mod 16.  Sort the batch's units by class and
    // deal them alternately to the two half-warps, so that the cells of one class are split evenly.
    __syncthreads();
    for (unsigned b = warp; b < NB; b += XCELLS / 32) {
        const size_t o = (size_t)(nb0 + b) * 32 + lane;
        const unsigned lw = blane[o], src = lsrc[o];
        const unsigned cell = lw & 0x1FFu;
        const unsigned key = (lw >> 16) == 0 ? 16u : (((cell >> 5) * (unsigned)boxw + (cell & 31u)) & 15u);   // idle lanes last
        unsigned r = 0;
        for (int q = 0; q < 32; ++q) {
            const unsigned kq = __shfl_sync(0xffffffffu, key, q);
            r += (kq < key || (kq == key && q < lane)) ? 1u : 0u;
        }
        const unsigned dstl = (r & 1u) * 16u + (r >> 1);
        __syncwarp();
        blane[(size_t)(nb0 + b) * 32 + dstl] = lw;
        lsrc[(size_t)(nb0 + b) * 32 + dstl] = src;
    }
    }
}

__global__ void split_totals_kernel(const BandTotals* __restrict__ t, int n_bands, unsigned* __restrict__ nb,
                                    unsigned* __restrict__ iters, unsigned* __restrict__ items, unsigned* __restrict__ nonempty) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n_bands) return;
    if (i == n_bands) { nb[i] = 0; iters[i] = 0; items[i] = 0; return; }
    nb[i] = t[i].nb; iters[i] = t[i].iters; items[i] = t[i].items;
    if (t[i].nb) atomicAdd(nonempty, 1u);
}

// a0.4: fill the slots of every batch (one warp per batch): permutation and the per-iteration
// records (reduced (u, v), weights).
template <typename F>
__global__ void __launch_bounds__(256)
slot_fill_kernel(const uint2* __restrict__ bhdr, const unsigned* __restrict__ blane, const unsigned* __restrict__ lsrc,
                 unsigned n_batches, const unsigned* __restrict__ perm0, const typename Cplx<F>::type* __restrict__ uv,
                 const F* __restrict__ w, int K, unsigned* __restrict__ perm, F* __restrict__ rec) {
    const unsigned warps = (gridDim.x * blockDim.x) >> 5;
    const int lane = threadIdx.x & 31;
    for (unsigned b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; b < n_batches; b += warps) {
        const uint2 h = bhdr[b];
        const unsigned n_iter = h.y & 0xFFFFu;
        const unsigned lw = blane[(size_t)b * 32 + lane], src = lsrc[(size_t)b * 32 + lane];
        const unsigned cnt = lw >> 16;
        typename Cplx<F>::type pad = mk2<F>((F)0, (F)0);
        if (cnt > 0) {                                     // padding coordinate: the unit's first visibility
            const typename Cplx<F>::type c = uv[perm0[src]];
            pad = mk2<F>(x_reduce<F>(c.x, K), x_reduce<F>(c.y, K));
        }
        for (unsigned i = 0; i < n_iter; ++i) {
            const size_t it = (size_t)h.x + i;
            F* r = rec + it * REC_FLOATS;
            typename Cplx<F>::type c = pad;
            F wv = (F)0;
            unsigned pi = PERM_PAD;
            if (i < cnt) {
                pi = perm0[src + i];
                const typename Cplx<F>::type c0 = uv[pi];
                c = mk2<F>(x_reduce<F>(c0.x, K), x_reduce<F>(c0.y, K));
                wv = w ? w[pi] : (F)1;
            }
            perm[it * 32 + lane] = pi;
            reinterpret_cast<typename Cplx<F>::type*>(r)[lane] = c;
            r[64 + lane] = wv;
        }
    }
}

// a0.5: iteration count of every item (its slots are one contiguous stream of `iters` x 32 slots).
__global__ void item_iters_kernel(XItem* __restrict__ items, int n_items, const uint2* __restrict__ bhdr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_items) return;
    const uint2 h = bhdr[items[i].end - 1];
    items[i].iters = h.x + (h.y & 0xFFFFu) - items[i].iter0;
}

template <typename F> using C2 = typename Cplx<F>::type;

// ---------------------------------------------------------------------------------------------
// packed fp32 helpers (sm_100 FFMA2 / FMUL2 / FADD2)
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 dup2(float a) { return make_float2(a, a); }
// the same vocabulary for complex128 (component-wise fp64; no packed instructions exist)
__device__ __forceinline__ double2 fma2(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ double2 mul2(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ double2 add2(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 dup2(double a) { return make_double2(a, a); }

// Kernel weights of both axes of one visibility in a known cell: g[j] = (g_x[j], g_y[j]) for the taps
// c_j = cell - J/2 + 1 + j.  ANALYTIC: t = (u - cell) - 1/2 per axis, the even / odd Horner chains of
// the two axes run as one packed chain.  TABLE: T[floor(|u - c_j| R + 1/2)], one IEEE op per step.
template <typename F, int J, int DEG, int MODE>
__device__ __forceinline__ void x_weights(C2<F> uv, C2<F> cellf, int cx, int cy, const XParamsT<F>& p, const F* tab,
                                          C2<F> (&g)[J]) {
    if (MODE == 0) {
        constexpr int NE = DEG / 2 + 1, NO = (DEG + 1) / 2;
        const C2<F> t = add2(uv, mk2<F>(-cellf.x - (F)0.5, -cellf.y - (F)0.5));     // cell + 1/2 is exact; so is u - cell
        const C2<F> t2 = mul2(t, t), nt = mk2<F>(-t.x, -t.y);
#pragma unroll
        for (int j = 0; j < J / 2; ++j) {
            C2<F> E = dup2(p.coef.e[j][NE - 1]), O = dup2(p.coef.o[j][NO - 1]);
#pragma unroll
            for (int m = NE - 2; m >= 0; --m) E = fma2(E, t2, dup2(p.coef.e[j][m]));
#pragma unroll
            for (int m = NO - 2; m >= 0; --m) O = fma2(O, t2, dup2(p.coef.o[j][m]));
            g[j] = fma2(t, O, E);
            g[J - 1 - j] = fma2(nt, O, E);
        }
    } else {
#pragma unroll
        for (int j = 0; j < J; ++j) {
            const int ox = cx - J / 2 + 1 + j, oy = cy - J / 2 + 1 + j;
            const F dx = sub_rn(uv.x, (F)ox), dy = sub_rn(uv.y, (F)oy);
            const int ix = (int)floor_r(add_rn(mul_rn(fabs(dx), p.table_R), (F)0.5));
            const int iy = (int)floor_r(add_rn(mul_rn(fabs(dy), p.table_R), (F)0.5));
            // MODE 1: table in global memory (read through L1); MODE 2: the CTA's copy in shared memory.  A real slot's
            // (u, v) lies in its unit's cell, so |d| <= J/2 and the index is at most R J/2; the clamp only serves the
            // slots of idle lanes (no unit, w = 0): the last table entry is g beyond the support, 0.
            const int jx = min(ix, p.table_len - 1), jy = min(iy, p.table_len - 1);
            g[j].x = MODE == 2 ? tab[jx] : __ldg(tab + jx);
            g[j].y = MODE == 2 ? tab[jy] : __ldg(tab + jy);
        }
    }
}

// Kernel weights of V visibilities of one cell, written statement-interleaved so that the V dependency
// graphs advance together (ANALYTIC; TABLE evaluates visibility by visibility).
template <typename F, int J, int DEG, int MODE, int V>
__device__ __forceinline__ void x_weights_v(const C2<F> (&uv)[V], C2<F> cellf, int cx, int cy, const XParamsT<F>& p,
                                            const F* tab, C2<F> (&g)[V][J]) {
    if (MODE == 0) {
        constexpr int NE = DEG / 2 + 1, NO = (DEG + 1) / 2;
        C2<F> t[V], t2[V], nt[V];
#pragma unroll
        for (int v = 0; v < V; ++v) {
            t[v] = add2(uv[v], mk2<F>(-cellf.x - (F)0.5, -cellf.y - (F)0.5));       // cell + 1/2 is exact; so is u - cell
            t2[v] = mul2(t[v], t[v]);
            nt[v] = mk2<F>(-t[v].x, -t[v].y);
        }
#pragma unroll
        for (int j = 0; j < J / 2; ++j) {
            C2<F> E[V], O[V];
#pragma unroll
            for (int v = 0; v < V; ++v) { E[v] = dup2(p.coef.e[j][NE - 1]); O[v] = dup2(p.coef.o[j][NO - 1]); }
#pragma unroll
            for (int m = NE - 2; m >= 0; --m)
#pragma unroll
                for (int v = 0; v < V; ++v) E[v] = fma2(E[v], t2[v], dup2(p.coef.e[j][m]));
#pragma unroll
            for (int m = NO - 2; m >= 0; --m)
#pragma unroll
                for (int v = 0; v < V; ++v) O[v] = fma2(O[v], t2[v], dup2(p.coef.o[j][m]));
#pragma unroll
            for (int v = 0; v < V; ++v) { g[v][j] = fma2(t[v], O[v], E[v]); g[v][J - 1 - j] = fma2(nt[v], O[v], E[v]); }
        }
    } else {
#pragma unroll
        for (int v = 0; v < V; ++v) x_weights<F, J, DEG, MODE>(uv[v], cellf, cx, cy, p, tab, g[v]);
    }
}

// a3 arithmetic for V visibilities of one cell: J independent row chains per visibility (a dependent FFMA2 is
// V J instructions away), two column chains.
template <typename F, int J, int DEG, int MODE, int V>
__device__ __forceinline__ void x_degrid_vis(const C2<F> (&uv)[V], const F (&w)[V], C2<F> cellf, int cx, int cy,
                                             const XParamsT<F>& p, const F* tab, const C2<F> (&B)[J][J], C2<F> (&out)[V]) {
    C2<F> g[V][J];
    x_weights_v<F, J, DEG, MODE, V>(uv, cellf, cx, cy, p, tab, g);
    C2<F> r[V][J];
#pragma unroll
    for (int a = 0; a < J; ++a)
#pragma unroll
        for (int v = 0; v < V; ++v) r[v][a] = mul2(dup2(g[v][0].x), B[a][0]);
#pragma unroll
    for (int c = 1; c < J; ++c)
#pragma unroll
        for (int a = 0; a < J; ++a)
#pragma unroll
            for (int v = 0; v < V; ++v) r[v][a] = fma2(dup2(g[v][c].x), B[a][c], r[v][a]);
    C2<F> acc0[V], acc1[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { acc0[v] = mul2(dup2(g[v][0].y), r[v][0]); acc1[v] = mul2(dup2(g[v][1].y), r[v][1]); }
#pragma unroll
    for (int a = 2; a < J; a += 2)
#pragma unroll
        for (int v = 0; v < V; ++v) {
            acc0[v] = fma2(dup2(g[v][a].y), r[v][a], acc0[v]);
            acc1[v] = fma2(dup2(g[v][a + 1].y), r[v][a + 1], acc1[v]);
        }
#pragma unroll
    for (int v = 0; v < V; ++v) out[v] = mul2(dup2(w[v]), add2(acc0[v], acc1[v]));      // padding slots: w = 0 -> 0
}

// a4 arithmetic for V visibilities of one cell: A[a][c] += g_x[c] (g_y[a] w y), visibility by visibility per tap
template <typename F, int J, int DEG, int MODE, int V>
__device__ __forceinline__ void x_grid_vis(const C2<F> (&uv)[V], const F (&w)[V], const C2<F> (&yv)[V], C2<F> cellf,
                                           int cx, int cy, const XParamsT<F>& p, const F* tab, C2<F> (&A)[J][J]) {
    C2<F> g[V][J];
    x_weights_v<F, J, DEG, MODE, V>(uv, cellf, cx, cy, p, tab, g);
    C2<F> z[V];
#pragma unroll
    for (int v = 0; v < V; ++v) z[v] = mul2(dup2(w[v]), yv[v]);
#pragma unroll
    for (int a = 0; a < J; ++a) {
        C2<F> q[V];
#pragma unroll
        for (int v = 0; v < V; ++v) q[v] = mul2(dup2(g[v][a].y), z[v]);
#pragma unroll
        for (int v = 0; v < V; ++v)
#pragma unroll
            for (int c = 0; c < J; ++c) A[a][c] = fma2(dup2(g[v][c].x), q[v], A[a][c]);
    }
}

__device__ __forceinline__ unsigned x_next_item(unsigned* counter, int lane) {
    unsigned it = 0;
    if (lane == 0) it = atomicAdd(counter, 1u);
    return __shfl_sync(0xffffffffu, it, 0);
}
// Kernel tail: the last persistent warp to leave resets the queue, so that launches need no memset in between
// (every warp's pops precede its own arrival here; launches of one handle are ordered by the stream).
__device__ __forceinline__ void x_queue_finish(unsigned* counter, int n_warps, int lane) {
    if (lane == 0) {
        __threadfence();
        if (atomicAdd(counter + 1, 1u) == (unsigned)n_warps - 1u) {
            counter[0] = 0;
            counter[1] = 0;
            __threadfence();
        }
    }
}

// a0.6: longest items first (LPT order of the dynamic queue: the tail of a launch then consists of short items).
__global__ void item_key_kernel(const XItem* __restrict__ items, int n_items, unsigned* __restrict__ key, unsigned* __restrict__ idx) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_items) return;
    key[i] = 0xFFFFu - min(items[i].iters, 0xFFFFu);
    idx[i] = (unsigned)i;
}
__global__ void item_gather_kernel(const XItem* __restrict__ in, const unsigned* __restrict__ idx, int n_items, XItem* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_items) out[i] = in[idx[i]];
}

// ---------------------------------------------------------------------------------------------
// Visibility stream ring.  The slots of one item are contiguous in HBM, so every warp streams them
// through a private ring of S stages in shared memory, each filled by 1-D bulk copies
// (cp.async.bulk, mbarrier completion) of CH iterations: the records (uv, w) and - for the
// adjoint - y.  The copies run S-1 chunks ahead of the arithmetic, which is what hides the HBM
// latency (profiles/r1b_summary.md: with a one-deep register prefetch both kernels were
// long-scoreboard bound at 32 % issue utilisation).
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <typename F> __device__ __forceinline__ C2<F> lds_v2(uint32_t a);
template <> __device__ __forceinline__ float2 lds_v2<float>(uint32_t a) {
    float2 v;
    asm volatile("ld.volatile.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory");
    return v;
}
template <> __device__ __forceinline__ double2 lds_v2<double>(uint32_t a) {
    double2 v;
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_v2(uint32_t a, float2 v) {
    asm volatile("st.volatile.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void sts_v2(uint32_t a, double2 v) {
    asm volatile("st.volatile.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}
// grid[idx] += v: one 8-byte vector reduction for complex64, two fp64 reductions for complex128
__device__ __forceinline__ void atomic_add2(float2* addr, float2 v) { atomicAdd(addr, v); }
__device__ __forceinline__ void atomic_add2(double2* addr, double2 v) { atomicAdd(&addr->x, v.x); atomicAdd(&addr->y, v.y); }

// NY = number of complex64 native-order vectors streamed next to the records: 0 (degridding), 1 (gridding: y),
// 2 (degridding + residual norm of the ADMM step: s, y), 3 (gridding of the ADMM step: v, s, y)
template <typename F, int CH, int NY> struct RingCfg {
    static constexpr int REC_B = REC_FLOATS * (int)sizeof(F), Y_B = 64 * (int)sizeof(F);   // bytes per iteration
    static constexpr int REC = CH * REC_B, Y = CH * Y_B;
    static constexpr int STAGE = REC + NY * Y;
};

// warps per CTA: 4; 8 for the shared-memory-table kernels (MODE 2), so that one copy of the table serves more warps
__host__ __device__ constexpr int x_warps(int MODE) { return MODE == 2 ? 8 : 4; }

template <typename F, int J, int CH, int S, int NY, int NW = 4> struct XSmem {
    static constexpr int BOX_BYTES = XCfg<J>::REGION_BYTES * ((int)sizeof(F) / 4);
    static constexpr int WARP_BYTES = BOX_BYTES + S * RingCfg<F, CH, NY>::STAGE;
    static constexpr int BARS = S + 1;                   // per warp: the box + the ring stages
    static constexpr size_t TOTAL = (size_t)NW * WARP_BYTES + NW * BARS * sizeof(uint64_t);   // (+ the table, MODE 2)
};

// one lane: start the copies of chunk c (iterations [c CH, c CH + n)) of the item into `stage`.
// (No proxy fence: the stage was only READ through the generic proxy, and those reads are ordered
// before this call by the __syncwarp() that precedes it.)
template <typename F, int CH, int NY>
__device__ __forceinline__ void ring_issue(unsigned char* ring, uint64_t* rbar, int stage, const XParamsT<F>& p,
                                           const C2<F>* y0, const C2<F>* y1, const C2<F>* y2, unsigned iter0, int c, int T) {
    typedef RingCfg<F, CH, NY> R;
    const int n = min(CH, T - c * CH);
    const size_t i0 = (size_t)iter0 + (size_t)c * CH;
    unsigned char* st = ring + stage * R::STAGE;
    mbar_expect_tx(rbar + stage, (uint32_t)(n * (R::REC_B + NY * R::Y_B)));
    bulk_g2s(st, p.rec + i0 * REC_FLOATS, (uint32_t)(n * R::REC_B), rbar + stage);
    if (NY >= 1) bulk_g2s(st + R::REC, y0 + i0 * 32, (uint32_t)(n * R::Y_B), rbar + stage);
    if (NY >= 2) bulk_g2s(st + R::REC + R::Y, y1 + i0 * 32, (uint32_t)(n * R::Y_B), rbar + stage);
    if (NY >= 3) bulk_g2s(st + R::REC + 2 * R::Y, y2 + i0 * 32, (uint32_t)(n * R::Y_B), rbar + stage);
}

// ---------------------------------------------------------------------------------------------
// a3 (complex64): W G.  Persistent warps; per item the band's box is staged by one TMA load into the
// warp's private shared-memory region and the item's visibility stream runs through the warp's ring;
// per batch every lane loads its cell's J x J patch into registers and then runs its unit's
// visibilities out of registers.  HBM per slot: uv 8 + w 4 read, y 8 written (native order).
// FUSE = 1 (f1): additionally streams s and y and accumulates ||v + s - y||^2 over the real slots into *p.norm2 (fp64).
template <typename F, int J, int DEG, int MODE, int CH, int S, int FUSE = 0>
__global__ void __launch_bounds__(x_warps(MODE) * 32, (MODE == 2 || sizeof(F) == 8) ? 1 : (J <= 6 ? (XVD == 1 ? 4 : (XVD == 2 ? 3 : 2)) : 1))
degrid_x_kernel(const __grid_constant__ CUtensorMap tmap, const XParamsT<F> p, C2<F>* __restrict__ y) {
    typedef XCfg<J> Cfg;
    constexpr int XVK = sizeof(F) == 4 ? XVD : 1;        // visibilities per trip (complex128: 1, registers)
    constexpr int NY = FUSE ? 2 : 0;
    typedef RingCfg<F, CH, NY> R;
    constexpr int NW = x_warps(MODE);
    typedef XSmem<F, J, CH, S, NY, NW> SM;
    constexpr int BOXW = Cfg::BOXW, BOXH = Cfg::BOXH, XOFF = Cfg::XOFF;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    C2<F>* tile = reinterpret_cast<C2<F>*>(smem_raw + warp * SM::WARP_BYTES);
    unsigned char* ring = smem_raw + warp * SM::WARP_BYTES + SM::BOX_BYTES;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + NW * SM::WARP_BYTES) + warp * SM::BARS;
    uint64_t* rbar = bar + 1;
    const F* tab = p.table;
    if (MODE == 2) {                                    // the CTA's copy of the pre-sampled table (the only CTA-wide step)
        F* ts = reinterpret_cast<F*>(smem_raw + SM::TOTAL);
        for (int i = threadIdx.x; i < p.table_len; i += NW * 32) ts[i] = __ldg(p.table + i);
        __syncthreads();
        tab = ts;
    }
    if (lane == 0) {
        for (int i = 0; i < SM::BARS; ++i) mbar_init(bar + i, 1);
        fence_barrier_init();
    }
    __syncwarp();
    uint32_t box_phase = 0, ring_phase = 0;
    int stage = 0;
    double nacc = 0.0;                                  // FUSE: this lane's share of ||v + s - y||^2

    // the NEXT item (index and descriptor) is fetched while the current one is processed
    unsigned item = x_next_item(p.counter, lane);
    XItem nit = p.items[min(item, (unsigned)p.n_items - 1)];
    uint2 hn = p.bhdr[nit.begin];
    unsigned lwn = p.blane[(size_t)nit.begin * 32 + lane];
    while (item < (unsigned)p.n_items) {
        const XItem it = nit;
        item = x_next_item(p.counter, lane);
        nit = p.items[min(item, (unsigned)p.n_items - 1)];
        const int T = (int)it.iters, nch = (T + CH - 1) / CH;
        const int bx0 = it.x0 - (J / 2 - 1) - XOFF, by0 = it.y0 - (J / 2 - 1);
        const bool interior = bx0 >= 0 && by0 >= 0 && bx0 + BOXW <= p.K && by0 + BOXH <= p.K;
        __syncwarp();                                   // every lane is done with the previous box
        if (lane == 0) {
            if (interior) {
                fence_proxy_async();
                mbar_expect_tx(bar, (uint32_t)(sizeof(C2<F>) * BOXW * BOXH));
                tma_load_2d(tile, &tmap, 2 * bx0, by0, bar);
            }
            int st = stage;
            for (int c = 0; c < S && c < nch; ++c) {
                ring_issue<F, CH, NY>(ring, rbar, st, p, p.s_in, p.yobs, nullptr, it.iter0, c, T);
                st = st + 1 == S ? 0 : st + 1;
            }
        }
        int cnext = S;                                  // next chunk to start
        if (interior) {
            mbar_wait(bar, box_phase);
            box_phase ^= 1;
        } else {
            for (int i = lane; i < BOXW * BOXH; i += 32) {
                const int r = wrap_idx(by0 + i / BOXW, p.K, p.kmask), c = wrap_idx(bx0 + i % BOXW, p.K, p.kmask);
                tile[i] = p.grid[(long long)r * p.K + c];
            }
            __syncwarp();
        }
        int left = T;                                   // iterations of the item not yet started
        int rem = 0;                                    // iterations left in the current chunk
        const F* rp = nullptr;                      // this lane's view of the current record
        const C2<F>* sp = nullptr;                     // FUSE: this lane's s of the current slot (y is CH*32 entries further)
        C2<F>* yout = y + (size_t)it.iter0 * 32 + lane;
        for (int b = it.begin; b < it.end; ++b) {
            const uint2 h = hn;
            const unsigned lw = lwn;
            {                                           // header of the next batch (of this or of the next item)
                const int bn = b + 1 < it.end ? b + 1 : nit.begin;
                hn = p.bhdr[bn];
                lwn = p.blane[(size_t)bn * 32 + lane];
            }
            const int n_iter = (int)(h.y & 0xFFFFu);
            const int cnt = (int)(lw >> 16);
            const int ly = (lw >> 5) & 15, lx = lw & 31;
            const int cx = it.x0 + lx - p.Kh, cy = it.y0 + ly - p.Kh;       // cell = floor(u'), floor(v')
            const C2<F> cellf = mk2<F>((F)cx, (F)cy);
            C2<F> B[J][J];
            {
                const C2<F>* src = tile + ly * BOXW + lx + XOFF;
#pragma unroll
                for (int a = 0; a < J; ++a)
#pragma unroll
                    for (int c = 0; c < J; ++c) B[a][c] = src[a * BOXW + c];
            }
            // the batch's iterations, cut into segments at the ring's chunk boundaries: the inner loop
            // carries no ring logic
            for (int i = 0; i < n_iter;) {
                if (rem == 0) {
                    mbar_wait(rbar + stage, ring_phase);
                    rem = min(CH, left);
                    left -= rem;
                    rp = reinterpret_cast<const F*>(ring + stage * R::STAGE) + lane;
                    if (FUSE) sp = reinterpret_cast<const C2<F>*>(ring + stage * R::STAGE + R::REC) + lane;
                }
                const int seg = min(rem, n_iter - i);
                int k = 0;
#pragma unroll 1
                for (; k + XVK <= seg; k += XVK) {            // XVK visibilities per trip: XVK interleaved dependency graphs
                    C2<F> uvk[XVK], o[XVK];
                    F wk[XVK];
#pragma unroll
                    for (int v = 0; v < XVK; ++v) {
                        uvk[v] = *reinterpret_cast<const C2<F>*>(rp + v * REC_FLOATS + lane);
                        wk[v] = rp[v * REC_FLOATS + 64];
                    }
                    rp += XVK * REC_FLOATS;
                    x_degrid_vis<F, J, DEG, MODE, XVK>(uvk, wk, cellf, cx, cy, p, tab, B, o);
#pragma unroll
                    for (int v = 0; v < XVK; ++v) yout[v * 32] = o[v];
                    yout += XVK * 32;
                    if (FUSE) {
#pragma unroll
                        for (int v = 0; v < XVK; ++v)
                            if (i + k + v < cnt) {                          // a real slot: d = v + s - y
                                const C2<F> sv = sp[v * 32], yv = sp[CH * 32 + v * 32];
                                const F dx = (o[v].x + sv.x) - yv.x, dy = (o[v].y + sv.y) - yv.y;
                                nacc += (double)dx * (double)dx + (double)dy * (double)dy;
                            }
                        sp += XVK * 32;
                    }
                }
                for (; XVK > 1 && k < seg; ++k) {            // tail of the segment, one visibility at a time
                    const C2<F> uv1[1] = {*reinterpret_cast<const C2<F>*>(rp + lane)};
                    const F w1[1] = {rp[64]};
                    C2<F> o1[1];
                    rp += REC_FLOATS;
                    x_degrid_vis<F, J, DEG, MODE, 1>(uv1, w1, cellf, cx, cy, p, tab, B, o1);
                    *yout = o1[0];
                    yout += 32;
                    if (FUSE) {
                        if (i + k < cnt) {
                            const C2<F> sv = sp[0], yv = sp[CH * 32];
                            const F dx = (o1[0].x + sv.x) - yv.x, dy = (o1[0].y + sv.y) - yv.y;
                            nacc += (double)dx * (double)dx + (double)dy * (double)dy;
                        }
                        sp += 32;
                    }
                }
                i += seg;
                rem -= seg;
                if (rem == 0) {                                             // chunk consumed: refill its stage
                    __syncwarp();
                    if (cnext < nch) {
                        if (lane == 0) ring_issue<F, CH, NY>(ring, rbar, stage, p, p.s_in, p.yobs, nullptr, it.iter0, cnext, T);
                        ++cnext;
                    }
                    if (++stage == S) { stage = 0; ring_phase ^= 1; }
                }
            }
        }
    }
    if (FUSE) {                                         // one fp64 atomic per warp
        for (int o = 16; o > 0; o >>= 1) nacc += __shfl_down_sync(0xffffffffu, nacc, o);
        if (lane == 0) atomicAdd(p.norm2, nacc);
    }
    x_queue_finish(p.counter, p.n_warps, lane);
}

// ---------------------------------------------------------------------------------------------
// a4 (complex64): G^dagger W^dagger.  Same items / batches / ring (with y).  Every lane accumulates
// its unit's J x J outer products in registers; at the end of the batch the accumulators are added
// into the warp's private shared-memory box: lanes of an unflagged batch hold distinct cells =>
// distinct addresses in every step, plain read-modify-writes (__syncwarp orders the steps because
// footprints of different lanes overlap); a flagged batch (a cell may occur twice) uses
// shared-memory atomics.  At the end of the item the box is added to the global grid with one
// 8-byte reduction per non-zero cell (RED.ADD.F32x2; halos of neighbouring bands and the items of
// one band meet there).
// FUSE = 1 (f1): y is v = Phi x; s and the measurements are streamed too, the gridded vector z = v - r + s_new is formed
// slot by slot (never stored) and s_new is written to p.s_out (kernels.cuh: admm_update_kernel has the formulas).
template <typename F, int J, int DEG, int MODE, int CH, int S, int FUSE = 0>
__global__ void __launch_bounds__(x_warps(MODE) * 32, (MODE == 2 || sizeof(F) == 8) ? 1 : (J <= 6 ? ((J == 4 ? XVG4 : XVG6) == 1 ? 4 : 3) : 1))
grid_x_kernel(const __grid_constant__ CUtensorMap tmap, const XParamsT<F> p, const C2<F>* __restrict__ y) {
    typedef XCfg<J> Cfg;
    constexpr int NY = FUSE ? 3 : 1;
    typedef RingCfg<F, CH, NY> R;
    constexpr int XVG = sizeof(F) == 8 ? 1 : (J == 4 ? XVG4 : XVG6);   // visibilities per trip
    constexpr int NW = x_warps(MODE);
    typedef XSmem<F, J, CH, S, NY, NW> SM;
    constexpr int BOXW = Cfg::BOXW, BOXH = Cfg::BOXH, XOFF = Cfg::XOFF;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    C2<F>* tile = reinterpret_cast<C2<F>*>(smem_raw + warp * SM::WARP_BYTES);
    unsigned char* ring = smem_raw + warp * SM::WARP_BYTES + SM::BOX_BYTES;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + NW * SM::WARP_BYTES) + warp * SM::BARS;
    uint64_t* rbar = bar + 1;
    const F* tab = p.table;
    if (MODE == 2) {                                    // the CTA's copy of the pre-sampled table (the only CTA-wide step)
        F* ts = reinterpret_cast<F*>(smem_raw + SM::TOTAL);
        for (int i = threadIdx.x; i < p.table_len; i += NW * 32) ts[i] = __ldg(p.table + i);
        __syncthreads();
        tab = ts;
    }
    if (lane == 0) {
        for (int i = 0; i < SM::BARS; ++i) mbar_init(bar + i, 1);
        fence_barrier_init();
    }
    __syncwarp();
    uint32_t ring_phase = 0;
    int stage = 0;
    const F oma = FUSE ? (F)(1.0 - admm_alpha(*p.norm2, p.eps)) : (F)0, vrho = (F)p.varrho;
    // one slot of the fused ADMM step: (v, s, y) -> z = v - r + s_new, s_new stored; padding slots give 0
    auto admm_slot = [&](const C2<F>* q, bool real_slot, C2<F>* sdst) -> C2<F> {
        C2<F> z = mk2<F>((F)0, (F)0), sn = z;
        if (real_slot) {
            const C2<F> vv = q[0], sv = q[CH * 32], yv = q[2 * CH * 32];
            const F dx = (vv.x + sv.x) - yv.x, dy = (vv.y + sv.y) - yv.y;
            const F vrx = oma * dx - sv.x, vry = oma * dy - sv.y;
            sn = mk2<F>(sv.x + vrho * vrx, sv.y + vrho * vry);
            z = mk2<F>(vrx + sn.x, vry + sn.y);
        }
        *sdst = sn;
        return z;
    };

    unsigned item = x_next_item(p.counter, lane);
    XItem nit = p.items[min(item, (unsigned)p.n_items - 1)];
    uint2 hn = p.bhdr[nit.begin];
    unsigned lwn = p.blane[(size_t)nit.begin * 32 + lane];
    while (item < (unsigned)p.n_items) {
        const XItem it = nit;
        item = x_next_item(p.counter, lane);
        nit = p.items[min(item, (unsigned)p.n_items - 1)];
        const int T = (int)it.iters, nch = (T + CH - 1) / CH;
        if (lane == 0) {
            int st = stage;
            for (int c = 0; c < S && c < nch; ++c) {
                ring_issue<F, CH, NY>(ring, rbar, st, p, y, p.s_in, p.yobs, it.iter0, c, T);
                st = st + 1 == S ? 0 : st + 1;
            }
        }
        int cnext = S;
        if (lane == 0) bulk_wait_group_read0();         // the previous item's box reduction has read the box
        __syncwarp();
        for (int i = lane; i < BOXW * BOXH; i += 32) tile[i] = mk2<F>((F)0, (F)0);
        __syncwarp();
        C2<F>* sout = FUSE ? p.s_out + (size_t)it.iter0 * 32 + lane : nullptr;
        int left = T, rem = 0;
        const F* rp = nullptr;
        const C2<F>* yp = nullptr;
        for (int b = it.begin; b < it.end; ++b) {
            const uint2 h = hn;
            const unsigned lw = lwn;
            {
                const int bn = b + 1 < it.end ? b + 1 : nit.begin;
                hn = p.bhdr[bn];
                lwn = p.blane[(size_t)bn * 32 + lane];
            }
            const int n_iter = (int)(h.y & 0xFFFFu);
            const bool dup = (h.y >> 16) & 1u;
            const int cnt = (int)(lw >> 16);
            const int ly = (lw >> 5) & 15, lx = lw & 31;
            const int cx = it.x0 + lx - p.Kh, cy = it.y0 + ly - p.Kh;
            const C2<F> cellf = mk2<F>((F)cx, (F)cy);
            C2<F> A[J][J];
#pragma unroll
            for (int a = 0; a < J; ++a)
#pragma unroll
                for (int c = 0; c < J; ++c) A[a][c] = mk2<F>((F)0, (F)0);

            for (int i = 0; i < n_iter;) {
                if (rem == 0) {
                    mbar_wait(rbar + stage, ring_phase);
                    rem = min(CH, left);
                    left -= rem;
                    rp = reinterpret_cast<const F*>(ring + stage * R::STAGE) + lane;
                    yp = reinterpret_cast<const C2<F>*>(ring + stage * R::STAGE + R::REC) + lane;
                }
                const int seg = min(rem, n_iter - i);
                int live = cnt - i;                                         // slots of this segment that hold a visibility
                int k = 0;
#pragma unroll 1
                for (; k + XVG <= seg; k += XVG, live -= XVG) {
                    C2<F> uvk[XVG], yk[XVG];
                    F wk[XVG];
#pragma unroll
                    for (int v = 0; v < XVG; ++v) {
                        uvk[v] = *reinterpret_cast<const C2<F>*>(rp + v * REC_FLOATS + lane);
                        wk[v] = rp[v * REC_FLOATS + 64];
                        if (FUSE) {
                            yk[v] = admm_slot(yp + v * 32, live > v, sout + v * 32);
                        } else {
                            yk[v] = yp[v * 32];
                            if (live <= v) yk[v] = mk2<F>((F)0, (F)0);   // padding slot: whatever y holds there is ignored
                        }
                    }
                    rp += XVG * REC_FLOATS;
                    yp += XVG * 32;
                    if (FUSE) sout += XVG * 32;
                    x_grid_vis<F, J, DEG, MODE, XVG>(uvk, wk, yk, cellf, cx, cy, p, tab, A);
                }
                for (; XVG > 1 && k < seg; ++k, --live) {
                    const C2<F> uv1[1] = {*reinterpret_cast<const C2<F>*>(rp + lane)};
                    const F w1[1] = {rp[64]};
                    C2<F> y1[1];
                    if (FUSE) {
                        y1[0] = admm_slot(yp, live > 0, sout);
                        sout += 32;
                    } else {
                        y1[0] = *yp;
                        if (live <= 0) y1[0] = mk2<F>((F)0, (F)0);
                    }
                    rp += REC_FLOATS;
                    yp += 32;
                    x_grid_vis<F, J, DEG, MODE, 1>(uv1, w1, y1, cellf, cx, cy, p, tab, A);
                }
                i += seg;
                rem -= seg;
                if (rem == 0) {
                    __syncwarp();
                    if (cnext < nch) {
                        if (lane == 0) ring_issue<F, CH, NY>(ring, rbar, stage, p, y, p.s_in, p.yobs, it.iter0, cnext, T);
                        ++cnext;
                    }
                    if (++stage == S) { stage = 0; ring_phase ^= 1; }
                }
            }
            // ---- flush the accumulators into the warp's box; idle lanes (no unit) stay out
            C2<F>* dst = tile + ly * BOXW + lx + XOFF;
            if (!dup) {
                // One read-modify-write per tap.  In step (a, c) the lanes touch distinct addresses (distinct
                // cells); the footprints of different lanes overlap ACROSS steps, so step s+1 must see step s.
                // The warp is converged here and the block below is straight-line code, so every lane issues
                // each shared-memory instruction together and the LSU performs a warp's shared-memory
                // instructions in issue order; the volatile asm keeps the compiler from reordering them.
                // (A __syncwarp() per step is semantically the same and costs a BRA.DIV + NOP per tap.)
                __syncwarp();
                {
                    const uint32_t da = smem_u32(dst);
#pragma unroll
                    for (int a = 0; a < J; ++a)
#pragma unroll
                        for (int c = 0; c < J; ++c) {
                            const uint32_t ad = da + (uint32_t)(a * BOXW + c) * (uint32_t)sizeof(C2<F>);
                            if (cnt > 0) sts_v2(ad, add2(lds_v2<F>(ad), A[a][c]));
                            __syncwarp();
                        }
                }
            } else {
                if (cnt > 0) {
#pragma unroll
                    for (int a = 0; a < J; ++a)
#pragma unroll
                        for (int c = 0; c < J; ++c) {
                            atomicAdd(&dst[a * BOXW + c].x, A[a][c].x);
                            atomicAdd(&dst[a * BOXW + c].y, A[a][c].y);
                        }
                }
                __syncwarp();
            }
        }
        // ---- add the box to the global grid: one TMA reduction (element-wise fp32 adds at L2) for a box in the
        // interior, 8-byte reductions with periodic wrap for a box that crosses the grid edge.  Halos of
        // neighbouring bands and the items of one band meet here.
        __syncwarp();
        const int bx0 = it.x0 - (J / 2 - 1) - XOFF, by0 = it.y0 - (J / 2 - 1);
        const bool interior = bx0 >= 0 && by0 >= 0 && bx0 + BOXW <= p.K && by0 + BOXH <= p.K;
        if (interior && sizeof(F) == 4) {                // (no fp64 add in the TMA reduction: complex128 uses the loop below)
            if (lane == 0) {
                fence_proxy_async();
                tma_reduce_add_2d(&tmap, 2 * bx0, by0, tile);
                bulk_commit_group();
            }
        } else {
            for (int i = lane; i < BOXW * BOXH; i += 32) {
                const C2<F> v = tile[i];
                if (v.x != (F)0 || v.y != (F)0) {
                    const int r = wrap_idx(by0 + i / BOXW, p.K, p.kmask), c = wrap_idx(bx0 + i % BOXW, p.K, p.kmask);
                    atomic_add2(p.grid + (long long)r * p.K + c, v);
                }
            }
        }
        __syncwarp();
    }
    if (lane == 0) bulk_wait_group_read0();             // shared memory must outlive the last reduction's reads
    x_queue_finish(p.counter, p.n_warps, lane);
}

}  // namespace pk
