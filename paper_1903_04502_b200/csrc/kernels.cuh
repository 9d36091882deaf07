// Device kernels of the measurement operator (sm_100a).  DESIGN.md "Kernels" describes each one,
// the roofline that bounds it and its algorithmic bytes per visibility.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pk {

constexpr int TILE = 32;   // tile side in grid cells (T)

template <typename R> struct Cplx;
template <> struct Cplx<float> { typedef float2 type; };
template <> struct Cplx<double> { typedef double2 type; };

template <typename R> __device__ __forceinline__ typename Cplx<R>::type mk2(R a, R b);
template <> __device__ __forceinline__ float2 mk2<float>(float a, float b) { return make_float2(a, b); }
template <> __device__ __forceinline__ double2 mk2<double>(double a, double b) { return make_double2(a, b); }

// Polynomial coefficients of the kernel taps (kb_host.hpp PolyFit), passed by value in the
// kernel parameter (constant) bank so that Horner steps read them as immediate c[][] operands.
template <typename R> struct KbCoef {
    R e[4][9];
    R o[4][9];
};

// One work item = one chunk of one tile's visibilities (native order range [start, start+count)).
struct Item {
    int x0, y0;      // tile origin in the internal (DC-centred) grid layout
    int start, count;
};

template <typename R> struct OpParams {
    typename Cplx<R>::type* grid;   // K*K internal layout: index (cy + K/2 mod K)*K + (cx + K/2 mod K)
    int K, Kh, kmask;               // Kh = K/2; kmask = K-1 if K is a power of two else 0
    const Item* items;
    const typename Cplx<R>::type* uv;   // native order (u, v)
    const R* w;                         // native order weights
    const unsigned* perm;               // native -> caller index, or nullptr for native-order y
    KbCoef<R> coef;
    const R* table;                     // TABLE mode
    R table_R;
    int table_len;
};

__device__ __forceinline__ int wrap_idx(int a, int K, int kmask) {
    if (kmask) return a & kmask;
    int r = a % K;
    return r < 0 ? r + K : r;
}

__device__ __forceinline__ float floor_r(float a) { return floorf(a); }
__device__ __forceinline__ double floor_r(double a) { return floor(a); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float fma_r(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_r(double a, double b, double c) { return fma(a, b, c); }

// Kernel weights of the J taps c_j = cell - J/2 + 1 + j of one coordinate.
//   ANALYTIC (MODE 0): per-tap-pair even/odd polynomials in t = (u - cell) - 1/2.
//   TABLE    (MODE 1): T[floor(|u - c| R + 1/2)], each step one IEEE operation in R's precision
//                      (reading R11; the oracle decides the index in the same precision).
template <typename R, int J, int DEG, int MODE>
__device__ __forceinline__ void kb_weights(R u, R cellf, int cell, const OpParams<R>& p, R (&g)[J]) {
    if (MODE == 0) {
        constexpr int NE = DEG / 2 + 1, NO = (DEG + 1) / 2;
        const R t = (u - cellf) - (R)0.5;
        const R t2 = t * t;
#pragma unroll
        for (int j = 0; j < J / 2; ++j) {
            R E = p.coef.e[j][NE - 1], O = p.coef.o[j][NO - 1];
#pragma unroll
            for (int m = NE - 2; m >= 0; --m) E = fma_r(E, t2, p.coef.e[j][m]);
#pragma unroll
            for (int m = NO - 2; m >= 0; --m) O = fma_r(O, t2, p.coef.o[j][m]);
            const R tO = t * O;
            g[j] = E + tO;
            g[J - 1 - j] = E - tO;
        }
    } else {
#pragma unroll
        for (int j = 0; j < J; ++j) {
            const int c = cell - J / 2 + 1 + j;
            const R d = sub_rn(u, (R)c);
            const R a = mul_rn(fabs(d), p.table_R);
            const R b = add_rn(a, (R)0.5);
            const int idx = (int)floor_r(b);
            g[j] = idx < p.table_len ? __ldg(p.table + idx) : (R)0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// mbarrier / TMA helpers (inline PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase) {
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(phase) : "memory");
    }
}
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* tmap, int x, int y, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(smem_u32(smem_dst)), "l"(tmap), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}

// TMA reduction: global[box at (x, y)] += smem box, element-wise fp32 adds performed at L2 (no return value)
__device__ __forceinline__ void tma_reduce_add_2d(const CUtensorMap* tmap, int x, int y, const void* smem_src) {
    asm volatile(
        "cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2}], [%3];"
        ::"l"(tmap), "r"(x), "r"(y), "r"(smem_u32(smem_src)) : "memory");
}
__device__ __forceinline__ void bulk_commit_group() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_group_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------
// a1: S + Z fused.  Writes the WHOLE K x K grid: b[p^ mod K] = sign s[py] s[px] x[py,px], 0 elsewhere,
// with sign = (-1)^(p^x + p^y) so that the FFT output lands DC-centred (index c + K/2): the dense
// part of the uv plane is then in the interior of the grid and tiles there never wrap.
// One thread per 16 bytes of grid (2 complex64 / 1 complex128), fully coalesced vector stores.
template <typename R>
__global__ void __launch_bounds__(256) pad_kernel(const typename Cplx<R>::type* __restrict__ x,
                                                  const R* __restrict__ s, typename Cplx<R>::type* __restrict__ b,
                                                  int n, int K) {
    typedef typename Cplx<R>::type C;
    constexpr int V = 16 / sizeof(C);           // complex elements per thread
    const int vec_per_row = K / V;
    const long long total = (long long)K * vec_per_row;
    const int nh = n / 2;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int jy = (int)(i / vec_per_row);
        const int jx0 = (int)(i % vec_per_row) * V;
        const int py = jy < nh ? jy + nh : (jy >= K - nh ? jy - (K - nh) : -1);
        C out[V];
#pragma unroll
        for (int e = 0; e < V; ++e) {
            const int jx = jx0 + e;
            const int px = jx < nh ? jx + nh : (jx >= K - nh ? jx - (K - nh) : -1);
            if (py >= 0 && px >= 0) {
                const C v = x[(long long)py * n + px];
                R f = s[py] * s[px];
                if ((jx + jy) & 1) f = -f;
                out[e] = mk2<R>(f * v.x, f * v.y);
            } else {
                out[e] = mk2<R>((R)0, (R)0);
            }
        }
        if constexpr (V == 2) {
            reinterpret_cast<float4*>(b)[i] = make_float4(out[0].x, out[0].y, out[1].x, out[1].y);
        } else {
            b[i] = out[0];
        }
    }
}

// a6: Z^dagger S^dagger fused: x'[py,px] = sign s[py] s[px] b'[p^y mod K, p^x mod K], image rows [row0, row1)
// (the whole image, or one band of it when the bands are handed to an all-reduce one by one, f3).
template <typename R>
__global__ void __launch_bounds__(256) crop_kernel(const typename Cplx<R>::type* __restrict__ b,
                                                   const R* __restrict__ s, typename Cplx<R>::type* __restrict__ x,
                                                   int n, int K, int row0, int row1) {
    typedef typename Cplx<R>::type C;
    const int nh = n / 2;
    const long long first = (long long)row0 * n, total = (long long)row1 * n;
    for (long long i = first + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int py = (int)(i / n), px = (int)(i % n);
        const int jy = py >= nh ? py - nh : py + K - nh;
        const int jx = px >= nh ? px - nh : px + K - nh;
        const C v = b[(long long)jy * K + jx];
        R f = s[py] * s[px];
        if ((jx + jy) & 1) f = -f;
        x[i] = mk2<R>(f * v.x, f * v.y);
    }
}

// Internal (DC-centred) layout <-> mathematical layout B[ky*K+kx] (test/stage access only).
template <typename R>
__global__ void relayout_kernel(const typename Cplx<R>::type* __restrict__ in, typename Cplx<R>::type* __restrict__ out,
                                int K, int to_math) {
    const long long total = (long long)K * K;
    const int Kh = K / 2;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(i / K), c = (int)(i % K);
        const int r2 = (r + Kh) % K, c2 = (c + Kh) % K;      // K even: the shift is its own inverse
        (void)to_math;
        out[(long long)r2 * K + c2] = in[i];
    }
}

// ---------------------------------------------------------------------------------------------
// a0: sort key per visibility: (tile, cell-in-tile), tile-major then row-major cell order.
template <typename R>
__global__ void key_kernel(const typename Cplx<R>::type* __restrict__ uv, long long M, int K, int kmask, int ntx,
                           unsigned* __restrict__ keys, unsigned* __restrict__ idx, int* __restrict__ bad) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const typename Cplx<R>::type c = uv[k];
        unsigned key = 0;
        if (!(fabs(c.x) < (R)1073741824.0) || !(fabs(c.y) < (R)1073741824.0)) {   // NaN, Inf, too large
            atomicOr(bad, 1);
        } else {
            const int gx = wrap_idx((int)floor_r(c.x) + K / 2, K, kmask);
            const int gy = wrap_idx((int)floor_r(c.y) + K / 2, K, kmask);
            const unsigned tile = (unsigned)(gy / TILE) * ntx + (unsigned)(gx / TILE);
            key = (tile * TILE + (unsigned)(gy % TILE)) * TILE + (unsigned)(gx % TILE);
        }
        keys[k] = key;
        idx[k] = (unsigned)k;
    }
}

template <typename R>
__global__ void gather_kernel(const typename Cplx<R>::type* __restrict__ uv, const R* __restrict__ w,
                              const unsigned* __restrict__ perm, long long M,
                              typename Cplx<R>::type* __restrict__ uv_s, R* __restrict__ w_s) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const unsigned src = perm[k];
        uv_s[k] = uv[src];
        w_s[k] = w ? w[src] : (R)1;
    }
}

// tile_start[t] = first native index whose key >= t*TILE*TILE (binary search), t = 0..n_tiles.
__global__ void tile_start_kernel(const unsigned* __restrict__ keys, long long M, int n_tiles, int* __restrict__ tile_start) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > n_tiles) return;
    const unsigned long long target = (unsigned long long)t * TILE * TILE;
    long long lo = 0, hi = M;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if ((unsigned long long)keys[mid] < target) lo = mid + 1; else hi = mid;
    }
    tile_start[t] = (int)lo;
}

__global__ void tile_chunks_kernel(const int* __restrict__ tile_start, int n_tiles, int chunk, int* __restrict__ n_chunks) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tiles) return;
    const int cnt = tile_start[t + 1] - tile_start[t];
    n_chunks[t] = (cnt + chunk - 1) / chunk;
}

__global__ void fill_items_kernel(const int* __restrict__ tile_start, const int* __restrict__ chunk_off, int n_tiles,
                                  int ntx, int chunk, Item* __restrict__ items) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tiles) return;
    const int s = tile_start[t], e = tile_start[t + 1];
    int o = chunk_off[t];
    for (int a = s; a < e; a += chunk) {
        Item it;
        it.x0 = (t % ntx) * TILE;
        it.y0 = (t / ntx) * TILE;
        it.start = a;
        it.count = min(chunk, e - a);
        items[o++] = it;
    }
}

template <typename C>
__global__ void permute_kernel(const C* __restrict__ in, C* __restrict__ out, const unsigned* __restrict__ perm,
                               long long M_native, int to_native) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M_native; k += (long long)gridDim.x * blockDim.x) {
        const unsigned pi = perm[k];
        if (to_native) { C z; z.x = 0; z.y = 0; out[k] = pi == 0xFFFFFFFFu ? z : in[pi]; }
        else if (pi != 0xFFFFFFFFu) out[pi] = in[k];
    }
}

// inverse of the native -> caller permutation (padding entries skipped): inv[perm[k]] = k
__global__ void invert_perm_kernel(const unsigned* __restrict__ perm, long long M_native, unsigned* __restrict__ inv) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M_native; k += (long long)gridDim.x * blockDim.x) {
        const unsigned pi = perm[k];
        if (pi != 0xFFFFFFFFu) inv[pi] = (unsigned)k;
    }
}

// native -> caller order as a GATHER (coalesced 8/16-byte stores, scattered loads): measurably cheaper than
// the scatter form, whose partial-sector stores cost a read-modify-write each
template <typename C>
__global__ void gather_from_native_kernel(const C* __restrict__ in, C* __restrict__ out, const unsigned* __restrict__ inv,
                                          long long M) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < M; i += (long long)gridDim.x * blockDim.x)
        out[i] = in[inv[i]];
}

// ---------------------------------------------------------------------------------------------
// Routed permutation native <-> caller order (the caller-order entry points purify_degrid / purify_grid).
// One gather over M = 1e8 elements pays one DRAM access AND one L2 request per 8-byte element (2.2 ms at config 4;
// with DRAM locality restored, scattered 8-byte accesses still run at only ~8e10 per second).  So the permutation is
// routed like the passes of a radix sort whose ranks are all known at create: every pass loads a BLOCK of consecutive
// elements with coalesced accesses, permutes it in shared memory, and writes runs of consecutive elements:
//   pass A  native order -> "A order": grouped by COARSE bucket (a range of 2^cs caller indices, at most 256 buckets),
//           native order inside a bucket.  A block's elements for one bucket form one run (about 32 elements).
//   pass B  A order -> "mid" order: grouped by caller TILE (PERM_TILE consecutive caller indices), runs of ~85 elements.
//   pass C  mid -> caller order: a permutation inside each tile, in shared memory, in place.
// and the inverse passes in the other direction.  Index arrays (create): per pass a 16-bit rank inside the block for
// every input element (0xFFFF: padding slot) and a 32-bit destination for every sorted rank (0xFFFFFFFF: none).
constexpr int PERM_TILE_SHIFT = 12, PERM_TILE = 1 << PERM_TILE_SHIFT, PERM_THREADS = 512;
constexpr unsigned NONE32 = 0xFFFFFFFFu;
constexpr unsigned short NONE16 = 0xFFFFu;

// key = caller tile, padding slots behind the last tile
__global__ void tile_key_kernel(const unsigned* __restrict__ perm, long long S, unsigned n_tiles,
                                unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
    for (long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x; s < S; s += (long long)gridDim.x * blockDim.x) {
        const unsigned pi = perm[s];
        keys[s] = pi == NONE32 ? n_tiles : (pi >> PERM_TILE_SHIFT);
        vals[s] = (unsigned)s;
    }
}
// after the stable sort by tile: slot_of[k] is the native slot of mid element k (k < M)
__global__ void mid_fill_kernel(const unsigned* __restrict__ slot_of, const unsigned* __restrict__ perm, long long M,
                                unsigned* __restrict__ q, unsigned short* __restrict__ loc) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const unsigned s = slot_of[k];
        q[s] = (unsigned)k;
        loc[k] = (unsigned short)(perm[s] & (unsigned)(PERM_TILE - 1));
    }
}
// key = coarse bucket (9 bits, 511 = padding), optionally below the native block: (s >> bs) << 9 | bucket
__global__ void coarse_key_kernel(const unsigned* __restrict__ perm, long long S, int cs, int bs, int with_block,
                                  unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
    for (long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x; s < S; s += (long long)gridDim.x * blockDim.x) {
        const unsigned pi = perm[s];
        const unsigned g = pi == NONE32 ? 511u : (pi >> cs);
        keys[s] = with_block ? ((unsigned)(s >> bs) << 9) | g : g;
        vals[s] = (unsigned)s;
    }
}
// after the stable sort by bucket: slot_of_a[k] is the native slot of A-order element k; a[s] = k
__global__ void a_pos_kernel(const unsigned* __restrict__ slot_of_a, long long M, unsigned* __restrict__ a) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x)
        a[slot_of_a[k]] = (unsigned)k;
}
// pass A index arrays from the (block, bucket) order: order1[p] = slot; block b owns p in [b B, (b + 1) B)
__global__ void pass_a_fill_kernel(const unsigned* __restrict__ order1, const unsigned* __restrict__ perm,
                                   const unsigned* __restrict__ a, long long S, int bs,
                                   unsigned short* __restrict__ loc_a, unsigned* __restrict__ dst_a) {
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < S; p += (long long)gridDim.x * blockDim.x) {
        const unsigned s = order1[p];
        const bool real = perm[s] != NONE32;
        loc_a[s] = real ? (unsigned short)(p & ((1ll << bs) - 1)) : NONE16;
        dst_a[p] = real ? a[s] : NONE32;
    }
}
// key of A-order element k: (A block) << kb | (tile relative to the first tile of the bucket the block starts in)
__global__ void pass_b_key_kernel(const unsigned* __restrict__ slot_of_a, const unsigned* __restrict__ perm, long long M,
                                  int cs, int bs, int kb, unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const unsigned blk = (unsigned)(k >> bs);
        const unsigned tile = perm[slot_of_a[k]] >> PERM_TILE_SHIFT;
        const unsigned g0 = perm[slot_of_a[(long long)blk << bs]] >> cs;
        keys[k] = (blk << kb) | (tile - (g0 << (cs - PERM_TILE_SHIFT)));
        vals[k] = (unsigned)k;
    }
}
__global__ void pass_b_fill_kernel(const unsigned* __restrict__ order2, const unsigned* __restrict__ slot_of_a,
                                   const unsigned* __restrict__ q, long long M, int bs,
                                   unsigned short* __restrict__ loc_b, unsigned* __restrict__ dst_b) {
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < M; p += (long long)gridDim.x * blockDim.x) {
        const unsigned k = order2[p];
        loc_b[k] = (unsigned short)(p & ((1ll << bs) - 1));
        dst_b[p] = q[slot_of_a[k]];
    }
}

// One routing pass over blocks of 2^BS elements.  DIR 0: blk[i] -> shared[loc[i]], far[dst[j]] <- shared[j];
// DIR 1 (the inverse): shared[j] <- far[dst[j]], blk[i] <- shared[loc[i]] (0 where loc is NONE16).
template <typename C, int BS, int DIR>
__global__ void __launch_bounds__(PERM_THREADS) route_kernel(const C* __restrict__ src, C* __restrict__ dstv,
                                                              const unsigned short* __restrict__ loc,
                                                              const unsigned* __restrict__ dst, long long n_blk_domain) {
    extern __shared__ __align__(16) unsigned char perm_smem[];
    C* sh = reinterpret_cast<C*>(perm_smem);
    constexpr int B = 1 << BS, EPT = B / PERM_THREADS;
    const long long base = (long long)blockIdx.x * B;
    const int n = (int)((n_blk_domain - base) < (long long)B ? (n_blk_domain - base) : (long long)B);
    // Every index this CTA needs is requested up front, and nothing that depends on one of them is issued before all
    // of them are: the dependent addresses carry a term that is always 0 but is computed from ALL the indices
    // (ptxas otherwise interleaves dependent loads one element at a time - 16 serial DRAM latencies instead of one;
    // measured 0.81 ms against 0.37 ms per pass).
    unsigned d[EPT];
    unsigned l[EPT];
    C v[EPT];
    unsigned fold_d = 0xFFFFFFFFu, fold_l = 0xFFFFFFFFu;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int i = threadIdx.x + e * PERM_THREADS;
        d[e] = NONE32;
        l[e] = NONE16;
        if (i < n) { d[e] = dst[base + i]; l[e] = loc[base + i]; }
        fold_d &= d[e];
        fold_l &= l[e];
    }
    // d is NONE32 or below 2^31, l is at most 0xFFFF: neither comparison can hold
    const unsigned zero_d = fold_d == 0x80000000u ? 1u : 0u, zero_l = fold_l == 0x10000u ? 1u : 0u;
    if (DIR == 0) {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int i = threadIdx.x + e * PERM_THREADS;
            if (i < n) v[e] = src[base + i];
        }
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            if (l[e] != NONE16) sh[l[e] + zero_l] = v[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            if (d[e] != NONE32) dstv[d[e] + zero_d] = sh[threadIdx.x + e * PERM_THREADS];
    } else {
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            if (d[e] != NONE32) v[e] = src[d[e] + zero_d];
        unsigned fold_v = 0xFFFFFFFFu;          // likewise: no store to shared memory before every load is in flight
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            if (d[e] != NONE32) fold_v &= __float_as_uint((float)v[e].x) | 1u;
        const unsigned zero_v = fold_v == 0u ? 1u : 0u;
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            if (d[e] != NONE32) sh[threadIdx.x + e * PERM_THREADS + zero_v] = v[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int i = threadIdx.x + e * PERM_THREADS;
            if (i < n) {
                C z; z.x = 0; z.y = 0;
                dstv[base + i] = l[e] != NONE16 ? sh[l[e] + zero_l] : z;
            }
        }
    }
}

// pass C: one CTA per caller tile.  DIR 0: mid -> caller (out may be the same buffer as in), DIR 1: caller -> mid.
template <typename C, int DIR>
__global__ void __launch_bounds__(PERM_THREADS) tile_permute_kernel(const C* in, C* out, const unsigned short* __restrict__ loc,
                                                                     long long M) {
    extern __shared__ __align__(16) unsigned char perm_smem[];
    C* tile = reinterpret_cast<C*>(perm_smem);
    constexpr int EPT = PERM_TILE / PERM_THREADS;
    const long long base = (long long)blockIdx.x * PERM_TILE;
    const int n = (int)((M - base) < (long long)PERM_TILE ? (M - base) : (long long)PERM_TILE);
    C v[EPT];
    unsigned short l[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int j = threadIdx.x + e * PERM_THREADS;
        if (j < n) { v[e] = in[base + j]; l[e] = loc[base + j]; }
    }
    if (DIR == 0) {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int j = threadIdx.x + e * PERM_THREADS;
            if (j < n) tile[l[e]] = v[e];
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int j = threadIdx.x + e * PERM_THREADS;
            if (j < n) out[base + j] = tile[j];
        }
    } else {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int j = threadIdx.x + e * PERM_THREADS;
            if (j < n) tile[j] = v[e];
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int j = threadIdx.x + e * PERM_THREADS;
            if (j < n) out[base + j] = tile[l[e]];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// f2: pieces of the power method on Phi^dagger Phi.
// sum of |x_i|^2 over a complex vector, accumulated in fp64 into *out (zeroed by the caller)
template <typename R>
__global__ void __launch_bounds__(256) norm2_kernel(const typename Cplx<R>::type* __restrict__ x, long long count,
                                                    double* __restrict__ out) {
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const typename Cplx<R>::type v = x[i];
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += part[w];
        atomicAdd(out, t);
    }
}

template <typename R>
__global__ void __launch_bounds__(256) fill_ones_kernel(typename Cplx<R>::type* __restrict__ x, long long count) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x)
        x[i] = mk2<R>((R)1, (R)0);
}

// y = x / sqrt(*norm2) (y may alias x); a zero vector is left unchanged
template <typename R>
__global__ void __launch_bounds__(256) normalise_kernel(const typename Cplx<R>::type* __restrict__ x,
                                                        typename Cplx<R>::type* __restrict__ y, long long count,
                                                        const double* __restrict__ norm2) {
    const double n2 = *norm2;
    const double f = n2 > 0.0 ? 1.0 / sqrt(n2) : 1.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const typename Cplx<R>::type v = x[i];
        y[i] = mk2<R>((R)((double)v.x * f), (R)((double)v.y * f));
    }
}

// ---------------------------------------------------------------------------------------------
// f1: the data-fidelity half of one ADMM iteration around the operator (Algorithm 1 lines 3-6,
// PAPER.md:224-231; Eq. 23), on native-order vectors.  With d = v + s - y and
// alpha = 1 if ||d|| <= eps else eps / ||d||:   r = y + alpha d  (projection onto the l2 ball of radius eps around y),
// v - r = (1 - alpha) d - s,   s_new = s + varrho (v - r),   z = v - r + s_new  (what Phi^dagger is applied to).
// Padding entries of the complex64 layout (perm = 0xFFFFFFFF) count as 0 and are written as 0.
template <typename R>
__global__ void __launch_bounds__(256) admm_norm2_kernel(const typename Cplx<R>::type* __restrict__ v,
                                                         const typename Cplx<R>::type* __restrict__ s,
                                                         const typename Cplx<R>::type* __restrict__ y,
                                                         const unsigned* __restrict__ perm, long long count,
                                                         double* __restrict__ out) {
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        if (perm && perm[i] == 0xFFFFFFFFu) continue;
        const typename Cplx<R>::type a = v[i], b = s[i], c = y[i];
        const R dx = (a.x + b.x) - c.x, dy = (a.y + b.y) - c.y;
        acc += (double)dx * (double)dx + (double)dy * (double)dy;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += part[w];
        atomicAdd(out, t);
    }
}

// alpha of the projection from the device-resident ||d||^2 (the same expression in every kernel that needs it)
__device__ __forceinline__ double admm_alpha(double norm2, double eps) {
    const double nrm = sqrt(norm2);
    return nrm <= eps ? 1.0 : eps / nrm;
}

template <typename R>
__global__ void __launch_bounds__(256) admm_update_kernel(const typename Cplx<R>::type* __restrict__ v,
                                                          typename Cplx<R>::type* __restrict__ s,      // in / out
                                                          const typename Cplx<R>::type* __restrict__ y,
                                                          const unsigned* __restrict__ perm, long long count,
                                                          const double* __restrict__ norm2, double eps, double varrho,
                                                          typename Cplx<R>::type* __restrict__ z) {
    const R oma = (R)(1.0 - admm_alpha(*norm2, eps)), rho = (R)varrho;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        if (perm && perm[i] == 0xFFFFFFFFu) { s[i] = mk2<R>((R)0, (R)0); z[i] = mk2<R>((R)0, (R)0); continue; }
        const typename Cplx<R>::type a = v[i], b = s[i], c = y[i];
        const R dx = (a.x + b.x) - c.x, dy = (a.y + b.y) - c.y;
        const R vrx = oma * dx - b.x, vry = oma * dy - b.y;          // v - r
        const R sx = b.x + rho * vrx, sy = b.y + rho * vry;          // s_new
        s[i] = mk2<R>(sx, sy);
        z[i] = mk2<R>(vrx + sx, vry + sy);
    }
}

}  // namespace pk
