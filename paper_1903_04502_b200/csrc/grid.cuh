// a4: G^dagger W^dagger - weighted gridding (the
// paper keeps a second row-major copy of G for this; here nothing is stored).
//
// One CTA per work item (the same tile chunks as degridding).  No per-visibility atomics anywhere:
//   * every WARP owns a private (T+J) x (T+J) accumulation tile in shared memory;
//   * phase 1 (lane = visibility): kernel weights, z = w y, stage gx[.] and gy[.] z for 32
//     visibilities in the warp's staging area, and find the runs of equal cell (the native order
//     is cell-sorted inside a tile, so equal cells are adjacent);
//   * phase 2 (lane = (tap row a, tap column pair p)): walk the 32 visibilities, accumulate
//     gx[b] * (gy[a] z) in registers while the cell stays the same, and add the run's sum into the
//     warp's tile when the cell changes - lanes hold distinct taps, so plain read-modify-write;
//   * at the end the warps' tiles are summed and the box is flushed to the global grid ONCE per
//     work item with one floating-point atomic per touched cell component (halo cells of
//     neighbouring tiles and the chunks of one tile meet there; periodic wrap applied here).
#pragma once
#include "kernels.cuh"

namespace pk {

template <int J> struct GridCfg {
    static constexpr int BOX = TILE + J;
    static constexpr int WARPS = 4;
    static constexpr int THREADS = WARPS * 32;
};

template <typename R> __device__ __forceinline__ void atomic_add_r(R* addr, R v) { atomicAdd(addr, v); }

template <typename R, int J>
constexpr size_t grid_smem_bytes() {
    typedef typename Cplx<R>::type C;
    return (size_t)GridCfg<J>::WARPS * (sizeof(C) * GridCfg<J>::BOX * GridCfg<J>::BOX      // tiles
                                        + sizeof(R) * 32 * J                                // gx staging
                                        + sizeof(C) * 32 * J);                              // gy z staging
}

template <typename R, int J, int DEG, int MODE>
__global__ void __launch_bounds__(GridCfg<J>::THREADS)
grid_kernel(const OpParams<R> p, const typename Cplx<R>::type* __restrict__ y) {
    typedef typename Cplx<R>::type C;
    constexpr int BOX = GridCfg<J>::BOX, NW = GridCfg<J>::WARPS, HP = J / 2;
    constexpr int NACT = J * HP;                   // active lanes in phase 2
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* tiles = reinterpret_cast<C*>(smem_raw);                              // [NW][BOX*BOX]
    C* sqy_all = tiles + NW * BOX * BOX;                                    // [NW][J][32]   gy[a] z
    C* spx_all = sqy_all + NW * J * 32;                                     // [NW][HP][32]  (gx[2p], gx[2p+1])

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    C* mytile = tiles + warp * BOX * BOX;
    C* sqy = sqy_all + warp * J * 32;
    C* spx = spx_all + warp * HP * 32;

    for (int i = threadIdx.x; i < NW * BOX * BOX; i += blockDim.x) tiles[i] = mk2<R>((R)0, (R)0);
    __syncthreads();

    const Item it = p.items[blockIdx.x];
    const int end = it.start + it.count;
    const int a_tap = lane / HP, p_tap = lane % HP;          // phase-2 role
    const bool act = lane < NACT;

    for (int base = it.start + warp * 32; base < end; base += NW * 32) {
        // ---------------- phase 1: lane = visibility
        const int k = base + lane;
        const bool valid = k < end;
        int off = 0;
        {
            C uvk = mk2<R>((R)0, (R)0), yk = mk2<R>((R)0, (R)0);
            R wk = (R)0;
            if (valid) {
                uvk = p.uv[k];
                wk = p.w[k];
                yk = p.perm ? y[p.perm[k]] : y[k];
            }
            const R fu = floor_r(uvk.x), fv = floor_r(uvk.y);
            const int cx = (int)fu, cy = (int)fv;
            R gx[J], gy[J];
            kb_weights<R, J, DEG, MODE>(uvk.x, fu, cx, p, gx);
            kb_weights<R, J, DEG, MODE>(uvk.y, fv, cy, p, gy);
            const R zr = wk * yk.x, zi = wk * yk.y;          // invalid lanes: z = 0
            if (valid) {
                const int lx = wrap_idx(cx + p.Kh, p.K, p.kmask) - it.x0;
                const int ly = wrap_idx(cy + p.Kh, p.K, p.kmask) - it.y0;
                off = ly * BOX + lx;
            }
#pragma unroll
            for (int j = 0; j < HP; ++j) spx[j * 32 + lane] = mk2<R>(gx[2 * j], gx[2 * j + 1]);
#pragma unroll
            for (int a = 0; a < J; ++a) sqy[a * 32 + lane] = mk2<R>(gy[a] * zr, gy[a] * zi);
        }
        // invalid tail lanes inherit the last valid lane's cell so that they open no new run
        const int nvalid = min(32, end - base);
        off = __shfl_sync(0xffffffffu, off, min(lane, nvalid - 1));
        const int prev = __shfl_up_sync(0xffffffffu, off, 1);
        const unsigned newrun = __ballot_sync(0xffffffffu, lane == 0 || off != prev);
        __syncwarp();

        // ---------------- phase 2: lane = (a_tap, p_tap); sequential over the 32 visibilities
        R a0r = (R)0, a0i = (R)0, a1r = (R)0, a1i = (R)0;
        int cur = __shfl_sync(0xffffffffu, off, 0);
#pragma unroll
        for (int kk = 0; kk < 32; ++kk) {
            if (kk > 0 && ((newrun >> kk) & 1u)) {
                if (act) {
                    C* d = mytile + cur + a_tap * BOX + 2 * p_tap;
                    C t0 = d[0], t1 = d[1];
                    t0.x += a0r; t0.y += a0i; t1.x += a1r; t1.y += a1i;
                    d[0] = t0; d[1] = t1;
                }
                // (the branch is warp-uniform: `newrun` is a ballot.)  The next run's flush may touch, from ANOTHER lane,
                // an address this flush has just written: order the two read-modify-write rounds.
                __syncwarp();
                a0r = a0i = a1r = a1i = (R)0;
                cur = __shfl_sync(0xffffffffu, off, kk);
            }
            if (act) {
                const C gp = spx[p_tap * 32 + kk];
                const R g0 = gp.x, g1 = gp.y;
                const C q = sqy[a_tap * 32 + kk];
                a0r = fma_r(g0, q.x, a0r); a0i = fma_r(g0, q.y, a0i);
                a1r = fma_r(g1, q.x, a1r); a1i = fma_r(g1, q.y, a1i);
            }
        }
        if (act) {
            C* d = mytile + cur + a_tap * BOX + 2 * p_tap;
            C t0 = d[0], t1 = d[1];
            t0.x += a0r; t0.y += a0i; t1.x += a1r; t1.y += a1i;
            d[0] = t0; d[1] = t1;
        }
        __syncwarp();
    }
    __syncthreads();

    // ---------------- merge the warps' tiles and flush the box once
    const int bx0 = it.x0 - J / 2 + 1, by0 = it.y0 - J / 2 + 1;
    for (int i = threadIdx.x; i < BOX * BOX; i += blockDim.x) {
        R sr = (R)0, si = (R)0;
#pragma unroll
        for (int w = 0; w < NW; ++w) { const C v = tiles[w * BOX * BOX + i]; sr += v.x; si += v.y; }
        if (sr != (R)0 || si != (R)0) {
            const int r = wrap_idx(by0 + i / BOX, p.K, p.kmask), c = wrap_idx(bx0 + i % BOX, p.K, p.kmask);
            R* g = reinterpret_cast<R*>(p.grid + (long long)r * p.K + c);
            atomic_add_r(g, sr);
            atomic_add_r(g + 1, si);
        }
    }
}

}  // namespace pk
