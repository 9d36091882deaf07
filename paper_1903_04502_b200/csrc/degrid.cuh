// a3: W G - degridding ("G represents a convolution matrix that
// interpolates measurements off the grid", cost O(M J^2)).
//
// One CTA per work item (a chunk of one tile's visibilities, native = tile/cell-sorted order).
//   1. the (T+J) x (T+J) box of the Fourier grid that the tile's footprints can touch is staged
//      into shared memory by ONE TMA load (cp.async.bulk.tensor.2d, mbarrier completion); boxes that
//      cross the grid edge (periodic wrap, reading R8) are staged by wrapped cooperative loads;
//   2. one thread per visibility: 2J kernel weights in registers, J x J complex dot product
//      against the staged tile (lanes are sorted by cell, so a warp's shared-memory reads hit a
//      handful of addresses -> broadcast, no bank conflicts), times w, one 8/16-byte store.
// HBM traffic per visibility: uv + w read, y written = 20 B (c64) / 40 B (c128) in native order.
#pragma once
#include "kernels.cuh"

namespace pk {

template <int J> struct DegridCfg {
    static constexpr int BOX = TILE + J;          // box side (even => TMA inner extent multiple of 16 B)
    static constexpr int THREADS = 256;
};

template <typename R, int J, int DEG, int MODE>
__global__ void __launch_bounds__(DegridCfg<J>::THREADS)
degrid_kernel(const __grid_constant__ CUtensorMap tmap, const OpParams<R> p, typename Cplx<R>::type* __restrict__ y) {
    typedef typename Cplx<R>::type C;
    constexpr int BOX = DegridCfg<J>::BOX;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* tile = reinterpret_cast<C*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + sizeof(C) * BOX * BOX);

    const Item it = p.items[blockIdx.x];
    // box origin (internal layout).  The first column is shifted left by XOFF so that it is EVEN:
    // a complex64 box must start on a 16-byte boundary for the TMA engine (an odd start column
    // faults with "illegal instruction" on sm_100a).
    constexpr int XOFF = (J / 2 - 1) & 1;
    const int bx0 = it.x0 - J / 2 + 1 - XOFF, by0 = it.y0 - J / 2 + 1;
    const bool interior = bx0 >= 0 && by0 >= 0 && bx0 + BOX <= p.K && by0 + BOX <= p.K;

    if (interior) {
        if (threadIdx.x == 0) {
            mbar_init(bar, 1);
            fence_barrier_init();
            fence_proxy_async();
            mbar_expect_tx(bar, (uint32_t)(sizeof(C) * BOX * BOX));
            tma_load_2d(tile, &tmap, 2 * bx0, by0, bar);               // inner coordinate in reals
        }
    } else {
        for (int i = threadIdx.x; i < BOX * BOX; i += blockDim.x) {
            const int r = wrap_idx(by0 + i / BOX, p.K, p.kmask), c = wrap_idx(bx0 + i % BOX, p.K, p.kmask);
            tile[i] = p.grid[(long long)r * p.K + c];
        }
    }

    // prefetch this thread's first visibility while the tile is in flight
    const int end = it.start + it.count;
    int k = it.start + threadIdx.x;
    C uvk = mk2<R>((R)0, (R)0);
    R wk = (R)0;
    if (k < end) { uvk = p.uv[k]; wk = p.w[k]; }

    __syncthreads();                       // mbarrier init visible / manual tile complete
    if (interior) mbar_wait(bar, 0);

    while (k < end) {
        const int kn = k + blockDim.x;
        C uvn = mk2<R>((R)0, (R)0);
        R wn = (R)0;
        if (kn < end) { uvn = p.uv[kn]; wn = p.w[kn]; }

        const R fu = floor_r(uvk.x), fv = floor_r(uvk.y);
        const int cx = (int)fu, cy = (int)fv;
        R gx[J], gy[J];
        kb_weights<R, J, DEG, MODE>(uvk.x, fu, cx, p, gx);
        kb_weights<R, J, DEG, MODE>(uvk.y, fv, cy, p, gy);
        const int lx = wrap_idx(cx + p.Kh, p.K, p.kmask) - it.x0;
        const int ly = wrap_idx(cy + p.Kh, p.K, p.kmask) - it.y0;
        const C* row = tile + ly * BOX + lx + XOFF;
        R yr = (R)0, yi = (R)0;
#pragma unroll
        for (int a = 0; a < J; ++a) {
            R ar = (R)0, ai = (R)0;
#pragma unroll
            for (int b = 0; b < J; ++b) {
                const C v = row[a * BOX + b];
                ar = fma_r(gx[b], v.x, ar);
                ai = fma_r(gx[b], v.y, ai);
            }
            yr = fma_r(gy[a], ar, yr);
            yi = fma_r(gy[a], ai, yi);
        }
        const C out = mk2<R>(wk * yr, wk * yi);
        if (p.perm) y[p.perm[k]] = out; else y[k] = out;

        k = kn; uvk = uvn; wk = wn;
    }
}

}  // namespace pk
