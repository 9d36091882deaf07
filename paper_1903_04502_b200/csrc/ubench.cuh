// Issue-rate probe of the packed fp32 instruction forms the two hot kernels are made of ("which roofline
// binds").  Every warp runs a long, fully unrolled block of independent instructions of ONE form; clock64() inside the
// kernel gives SM cycles, so the result (cycles per instruction per SM sub-partition) does not depend on what the
// clock does under the load.  The forms differ in how many 32-bit register-file reads an instruction needs beyond
// what the operand-reuse cache and the uniform / constant operand path supply - that, not the FMA pipe, is what
// bounds the kernels (purify_ubench_fma; bench.py --ubench; tests/test_gpu_parity.py::test_ubench_fma_forms).
#pragma once
#include <cuda_runtime.h>

namespace pk {

constexpr int UB_NA = 16, UB_REP = 4;       // independent accumulators, repetitions per loop trip

// FORM 0  2 x FFMA   acc = g * b[i] + acc          scalar, 3 register operands (g reused)
// FORM 1  FFMA2      acc = (g, g) * b[i] + acc     broadcast scalar x pair + pair   (degridding row pass: g[c] x B[a][c] + r[a])
// FORM 2  FFMA2      acc = gpair * b[i] + acc      pair x pair + pair               (weight combination t x O + E)
// FORM 3  FFMA2      acc = acc * gpair + const     pair x pair + uniform constant   (Horner step)
// FORM 4  FFMA2      acc = (b[i].x, b[i].x) * gpair + acc   varying scalar x shared pair + pair   (gridding: g[c] x q + A[a][c])
template <int FORM>
__global__ void __launch_bounds__(1024) ubench_fma_kernel(float* out, long long* cyc, int iters, float a0, float c0) {
    float2 acc[UB_NA], b[UB_NA];
    for (int i = 0; i < UB_NA; ++i) {
        acc[i] = make_float2(threadIdx.x * 0.001f + i, 1.f);
        b[i] = make_float2(0.5f + i * 0.01f + threadIdx.x * 1e-5f, 0.25f + i * 0.02f);
    }
    const float2 g = make_float2(a0, a0 * 0.5f);
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < UB_REP; ++r) {
#pragma unroll
            for (int i = 0; i < UB_NA; ++i) {
                if (FORM == 0) { acc[i].x = fmaf(g.x, b[i].x, acc[i].x); acc[i].y = fmaf(g.x, b[i].y, acc[i].y); }
                else if (FORM == 1) acc[i] = __ffma2_rn(make_float2(g.x, g.x), b[i], acc[i]);
                else if (FORM == 2) acc[i] = __ffma2_rn(g, b[i], acc[i]);
                else if (FORM == 3) acc[i] = __ffma2_rn(acc[i], g, make_float2(c0, c0));
                else acc[i] = __ffma2_rn(make_float2(b[i].x, b[i].x), g, acc[i]);
            }
        }
    }
    const long long t1 = clock64();
    float s = 0;
    for (int i = 0; i < UB_NA; ++i) s += acc[i].x + acc[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

}  // namespace pk
