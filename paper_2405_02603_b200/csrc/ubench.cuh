// ubench.cuh -- the issue cost of one fp64 warp-instruction, measured on the device the library runs on (bench.py reports
// it beside the ALU roofline).  What it shows on B200: the fp64 pipe takes a DADD or a DFMA every
// 2 clocks per scheduler ONLY while at most two of its 64-bit sources are new register reads; a DFMA whose three sources
// are three registers none of which the previous instruction used in the same operand slot (no operand-reuse-cache hit)
// issues every 3 clocks.  The stage-2 butterflies of the transforms (lane-constant twiddles: all three sources are
// registers) therefore cost up to 1.5 x what the "64 fp64 ops/clk/SM" roof assumes.
#pragma once
#include <cuda_runtime.h>

namespace fsp {

// MODE 0: c_i = fma(a_i, b_i, c_i), all sources different from the previous instruction's   (3 new register reads)
// MODE 1: c_i = fma(a_0, b_0, c_i)                                                         (1 new read, 2 reuse hits)
// MODE 2: c_i = fma(a_0, b_i, c_i)                                                         (2 new reads, 1 reuse hit)
// MODE 3: c_i = c_i + a_i                                                                  (DADD, 2 new reads)
template <int MODE>
__global__ void k_ubench_fp64(double* out, const double* in, int iters, long long* clk) {
    double a[16], b[16], c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        a[i] = in[i + threadIdx.x]; b[i] = in[16 + i + threadIdx.x]; c[i] = in[32 + i + threadIdx.x];
    }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            if (MODE == 0) c[i] = fma(a[i], b[i], c[i]);
            if (MODE == 1) c[i] = fma(a[0], b[0], c[i]);
            if (MODE == 2) c[i] = fma(a[0], b[i], c[i]);
            if (MODE == 3) c[i] = c[i] + a[i];
        }
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i] + a[i] + b[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = t1 - t0;
}

}  // namespace fsp
