// peak.cuh -- FMA-chain microbenchmark: the measured ALU peak the roofline fractions are quoted
// against beside the nominal one (MEASURED_PEAKS.json has HBM and bf16 entries only).
// FP32 uses the packed two-wide FMA (SASS FFMA2) the pair kernel uses; FP64 uses DFMA.
// Measurement infrastructure: it holds none of the method's arithmetic.
#pragma once
#include <cuda_runtime.h>

#include "pack.cuh"

namespace ds {

template <typename T, int CHAINS>
__global__ void __launch_bounds__(256) fma_chain_kernel(T *out, int iters, T a0, T b0) {
    typedef Pack<T> P;
    typedef typename P::V V;
    V acc[CHAINS];
    const V a = P::bc(a0), b = P::bc(b0);
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) acc[k] = P::bc((T)(threadIdx.x + k));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int k = 0; k < CHAINS; ++k) acc[k] = P::fma(acc[k], a, b);
    }
    V s = acc[0];
#pragma unroll
    for (int k = 1; k < CHAINS; ++k) s = P::fma(s, a, acc[k]);
    if (P::hsum(s) == (T)123456.789) out[blockIdx.x * blockDim.x + threadIdx.x] = P::hsum(s);  // keeps the chain live
}

}  // namespace ds
