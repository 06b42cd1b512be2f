// pack.cuh -- arithmetic "packs" the pair kernel is written in.
//
// The O(N^2) pair sum of Eq. (3b) is bound by the FP32 / FP64 FMA pipes, not by
// memory.  On sm_100a the FP32 pipe has packed two-wide forms (SASS FFMA2 / FMUL2 / FADD2, PTX
// fma.rn.f32x2 ...) that retire two FMAs per issue slot, so the FP32 kernel processes TWO
// j-spheres per instruction: Pack<float>::V is a float2 whose .x/.y lanes are j and j+1.
// The FP64 kernel processes one j per instruction: Pack<double>::V is a double.  Both V are
// 8 bytes, so the shared-memory j-tile layout (6 V per "unit" of W j-spheres) is common.
#pragma once
#include <cuda_runtime.h>

namespace ds {

template <typename T> struct Pack;

template <> struct Pack<float> {
    typedef float2 V;
    typedef float4 T4;
    static constexpr int W = 2;  // j-spheres per pack
    static __device__ __forceinline__ V bc(float s) { return make_float2(s, s); }
    static __device__ __forceinline__ T4 make4(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
    static __device__ __forceinline__ V sub(V a, V b) {
        // sub.f32x2 -> FADD2 with a negated source modifier (no extra instruction)
        unsigned long long r;
        asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<unsigned long long *>(&a)),
            "l"(*reinterpret_cast<unsigned long long *>(&b)));
        return *reinterpret_cast<V *>(&r);
    }
    static __device__ __forceinline__ V mul(V a, V b) { return __fmul2_rn(a, b); }
    static __device__ __forceinline__ V fma(V a, V b, V c) { return __ffma2_rn(a, b, c); }
    static __device__ __forceinline__ float rsq1(float x) {
        float y;  // one MUFU.RSQ; inputs are finite, positive, normal (r^2 of distinct spheres)
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
        return y;
    }
    template <bool GUARD> static __device__ __forceinline__ V rsq(V r2) {
        V y = make_float2(rsq1(r2.x), rsq1(r2.y));
        if (GUARD) {  // alpha == beta (r = 0) is not a pair: Eq. (3b) holds for alpha != beta only
            y.x = r2.x > 0.f ? y.x : 0.f;
            y.y = r2.y > 0.f ? y.y : 0.f;
        }
        return y;
    }
    static __device__ __forceinline__ float hsum(V a) { return a.x + a.y; }
    static __device__ __forceinline__ float dummy() { return 1.0e18f; }  // far-away pad sphere, F = 0
};

template <> struct Pack<double> {
    typedef double V;
    typedef double4 T4;
    static constexpr int W = 1;
    static __device__ __forceinline__ V bc(double s) { return s; }
    static __device__ __forceinline__ T4 make4(double a, double b, double c, double d) { return make_double4(a, b, c, d); }
    static __device__ __forceinline__ V sub(V a, V b) { return a - b; }
    static __device__ __forceinline__ V mul(V a, V b) { return a * b; }
    static __device__ __forceinline__ V fma(V a, V b, V c) { return ::fma(a, b, c); }
    template <bool GUARD> static __device__ __forceinline__ V rsq(V x) {
        // There is no full-precision FP64 rsqrt in hardware.  Seed: MUFU.RSQ64H (about 2^-20);
        // one third-order step y <- y (1 + e/2 + 3 e^2/8), e = 1 - x y^2, leaves a relative error
        // of (5/16) e^3 < 2^-60.  5 DFMA-pipe instructions, no slow path (x is finite, positive, normal).
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        double xy = x * y;
        double e = ::fma(-xy, y, 1.0);
        double p = ::fma(0.375, e, 0.5);
        double pe = p * e;
        y = ::fma(y, pe, y);
        if (GUARD) y = x > 0.0 ? y : 0.0;
        return y;
    }
    static __device__ __forceinline__ double hsum(V a) { return a; }
    static __device__ __forceinline__ double dummy() { return 1.0e18; }
};

}  // namespace ds
