// state.cuh -- O(N) kernels around the state: initialisation (ds_set_state), force output
// (ds_forces), state read-back (ds_get_state) and the stream packing of the stateless apply.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "mobility.cuh"

namespace ds {

struct StateArgs {
    int N, B;
    const void *user_pos;   // [B][N][3] user precision (ds_set_state) or NULL
    void *user_out;         // [B][N][3] user precision (ds_forces)
    double *X;              // [B][N][3]
    const double *phase;    // [B][S]
    double t, ell, lambda, omega, k0;
};

// ds_set_state: X <- user positions (widened to FP64: the state is FP64 in both precisions).
template <typename T> __global__ void state_init_kernel(const StateArgs A) {
    const long long n3 = (long long)A.B * A.N * 3;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid < n3) A.X[gid] = (double)reinterpret_cast<const T *>(A.user_pos)[gid];
}

// Pad units [U, unit_stride) of every system's stream: far-away spheres with zero force (they
// contribute exactly 0 to every sum); written once, never touched afterwards.
template <typename T> __global__ void pad_init_kernel(void *units, int U, long long unit_stride, int B) {
    constexpr int W = Pack<T>::W;
    const long long npad = unit_stride - U;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)B * npad) return;
    const long long b = gid / npad, k = gid % npad;
    T *un = reinterpret_cast<T *>(units) + ((size_t)b * unit_stride + U + k) * (6 * W);
#pragma unroll
    for (int e = 0; e < 6 * W; ++e) un[e] = e < 3 * W ? Pack<T>::dummy() : T(0);
}

// ds_mobility_apply: user arrays pos, F [n][3] -> one stream of U + PAD_UNITS units (a tail lane of
// the last unit when n is odd, and all pad units, are far-away zero-force spheres).
template <typename T> __global__ void pack_user_kernel(const T *__restrict__ pos, const T *__restrict__ F, T *units,
                                                       int n, long long n_units) {
    constexpr int W = Pack<T>::W;
    const long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= n_units) return;
    T *un = units + (size_t)u * (6 * W);
#pragma unroll
    for (int l = 0; l < W; ++l) {
        const long long i = u * W + l;
        const bool real = i < n;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            un[c * W + l] = real ? pos[i * 3 + c] : Pack<T>::dummy();
            un[(3 + c) * W + l] = real ? F[i * 3 + c] : T(0);
        }
    }
}

// ds_forces: Eq. (4) at the current X and t, written in user precision.  One thread per dumbbell.
template <typename T> __global__ void forces_out_kernel(const StateArgs A) {
    const int S = A.N / 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)A.B * S) return;
    const int b = (int)(gid / S), s = (int)(gid % S);
    const size_t g3 = ((size_t)b * A.N + 2 * s) * 3;
    double x0[3], x1[3], F0[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { x0[c] = A.X[g3 + c]; x1[c] = A.X[g3 + 3 + c]; }
    dumbbell_force(x0, x1, stroke_length(A.t, A.phase[(size_t)b * S + s], A.ell, A.lambda, A.omega), A.k0, F0);
    T *out = reinterpret_cast<T *>(A.user_out) + g3;
#pragma unroll
    for (int c = 0; c < 3; ++c) { out[c] = (T)F0[c]; out[3 + c] = (T)(-F0[c]); }
}

// ds_get_state: X (double) -> user precision.
template <typename T> __global__ void state_out_kernel(const double *X, void *out, long long n3) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid < n3) reinterpret_cast<T *>(out)[gid] = (T)X[gid];
}

}  // namespace ds

namespace ds {

// ---------------------------------------------------------------------------------------------
// Observables.  Dumbbell coordinates, Eq. (6a), (6b), from the FP64 state:
//   N^s = (X_{2s+1} - X_{2s}) / |X_{2s+1} - X_{2s}|,   R^s = (X_{2s+1} + X_{2s}) / 2.
// One thread per dumbbell.  outR / outN in user precision (either may be NULL); Rref (FP64, may be NULL) receives
// the centres as the reference R(0; w) of Eq. (13).
template <typename T>
__global__ void coords_kernel(const double *__restrict__ X, long long n_db, T *outR, T *outN, double *Rref) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_db) return;
    const double *x1 = X + 6 * s, *x2 = x1 + 3;
    double d[3], len2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) { d[c] = x2[c] - x1[c]; len2 += d[c] * d[c]; }
    const double len = sqrt(len2);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double r = 0.5 * (x2[c] + x1[c]);
        if (outR) outR[3 * s + c] = (T)r;
        if (outN) outN[3 * s + c] = (T)(d[c] / len);
        if (Rref) Rref[3 * s + c] = r;
    }
}

// Eq. (13), first pass: block (chunk, w) adds |R^s(t; w) - R^s(0; w)|^2 over its <= 256 dumbbells
// (shared-memory tree, fixed order) -> partial[w][chunk].
__global__ void __launch_bounds__(256) msd_partial_kernel(const double *__restrict__ X, const double *__restrict__ Rref, int S,
                                                          double *partial) {
    __shared__ double sh[256];
    const int w = blockIdx.y, s = blockIdx.x * 256 + threadIdx.x;
    double q = 0.0;
    if (s < S) {
        const size_t k = (size_t)w * S + s;
        const double *x1 = X + 6 * k, *x2 = x1 + 3, *r0 = Rref + 3 * k;
#pragma unroll
        for (int c = 0; c < 3; ++c) { const double d = 0.5 * (x2[c] + x1[c]) - r0[c]; q += d * d; }
    }
    sh[threadIdx.x] = q;
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) sh[threadIdx.x] += sh[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(size_t)w * gridDim.x + blockIdx.x] = sh[0];
}
// second pass (one block): (1/W) sum_w (1/S) sum_chunks partial[w][chunk], fixed order.
__global__ void __launch_bounds__(256) msd_final_kernel(const double *__restrict__ partial, int W, int S, int n_chunk, double *out) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (int w = threadIdx.x; w < W; w += 256) {
        double inner = 0.0;
        for (int c = 0; c < n_chunk; ++c) inner += partial[(size_t)w * n_chunk + c];
        acc += inner / (double)S;
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) sh[threadIdx.x] += sh[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0] / (double)W;
}

}  // namespace ds
