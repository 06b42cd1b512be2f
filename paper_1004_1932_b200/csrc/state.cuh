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
