// state.cuh -- O(N) kernels around the state: initialisation (ds_set_state), force output
// (ds_forces) and state read-back (ds_get_state).  One thread per dumbbell.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "mobility.cuh"

namespace ds {

struct StateArgs {
    int N, B;
    long long unit_stride;  // units per system in the stream
    const void *user_pos;   // [B][N][3] user precision (init) or NULL
    void *user_out;         // [B][N][3] user precision (forces / get_state)
    double *X;              // [B][N][3]
    void *units;            // beta-stream T[B][unit_stride][6][W] (mobility.cuh)
    double *Fd;             // [B][N][3]
    const double *phase;    // [B][S]
    long long *counters;    // step counters c[0], c[1]
    double t, ell, lambda, omega, k0;
};

// Eq. (4), PAPER.md:63-67 for dumbbell s of system b (spheres 2s, 2s+1): F_{2s} = +g n, F_{2s+1} = -g n.
__device__ __forceinline__ void dumbbell_force(const double (&x1)[3], const double (&x2)[3], double phi, double t,
                                               const StateArgs &A, double (&F1)[3]) {
    const double s0 = x2[0] - x1[0], s1 = x2[1] - x1[1], s2 = x2[2] - x1[2];
    const double d = sqrt(s0 * s0 + s1 * s1 + s2 * s2);
    const double L = A.ell + A.lambda * sin(A.omega * t + phi);
    const double g = A.k0 * (d - L);
    F1[0] = g * (s0 / d);
    F1[1] = g * (s1 / d);
    F1[2] = g * (s2 / d);
}

// ds_set_state: X <- user positions; packed copies; forces at t = t0 (step index 0); counters <- 0.
template <typename T> __global__ void state_init_kernel(const StateArgs A) {
    constexpr int W = Pack<T>::W;
    const int S = A.N / 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid == 0) { A.counters[0] = 0; A.counters[1] = 0; }
    if (gid >= (long long)A.B * S) return;
    const int b = (int)(gid / S), s = (int)(gid % S);
    const size_t g3 = ((size_t)b * A.N + 2 * s) * 3;
    const T *up = reinterpret_cast<const T *>(A.user_pos) + g3;
    double x1[3], x2[3], F1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { x1[c] = (double)up[c]; x2[c] = (double)up[3 + c]; }
    dumbbell_force(x1, x2, A.phase[(size_t)b * S + s], A.t, A, F1);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        A.X[g3 + c] = x1[c]; A.X[g3 + 3 + c] = x2[c];
        A.Fd[g3 + c] = F1[c]; A.Fd[g3 + 3 + c] = -F1[c];
    }
    T *un = reinterpret_cast<T *>(A.units) + (size_t)b * A.unit_stride * (6 * W);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        un[unit_index<T>(2LL * s, c)] = (T)x1[c];
        un[unit_index<T>(2LL * s + 1, c)] = (T)x2[c];
        un[unit_index<T>(2LL * s, 3 + c)] = (T)F1[c];
        un[unit_index<T>(2LL * s + 1, 3 + c)] = (T)(-F1[c]);
    }
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

// ds_forces: Eq. (4) at the current X and t, written in user precision.
template <typename T> __global__ void forces_out_kernel(const StateArgs A) {
    const int S = A.N / 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)A.B * S) return;
    const int b = (int)(gid / S), s = (int)(gid % S);
    const size_t g3 = ((size_t)b * A.N + 2 * s) * 3;
    double x1[3], x2[3], F1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { x1[c] = A.X[g3 + c]; x2[c] = A.X[g3 + 3 + c]; }
    dumbbell_force(x1, x2, A.phase[(size_t)b * S + s], A.t, A, F1);
    T *out = reinterpret_cast<T *>(A.user_out) + g3;
#pragma unroll
    for (int c = 0; c < 3; ++c) { out[c] = (T)F1[c]; out[3 + c] = (T)(-F1[c]); }
}

// ds_get_state: X (double) -> user precision.
template <typename T> __global__ void state_out_kernel(const double *X, void *out, long long n3) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid < n3) reinterpret_cast<T *>(out)[gid] = (T)X[gid];
}

}  // namespace ds
