// state.cuh -- O(N) kernels around the state: initialisation (ds_set_state), force output
// (ds_forces) and state read-back (ds_get_state).  One thread per dumbbell.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "mobility.cuh"

namespace ds {

struct StateArgs {
    int N, B, Npad;
    const void *user_pos;   // [B][N][3] user precision (init) or NULL
    void *user_out;         // [B][N][3] user precision (forces / get_state)
    double *X;              // [B][N][3]
    void *pos4, *F4;        // packed T4 [B][Npad]
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
    typedef typename Pack<T>::T4 T4;
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
    T4 *p4 = reinterpret_cast<T4 *>(A.pos4) + (size_t)b * A.Npad + 2 * s;
    T4 *f4 = reinterpret_cast<T4 *>(A.F4) + (size_t)b * A.Npad + 2 * s;
    p4[0] = MakeT4<T>::make(x1[0], x1[1], x1[2]);
    p4[1] = MakeT4<T>::make(x2[0], x2[1], x2[2]);
    f4[0] = MakeT4<T>::make(F1[0], F1[1], F1[2]);
    f4[1] = MakeT4<T>::make(-F1[0], -F1[1], -F1[2]);
}

// pad entries of the packed arrays: far-away sphere, zero force (never touched afterwards)
template <typename T> __global__ void pad_init_kernel(void *pos4, void *F4, int N, int Npad, int B) {
    typedef typename Pack<T>::T4 T4;
    const int npad = Npad - N;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)B * npad) return;
    const int b = (int)(gid / npad), k = (int)(gid % npad);
    const double far = (double)Pack<T>::dummy();
    reinterpret_cast<T4 *>(pos4)[(size_t)b * Npad + N + k] = MakeT4<T>::make(far, far, far);
    reinterpret_cast<T4 *>(F4)[(size_t)b * Npad + N + k] = MakeT4<T>::make(0.0, 0.0, 0.0);
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
