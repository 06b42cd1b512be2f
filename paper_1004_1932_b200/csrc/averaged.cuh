// averaged.cuh -- the stroke-averaged far-field model, Eq. (9a)-(9d): a second
// O(S^2) pair sum, over dumbbells instead of spheres:
//   dR^s/dt = sum_{r != s} J^{sr},      dN^s/dt = -(1 - N^s N^s) sum_{r != s} K^{sr},
//   J^{sr} = a w sin(phi^s - phi^r) (9/64) (lam/ell)^2 (ell/|D|)^4 { N^s (2s + 4qr - 10 s r^2)
//                                  + Dh (1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2) },
//   K^{sr} = w sin(phi^s - phi^r) (15/64) (a/ell) (lam/ell)^2 (ell/|D|)^5 Dh (3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2
//                                  - 42 q s^2 r + 63 s^3 r^2),
//   D = R^s - R^r, Dh = D/|D|, s = Dh.N^s, r = Dh.N^r, q = N^s.N^r.
// The state (R, N) is FP64 (the increments per step are ~1e-7 of |R|: below FP32 resolution); the pair
// arithmetic runs in T.  Block = 16 dumbbells s x 16 slices of the r loop; r tiles of 256 staged in shared memory with
// sin/cos of the phases (sin(phi^s - phi^r) by the addition theorem: no transcendental per pair).
#pragma once
#include <cuda_runtime.h>

namespace ds {

struct AvgConsts {
    double cj;   // a w (9/64) (lam/ell)^2 ell^4
    double ck;   // w (15/64) (a/ell) (lam/ell)^2 ell^5
};

constexpr int AVG_SB = 16, AVG_SL = 16, AVG_TILE = 256;

__device__ __forceinline__ float inv_sqrt(float x) { return rsqrtf(x); }
__device__ __forceinline__ double inv_sqrt(double x) { return 1.0 / sqrt(x); }

// T: type of the pair arithmetic; IO: element type of R, N, dR, dN (double for the FP64 state of ds_avg_step, the user's
// type for the stateless ds_avg_rhs)
template <typename T, typename IO>
__global__ void __launch_bounds__(AVG_SB *AVG_SL) avg_rhs_kernel(const IO *__restrict__ R, const IO *__restrict__ N,
                                                                  const double *__restrict__ phi, int S, AvgConsts C,
                                                                  IO *__restrict__ dR, IO *__restrict__ dN) {
    __shared__ T tR[AVG_TILE][3], tN[AVG_TILE][3], tS[AVG_TILE], tC[AVG_TILE];
    __shared__ T part[AVG_SL][AVG_SB][6];
    const int ls = threadIdx.x, sl = threadIdx.y, tid = sl * AVG_SB + ls;
    const int s_ = blockIdx.x * AVG_SB + ls;
    const bool live = s_ < S;
    T Rs[3] = {0, 0, 0}, Ns[3] = {1, 0, 0}, ss = 0, cs = 1;
    if (live) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { Rs[c] = (T)R[3 * (size_t)s_ + c]; Ns[c] = (T)N[3 * (size_t)s_ + c]; }
        ss = (T)sin(phi[s_]); cs = (T)cos(phi[s_]);
    }
    T J[3] = {0, 0, 0}, K[3] = {0, 0, 0};
    for (int t0 = 0; t0 < S; t0 += AVG_TILE) {
        __syncthreads();
        {
            const int r_ = t0 + tid;
            if (r_ < S) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { tR[tid][c] = (T)R[3 * (size_t)r_ + c]; tN[tid][c] = (T)N[3 * (size_t)r_ + c]; }
                tS[tid] = (T)sin(phi[r_]); tC[tid] = (T)cos(phi[r_]);
            }
        }
        __syncthreads();
        const int nt = S - t0 < AVG_TILE ? S - t0 : AVG_TILE;
        for (int k = sl; k < nt; k += AVG_SL) {
            if (t0 + k == s_ || !live) continue;
            const T D0 = Rs[0] - tR[k][0], D1 = Rs[1] - tR[k][1], D2 = Rs[2] - tR[k][2];
            const T d2 = D0 * D0 + D1 * D1 + D2 * D2;
            const T di = inv_sqrt(d2);
            const T h0 = D0 * di, h1 = D1 * di, h2 = D2 * di;
            const T s = h0 * Ns[0] + h1 * Ns[1] + h2 * Ns[2];
            const T r = h0 * tN[k][0] + h1 * tN[k][1] + h2 * tN[k][2];
            const T q = Ns[0] * tN[k][0] + Ns[1] * tN[k][1] + Ns[2] * tN[k][2];
            const T sn = ss * tC[k] - cs * tS[k];          // sin(phi^s - phi^r)
            const T di2 = di * di, di4 = di2 * di2;
            const T cj = (T)C.cj * sn * di4, ck = (T)C.ck * sn * di4 * di;
            const T jn = (T)2 * s + (T)4 * q * r - (T)10 * s * r * r;
            const T jd = (T)1 + (T)2 * q * q - (T)5 * s * s - (T)5 * r * r - (T)20 * q * s * r + (T)35 * s * s * r * r;
            const T kd = (T)3 * s + (T)6 * r * q + (T)6 * s * q * q - (T)7 * s * s * s - (T)21 * s * r * r - (T)42 * q * s * s * r +
                         (T)63 * s * s * s * r * r;
            J[0] += cj * (Ns[0] * jn + h0 * jd); J[1] += cj * (Ns[1] * jn + h1 * jd); J[2] += cj * (Ns[2] * jn + h2 * jd);
            K[0] += ck * h0 * kd; K[1] += ck * h1 * kd; K[2] += ck * h2 * kd;
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) { part[sl][ls][c] = J[c]; part[sl][ls][3 + c] = K[c]; }
    __syncthreads();
    if (sl == 0 && live) {
        double Js[3], Ks[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double a = 0.0, b = 0.0;
            for (int m = 0; m < AVG_SL; ++m) { a += (double)part[m][ls][c]; b += (double)part[m][ls][3 + c]; }
            Js[c] = a; Ks[c] = b;
        }
        const double n0 = (double)N[3 * (size_t)s_], n1 = (double)N[3 * (size_t)s_ + 1], n2 = (double)N[3 * (size_t)s_ + 2];
        const double nk = n0 * Ks[0] + n1 * Ks[1] + n2 * Ks[2];
        dR[3 * (size_t)s_] = (IO)Js[0]; dR[3 * (size_t)s_ + 1] = (IO)Js[1]; dR[3 * (size_t)s_ + 2] = (IO)Js[2];
        dN[3 * (size_t)s_] = (IO)(-(Ks[0] - n0 * nk)); dN[3 * (size_t)s_ + 1] = (IO)(-(Ks[1] - n1 * nk));
        dN[3 * (size_t)s_ + 2] = (IO)(-(Ks[2] - n2 * nk));
    }
}

// user precision <-> FP64
template <typename T> __global__ void widen_kernel(const T *in, double *out, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (double)in[i];
}
template <typename T> __global__ void narrow_kernel(const double *in, T *out, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (T)in[i];
}

// One Heun stage of Eq. (9) on the FP64 state, one thread per dumbbell:
//   predictor (second == 0): Rout = R + dt dR1, Nout = (N + dt dN1) / |.|
//   corrector (second == 1): Rout = R + (dt/2)(dR1 + dR2), Nout = (N + (dt/2)(dN1 + dN2)) / |.|
// N is renormalised after every stage: the projector of (9b) keeps |N| = 1 only to first order in dt.
__global__ void avg_update_kernel(const double *R, const double *N, const double *dR1, const double *dN1, const double *dR2,
                                  const double *dN2, double dt, int second, int S, double *Rout, double *Nout) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    double v[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)s + c;
        const double fr = second ? 0.5 * (dR1[k] + dR2[k]) : dR1[k], fn = second ? 0.5 * (dN1[k] + dN2[k]) : dN1[k];
        Rout[k] = R[k] + dt * fr;
        v[c] = N[k] + dt * fn;
    }
    const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
#pragma unroll
    for (int c = 0; c < 3; ++c) Nout[3 * (size_t)s + c] = v[c] / len;
}

}  // namespace ds
