// averaged.cuh -- the stroke-averaged far-field model, Eq. (9a)-(9d): a second
// O(S^2) pair sum, over dumbbells instead of spheres:
//   dR^s/dt = sum_{r != s} J^{sr},      dN^s/dt = -(1 - N^s N^s) sum_{r != s} K^{sr},
//   J^{sr} = a w sin(phi^s - phi^r) (9/64) (lam/ell)^2 (ell/|D|)^4 { N^s (2s + 4qr - 10 s r^2)
//                                  + Dh (1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2) },
//   K^{sr} = w sin(phi^s - phi^r) (15/64) (a/ell) (lam/ell)^2 (ell/|D|)^5 Dh (3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2
//                                  - 42 q s^2 r + 63 s^3 r^2),
//   D = R^s - R^r, Dh = D/|D|, s = Dh.N^s, r = Dh.N^r, q = N^s.N^r.
// The state (R, N) is FP64 (the increments per step are ~1e-7 of |R|: below FP32 resolution); the pair
// arithmetic runs in T.  Grid = (s blocks of 32 dumbbells) x (Y chunks of the r sum); in a CTA lane = s, warp = slice
// of the chunk, so every shared-memory read of an r record is a broadcast.  sin/cos of the phases come from a table
// (avg_sincos_kernel, once per call: the phases are constants of the motion) and sin(phi^s - phi^r) from the addition
// theorem: no transcendental per pair.  The Y <= 8 CTAs of an s block are one thread-block cluster: their partial sums
// are added in the order of the chunks through distributed shared memory (no global partials, no atomics; results
// independent of the schedule).  Launched with programmatic stream serialisation: the CTAs become resident while the
// previous kernel of the stream drains and wait (griddepcontrol.wait) before their first global access.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>

namespace ds {

namespace cg = cooperative_groups;

struct AvgConsts {
    double cj;   // a w (9/64) (lam/ell)^2 ell^4
    double ck;   // w (15/64) (a/ell) (lam/ell)^2 ell^5
};

constexpr int AVG_SB = 32, AVG_W = 8, AVG_NT = AVG_SB * AVG_W, AVG_TILE = 256, AVG_YMAX = 8;

// What the CTA that completes an s block does with the right-hand sides (dR, dN) of its 32 dumbbells:
//   AVG_RHS : write them out (ds_avg_rhs);
//   AVG_PRED: Heun predictor: keep them in d1R, d1N; Rout = R0 + dt dR, Nout = (N0 + dt dN) / |.|;
//   AVG_CORR: corrector: Rout = R0 + (dt/2)(d1R + dR), Nout = (N0 + (dt/2)(d1N + dN)) / |.|.
// N is renormalised after every stage: the projector of (9b) keeps |N| = 1 only to first order in dt.  (R0, N0) is
// the state at the start of the step: the kernel's own input in the predictor, and in the corrector (whose input is the
// predicted state) it may be the same array as (Rout, Nout), each element being read and written by one thread.
enum AvgMode { AVG_RHS = 0, AVG_PRED = 1, AVG_CORR = 2 };
struct AvgUpdate {
    int mode;
    double dt;
    const double *R0, *N0;
    double *d1R, *d1N, *Rout, *Nout;
};

__device__ __forceinline__ float inv_sqrt(float x) { return rsqrtf(x); }
__device__ __forceinline__ double inv_sqrt(double x) { return 1.0 / sqrt(x); }

__global__ void avg_sincos_kernel(const double *__restrict__ phi, int S, double2 *__restrict__ sc) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    double sn, cs;
    sincos(phi[s], &sn, &cs);
    sc[s] = make_double2(sn, cs);
}

// T: type of the pair arithmetic; IO: element type of R, N, dR, dN (double for the FP64 state of ds_avg_step, the user's
// type for the stateless ds_avg_rhs).  gridDim = (ceil(S/32), Y), cluster = (1, Y, 1), chunk = r's per CTA.
template <typename T, typename IO>
__global__ void __launch_bounds__(AVG_NT) avg_rhs_kernel(const IO *__restrict__ R, const IO *__restrict__ N,
                                                         const double2 *__restrict__ sc, int S, int chunk, AvgConsts C,
                                                         IO *__restrict__ dR, IO *__restrict__ dN, AvgUpdate U) {
    __shared__ T tile[AVG_TILE][8];              // R0 R1 R2 N0 | N1 N2 sin cos
    __shared__ T red[AVG_W][6][AVG_SB];
    __shared__ double csum[6][AVG_SB];
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, tid = threadIdx.x;
    const int s_ = blockIdx.x * AVG_SB + lane;
    const bool live = s_ < S;
    const int r_lo = blockIdx.y * chunk, r_hi = min(S, r_lo + chunk);
    T Rs[3] = {0, 0, 0}, Ns[3] = {1, 0, 0}, ss = 0, cs = 1;
    if (live) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { Rs[c] = (T)R[3 * (size_t)s_ + c]; Ns[c] = (T)N[3 * (size_t)s_ + c]; }
        const double2 v = sc[s_];
        ss = (T)v.x; cs = (T)v.y;
    }
    const T Cj = (T)C.cj, Ck = (T)C.ck;
    T J[3] = {0, 0, 0}, K[3] = {0, 0, 0};
    for (int t0 = r_lo; t0 < r_hi; t0 += AVG_TILE) {
        if (t0 != r_lo) __syncthreads();
        {
            const int r_ = t0 + tid;
            if (r_ < r_hi) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { tile[tid][c] = (T)R[3 * (size_t)r_ + c]; tile[tid][3 + c] = (T)N[3 * (size_t)r_ + c]; }
                const double2 v = sc[r_];
                tile[tid][6] = (T)v.x; tile[tid][7] = (T)v.y;
            }
        }
        __syncthreads();
        const int nt = min(r_hi - t0, AVG_TILE);
#pragma unroll 2
        for (int k = w; k < nt; k += AVG_W) {
            const bool on = live && (t0 + k != s_);            // no self term (r != s)
            const T *q_ = tile[k];
            const T D0 = Rs[0] - q_[0], D1 = Rs[1] - q_[1], D2 = Rs[2] - q_[2];
            const T d2 = on ? D0 * D0 + D1 * D1 + D2 * D2 : (T)1;
            const T di = inv_sqrt(d2);
            const T h0 = D0 * di, h1 = D1 * di, h2 = D2 * di;
            const T s = h0 * Ns[0] + h1 * Ns[1] + h2 * Ns[2];
            const T r = h0 * q_[3] + h1 * q_[4] + h2 * q_[5];
            const T q = Ns[0] * q_[3] + Ns[1] * q_[4] + Ns[2] * q_[5];
            const T sn = on ? ss * q_[7] - cs * q_[6] : (T)0;   // sin(phi^s - phi^r)
            const T di2 = di * di, di4 = di2 * di2;
            const T cj = Cj * sn * di4, ck = Ck * sn * (di4 * di);
            const T sr = s * r, r2 = r * r, s2 = s * s, q2 = q * q;
            // (9c): 2s + 4qr - 10 s r^2 and 1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2
            const T jn = s * ((T)2 - (T)10 * r2) + (T)4 * q * r;
            const T jd = (T)1 + (T)2 * q2 - (T)5 * (s2 + r2) + sr * ((T)35 * sr - (T)20 * q);
            // (9d): 3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2 - 42 q s^2 r + 63 s^3 r^2
            const T kd = s * ((T)3 + (T)6 * q2 - (T)7 * s2 - (T)21 * r2 + sr * ((T)63 * sr - (T)42 * q)) + (T)6 * r * q;
            const T cjd = cj * jd, cjn = cj * jn, ckd = ck * kd;
            J[0] += Ns[0] * cjn + h0 * cjd; J[1] += Ns[1] * cjn + h1 * cjd; J[2] += Ns[2] * cjn + h2 * cjd;
            K[0] += h0 * ckd; K[1] += h1 * ckd; K[2] += h2 * ckd;
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) { red[w][c][lane] = J[c]; red[w][3 + c][lane] = K[c]; }
    __syncthreads();
    double acc[6] = {0, 0, 0, 0, 0, 0};
    if (w == 0) {
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            double a = 0.0;
#pragma unroll
            for (int m = 0; m < AVG_W; ++m) a += (double)red[m][c][lane];
            acc[c] = a;
        }
    }
    const int Y = gridDim.y;
    if (Y > 1) {
        // the Y CTAs of an s block form a cluster (1, Y, 1); CTA 0 adds their sums through distributed shared memory,
        // in the order of the chunks
        cg::cluster_group cl = cg::this_cluster();
        if (w == 0) {
#pragma unroll
            for (int c = 0; c < 6; ++c) csum[c][lane] = acc[c];
        }
        cl.sync();
        if (blockIdx.y == 0 && w == 0) {
#pragma unroll
            for (int y = 1; y < AVG_YMAX; ++y) {
                if (y < Y) {
                    const double *rc = cl.map_shared_rank(&csum[0][0], y);
#pragma unroll
                    for (int c = 0; c < 6; ++c) acc[c] += rc[c * AVG_SB + lane];
                }
            }
        }
        cl.sync();                                   // no CTA leaves while its sums may still be read
    }
    if (w != 0 || blockIdx.y != 0) return;
    if (live) {
        const double n0 = (double)N[3 * (size_t)s_], n1 = (double)N[3 * (size_t)s_ + 1], n2 = (double)N[3 * (size_t)s_ + 2];
        const double nk = n0 * acc[3] + n1 * acc[4] + n2 * acc[5];
        const double vN[3] = {-(acc[3] - n0 * nk), -(acc[4] - n1 * nk), -(acc[5] - n2 * nk)};
        const size_t k0 = 3 * (size_t)s_;
        if (U.mode == AVG_RHS) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { dR[k0 + c] = (IO)acc[c]; dN[k0 + c] = (IO)vN[c]; }
        } else {
            double v[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double fr = acc[c], fn = vN[c];
                if (U.mode == AVG_PRED) { U.d1R[k0 + c] = fr; U.d1N[k0 + c] = fn; }
                else { fr = 0.5 * (U.d1R[k0 + c] + fr); fn = 0.5 * (U.d1N[k0 + c] + fn); }
                const double r0 = U.R0[k0 + c];
                v[c] = U.N0[k0 + c] + U.dt * fn;
                U.Rout[k0 + c] = r0 + U.dt * fr;
            }
            const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
#pragma unroll
            for (int c = 0; c < 3; ++c) U.Nout[k0 + c] = v[c] / len;
        }
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

}  // namespace ds
