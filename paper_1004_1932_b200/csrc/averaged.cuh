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
// theorem: no transcendental per pair.  The Y <= 8 CTAs of an s block are one thread-block cluster: each writes its
// partial sums into the shared memory of CTA 0 (distributed shared memory), arrives at the cluster barrier and leaves;
// CTA 0 adds them in the order of the chunks (no global partials, no atomics; results independent of the schedule).  Launched with programmatic stream serialisation: the CTAs become resident while the
// previous kernel of the stream drains and wait (griddepcontrol.wait) before their first global access.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "pack.cuh"

namespace ds {

namespace cg = cooperative_groups;

struct AvgConsts {
    double cj;   // a w (9/64) (lam/ell)^2 ell^4
    double ck;   // w (15/64) (a/ell) (lam/ell)^2 ell^5
};

constexpr int AVG_SB = 32, AVG_W = 16, AVG_NT = AVG_SB * AVG_W, AVG_TILE = 512, AVG_YMAX = 8;

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


// Cluster barrier, split: arrive (release: earlier writes, also those into another CTA's shared memory, are visible to
// whoever completes the wait) and wait (acquire).  A CTA may leave after arriving.
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive_release() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

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
    // tile: units of W dumbbells r (the lanes of a pack, pack.cuh), 8 packs each: R0 R1 R2 N0 N1 N2 sin cos;
    // red (the warps' sums) takes its place after the pair loop
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;
    constexpr size_t BUF = sizeof(T) * (AVG_TILE * 8 > AVG_W * 6 * AVG_SB ? AVG_TILE * 8 : AVG_W * 6 * AVG_SB);
    __shared__ __align__(16) unsigned char buf[BUF];
    V(*tile)[8] = reinterpret_cast<V(*)[8]>(buf);
    T(*red)[6][AVG_SB] = reinterpret_cast<T(*)[6][AVG_SB]>(buf);
    __shared__ double csum[AVG_YMAX][6][AVG_SB];   // used in CTA 0 of the cluster: the sums of all its CTAs
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int Y = gridDim.y;
    if (Y > 1) cluster_arrive_relaxed();         // phase 1: "this CTA runs" (its shared memory may be written)
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
    const V Rv0 = P::bc(Rs[0]), Rv1 = P::bc(Rs[1]), Rv2 = P::bc(Rs[2]), Nv0 = P::bc(Ns[0]), Nv1 = P::bc(Ns[1]), Nv2 = P::bc(Ns[2]);
    const V ssv = P::bc(ss), ncs = P::bc(-cs), Cjv = P::bc((T)C.cj), Ckv = P::bc((T)C.ck);
    const V c1 = P::bc((T)1), c2 = P::bc((T)2), c3 = P::bc((T)3), c4 = P::bc((T)4), c6 = P::bc((T)6), c35 = P::bc((T)35),
            c63 = P::bc((T)63), cm5 = P::bc((T)-5), cm7 = P::bc((T)-7), cm10 = P::bc((T)-10), cm20 = P::bc((T)-20),
            cm21 = P::bc((T)-21), cm42 = P::bc((T)-42);
    V J0 = P::bc((T)0), J1 = J0, J2 = J0, K0 = J0, K1 = J0, K2 = J0;
    for (int t0 = r_lo; t0 < r_hi; t0 += AVG_TILE) {
        if (t0 != r_lo) __syncthreads();
        const int nt = min(r_hi - t0, AVG_TILE), nu = (nt + W - 1) / W;
        if (tid < nu * W) {
            const int r_ = t0 + tid;
            T *slot = reinterpret_cast<T *>(&tile[tid / W][0]) + tid % W;      // component c of r at slot[c * W]
            if (r_ < r_hi) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { slot[c * W] = (T)R[3 * (size_t)r_ + c]; slot[(3 + c) * W] = (T)N[3 * (size_t)r_ + c]; }
                const double2 v = sc[r_];
                slot[6 * W] = (T)v.x; slot[7 * W] = (T)v.y;
            } else {   // the odd lane of the last pack: far away, sin = cos = 0: contributes exactly nothing
#pragma unroll
                for (int c = 0; c < 3; ++c) { slot[c * W] = (T)1e9; slot[(3 + c) * W] = (T)(c == 0); }
                slot[6 * W] = (T)0; slot[7 * W] = (T)0;
            }
        }
        __syncthreads();
#pragma unroll 2
        for (int u = w; u < nu; u += AVG_W) {
            const V *q_ = tile[u];
            const V D0 = P::sub(Rv0, q_[0]), D1 = P::sub(Rv1, q_[1]), D2 = P::sub(Rv2, q_[2]);
            const V d2 = P::fma(D2, D2, P::fma(D1, D1, P::mul(D0, D0)));
            const V di = P::template rsq<true>(d2);          // 0 for r == s (D = 0): no self term
            const V h0 = P::mul(D0, di), h1 = P::mul(D1, di), h2 = P::mul(D2, di);
            const V s = P::fma(h2, Nv2, P::fma(h1, Nv1, P::mul(h0, Nv0)));
            const V r = P::fma(h2, q_[5], P::fma(h1, q_[4], P::mul(h0, q_[3])));
            const V q = P::fma(Nv2, q_[5], P::fma(Nv1, q_[4], P::mul(Nv0, q_[3])));
            const V sn = P::fma(ssv, q_[7], P::mul(ncs, q_[6]));          // sin(phi^s - phi^r)
            const V di2 = P::mul(di, di), di4 = P::mul(di2, di2);
            const V cj = P::mul(P::mul(Cjv, sn), di4), ck = P::mul(P::mul(Ckv, sn), P::mul(di4, di));
            const V sr = P::mul(s, r), r2 = P::mul(r, r), s2 = P::mul(s, s), q2 = P::mul(q, q);
            // (9c): 2s + 4qr - 10 s r^2 and 1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2
            const V jn = P::fma(P::mul(c4, q), r, P::mul(s, P::fma(cm10, r2, c2)));
            const V jd = P::fma(cm5, P::fma(s, s, r2), P::fma(sr, P::fma(c35, sr, P::mul(cm20, q)), P::fma(c2, q2, c1)));
            // (9d): 3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2 - 42 q s^2 r + 63 s^3 r^2
            const V kp = P::fma(sr, P::fma(c63, sr, P::mul(cm42, q)), P::fma(c6, q2, c3));
            const V kd = P::fma(s, P::fma(cm21, r2, P::fma(cm7, s2, kp)), P::mul(P::mul(c6, r), q));
            const V cjd = P::mul(cj, jd), cjn = P::mul(cj, jn), ckd = P::mul(ck, kd);
            J0 = P::fma(Nv0, cjn, P::fma(h0, cjd, J0)); J1 = P::fma(Nv1, cjn, P::fma(h1, cjd, J1));
            J2 = P::fma(Nv2, cjn, P::fma(h2, cjd, J2));
            K0 = P::fma(h0, ckd, K0); K1 = P::fma(h1, ckd, K1); K2 = P::fma(h2, ckd, K2);
        }
    }
    const T J[3] = {P::hsum(J0), P::hsum(J1), P::hsum(J2)}, K[3] = {P::hsum(K0), P::hsum(K1), P::hsum(K2)};
    __syncthreads();                                 // the tile is done with
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
    // what the finishing warp needs from global memory, fetched before it waits for the other CTAs
    const bool fin = w == 0 && blockIdx.y == 0 && live;
    const size_t k0 = 3 * (size_t)s_;
    double n_[3] = {0, 0, 0}, r0_[3] = {0, 0, 0}, n0_[3] = {0, 0, 0}, d1r_[3] = {0, 0, 0}, d1n_[3] = {0, 0, 0};
    if (fin) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            n_[c] = (double)N[k0 + c];
            if (U.mode != AVG_RHS) { r0_[c] = U.R0[k0 + c]; n0_[c] = U.N0[k0 + c]; }
            if (U.mode == AVG_CORR) { d1r_[c] = U.d1R[k0 + c]; d1n_[c] = U.d1N[k0 + c]; }
        }
    }
    if (Y > 1) {
        cluster_wait_acquire();                      // phase 1: every CTA of the cluster runs
        if (w == 0) {
            cg::cluster_group cl = cg::this_cluster();
            double *dst = cl.map_shared_rank(&csum[0][0][0], 0) + (size_t)blockIdx.y * 6 * AVG_SB;
#pragma unroll
            for (int c = 0; c < 6; ++c) dst[c * AVG_SB + lane] = acc[c];
        }
        cluster_arrive_release();                    // phase 2: the sums are in CTA 0
        if (blockIdx.y != 0) return;
        cluster_wait_acquire();
        if (w == 0) {
#pragma unroll
            for (int c = 0; c < 6; ++c) acc[c] = csum[0][c][lane];
#pragma unroll
            for (int y = 1; y < AVG_YMAX; ++y) {
                if (y < Y) {
#pragma unroll
                    for (int c = 0; c < 6; ++c) acc[c] += csum[y][c][lane];
                }
            }
        }
    }
    if (!fin) return;
    {
        const double n0 = n_[0], n1 = n_[1], n2 = n_[2];
        const double nk = n0 * acc[3] + n1 * acc[4] + n2 * acc[5];
        const double vN[3] = {-(acc[3] - n0 * nk), -(acc[4] - n1 * nk), -(acc[5] - n2 * nk)};
        if (U.mode == AVG_RHS) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { dR[k0 + c] = (IO)acc[c]; dN[k0 + c] = (IO)vN[c]; }
        } else {
            double v[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double fr = acc[c], fn = vN[c];
                if (U.mode == AVG_PRED) { U.d1R[k0 + c] = fr; U.d1N[k0 + c] = fn; }
                else { fr = 0.5 * (d1r_[c] + fr); fn = 0.5 * (d1n_[c] + fn); }
                v[c] = n0_[c] + U.dt * fn;
                U.Rout[k0 + c] = r0_[c] + U.dt * fr;
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
