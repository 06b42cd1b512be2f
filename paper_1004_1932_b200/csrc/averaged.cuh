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
#include <stdint.h>

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

// The s side of a pair and the constants of Eq. (9c,d), broadcast to the lanes of a pack.
template <typename T> struct AvgRegs {
    typedef Pack<T> P;
    typedef typename P::V V;
    V Rv0, Rv1, Rv2, Nv0, Nv1, Nv2, ssv, ncs, Cjv, Ckv;
    __device__ __forceinline__ AvgRegs(const T (&Rs)[3], const T (&Ns)[3], T ss, T cs, const AvgConsts &C)
        : Rv0(P::bc(Rs[0])), Rv1(P::bc(Rs[1])), Rv2(P::bc(Rs[2])), Nv0(P::bc(Ns[0])), Nv1(P::bc(Ns[1])), Nv2(P::bc(Ns[2])),
          ssv(P::bc(ss)), ncs(P::bc(-cs)), Cjv(P::bc((T)C.cj)), Ckv(P::bc((T)C.ck)) {}
};

// One unit of W dumbbells r (8 packs: R0 R1 R2 N0 N1 N2 sin cos) against dumbbell s: J and K of Eq. (9c), (9d) added to the sums.
template <typename T>
__device__ __forceinline__ void avg_pair(const typename Pack<T>::V *__restrict__ q_, const AvgRegs<T> &A, typename Pack<T>::V &J0,
                                         typename Pack<T>::V &J1, typename Pack<T>::V &J2, typename Pack<T>::V &K0,
                                         typename Pack<T>::V &K1, typename Pack<T>::V &K2) {
    typedef Pack<T> P;
    typedef typename P::V V;
    const V c1 = P::bc((T)1), c2 = P::bc((T)2), c3 = P::bc((T)3), c4 = P::bc((T)4), c6 = P::bc((T)6), c35 = P::bc((T)35),
            c63 = P::bc((T)63), cm5 = P::bc((T)-5), cm7 = P::bc((T)-7), cm10 = P::bc((T)-10), cm20 = P::bc((T)-20),
            cm21 = P::bc((T)-21), cm42 = P::bc((T)-42);
    const V D0 = P::sub(A.Rv0, q_[0]), D1 = P::sub(A.Rv1, q_[1]), D2 = P::sub(A.Rv2, q_[2]);
    const V d2 = P::fma(D2, D2, P::fma(D1, D1, P::mul(D0, D0)));
    const V di = P::template rsq<true>(d2);          // 0 for r == s (D = 0): no self term
    const V h0 = P::mul(D0, di), h1 = P::mul(D1, di), h2 = P::mul(D2, di);
    const V s = P::fma(h2, A.Nv2, P::fma(h1, A.Nv1, P::mul(h0, A.Nv0)));
    const V r = P::fma(h2, q_[5], P::fma(h1, q_[4], P::mul(h0, q_[3])));
    const V q = P::fma(A.Nv2, q_[5], P::fma(A.Nv1, q_[4], P::mul(A.Nv0, q_[3])));
    const V sn = P::fma(A.ssv, q_[7], P::mul(A.ncs, q_[6]));          // sin(phi^s - phi^r)
    const V di2 = P::mul(di, di), di4 = P::mul(di2, di2);
    const V cj = P::mul(P::mul(A.Cjv, sn), di4), ck = P::mul(P::mul(A.Ckv, sn), P::mul(di4, di));
    const V sr = P::mul(s, r), r2 = P::mul(r, r), s2 = P::mul(s, s), q2 = P::mul(q, q);
    // (9c): 2s + 4qr - 10 s r^2 and 1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2
    const V jn = P::fma(P::mul(c4, q), r, P::mul(s, P::fma(cm10, r2, c2)));
    const V jd = P::fma(cm5, P::fma(s, s, r2), P::fma(sr, P::fma(c35, sr, P::mul(cm20, q)), P::fma(c2, q2, c1)));
    // (9d): 3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2 - 42 q s^2 r + 63 s^3 r^2
    const V kp = P::fma(sr, P::fma(c63, sr, P::mul(cm42, q)), P::fma(c6, q2, c3));
    const V kd = P::fma(s, P::fma(cm21, r2, P::fma(cm7, s2, kp)), P::mul(P::mul(c6, r), q));
    const V cjd = P::mul(cj, jd), cjn = P::mul(cj, jn), ckd = P::mul(ck, kd);
    J0 = P::fma(A.Nv0, cjn, P::fma(h0, cjd, J0)); J1 = P::fma(A.Nv1, cjn, P::fma(h1, cjd, J1));
    J2 = P::fma(A.Nv2, cjn, P::fma(h2, cjd, J2));
    K0 = P::fma(h0, ckd, K0); K1 = P::fma(h1, ckd, K1); K2 = P::fma(h2, ckd, K2);
}

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
    const AvgRegs<T> A_(Rs, Ns, ss, cs, C);
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
            avg_pair<T>(tile[u], A_, J0, J1, J2, K0, K1, K2);
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

// ---------------------------------------------------------------------------------------------------------------------
// Device-resident Heun stepping of Eq. (9) for the paper's sizes (S up to a few thousand): ONE
// cooperative launch runs all n_steps; no host round trip, no kernel boundary per stage.
//   grid = G CTAs, CTA c owns the dumbbells [c ns, (c + 1) ns); thread = (own dumbbell, slice of the r sum).
//   The FP64 state of a dumbbell (R, N, the predictor's right-hand sides) lives in the registers of ONE owner thread for
//   the whole launch.  A stage: every CTA fills its shared-memory tile with the T-rounded records (R, N, sin, cos) of ALL
//   S dumbbells of the stage's input -> pair sums -> fixed-order sum over the slices -> the owner applies the Heun
//   predictor / corrector (N renormalised, reading R16) -> publishes its record of the next stage.
//   Hand-over without a barrier or a fence: a record is published as (word, tag) pairs, 8 bytes each (single-copy
//   atomic), tag = number of the stage that reads it; readers poll a 16-byte piece until both tags show.  Two ping-pong
//   buffers suffice: nobody can publish stage g + 2 before it has read ALL of stage g + 1, which nobody publishes
//   before it has finished reading stage g.
struct AvgPersistArgs {
    int S, ns;                       // dumbbells; dumbbells per CTA
    double *R, *N;                   // FP64 state [S][3], read at the start, written at the end
    const double2 *sc;               // sin / cos of the phases
    AvgConsts C;
    double dt;
    long long n_steps;
    uint4 *xch[2];                   // ping-pong exchange buffers: S records of 8 T words, every 32-bit word beside a tag
    unsigned int tag0;               // tag of the first stage's input; stage g reads tag0 + g
    long long *probe;                // dev instrumentation (DS_ENABLE_PROBE builds) or NULL
};

#ifdef DS_ENABLE_PROBE
#define AVG_PROBE(slot) do { if (A.probe != nullptr && tid == 0 && g == n_stage - 2) A.probe[blockIdx.x * 16 + (slot)] = clock64(); } while (0)
#else
#define AVG_PROBE(slot) do { } while (0)
#endif

template <typename T> __global__ void __launch_bounds__(AVG_NT, 1) avg_persist_kernel(const AvgPersistArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;
    constexpr int PPR = 8 * (int)sizeof(T) / 8;          // 16-byte tagged pieces per record: 4 (FP32), 8 (FP64)
    extern __shared__ __align__(16) unsigned char avg_smem[];
    const int S = A.S, ns = A.ns, tid = threadIdx.x;
    const int nu = (S + W - 1) / W;
    V(*tile)[8] = reinterpret_cast<V(*)[8]>(avg_smem);                          // [nu][8]
    T *red = reinterpret_cast<T *>(avg_smem + (size_t)nu * 8 * sizeof(V));      // [n_sl][6 ns]
    const int s0 = blockIdx.x * ns, nown = min(ns, S - s0);                     // own dumbbells (>= 1 by the grid size)
    const int n_sl = AVG_NT / ns;                                               // slices of the r sum
    const int sl = tid / ns, is = tid - sl * ns;                                // thread = (slice, own dumbbell)
    const bool active = sl < n_sl && is < nown;
    double *red2 = reinterpret_cast<double *>(red + (size_t)n_sl * 6 * ns);     // [6 ns]
    const int n_out = 6 * ns;
    // owner thread of dumbbell s0 + tid (tid < nown): its FP64 state
    const bool owner = tid < nown;
    // (in shared memory, one row of 20 doubles per own dumbbell, so that the pair loop has the registers to itself)
    double *const own_st = red2 + n_out + 20 * (owner ? tid : 0);
    double *const R0 = own_st, *const N0 = own_st + 3, *const Rc = own_st + 6, *const Nc = own_st + 9, *const d1R = own_st + 12,
                 *const d1N = own_st + 15;
    T sn_ = 0, cs_ = 0;
    auto publish = [&](int buf, unsigned int tag) {          // the owner's record of (Rc, Nc): R N sin cos, rounded to T
        const T rec[8] = {(T)Rc[0], (T)Rc[1], (T)Rc[2], (T)Nc[0], (T)Nc[1], (T)Nc[2], sn_, cs_};
        uint4 *q = A.xch[buf] + (size_t)(s0 + tid) * PPR;
        if (sizeof(T) == 4) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                q[k] = make_uint4(__float_as_uint((float)rec[2 * k]), tag, __float_as_uint((float)rec[2 * k + 1]), tag);
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                q[k] = make_uint4((uint32_t)__double2loint((double)rec[k]), tag, (uint32_t)__double2hiint((double)rec[k]), tag);
        }
    };
    if (owner) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { R0[c] = Rc[c] = A.R[3 * (size_t)(s0 + tid) + c]; N0[c] = Nc[c] = A.N[3 * (size_t)(s0 + tid) + c]; }
        const double2 v = A.sc[s0 + tid];
        sn_ = (T)v.x; cs_ = (T)v.y;
        publish(0, A.tag0);
    }
    if (W == 2 && (S & 1) && tid == 0) {   // the odd lane of the last pack: far away, sin = cos = 0: contributes exactly nothing
        T *slot = reinterpret_cast<T *>(&tile[nu - 1][0]) + 1;
#pragma unroll
        for (int c = 0; c < 3; ++c) { slot[c * W] = (T)1e9; slot[(3 + c) * W] = (T)(c == 0); }
        slot[6 * W] = (T)0; slot[7 * W] = (T)0;
    }
    const long long n_stage = 2 * A.n_steps;
    for (long long g = 0; g < n_stage; ++g) {
        const unsigned int tag = A.tag0 + (unsigned int)g;
        const uint4 *src = A.xch[g & 1];
        AVG_PROBE(0);
        // ---- the stage's input: all S records, piece by piece as the owners' stores land ----
        // (a thread's loads are issued eight at a time before the first tag is looked at: one L2 round trip per batch)
        for (int pc0 = tid; pc0 < S * PPR; pc0 += 8 * AVG_NT) {
            uint4 v[8];
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                const int pc = pc0 + b * AVG_NT;
                if (pc < S * PPR)
                    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v[b].x), "=r"(v[b].y), "=r"(v[b].z), "=r"(v[b].w) : "l"(src + pc) : "memory");
            }
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                const int pc = pc0 + b * AVG_NT;
                if (pc >= S * PPR) continue;
                while (v[b].y != tag || v[b].w != tag)
                    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v[b].x), "=r"(v[b].y), "=r"(v[b].z), "=r"(v[b].w) : "l"(src + pc) : "memory");
                const int r_ = pc / PPR, k = pc - r_ * PPR;
                if (sizeof(T) == 4) {      // words 2k, 2k + 1 of the record = components 2k, 2k + 1 of dumbbell r
                    T *slot = reinterpret_cast<T *>(&tile[r_ / W][0]) + r_ % W;
                    slot[(2 * k) * W] = (T)__uint_as_float(v[b].x);
                    slot[(2 * k + 1) * W] = (T)__uint_as_float(v[b].z);
                } else {
                    reinterpret_cast<T *>(&tile[r_][0])[k] = (T)__hiloint2double((int)v[b].z, (int)v[b].x);
                }
            }
        }
        AVG_PROBE(1);
        __syncthreads();
        AVG_PROBE(2);
        // ---- pair sums of the own dumbbells over this thread's slice of r ----
        V J0 = P::bc((T)0), J1 = J0, J2 = J0, K0 = J0, K1 = J0, K2 = J0;
        if (active) {
            const T *own = reinterpret_cast<const T *>(&tile[(s0 + is) / W][0]) + (s0 + is) % W;
            const T Rs[3] = {own[0], own[W], own[2 * W]}, Ns[3] = {own[3 * W], own[4 * W], own[5 * W]};
            const AvgRegs<T> A_(Rs, Ns, own[6 * W], own[7 * W], A.C);
#pragma unroll 2
            for (int u = sl; u < nu; u += n_sl) avg_pair<T>(tile[u], A_, J0, J1, J2, K0, K1, K2);
            T *o = red + (size_t)sl * n_out + is;
            o[0] = P::hsum(J0); o[ns] = P::hsum(J1); o[2 * ns] = P::hsum(J2);
            o[3 * ns] = P::hsum(K0); o[4 * ns] = P::hsum(K1); o[5 * ns] = P::hsum(K2);
        }
        AVG_PROBE(3);
        __syncthreads();
        AVG_PROBE(4);
        // ---- sum over the slices in a fixed order: a warp per output, lanes take every 32nd slice, then a shuffle tree ----
        for (int o = tid >> 5; o < n_out; o += AVG_NT / 32) {
            T a = T(0);
            for (int j = tid & 31; j < n_sl; j += 32) a += red[(size_t)j * n_out + o];
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) a += __shfl_xor_sync(0xffffffffu, a, d);
            if ((tid & 31) == 0) red2[o] = (double)a;
        }
        AVG_PROBE(5);
        __syncthreads();
        AVG_PROBE(6);
        if (owner) {
            double acc[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) acc[c] = red2[c * ns + tid];
            // right-hand sides of (9a), (9b) at the stage's input (Rc, Nc); Heun
            const double nk = Nc[0] * acc[3] + Nc[1] * acc[4] + Nc[2] * acc[5];
            const double vN[3] = {-(acc[3] - Nc[0] * nk), -(acc[4] - Nc[1] * nk), -(acc[5] - Nc[2] * nk)};
            const bool predictor = (g & 1) == 0;
            double v[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double fr = acc[c], fn = vN[c];
                if (predictor) { d1R[c] = fr; d1N[c] = fn; }
                else { fr = 0.5 * (d1R[c] + fr); fn = 0.5 * (d1N[c] + fn); }
                v[c] = N0[c] + A.dt * fn;
                Rc[c] = R0[c] + A.dt * fr;
            }
            const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
#pragma unroll
            for (int c = 0; c < 3; ++c) Nc[c] = v[c] / len;
            if (!predictor) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { R0[c] = Rc[c]; N0[c] = Nc[c]; }
            }
            if (g + 1 < n_stage) publish((int)((g + 1) & 1), tag + 1u);
        }
        AVG_PROBE(7);
        // (the tile is rewritten only after the next stage's records arrive, which needs this CTA's own publish: all
        //  threads are past the pair loop by then because of the two barriers above)
    }
    if (owner) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { A.R[3 * (size_t)(s0 + tid) + c] = R0[c]; A.N[3 * (size_t)(s0 + tid) + c] = N0[c]; }
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
