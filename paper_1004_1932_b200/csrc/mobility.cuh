// mobility.cuh -- the hot kernel: matrix-free all-pairs mobility apply, Eq. (1a) deterministic
// part with the tensor of Eq. (3a,3b), fused with the O(N) rest of the time
// step (self term, reduction, integrator update, next force evaluation) and
// with the step loop itself: ONE launch runs all n_steps of ds_step / ds_batch_step.
//
// Decomposition ("row owner": no partial sum ever leaves the SM).
//   grid = (n_cta row tiles, systems), one CTA of NT = 512 threads per SM.
//   The N alpha-spheres of a system are cut into NQ = ceil(N/4) quads; CTA c owns the contiguous
//   quads [c NQ / n_cta, (c+1) NQ / n_cta) -- nq of them, chosen by the host so that
//   systems * n_cta fills the 148 SMs (N = 4096: 148 CTAs of 6 or 7 quads).
//   Thread t = (ith, jg) = (t % nq, t / nq): it keeps the I = 4 alpha-spheres of quad q0 + ith in
//   registers and belongs to beta-group jg of n_jg = NT / nq.  The split over beta is therefore
//   INSIDE the CTA; it is undone through shared memory in a fixed order (deterministic, no
//   floating-point atomics, no global scratch).
//   Every CTA streams ALL beta-spheres of its system through a ring of shared-memory slots filled
//   by TMA bulk copies (cp.async.bulk global -> shared, completion on an mbarrier; one elected
//   thread issues them, consumer warps release slots through a second mbarrier).  The beta-stream
//   lives in global memory (L2-resident) in the exact shared-memory layout ("units", see pack.cuh):
//   one unit = W beta-spheres = 6 packs = 48 bytes, so a chunk is one contiguous copy.  N = 4096
//   (FP32: 96 KB, FP64: 192 KB) is resident at once: all copies are issued up front.
//   Inside a chunk, group jg takes units jg, jg + n_jg, ... (consecutive groups read consecutive
//   48-byte units: conflict-free LDS.128, broadcast within a group); a chunk holds a multiple of
//   n_jg units (the stream is padded with far-away zero-force units), so every thread of the CTA
//   makes the same number of iterations.
//   r = 0 (alpha == beta) is excluded by a guarded rsqrt compiled only into the loop variant used
//   for chunks that intersect the CTA's own rows (CTA-uniform choice).
//
// Time stepping (RUN_STEP).  The CTA keeps its rows' state (X_n, V1, F; FP64) in shared memory for
// the whole launch.  A stage = pair sum over the input stream -> reduction -> Eq. (3a) self term ->
// integrator update -> Eq. (4) at the new positions -> publish the CTA's rows of the next stage's
// stream (ping-pong buffer in global memory) -> inter-CTA barrier (one arrival counter per system,
// release/acquire at gpu scope; the grid is launched cooperatively so all CTAs are co-resident).
// Heun = 2 stages per step, Euler = 1.  No host round trip, no kernel boundary per step.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pack.cuh"

namespace ds {

enum { TENSOR_OSEEN = 0, TENSOR_RPY = 1 };
enum RunMode { RUN_APPLY = 0, RUN_VELOCITY = 1, RUN_STEP = 2 };

constexpr int NT = 512;                  // threads per CTA: 16 warps, one CTA per SM
constexpr int QI = 4;                    // alpha-spheres per thread (one quad)
constexpr int UNIT_BYTES = 48;           // 6 packs of 8 bytes: x y z Fx Fy Fz of W beta-spheres
constexpr int CHU = 512;                 // units per ring slot (24 KB)
constexpr int SLOT_BYTES = CHU * UNIT_BYTES;
constexpr int NS_MAX = 8;                // ring slots (192 KB)
constexpr int NS_MIN = 4;                // the reduction scratch aliases the first 4 slots (96 KB)
constexpr int BAR_BYTES = 2 * NS_MAX * 8;
constexpr int SMEM_MAX = 232448;         // 227 KB opt-in limit per CTA on sm_100
constexpr int PAD_UNITS = CHU;           // dummy units appended to every system's stream
constexpr int STATE_BYTES_PER_ROW = 12 * 8 + 8;  // X_n, X of the stage, V1, F (3 doubles each) + (phase, L) per dumbbell = 16 B / 2 rows
constexpr int PROBE_SLOTS = 16;

struct RunArgs {
    // problem
    int N, NQ, U, n_cta;      // spheres, quads = ceil(N/4), units = ceil(N/W), row tiles per system
    int ns;                   // ring slots in use (NS_MIN..NS_MAX)
    int b0;                   // first system of this launch (blockIdx.y is relative to it)
    long long unit_stride;    // units per system in the streams (>= U + PAD_UNITS)
    void *units[2];           // beta-streams T[B][unit_stride][6][W]; stage g reads units[(cur+g)&1]
    int cur;
    // Eq. (3) constants
    double self_mob;  // 1/(6 pi eta a)   Eq. (3a)
    double pre;       // 1/(8 pi eta)     Eq. (3b)
    double c1, c2;    // 2a^2/3, 2a^2     second line of Eq. (3b), see pair body
    // what to run
    int mode;                 // RunMode
    int heun;                 // RUN_STEP: 1 = Heun (2 stages per step), 0 = Euler
    long long n0, n_steps;    // RUN_STEP: index of the first step, number of steps
    void *out_u;              // RUN_APPLY / RUN_VELOCITY: u [B][N][3] user precision
    double *X;                // state positions [B][N][3] (read at start; written at the end of RUN_STEP)
    const double *phase;      // [B][S]
    double t0, dt, ell, lambda, omega, k0;
    // inter-CTA barrier: one monotonic arrival counter per system; this launch starts at bar_base
    unsigned long long *bar;
    unsigned long long bar_base;
    // state rows in shared memory (1) or, for very large tiles, in these global arrays (0)
    int state_smem;
    double *Xcg, *V1g, *Fg, *Lg;  // [B][N][3] x 3, [B][S]
    long long *probe;         // dev instrumentation: PROBE_SLOTS clock samples per CTA, or NULL
};

template <typename T> struct alignas(16) V2 {
    typename Pack<T>::V a, b;
};

// ---------------------------------------------------------------------------------------------
// mbarrier / TMA bulk-copy primitives (PTX; sm_90+ forms, SASS: SYNCS.*, UBLKCP)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy of `bytes` (multiple of 16; both addresses 16-byte aligned), completing on bar
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// generic-proxy accesses (other CTAs' st.global seen through the acquire below; this CTA's own
// ld/st.shared to the ring while it served as scratch) ordered before later async-proxy (TMA) accesses
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_shared() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu(unsigned long long *p, unsigned long long v) {
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---------------------------------------------------------------------------------------------
// The pair body.  With r = x_a - x_b, w = 1/r^2, Eq. (3b) contracted with F_b is
//   Oseen: (1/8 pi mu) (1/r) [ F_b + (r.F_b) w r ]
//   RPY  : (1/8 pi mu) { (1/r + c1/r^3) F_b + (r.F_b) (1/r^3) (1 - c2 w) r },  c1 = 2a^2/3, c2 = 2a^2
// (second line of (3b): 2a^2/(24 pi mu r^3) (delta - 3 rr/r^2) = (1/8 pi mu)(1/r^3)[(2a^2/3) delta - 2a^2 rr/r^2]).
// The common factor 1/(8 pi mu) is applied once per alpha in the epilogue.
// FMA-pipe instruction count per pack: 3 sub + 3 (r^2) + 3 (r.F) + 2 + 6 = 17 (Oseen), 21 (RPY).
template <typename T, int TENSOR, bool GUARD>
__device__ __forceinline__ void pair_units(const V2<T> *__restrict__ p, int stride, int iters,
                                           const typename Pack<T>::V (&xi)[QI][3],
                                           typename Pack<T>::V (&acc)[QI][3], typename Pack<T>::V c1,
                                           typename Pack<T>::V negc2) {
    typedef Pack<T> P;
    typedef typename P::V V;
#pragma unroll 2
    for (int r = 0; r < iters; ++r, p += stride) {
        const V2<T> q0 = p[0], q1 = p[1], q2 = p[2];
        const V xj = q0.a, yj = q0.b, zj = q1.a, fx = q1.b, fy = q2.a, fz = q2.b;
#pragma unroll
        for (int k = 0; k < QI; ++k) {
            const V dx = P::sub(xi[k][0], xj), dy = P::sub(xi[k][1], yj), dz = P::sub(xi[k][2], zj);
            const V r2 = P::fma(dz, dz, P::fma(dy, dy, P::mul(dx, dx)));
            const V ri = P::template rsq<GUARD>(r2);
            const V rf = P::fma(dz, fz, P::fma(dy, fy, P::mul(dx, fx)));
            const V w = P::mul(ri, ri);
            if (TENSOR == TENSOR_OSEEN) {
                const V s2 = P::mul(rf, w);
                const V tx = P::fma(s2, dx, fx), ty = P::fma(s2, dy, fy), tz = P::fma(s2, dz, fz);
                acc[k][0] = P::fma(ri, tx, acc[k][0]);
                acc[k][1] = P::fma(ri, ty, acc[k][1]);
                acc[k][2] = P::fma(ri, tz, acc[k][2]);
            } else {
                const V ri3 = P::mul(ri, w);
                const V ca = P::fma(c1, ri3, ri);
                const V e = P::fma(negc2, w, P::bc(T(1)));
                const V g = P::mul(rf, ri3);
                const V cb = P::mul(g, e);
                acc[k][0] = P::fma(cb, dx, P::fma(ca, fx, acc[k][0]));
                acc[k][1] = P::fma(cb, dy, P::fma(ca, fy, acc[k][1]));
                acc[k][2] = P::fma(cb, dz, P::fma(ca, fz, acc[k][2]));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Eq. (4).  Explicit rounding (no contraction) so that every call site produces
// the same bits for the same inputs: ds_step(n) is bit-identical however the n steps are split.
//   L^s(t) = ell + lambda sin(omega t + phi^s)
__device__ __forceinline__ double stroke_length(double t, double phi, double ell, double lambda, double omega) {
    return __dadd_rn(ell, __dmul_rn(lambda, sin(__dadd_rn(__dmul_rn(omega, t), phi))));
}
//   n = (X_{2s+1} - X_{2s})/d, g = k0 (d - L), F_{2s} = +g n, F_{2s+1} = -g n   (F = -dU/dX)
__device__ __forceinline__ void dumbbell_force(const double (&x0)[3], const double (&x1)[3], double L, double k0,
                                               double (&F0)[3]) {
    const double s0 = __dsub_rn(x1[0], x0[0]), s1 = __dsub_rn(x1[1], x0[1]), s2 = __dsub_rn(x1[2], x0[2]);
    const double d = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(s0, s0), __dmul_rn(s1, s1)), __dmul_rn(s2, s2)));
    const double g = __dmul_rn(k0, __dsub_rn(d, L));
    F0[0] = __dmul_rn(g, __ddiv_rn(s0, d));
    F0[1] = __dmul_rn(g, __ddiv_rn(s1, d));
    F0[2] = __dmul_rn(g, __ddiv_rn(s2, d));
}
// t_n = t0 + n dt, formed from the step index (never accumulated), no contraction
__device__ __forceinline__ double time_of_step(double t0, long long n, double dt) {
    return __dadd_rn(t0, __dmul_rn((double)n, dt));
}

// element (sphere i, component c in 0..5 = x y z Fx Fy Fz) of a unit stream
template <typename T> __device__ __forceinline__ size_t unit_index(long long i, int c) {
    constexpr int W = Pack<T>::W;
    return (size_t)(i / W) * (6 * W) + (size_t)c * W + (size_t)(i % W);
}

// The two spheres i0 (even), i0 + 1 of one dumbbell -> their units of a stream, rounded to T.
__device__ __forceinline__ void publish_dumbbell(float *un, long long i0, const double (&x0)[3], const double (&x1)[3],
                                                 const double (&F0)[3]) {
    float4 *p = reinterpret_cast<float4 *>(un + (size_t)(i0 >> 1) * 12);  // one unit: [x0 x1][y0 y1][z0 z1][fx..][fy..][fz..]
    p[0] = make_float4((float)x0[0], (float)x1[0], (float)x0[1], (float)x1[1]);
    p[1] = make_float4((float)x0[2], (float)x1[2], (float)F0[0], (float)(-F0[0]));
    p[2] = make_float4((float)F0[1], (float)(-F0[1]), (float)F0[2], (float)(-F0[2]));
}
__device__ __forceinline__ void publish_dumbbell(double *un, long long i0, const double (&x0)[3], const double (&x1)[3],
                                                 const double (&F0)[3]) {
    double2 *p = reinterpret_cast<double2 *>(un + (size_t)i0 * 6);  // two units of one sphere each: [x y z fx fy fz]
    p[0] = make_double2(x0[0], x0[1]);
    p[1] = make_double2(x0[2], F0[0]);
    p[2] = make_double2(F0[1], F0[2]);
    p[3] = make_double2(x1[0], x1[1]);
    p[4] = make_double2(x1[2], -F0[0]);
    p[5] = make_double2(-F0[1], -F0[2]);
}

#define DS_PROBE(slot)                                                                          \
    do {                                                                                        \
        if (A.probe != nullptr && tid == 0 && probe_on)                                         \
            A.probe[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * PROBE_SLOTS + (slot)] = clock64(); \
    } while (0)

// ---------------------------------------------------------------------------------------------
template <typename T, int TENSOR>
__global__ void __launch_bounds__(NT, 1) run_kernel(const RunArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int ring_bytes = A.ns * SLOT_BYTES;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + ring_bytes);
    uint64_t *empty = full + NS_MAX;

    const int tid = threadIdx.x, lane = tid & 31;
    const int c = blockIdx.x, b = A.b0 + blockIdx.y;
    const int NS = A.ns;

    // rows of this CTA and the (alpha-thread, beta-group) shape
    const int q0 = (int)((long long)c * A.NQ / A.n_cta), q1 = (int)((long long)(c + 1) * A.NQ / A.n_cta);
    const int nq = q1 - q0;                 // 1 .. NT (host guarantees)
    const int n_jg = NT / nq;
    const int ith = tid % nq, jg = tid / nq;
    const bool active = jg < n_jg;
    const int chu = (CHU / n_jg) * n_jg;    // units per chunk: a multiple of n_jg, <= CHU (n_jg <= NT = CHU)
    const int nchunks = (A.U + chu - 1) / chu;
    const int rows = 4 * nq;
    const long long r0 = 4LL * q0;                                   // first sphere of this CTA
    const int nrows = (int)((A.N - r0) < rows ? (A.N - r0) : rows);  // real rows (N even in the step modes)
    const int nd = nrows >> 1;                                       // dumbbells owned (step modes)
    const size_t sys3 = (size_t)b * A.N * 3;

    // per-row state (step modes), FP64: X_n, Xc = positions the current stage evaluates (X_n or the
    // predictor's X*), V1, F(Xc); per dumbbell: phase, L(t_{n+1})
    double *Xs, *Xc, *V1s, *Fs, *Ls;
    const double *phs;
    if (A.state_smem) {
        double *st = reinterpret_cast<double *>(smem_raw + ring_bytes + BAR_BYTES);
        Xs = st; Xc = st + 3 * rows; V1s = st + 6 * rows; Fs = st + 9 * rows; Ls = st + 12 * rows;
        phs = st + 12 * rows + (rows >> 1);
    } else {
        Xs = A.X + sys3 + 3 * r0; Xc = A.Xcg + sys3 + 3 * r0; V1s = A.V1g + sys3 + 3 * r0; Fs = A.Fg + sys3 + 3 * r0;
        Ls = A.Lg + (size_t)b * (A.N / 2) + (r0 >> 1);
        phs = A.phase + (size_t)b * (A.N / 2) + (r0 >> 1);
    }

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, NT / 32);
        }
        mbar_fence_init();
    }

    const bool stepping = A.mode != RUN_APPLY;
    const int n_stage = A.mode == RUN_STEP ? (int)(A.n_steps * (A.heun ? 2 : 1)) : 1;
    unsigned long long *bar = A.bar != nullptr ? A.bar + b : nullptr;
    unsigned long long bar_target = A.bar_base;
    bool probe_on = false;

    // ---- prologue of the step modes: own rows X -> state, F(X_n, t_n), publish the stream rows ----
    if (stepping) {
        if (A.state_smem) {
            for (int e = tid; e < 3 * nrows; e += NT) Xs[e] = A.X[sys3 + 3 * r0 + e];
            for (int sl = tid; sl < nd; sl += NT) const_cast<double *>(phs)[sl] = A.phase[(size_t)b * (A.N / 2) + (r0 >> 1) + sl];
        }
        __syncthreads();
        for (int e = tid; e < 3 * nrows; e += NT) Xc[e] = Xs[e];
        const double tn = time_of_step(A.t0, A.n0, A.dt);
        T *un = reinterpret_cast<T *>(A.units[A.cur]) + (size_t)b * A.unit_stride * (6 * W);
        for (int sl = tid; sl < nd; sl += NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xs[6 * sl + cc]; x1[cc] = Xs[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, stroke_length(tn, phs[sl], A.ell, A.lambda, A.omega), A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            publish_dumbbell(un, r0 + 2 * sl, x0, x1, F0);
        }
        fence_proxy_async_global();
    }
    __syncthreads();  // mbarriers initialised; state and published rows written

    uint32_t seq0 = 0;  // chunk sequence number of the stage's first chunk (slot = seq % NS, parity = (seq / NS) & 1)
    for (int g = 0; g < n_stage; ++g, seq0 += (uint32_t)nchunks) {
        probe_on = (g == n_stage - 1);
        DS_PROBE(0);
        const T *units = reinterpret_cast<const T *>(A.units[(A.cur + g) & 1]) + (size_t)b * A.unit_stride * (6 * W);
        const int n_pre = nchunks < NS ? nchunks : NS;  // chunks in flight before the loop starts

        // chunk ch = units [ch chu, ch chu + cu): cu rounded up to a multiple of n_jg (the pad units exist)
        auto chunk_units = [&](int ch) {
            const int rem = A.U - ch * chu;
            return rem >= chu ? chu : (rem + n_jg - 1) / n_jg * n_jg;
        };
        auto issue = [&](int ch) {
            const uint32_t seq = seq0 + (uint32_t)ch;
            const int s = (int)(seq % (uint32_t)NS);
            if (seq >= (uint32_t)NS) mbar_wait(empty + s, ((seq / (uint32_t)NS) - 1u) & 1u);  // previous content consumed
            const uint32_t bytes = (uint32_t)chunk_units(ch) * UNIT_BYTES;
            mbar_expect_tx(full + s, bytes);
            bulk_g2s(smem_raw + (size_t)s * SLOT_BYTES, units + (size_t)ch * chu * (6 * W), bytes, full + s);
        };

        if (tid == 0) {
            if (stepping && A.n_cta > 1) {
                // inter-CTA barrier: every CTA of the system has published its rows of this stage's input
                __threadfence();
                red_release_gpu(bar, 1ULL);
                bar_target += (unsigned long long)A.n_cta;
                while (ld_acquire_gpu(bar) < bar_target) {}
            }
            DS_PROBE(1);
            fence_proxy_async();
            for (int ch = 0; ch < n_pre; ++ch) issue(ch);
        }

        // stroke length at the end of this step, L(t_{n+1}), once per step (warps 1.. while warp 0 waits)
        if (A.mode == RUN_STEP && (!A.heun || (g & 1) == 0) && tid >= 32) {
            const double t1 = time_of_step(A.t0, A.n0 + (A.heun ? (g >> 1) : g) + 1, A.dt);
            for (int sl = tid - 32; sl < nd; sl += NT - 32) Ls[sl] = stroke_length(t1, phs[sl], A.ell, A.lambda, A.omega);
        }

        // alpha-spheres of this thread: rows 4 (q0 + ith) + k, rounded exactly as the stream rounds them
        V xi[QI][3], acc[QI][3];
#pragma unroll
        for (int k = 0; k < QI; ++k) {
            const int il = 4 * ith + k;
            T x = T(0), y = T(0), z = T(0);
            if (il < nrows) {
                if (stepping) {
                    x = (T)Xc[3 * il]; y = (T)Xc[3 * il + 1]; z = (T)Xc[3 * il + 2];
                } else {
                    x = __ldg(units + unit_index<T>(r0 + il, 0));
                    y = __ldg(units + unit_index<T>(r0 + il, 1));
                    z = __ldg(units + unit_index<T>(r0 + il, 2));
                }
            }
            xi[k][0] = P::bc(x); xi[k][1] = P::bc(y); xi[k][2] = P::bc(z);
            acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
        }
        const V c1 = P::bc((T)A.c1), negc2 = P::bc((T)(-A.c2));
        const int d0 = (4 * q0) / W, d1 = (4 * q1 + W - 1) / W;  // units that hold this CTA's own rows

        for (int ch = 0; ch < nchunks; ++ch) {
            const uint32_t seq = seq0 + (uint32_t)ch;
            const int s = (int)(seq % (uint32_t)NS);
            mbar_wait(full + s, (seq / (uint32_t)NS) & 1u);
            if (ch == 0) DS_PROBE(2);
            if (active) {
                const int u0 = ch * chu, cu = chunk_units(ch);
                const V2<T> *p = reinterpret_cast<const V2<T> *>(smem_raw + (size_t)s * SLOT_BYTES) + 3 * jg;
                if (u0 < d1 && u0 + cu > d0)
                    pair_units<T, TENSOR, true>(p, 3 * n_jg, cu / n_jg, xi, acc, c1, negc2);
                else
                    pair_units<T, TENSOR, false>(p, 3 * n_jg, cu / n_jg, xi, acc, c1, negc2);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);                 // this warp is done with the slot
            if (tid == 0 && ch + NS < nchunks) issue(ch + NS);     // refill it once every warp is
        }
        DS_PROBE(3);
        __syncthreads();  // every chunk consumed by every warp: the ring is free and becomes scratch
        DS_PROBE(4);

        // ---- sum over the n_jg beta-groups (fixed order) ----
        T *red = reinterpret_cast<T *>(smem_raw);   // [n_jg][n_out]   <= 12 NT
        T *red2 = red + 12 * NT;                    // [nparts][n_out] <= 12 NT     (2 x 12 NT x 8 B = 96 KB = NS_MIN slots)
        const int n_out = 12 * nq;
        if (active) {
#pragma unroll
            for (int k = 0; k < QI; ++k)
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) red[(size_t)jg * n_out + (k * 3 + cc) * nq + ith] = P::hsum(acc[k][cc]);
        }
        __syncthreads();
        int nparts = NT / n_out;
        nparts = nparts < 1 ? 1 : (nparts > n_jg ? n_jg : nparts);
        for (int idx = tid; idx < n_out * nparts; idx += NT) {
            const int o = idx % n_out, part = idx / n_out;
            T sum = T(0);
            for (int gq = part; gq < n_jg; gq += nparts) sum += red[(size_t)gq * n_out + o];
            red2[(size_t)part * n_out + o] = sum;
        }
        __syncthreads();
        DS_PROBE(5);
        // u of local row il, component cc: the parts are added in FP64, then Eq. (3a) + the 1/(8 pi mu) factor
        auto velocity = [&](int il, int cc, double Fi) {
            const int o = ((il & 3) * 3 + cc) * nq + (il >> 2);
            double sum = (double)red2[o];
            for (int part = 1; part < nparts; ++part) sum += (double)red2[(size_t)part * n_out + o];
            return A.self_mob * Fi + A.pre * sum;
        };

        if (!stepping) {  // ---- RUN_APPLY: a2 + a3 with the stream's own F ----
            for (int il = tid; il < nrows; il += NT) {
                const long long i = r0 + il;
#pragma unroll
                for (int cc = 0; cc < 3; ++cc)
                    reinterpret_cast<T *>(A.out_u)[(size_t)i * 3 + cc] = (T)velocity(il, cc, (double)units[unit_index<T>(i, 3 + cc)]);
            }
        } else if (A.mode == RUN_VELOCITY) {
            for (int il = tid; il < nrows; il += NT)
#pragma unroll
                for (int cc = 0; cc < 3; ++cc)
                    reinterpret_cast<T *>(A.out_u)[sys3 + (size_t)(r0 + il) * 3 + cc] = (T)velocity(il, cc, Fs[3 * il + cc]);
        } else {  // ---- RUN_STEP: integrator, Eq. (4) at the new positions, publish ----
            const bool pred = A.heun && (g & 1) == 0, corr = A.heun && (g & 1) == 1;
            T *un = reinterpret_cast<T *>(A.units[(A.cur + g + 1) & 1]) + (size_t)b * A.unit_stride * (6 * W);
            for (int sl = tid; sl < nd; sl += NT) {
                double xs[2][3], F0[3];
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) {
                        const int e = 3 * (2 * sl + r) + cc;
                        const double v = velocity(2 * sl + r, cc, Fs[e]);
                        double xn;
                        if (pred) {            // X* = X_n + dt V1
                            V1s[e] = v;
                            xn = Xs[e] + A.dt * v;
                        } else if (corr) {     // X_{n+1} = X_n + (dt/2)(V1 + V2)
                            xn = Xs[e] + (0.5 * A.dt) * (V1s[e] + v);
                            Xs[e] = xn;
                        } else {               // Euler
                            xn = Xs[e] + A.dt * v;
                            Xs[e] = xn;
                        }
                        xs[r][cc] = xn;
                        Xc[e] = xn;
                    }
                dumbbell_force(xs[0], xs[1], Ls[sl], A.k0, F0);
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
                if (g + 1 < n_stage) publish_dumbbell(un, r0 + 2 * sl, xs[0], xs[1], F0);
            }
            fence_proxy_async_global();
        }
        DS_PROBE(6);
        fence_proxy_async_shared();
        __syncthreads();  // scratch reads done (the ring may be refilled); this CTA's published rows complete
        DS_PROBE(7);
    }

    if (A.mode == RUN_STEP && A.state_smem)
        for (int e = tid; e < 3 * nrows; e += NT) A.X[sys3 + 3 * r0 + e] = Xs[e];
}

}  // namespace ds
