// mobility.cuh -- the hot kernel: matrix-free all-pairs mobility apply, Eq. (1a) deterministic
// part with the tensor of Eq. (3a,3b), fused with the O(N) rest of the time
// step (self term, reduction, integrator update, next force evaluation) and
// with the step loop itself: ONE launch runs all n_steps of ds_step / ds_batch_step.
// (DESIGN.md section 6 is the long form of this comment.)
//
// Decomposition ("row owner": no partial sum ever leaves the SM).
//   grid = (n_cta row tiles, systems), one CTA of NT = 512 threads per SM.
//   The N alpha-spheres of a system are cut into NQ = ceil(N/4) quads; CTA c owns the contiguous
//   quads [c NQ / n_cta, (c+1) NQ / n_cta) -- nq of them (N = 4096: 147 CTAs of 7 or 6 quads).
//   Thread t = (ith, jg) = (t % nq, t / nq): it keeps the 4 alpha-spheres of quad q0 + ith in
//   registers and belongs to beta-group jg of n_jg = min(NT / nq, units).  The split over beta is
//   therefore INSIDE the CTA; it is undone through shared memory and shuffles in a fixed order
//   (deterministic, no floating-point atomics, no global scratch).
//   Every CTA walks ALL beta-spheres of its system.  The beta-stream lives in global memory
//   (L2-resident) in the exact shared-memory layout ("units", see pack.cuh): one unit = W
//   beta-spheres = 6 packs = 48 bytes; it ends with far-away zero-force pad units.  One iteration =
//   4 alpha x 1 unit per thread; the groups of an iteration read consecutive 48-byte units
//   (conflict-free LDS.128, broadcast within a group).
//     RESIDENT (the stream fits the CTA's shared memory: N <= 8192 FP32 / 4096 FP64): the stream sits in
//       shared memory in natural order and is consumed starting at the CTA's own rows, in three granules:
//       G0 by every thread (LDGSTS, or the tagged low-latency copy, see below), G1 and G2 by TMA bulk copies.
//     otherwise: a ring of 24 KB slots filled by TMA bulk copies (cp.async.bulk, completion on an mbarrier;
//       one thread issues them, consumer warps release slots through a second mbarrier).
//   r = 0 (alpha == beta) is excluded by a guarded rsqrt compiled only into the loop variant taken by the
//   warps that read an own unit, in the one or two iterations that hold the CTA's own rows.
//
// Time stepping.  The CTA keeps its rows' state (X_n, the stage's positions, V1, F; FP64) in shared
// memory for the whole launch.  A stage = pair sum over the input stream -> reduction -> Eq. (3a) self
// term -> integrator update -> Eq. (4) at the new positions -> publish the CTA's rows of the next
// stage's stream (ping-pong buffers in global memory, plain and tagged copy) -> inter-CTA barrier (one
// arrival counter per system, release/acquire at gpu scope; the grid is launched cooperatively so all
// CTAs are co-resident).  In low-latency mode the first granule of the next stage is read from the
// tagged copy as soon as the producers' stores land, and the barrier is passed later inside the stage.
// Heun = 2 stages per step, Euler = 1.  No host round trip, no kernel boundary per step.
// One CTA per system (local mode): the stream never leaves shared memory.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "noise.cuh"
#include "pack.cuh"

namespace ds {

enum { TENSOR_OSEEN = 0, TENSOR_RPY = 1 };
enum RunMode { RUN_APPLY = 0, RUN_VELOCITY = 1, RUN_STEP = 2 };
// kernel variants (template parameter): the stage's tail is compiled for one of these only
enum KernelMode { KM_APPLY = 0, KM_VELOCITY = 1, KM_EULER = 2, KM_HEUN = 3 };

constexpr int NT = 512;                  // threads per CTA: 16 warps, one CTA per SM
constexpr int QI = 4;                    // alpha-spheres per thread (one quad)
constexpr int UNIT_BYTES = 48;           // 6 packs of 8 bytes: x y z Fx Fy Fz of W beta-spheres
constexpr int CHU = 512;                 // units per ring slot (24 KB)
constexpr int SLOT_BYTES = CHU * UNIT_BYTES;
constexpr int NS_MAX = 8;                // ring slots (192 KB)
constexpr int NS_MIN = 4;                // the reduction scratch aliases the first 4 slots (96 KB)
constexpr int BAR_BYTES = 512;           // mbarriers (2 NS_MAX + 3) and the resident mode's segment table (12 x 16 B)
constexpr int SMEM_MAX = 232448;         // 227 KB opt-in limit per CTA on sm_100
constexpr int PAD_UNITS = CHU;           // dummy units appended to every system's stream
constexpr int STATE_BYTES_PER_ROW = 15 * 8 + 8;  // X_n, X of the stage (FP64 and rounded to T), V1, F (3 x 8 B each) + (phase, L) per dumbbell = 16 B / 2 rows
constexpr int PROBE_SLOTS = 32;

struct RunArgs {
    // problem
    int N, NQ, U, n_cta;      // spheres, quads = ceil(N/4), units = ceil(N/W), row tiles per system
    int buf_bytes;            // shared-memory stream buffer (multiple of 128, >= NS_MIN slots)
    int b0;                   // first system of this launch (blockIdx.y is relative to it)
    long long unit_stride;    // units per system in the streams (>= U + PAD_UNITS)
    void *units[2];           // beta-streams T[B][unit_stride][6][W]; stage g reads units[(cur+g)&1]
    int cur;                  // always 0 today (the prologue republishes the stream of the first stage)
    // Eq. (3) constants
    double self_mob;  // 1/(6 pi eta a)   Eq. (3a)
    double pre;       // 1/(8 pi eta)     Eq. (3b)
    double c1, c2;    // 2a^2/3, 2a^2     second line of Eq. (3b), see pair body
    float c1f, c2f;   // the same rounded to FP32 on the host (no FP64 -> FP32 conversion in the pair loop)
    // what to run
    int mode;                 // RunMode
    int heun;                 // RUN_STEP: 1 = Heun (2 stages per step), 0 = Euler
    long long n0, n_steps;    // RUN_STEP: index of the first step, number of steps
    void *out_u;              // RUN_APPLY / RUN_VELOCITY: u [B][N][3] user precision
    const void *raw_pos, *raw_F;  // RUN_APPLY with a resident stream: the user's [n][3] arrays (each CTA packs them itself)
    double *X;                // state positions [B][N][3] (read at start; written at the end of RUN_STEP)
    void *xu;                 // the same in user precision [B][N][3]: written at the end of RUN_STEP (ds_get_state reads it);
    int from_user;            // 1: the launch starts from xu (ds_set_state with a host buffer left X stale)
    const double *phase;      // [B][S]
    double t0, dt, ell, lambda, omega, k0;
    double noise_amp;         // sqrt(2 k_B T dt / (6 pi mu a)): Brownian increments (noise.cuh); 0 = deterministic
    unsigned long long seed;
    // inter-CTA barrier: one monotonic arrival counter per system; this launch starts at bar_base
    unsigned long long *bar;
    unsigned long long bar_base;
    // low-latency copy of the streams: every 32-bit word of a unit paired with a stage tag ({w0, tag, w1, tag} per
    // 16 bytes, 96 B per unit); a reader that sees the tag has the word (8-byte accesses are single-copy atomic)
    void *ll[2];
    int h0_ll;                // iterations of the first granule in low-latency mode
    unsigned int ll_tag0;     // tag of the stream the prologue publishes; stage g's output carries ll_tag0 + g + 1
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
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
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
__device__ __forceinline__ unsigned long long ld_relaxed_gpu(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// Ampere-style asynchronous copy, 16 bytes global (L2 only, .cg) -> shared, in the generic proxy (SASS: LDGSTS);
// the mbarrier form makes `bar` count this thread's arrival once all its earlier copies have landed
__device__ __forceinline__ void cp_async16(void *dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_arrive(uint64_t *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
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
template <typename T, int TENSOR, bool GUARD, int NA = QI>
__device__ __forceinline__ void pair_unit(const V2<T> *__restrict__ p, const typename Pack<T>::V (&xi)[NA][3],
                                          typename Pack<T>::V (&acc)[NA][3], typename Pack<T>::V c1,
                                          typename Pack<T>::V negc2) {
    typedef Pack<T> P;
    typedef typename P::V V;
    const V2<T> q0 = p[0], q1 = p[1], q2 = p[2];
    const V xj = q0.a, yj = q0.b, zj = q1.a, fx = q1.b, fy = q2.a, fz = q2.b;
#pragma unroll
    for (int k = 0; k < NA; ++k) {
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

// ---------------------------------------------------------------------------------------------
// Eq. (4).  Explicit rounding (no contraction) so that every call site produces
// the same bits for the same inputs: ds_step(n) is bit-identical however the n steps are split.
//   L^s(t) = ell + lambda sin(omega t + phi^s)
__device__ __noinline__ double stroke_length(double t, double phi, double ell, double lambda, double omega) {
    return __dadd_rn(ell, __dmul_rn(lambda, sin(__dadd_rn(__dmul_rn(omega, t), phi))));
}
//   n = (X_{2s+1} - X_{2s})/d, g = k0 (d - L), F_{2s} = +g n, F_{2s+1} = -g n   (F = -dU/dX)
// 1/d comes from the refined reciprocal square root of pack.cuh (relative error < 2^-60, no division, no
// slow path: d^2 is finite, positive, normal); d = d^2 (1/d) gets one correction step, which leaves it
// within a rounding of sqrt(d^2): g = k0 (d - L) cancels, so d has to be that accurate.
__device__ __forceinline__ void dumbbell_force(const double (&x0)[3], const double (&x1)[3], double L, double k0,
                                               double (&F0)[3]) {
    const double s0 = __dsub_rn(x1[0], x0[0]), s1 = __dsub_rn(x1[1], x0[1]), s2 = __dsub_rn(x1[2], x0[2]);
    const double d2 = __fma_rn(s2, s2, __fma_rn(s1, s1, __dmul_rn(s0, s0)));
    const double y = Pack<double>::rsq<false>(d2);
    double d = __dmul_rn(d2, y);
    d = __fma_rn(__fma_rn(-d, d, d2), __dmul_rn(0.5, y), d);
    const double cf = __dmul_rn(__dmul_rn(k0, __dsub_rn(d, L)), y);
    F0[0] = __dmul_rn(cf, s0);
    F0[1] = __dmul_rn(cf, s1);
    F0[2] = __dmul_rn(cf, s2);
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

__device__ __forceinline__ uint4 ld_volatile_v4(const uint4 *p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
// the 16-byte piece (w0 w1 w2 w3) of a unit -> its two tagged quads
__device__ __forceinline__ void publish_ll_piece(uint4 *q, uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, uint32_t tag) {
    q[0] = make_uint4(w0, tag, w1, tag);
    q[1] = make_uint4(w2, tag, w3, tag);
}
__device__ __forceinline__ void publish_ll(uint4 *ll_units, long long i0, const float4 (&u)[3], uint32_t tag) {
    uint4 *q = ll_units + (size_t)(i0 >> 1) * 6;       // FP32: one unit per dumbbell
#pragma unroll
    for (int k = 0; k < 3; ++k)
        publish_ll_piece(q + 2 * k, __float_as_uint(u[k].x), __float_as_uint(u[k].y), __float_as_uint(u[k].z), __float_as_uint(u[k].w), tag);
}
__device__ __forceinline__ void publish_ll(uint4 *ll_units, long long i0, const double2 (&u)[6], uint32_t tag) {
    uint4 *q = ll_units + (size_t)i0 * 6;              // FP64: two units (one sphere each) per dumbbell
#pragma unroll
    for (int k = 0; k < 6; ++k)
        publish_ll_piece(q + 2 * k, (uint32_t)__double2loint(u[k].x), (uint32_t)__double2hiint(u[k].x),
                         (uint32_t)__double2loint(u[k].y), (uint32_t)__double2hiint(u[k].y), tag);
}

// The two spheres i0 (even), i0 + 1 of one dumbbell -> their units of a stream, rounded to T.
__device__ __forceinline__ void publish_dumbbell(float *un, uint4 *ll_units, uint32_t tag, long long i0, const double (&x0)[3],
                                                 const double (&x1)[3], const double (&F0)[3]) {
    float4 *p = reinterpret_cast<float4 *>(un + (size_t)(i0 >> 1) * 12);  // one unit: [x0 x1][y0 y1][z0 z1][fx..][fy..][fz..]
    const float4 u[3] = {make_float4((float)x0[0], (float)x1[0], (float)x0[1], (float)x1[1]),
                         make_float4((float)x0[2], (float)x1[2], (float)F0[0], (float)(-F0[0])),
                         make_float4((float)F0[1], (float)(-F0[1]), (float)F0[2], (float)(-F0[2]))};
    p[0] = u[0]; p[1] = u[1]; p[2] = u[2];
    if (ll_units != nullptr) publish_ll(ll_units, i0, u, tag);
}
__device__ __forceinline__ void publish_dumbbell(double *un, uint4 *ll_units, uint32_t tag, long long i0, const double (&x0)[3],
                                                 const double (&x1)[3], const double (&F0)[3]) {
    double2 *p = reinterpret_cast<double2 *>(un + (size_t)i0 * 6);  // two units of one sphere each: [x y z fx fy fz]
    const double2 u[6] = {make_double2(x0[0], x0[1]), make_double2(x0[2], F0[0]), make_double2(F0[1], F0[2]),
                          make_double2(x1[0], x1[1]), make_double2(x1[2], -F0[0]), make_double2(-F0[1], -F0[2])};
#pragma unroll
    for (int k = 0; k < 6; ++k) p[k] = u[k];
    if (ll_units != nullptr) publish_ll(ll_units, i0, u, tag);
}

// Unit u of the stream built from the user's arrays pos, F [n][3] (RUN_APPLY): spheres beyond n are far-away
// zero-force dummies.  FP32: spheres 2u, 2u + 1 -> [x0 x1][y0 y1][z0 z1][fx0 fx1][fy0 fy1][fz0 fz1]; FP64: sphere u.
__device__ __forceinline__ void pack_unit(float4 *dst, const float *pos, const float *F, int u, int n) {
    const float D = Pack<float>::dummy();
    float a[6] = {D, D, D, D, D, D}, f[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (2 * u + 1 < n) {
        const float2 *pp = reinterpret_cast<const float2 *>(pos + 6 * (size_t)u), *fp = reinterpret_cast<const float2 *>(F + 6 * (size_t)u);
        const float2 p0 = __ldg(pp), p1 = __ldg(pp + 1), p2 = __ldg(pp + 2), f0 = __ldg(fp), f1 = __ldg(fp + 1), f2 = __ldg(fp + 2);
        a[0] = p0.x; a[1] = p0.y; a[2] = p1.x; a[3] = p1.y; a[4] = p2.x; a[5] = p2.y;
        f[0] = f0.x; f[1] = f0.y; f[2] = f1.x; f[3] = f1.y; f[4] = f2.x; f[5] = f2.y;
    } else if (2 * u < n) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { a[c] = __ldg(pos + 6 * (size_t)u + c); f[c] = __ldg(F + 6 * (size_t)u + c); }
    }
    dst[0] = make_float4(a[0], a[3], a[1], a[4]);
    dst[1] = make_float4(a[2], a[5], f[0], f[3]);
    dst[2] = make_float4(f[1], f[4], f[2], f[5]);
}
__device__ __forceinline__ void pack_unit(double2 *dst, const double *pos, const double *F, int u, int n) {
    const double D = Pack<double>::dummy();
    double a[3] = {D, D, D}, f[3] = {0.0, 0.0, 0.0};
    if (u < n) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { a[c] = __ldg(pos + 3 * (size_t)u + c); f[c] = __ldg(F + 3 * (size_t)u + c); }
    }
    dst[0] = make_double2(a[0], a[1]);
    dst[1] = make_double2(a[2], f[0]);
    dst[2] = make_double2(f[1], f[2]);
}

// 16-byte piece p (0..2) of a far-away zero-force pad unit, as raw words
template <typename T> __device__ __forceinline__ uint4 pad_piece(int p);
template <> __device__ __forceinline__ uint4 pad_piece<float>(int p) {
    const uint32_t D = __float_as_uint(Pack<float>::dummy());
    return p == 0 ? make_uint4(D, D, D, D) : (p == 1 ? make_uint4(D, D, 0u, 0u) : make_uint4(0u, 0u, 0u, 0u));
}
template <> __device__ __forceinline__ uint4 pad_piece<double>(int p) {
    const double Dd = Pack<double>::dummy();
    const uint32_t lo = (uint32_t)__double2loint(Dd), hi = (uint32_t)__double2hiint(Dd);
    return p == 0 ? make_uint4(lo, hi, lo, hi) : (p == 1 ? make_uint4(lo, hi, 0u, 0u) : make_uint4(0u, 0u, 0u, 0u));
}

#ifdef DS_ENABLE_PROBE
#define DS_PROBE(slot)                                                                          \
    do {                                                                                        \
        if (A.probe != nullptr && tid == 0 && probe_on)                                         \
            A.probe[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * PROBE_SLOTS + (slot)] = clock64(); \
    } while (0)
#else
#define DS_PROBE(slot) do { } while (0)
#endif

// ---------------------------------------------------------------------------------------------
template <typename T, int TENSOR, int MODE, bool RESIDENT>
__global__ void __launch_bounds__(NT, 1) run_kernel(const RunArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int buf_bytes = A.buf_bytes;   // stream buffer: the whole stage input if it fits (resident), else a ring of slots
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + buf_bytes);
    uint64_t *empty = full + NS_MAX;
    uint64_t *gran = empty + NS_MAX;     // resident mode: one barrier per granule of the stream (3)
    int4 *segs = reinterpret_cast<int4 *>(gran + 4);   // resident mode: the stage's tight loops (<= 8), see below

    const int tid = threadIdx.x, lane = tid & 31;
    const int c = blockIdx.x, b = A.b0 + blockIdx.y;

    // rows of this CTA and the (alpha-thread, beta-group) shape
    const int q0 = (int)((long long)c * A.NQ / A.n_cta), q1 = (int)((long long)(c + 1) * A.NQ / A.n_cta);
    const int nq = q1 - q0;                 // 1 .. NT (host guarantees)
    const int n_jg = NT / nq < A.U ? NT / nq : A.U;   // beta-groups: no more than there are units
    const int ith = tid % nq, jg = tid / nq;
    const bool active = jg < n_jg;
    const int rows = 4 * nq;
    const long long r0 = 4LL * q0;                                   // first sphere of this CTA
    const int nrows = (int)((A.N - r0) < rows ? (A.N - r0) : rows);  // real rows (N even in the step modes)
    const int nd = nrows >> 1;                                       // dumbbells owned (step modes)
    const size_t sys3 = (size_t)b * A.N * 3;
    constexpr bool stepping = MODE != KM_APPLY;

    // per-row state (step modes), FP64: X_n, Xc = positions the current stage evaluates (X_n or the
    // predictor's X*; XcT = the same rounded to T as the stream holds them), V1, F(Xc); per dumbbell: phase, L(t_{n+1})
    double *Xs, *Xc, *V1s, *Fs, *Ls;
    T *XcT = nullptr;
    const double *phs;
    if (A.state_smem) {
        double *st = reinterpret_cast<double *>(smem_raw + buf_bytes + BAR_BYTES);
        Xs = st; Xc = st + 3 * rows; V1s = st + 6 * rows; Fs = st + 9 * rows; Ls = st + 12 * rows;
        phs = st + 12 * rows + (rows >> 1);
        XcT = reinterpret_cast<T *>(st + 13 * rows);
    } else {
        Xs = A.X + sys3 + 3 * r0; Xc = A.Xcg + sys3 + 3 * r0; V1s = A.V1g + sys3 + 3 * r0; Fs = A.Fg + sys3 + 3 * r0;
        Ls = A.Lg + (size_t)b * (A.N / 2) + (r0 >> 1);
        phs = A.phase + (size_t)b * (A.N / 2) + (r0 >> 1);
    }


    // the stage's stream: total_it iterations of n_jg units each (tail padded with far-away zero-force units)
    const int total_it = (A.U + n_jg - 1) / n_jg;
    const int stride = 3 * n_jg;                               // 16-byte pieces per iteration
    const int tp = total_it * stride;                          // pieces of the whole stream
    // RESIDENT: the host checked tp * 16 <= buf_bytes (no ring, no refills)
    // resident mode.  The stream sits in shared memory in its natural order; the CTA consumes it starting at
    // the iteration that holds its own rows (so only the first n_guard iterations need the r = 0 guard, and
    // the 148 CTAs start at 148 different places of the L2-resident stream), wrapping around at the end.
    // Three granules in consumption order, each with its own mbarrier: G0 (h0 iterations, copied first),
    // G1 (h1), G2 (the rest, copied by the loop itself while it works on G0 and G1).
    const int d0 = (4 * q0) / W, d1 = (4 * q1 + W - 1) / W;    // units that hold this CTA's own rows
    const int it_own = d0 / n_jg;
    const int n_guard = (d1 - 1) / n_jg - it_own + 1;
    const int sp = it_own * stride;                            // first piece in consumption order
    const int h0w = (RESIDENT && MODE != KM_APPLY && A.n_cta > 1 && A.ll[0] != nullptr) ? A.h0_ll : 4;  // low-latency mode: G0 also covers the barrier
    const int h0 = total_it < h0w ? total_it : h0w;
    const int h1 = total_it - h0 < 6 ? total_it - h0 : 6;
    const int h2 = total_it - h0 - h1;
    const int pA = h0 * stride, pAB = (h0 + h1) * stride;      // piece index (consumption order) where G1 / G2 start
    // ring mode: chunks of cit iterations (<= one slot of CHU units)
    const int NS = buf_bytes / SLOT_BYTES < NS_MAX ? buf_bytes / SLOT_BYTES : NS_MAX;
    const int cit = CHU / n_jg;
    const int chu = cit * n_jg;
    const int nchunks = (total_it + cit - 1) / cit;
    const int rot = c % nchunks;                               // CTAs start at different chunks: no L2 convoy

    const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
    // reduction shape (stage-invariant index arithmetic is done once, here)
    // split-beta reduction: the partials of thread tid sit at red[12 tid + m], m = 3 k + cc (three 16-byte stores,
    // 48-byte thread stride: conflict-free); the sums of quad ith are elements 12 ith + m of the CTA's state.
    // A task = (quad ith, 4 consecutive m) is summed by RP consecutive lanes: lane part adds the groups
    // jg = part, part + RP, ... with one LDS.128 each, then log2(RP) shuffle steps.
    const int n_task = 3 * nq;                                  // tasks of the CTA
    // few groups: fewer lanes per task, more tasks per pass; many groups and few tasks (small systems spread over many
    // CTAs): up to a warp per task while a lane would otherwise add more than 8 groups and every task still gets its
    // lanes in one pass (N = 4096 on 147 CTAs, 73 groups, stays at 8 lanes: wider measured no gain there)
    int rp_log = n_jg >= 32 ? 3 : (n_jg >= 16 ? 2 : (n_jg >= 8 ? 1 : 0));
    while (rp_log < 5 && n_jg >= (16 << rp_log) && (n_task << (rp_log + 1)) <= NT) ++rp_log;
    const int RP = 1 << rp_log, tpw = 32 >> rp_log;                              // lanes per task, tasks per warp
    const int my_task = tid >> rp_log, my_part = tid & (RP - 1);
    if (tid == 0) {
        for (int s = 0; s < NS_MAX; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, NT / 32);
        }
        // G0: every thread's LDGSTS copies; in low-latency mode warps 1.. fill G0 and warp 0 (barrier arrival) only waits
        mbar_init(gran + 0, (RESIDENT && MODE != KM_APPLY && A.n_cta > 1 && A.ll[0] != nullptr) ? NT - 32 : NT);
        mbar_init(gran + 1, 1);    // G1, G2: thread 0's TMA bulk copies
        mbar_init(gran + 2, 1);
        mbar_fence_init();
    }
    if (tid == 64) {   // another warp than the one that initialises the barriers
        if (RESIDENT) {
            // a new tight loop starts where a granule begins, where the guard ends and where the stream wraps around
            const int wrapq = total_it - it_own;
            int q = 0, n = 0;
            while (q < total_it) {
                int qe = q < h0 ? h0 : (q < h0 + h1 ? h0 + h1 : total_it);
                if (q < n_guard && n_guard < qe) qe = n_guard;
                if (q < wrapq && wrapq < qe) qe = wrapq;
                if (h0w > 6 && q < h0 && q >= n_guard && q + 4 < qe) qe = q + 4;   // low-latency mode: thread 0 looks at the barrier between segments
                int it = it_own + q;
                it = it >= total_it ? it - total_it : it;
                const int w = (q == h0 && h1 > 0) ? 1 : ((q == h0 + h1 && h2 > 0) ? 2 : -1);
                const int tail = (it + (qe - q) == total_it) ? (1 << 30) : 0;   // the segment ends with the stream's last iteration
                segs[n++] = make_int4(it * stride, (qe - q) | tail, w, q < n_guard ? it + 1 : 0);
                q = qe;
            }
            segs[11].x = n;
        }
    }

    if (MODE == KM_APPLY) {
        // programmatic dependent launch (ds_api.cu): let the next kernel of the stream become resident as SMs free up,
        // and do not touch global memory before the previous kernel has completed
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        asm volatile("griddepcontrol.wait;" ::: "memory");
    }
    const int n_stage = MODE >= KM_EULER ? (int)(A.n_steps * (MODE == KM_HEUN ? 2 : 1)) : 1;
    // low-latency mode (resident step modes with several CTAs per system): the first granule of every stage comes
    // from the tagged copy of the stream, word by word as the producers' stores land; the inter-CTA barrier is only
    // passed later in the stage, before the rest of the stream is fetched by TMA
    const bool use_ll = RESIDENT && stepping && A.n_cta > 1 && A.ll[0] != nullptr;
    // local mode (one CTA per system, resident): the stream never leaves shared memory; the stage's tail writes
    // the next stage's units in place, no copy, no barrier
    const bool local = RESIDENT && stepping && A.n_cta == 1;
    auto ll_of = [&](int k) { return reinterpret_cast<uint4 *>(A.ll[k & 1]) + (size_t)b * A.unit_stride * 6; };
    unsigned long long *bar = A.bar != nullptr ? A.bar + b : nullptr;
    unsigned long long bar_target = A.bar_base;
    bool probe_on = false;

    // ---- prologue of the step modes: own rows X -> state, F(X_n, t_n), publish the stream rows ----
    if (stepping) {
        if (!A.state_smem && A.from_user)
            for (int e = tid; e < 3 * nrows; e += NT) Xs[e] = (double)reinterpret_cast<const T *>(A.xu)[sys3 + 3 * r0 + e];
        if (A.state_smem) {
            for (int e = tid; e < 3 * nrows; e += NT)
                Xs[e] = A.from_user ? (double)reinterpret_cast<const T *>(A.xu)[sys3 + 3 * r0 + e] : A.X[sys3 + 3 * r0 + e];
            for (int sl = tid; sl < nd; sl += NT) const_cast<double *>(phs)[sl] = A.phase[(size_t)b * (A.N / 2) + (r0 >> 1) + sl];
        }
        __syncthreads();
        for (int e = tid; e < 3 * nrows; e += NT) {
            Xc[e] = Xs[e];
            if (XcT != nullptr) XcT[e] = (T)Xs[e];
        }
        const double tn = time_of_step(A.t0, A.n0, A.dt);
        T *un = local ? reinterpret_cast<T *>(smem_raw) : reinterpret_cast<T *>(A.units[A.cur]) + (size_t)b * A.unit_stride * (6 * W);
        if (local)   // the tail of the stream: far-away zero-force pad units
            for (int j = 3 * A.U + tid; j < tp; j += NT) reinterpret_cast<uint4 *>(smem_raw)[j] = pad_piece<T>(j % 3);
        for (int sl = tid; sl < nd; sl += NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xs[6 * sl + cc]; x1[cc] = Xs[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, stroke_length(tn, phs[sl], A.ell, A.lambda, A.omega), A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            publish_dumbbell(un, use_ll ? ll_of(A.cur) : nullptr, A.ll_tag0, r0 + 2 * sl, x0, x1, F0);
        }
        fence_proxy_async_global();   // the stream is also read through the async proxy (TMA)
    }
    if (!(MODE == KM_APPLY && RESIDENT && A.raw_pos != nullptr))
        __syncthreads();  // mbarriers initialised; state and published rows written (the in-kernel pack of the apply ends with its own)


    // ring mode: k-th chunk in this CTA's consumption order -> chunk index, iterations; ring position of the next
    // chunk to consume / to fill (slot, and how often the ring has been gone around: fill parity = wraps & 1)
    auto chunk_of = [&](int k) { const int ch = k + rot; return ch >= nchunks ? ch - nchunks : ch; };
    auto chunk_iters = [&](int ch) { const int rem = total_it - ch * cit; return rem < cit ? rem : cit; };
    int cslot = 0, pslot = 0;
    uint32_t cwraps = 0, pwraps = 0;

    for (int g = 0; g < n_stage; ++g) {
        probe_on = (g == n_stage - 1);
        DS_PROBE(0);
        const T *units = reinterpret_cast<const T *>(A.units[(A.cur + g) & 1]) + (size_t)b * A.unit_stride * (6 * W);

        if (stepping && A.n_cta > 1) {
            bar_target += (unsigned long long)A.n_cta;
            if (tid == 0) {
                // inter-CTA barrier, arrival: this CTA has published its rows of this stage's input
                red_release_gpu(bar, 1ULL);
                DS_PROBE(12);
                if (!use_ll) {   // ... and wait: every CTA of the system has
                    while (ld_relaxed_gpu(bar) < bar_target) {}
                    fence_acq_rel_gpu();
                }
            }
        }
        DS_PROBE(1);
        // stroke length at the end of this step, L(t_{n+1}), once per step (lanes 1.. of warp 0, while thread 0 is busy
        // with the barrier)
        if (MODE >= KM_EULER && (MODE != KM_HEUN || (g & 1) == 0) && tid >= 1 && tid < 32) {
            const double t1 = time_of_step(A.t0, A.n0 + (MODE == KM_HEUN ? (g >> 1) : g) + 1, A.dt);
            for (int sl = tid - 1; sl < nd; sl += 31) Ls[sl] = stroke_length(t1, phs[sl], A.ell, A.lambda, A.omega);
        }
        if (stepping && A.n_cta > 1 && !use_ll) __syncthreads();   // the barrier has been passed (thread 0)
        DS_PROBE(9);

        // alpha-spheres of this thread: rows 4 (q0 + ith) + k, rounded exactly as the stream rounds them
        V xi[QI][3], acc[QI][3];
#pragma unroll
        for (int k = 0; k < QI; ++k) {
            const int il = 4 * ith + k;
            T x = T(0), y = T(0), z = T(0);
            if (il < nrows) {
                if (XcT != nullptr && stepping) {
                    x = XcT[3 * il]; y = XcT[3 * il + 1]; z = XcT[3 * il + 2];
                } else {
                    if (MODE == KM_APPLY && A.raw_pos != nullptr) {
                        const T *rp = reinterpret_cast<const T *>(A.raw_pos) + 3 * (r0 + il);
                        x = __ldg(rp); y = __ldg(rp + 1); z = __ldg(rp + 2);
                    } else {
                        // local mode keeps the stream in shared memory only (r0 = 0 there)
                        if (local) {
                            const T *us = reinterpret_cast<const T *>(smem_raw);
                            x = us[unit_index<T>(il, 0)]; y = us[unit_index<T>(il, 1)]; z = us[unit_index<T>(il, 2)];
                        } else {
                            x = __ldcg(units + unit_index<T>(r0 + il, 0));
                            y = __ldcg(units + unit_index<T>(r0 + il, 1));
                            z = __ldcg(units + unit_index<T>(r0 + il, 2));
                        }
                    }
                }
            }
            xi[k][0] = P::bc(x); xi[k][1] = P::bc(y); xi[k][2] = P::bc(z);
            acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
        }
        DS_PROBE(11);


        if constexpr (RESIDENT) {
            // ---- resident stream: LDGSTS copies (generic proxy, L2 -> shared, 16 bytes per thread and piece) ----
            const uint4 *gsrc = reinterpret_cast<const uint4 *>(units);
            uint4 *sdst = reinterpret_cast<uint4 *>(smem_raw);
            auto copy_piece = [&](int j) {          // j-th piece in consumption order
                int a = sp + j;
                a = a >= tp ? a - tp : a;
                cp_async16(sdst + a, gsrc + a);
            };
            const uint32_t par = (uint32_t)g & 1u;  // every granule barrier completes one phase per stage
            // G1, G2: TMA bulk copies of consumption pieces [j0, j1) (two copies where the range wraps), thread 0
            auto tma_range = [&](int j0, int j1, uint64_t *bar_) {
                int a0 = sp + j0;
                a0 = a0 >= tp ? a0 - tp : a0;
                const int len = j1 - j0, first = a0 + len <= tp ? len : tp - a0;
                mbar_expect_tx(bar_, (uint32_t)len * 16u);
                bulk_g2s(sdst + a0, gsrc + a0, (uint32_t)first * 16u, bar_);
                if (first < len) bulk_g2s(sdst, gsrc, (uint32_t)(len - first) * 16u, bar_);
            };
            auto issue_rest = [&]() {
                if (h1 > 0) tma_range(pA, pAB, gran + 1);
                if (h2 > 0) tma_range(pAB, tp, gran + 2);
            };
            if (local) {
                // the stream is in place (written by the previous stage's tail or the prologue)
            } else if (MODE == KM_APPLY && A.raw_pos != nullptr) {
                // stateless apply: the CTA packs the user's arrays into its resident stream itself (no pack kernel,
                // no global intermediate); CTAs start at different units so that they do not read L2 in a convoy
                typedef typename std::conditional<sizeof(T) == 4, float4, double2>::type Q;
                const int up = total_it * n_jg;
                int u = tid + (int)(((long long)c * up) / A.n_cta);
                for (int k = tid; k < up; k += NT, u += NT) {
                    u = u >= up ? u - up : u;
                    pack_unit(reinterpret_cast<Q *>(smem_raw) + 3 * u, reinterpret_cast<const T *>(A.raw_pos),
                              reinterpret_cast<const T *>(A.raw_F), u, A.N);
                }
                __syncthreads();
                mbar_arrive(gran + 0);
                if (tid == 0) { mbar_arrive(gran + 1); mbar_arrive(gran + 2); }
            } else {
                if (!use_ll) {
                    if (tid == 0) issue_rest();
                    for (int j = tid; j < pA; j += NT) copy_piece(j);   // G0: LDGSTS by every thread (lowest latency)
                    cp_async_arrive(gran + 0);
                } else {
                    // G0 from the tagged copy: warps 1.. poll their pieces until the stage's tag shows in all four words
                    if (tid >= 32) {
                        const uint4 *lsrc = ll_of(A.cur + g);
                        const uint32_t tag = A.ll_tag0 + (uint32_t)g;
                        for (int j = tid - 32; j < pA; j += NT - 32) {
                            int a = sp + j;
                            a = a >= tp ? a - tp : a;
                            uint4 w;
                            if (a < 3 * A.U) {
                                uint4 v0 = ld_volatile_v4(lsrc + 2 * a), v1 = ld_volatile_v4(lsrc + 2 * a + 1);
                                while (v0.y != tag || v0.w != tag || v1.y != tag || v1.w != tag) {
                                    const long long t_retry = clock64() + 256;   // back off: the pollers of 148 CTAs share the L2
                                    while (clock64() < t_retry) {}
                                    v0 = ld_volatile_v4(lsrc + 2 * a);
                                    v1 = ld_volatile_v4(lsrc + 2 * a + 1);
                                }
                                w = make_uint4(v0.x, v0.z, v1.x, v1.z);
                            } else {
                                w = pad_piece<T>(a % 3);   // far-away zero-force unit of the stream's tail
                            }
                            sdst[a] = w;
                        }
                        mbar_arrive(gran + 0);
                    }
                }
            }
            DS_PROBE(10);
            // groups take the units of an iteration in REVERSE order (group jg reads unit n_jg - 1 - jg), so that the
            // pad units of the stream's last iteration fall to the low warps, which skip them: warp 0 also carries the
            // barrier and the TMA issue
            const int jgr = n_jg - 1 - jg;
            const V2<T> *const base = reinterpret_cast<const V2<T> *>(smem_raw) + 3 * jgr;
            const bool skip_tail = jgr >= A.U - (total_it - 1) * n_jg;   // this thread's unit of the last iteration is a pad
            if (!local) mbar_wait(gran + 0, par);
            DS_PROBE(2);
            const int nseg = segs[11].x;
            bool rest_issued = false;
            unsigned long long bar_seen = 0;
            // the stage's total_it iterations (each: QI alpha x 1 unit per thread) as the few tight loops of the
            // segment table (built once, stage-invariant): {first piece, iterations, granule to wait for or -1,
            // first iteration + 1 if the segment holds own rows else 0}
            for (int sgi = 0; sgi < nseg; ++sgi) {
                const int4 sg = segs[sgi];
                if (use_ll && tid == 32 && !rest_issued) bar_seen = ld_acquire_gpu(bar);   // consumed after the segment
                if (sg.z >= 0 && !local) mbar_wait(gran + sg.z, par);
                const V2<T> *p = base + sg.x;
                const int its = sg.y & 0xffffff;
                const int its_mine = its - ((sg.y >> 30) && skip_tail ? 1 : 0);
                if (sg.w != 0) {
                    // iterations that hold the CTA's own rows: a warp takes the guarded variant (r = 0 excluded) only if
                    // one of its lanes reads a unit of ITS OWN quad in that iteration (alpha == beta is possible nowhere
                    // else; with many rows per CTA, e.g. 256 at B = 64 x N = 512, half the stream is "own" units)
                    int u = (sg.w - 1) * n_jg + jgr;
                    constexpr unsigned UPQ = QI / W;                       // units of a quad
                    const int uq0 = d0 + ith * (int)UPQ;                   // first unit of this thread's quad
#pragma unroll 1
                    for (int r = 0; r < its; ++r, p += stride, u += n_jg) {
                        const bool own = __any_sync(0xffffffffu, active && (unsigned)(u - uq0) < UPQ);
                        if (active && r < its_mine) {
                            if (own) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
                            else pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                        }
                    }
                } else if (active) {
#pragma unroll 1
                    for (int r = 0; r < its_mine; ++r, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                }
                if (use_ll && tid == 32 && !rest_issued) {   // warp 1: warp 0 already carries the arrival
                    // low-latency mode: the inter-CTA barrier is passed here (every CTA has published this stage's
                    // input, and nobody reads the buffers of two stages ago any more), then the rest of the stream is
                    // fetched.  The counter was read when the segment began; only the last chance blocks.
                    const bool last = sgi + 1 == nseg || segs[sgi + 1].z >= 0;
                    if (bar_seen >= bar_target || last) {
                        while (bar_seen < bar_target) bar_seen = ld_acquire_gpu(bar);   // acquire: pairs with every CTA's red.release
                        issue_rest();
                        rest_issued = true;
                    }
                }
            }
        } else {
            // ---- ring of slots filled by TMA bulk copies (thread 0), one tight loop per chunk ----
            auto issue_tma = [&](int k) {
                const int ch = chunk_of(k);
                if (pwraps > 0) mbar_wait(empty + pslot, (pwraps - 1u) & 1u);   // previous content consumed by every warp
                const uint32_t bytes = (uint32_t)(chunk_iters(ch) * n_jg) * UNIT_BYTES;
                mbar_expect_tx(full + pslot, bytes);
                bulk_g2s(smem_raw + (size_t)pslot * SLOT_BYTES, units + (size_t)ch * chu * (6 * W), bytes, full + pslot);
                if (++pslot == NS) { pslot = 0; ++pwraps; }
            };
            if (tid == 0) {
                fence_proxy_async();
                for (int k = 0; k < NS && k < nchunks; ++k) issue_tma(k);
            }
            DS_PROBE(10);
            for (int k = 0; k < nchunks; ++k) {
                const int ch = chunk_of(k);
                mbar_wait(full + cslot, cwraps & 1u);
                if (k == 0) DS_PROBE(2);
                if (active) {
                    const int u0 = ch * chu, its = chunk_iters(ch);
                    const V2<T> *p = reinterpret_cast<const V2<T> *>(smem_raw + (size_t)cslot * SLOT_BYTES) + 3 * jg;
                    if (u0 < d1 && u0 + its * n_jg > d0) {
#pragma unroll 1
                        for (int r = 0; r < its; ++r, p += stride) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
                    } else {
#pragma unroll 2
                        for (int r = 0; r < its; ++r, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + cslot);                 // this warp is done with the slot
                if (tid == 0 && k + NS < nchunks) issue_tma(k + NS);       // refill it once every warp is
                if (++cslot == NS) { cslot = 0; ++cwraps; }
            }
        }

        DS_PROBE(3);
        __syncthreads();  // every chunk consumed by every warp: the ring is free and becomes scratch
        DS_PROBE(4);

        // ---- sum over the n_jg beta-groups (fixed order) ----
        T *red = reinterpret_cast<T *>(smem_raw);   // [NT][12]  <= 48 KB
        if (active) {
            typename P::T4 *rw = reinterpret_cast<typename P::T4 *>(red + 12 * tid);
            rw[0] = P::make4(P::hsum(acc[0][0]), P::hsum(acc[0][1]), P::hsum(acc[0][2]), P::hsum(acc[1][0]));
            rw[1] = P::make4(P::hsum(acc[1][1]), P::hsum(acc[1][2]), P::hsum(acc[2][0]), P::hsum(acc[2][1]));
            rw[2] = P::make4(P::hsum(acc[2][2]), P::hsum(acc[3][0]), P::hsum(acc[3][1]), P::hsum(acc[3][2]));
        }
        __syncthreads();
        DS_PROBE(5);
        if (tid < ((n_task * RP + 31) & ~31)) {        // the warps that hold tasks
            const bool pred = MODE == KM_HEUN && (g & 1) == 0, corr = MODE == KM_HEUN && (g & 1) == 1;
            for (int task = my_task; task < ((n_task + tpw - 1) & ~(tpw - 1)); task += NT >> rp_log) {   // warp-uniform trip count
                T s0 = T(0), s1 = T(0), s2 = T(0), s3 = T(0);
                if (task < n_task) {
                    const int tq = task / 3, mq = task - 3 * tq;        // quad, which 4 of its 12 elements
                    const typename P::T4 *rp = reinterpret_cast<const typename P::T4 *>(red + 12 * tq + 4 * mq);
                    // two independent partial sums per element, loads four groups ahead of the adds
                    T t0 = T(0), t1 = T(0), t2 = T(0), t3 = T(0);
                    const int gstep = 3 * nq * RP;
                    rp += 3 * nq * my_part;
                    int gq = my_part;
                    for (; gq + 3 * RP < n_jg; gq += 4 * RP, rp += 4 * gstep) {
                        const typename P::T4 a = rp[0], bq = rp[gstep], cq = rp[2 * gstep], dq = rp[3 * gstep];
                        s0 += a.x; s1 += a.y; s2 += a.z; s3 += a.w;
                        t0 += bq.x; t1 += bq.y; t2 += bq.z; t3 += bq.w;
                        s0 += cq.x; s1 += cq.y; s2 += cq.z; s3 += cq.w;
                        t0 += dq.x; t1 += dq.y; t2 += dq.z; t3 += dq.w;
                    }
                    for (; gq < n_jg; gq += RP, rp += gstep) {
                        const typename P::T4 a = rp[0];
                        s0 += a.x; s1 += a.y; s2 += a.z; s3 += a.w;
                    }
                    s0 += t0; s1 += t1; s2 += t2; s3 += t3;
                }
                DS_PROBE(18);
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    if (d < RP) {   // CTA-uniform
                        s0 += __shfl_xor_sync(0xffffffffu, s0, d); s1 += __shfl_xor_sync(0xffffffffu, s1, d);
                        s2 += __shfl_xor_sync(0xffffffffu, s2, d); s3 += __shfl_xor_sync(0xffffffffu, s3, d);
                    }
                }
                DS_PROBE(19);
                if (my_part != 0 || task >= n_task) continue;
                // state elements e0 .. e0 + 3 of the CTA (e = 3 (local row) + component): Eq. (3a) and the
                // 1/(8 pi mu) factor in FP64, then the integrator.  Straight-line: the four elements
                // are independent.
                const int e0 = 4 * task;
                const T sums[4] = {s0, s1, s2, s3};
                if constexpr (!stepping) {               // RUN_APPLY: a2 + a3 with the stream's own F
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int e = e0 + j;
                        if (e < 3 * nrows) {
                            const double Fi = A.raw_F != nullptr ? (double)reinterpret_cast<const T *>(A.raw_F)[(size_t)3 * r0 + e]
                                                                 : (double)units[unit_index<T>(r0 + e / 3, 3 + e % 3)];
                            reinterpret_cast<T *>(A.out_u)[(size_t)3 * r0 + e] = (T)(A.self_mob * Fi + A.pre * (double)sums[j]);
                        }
                    }
                } else {
                // the shared-memory state is padded to whole quads; its global home (state_smem == 0) is not: a last quad
                // of two rows must neither read nor write past its system
                const int e_end = A.state_smem ? e0 + 4 : 3 * nrows;
                double v[4], xo[4], v1[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const bool in = e0 + j < e_end;
                    v[j] = A.self_mob * (in ? Fs[e0 + j] : 0.0) + A.pre * (double)sums[j]; xo[j] = in ? Xs[e0 + j] : 0.0; v1[j] = in ? V1s[e0 + j] : 0.0;
                }
                if (MODE == KM_VELOCITY) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        if (e0 + j < 3 * nrows) reinterpret_cast<T *>(A.out_u)[sys3 + (size_t)3 * r0 + e0 + j] = (T)v[j];
                    continue;
                }
                // predictor X* = X_n + dt V1;  corrector X_{n+1} = X_n + (dt/2)(V1 + V2);  Euler X_{n+1} = X_n + dt V
                // with k_B T > 0 the same increment dW enters the predictor and the corrector (stochastic Heun for
                // additive noise; "can easily incorporate additive noise")
                const double cdt = corr ? 0.5 * A.dt : A.dt;
                const long long nstep = A.n0 + (MODE == KM_HEUN ? (g >> 1) : g);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int e = e0 + j;
                    const double w = corr ? v1[j] + v[j] : v[j];
                    double xn = xo[j] + cdt * w;
                    if (A.noise_amp != 0.0) xn += A.noise_amp * noise_normal(A.seed, nstep, b, 3 * r0 + e);
                    if (e < e_end) {
                        if (pred) V1s[e] = v[j]; else Xs[e] = xn;
                        Xc[e] = xn;
                        if (XcT != nullptr) XcT[e] = (T)xn;
                    }
                }
                }
            }
        }
        if (MODE >= KM_EULER) {
            __syncthreads();
            DS_PROBE(17);
            // Eq. (4) at the new positions and time, one thread per dumbbell; publish the next stage's rows
            if (tid < ((nd + 31) & ~31)) {
                T *un = local ? reinterpret_cast<T *>(smem_raw)
                              : reinterpret_cast<T *>(A.units[(A.cur + g + 1) & 1]) + (size_t)b * A.unit_stride * (6 * W);
                for (int sl = tid; sl < nd; sl += NT) {
                    double x0[3], x1[3], F0[3];
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xc[6 * sl + cc]; x1[cc] = Xc[6 * sl + 3 + cc]; }
                    dumbbell_force(x0, x1, Ls[sl], A.k0, F0);
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
                    if (g + 1 < n_stage)
                        publish_dumbbell(un, use_ll ? ll_of(A.cur + g + 1) : nullptr, A.ll_tag0 + (uint32_t)g + 1u, r0 + 2 * sl, x0, x1, F0);
                }
                fence_proxy_async_global();   // the stream is also read through the async proxy (TMA)
            }
            if (local)   // the pad units share their shared memory with the reduction scratch: rewrite them
                for (int j = 3 * A.U + tid; j < tp; j += NT) reinterpret_cast<uint4 *>(smem_raw)[j] = pad_piece<T>(j % 3);
        }
        DS_PROBE(6);
        fence_proxy_async_shared();
        __syncthreads();  // scratch reads done (the ring may be refilled); this CTA's published rows complete
        DS_PROBE(7);
    }

    if (MODE >= KM_EULER) {   // the state leaves the launch in FP64 and in user precision
        for (int e = tid; e < 3 * nrows; e += NT) {
            const double x = Xs[e];
            if (A.state_smem) A.X[sys3 + 3 * r0 + e] = x;
            reinterpret_cast<T *>(A.xu)[sys3 + 3 * r0 + e] = (T)x;
        }
    }
}

}  // namespace ds
