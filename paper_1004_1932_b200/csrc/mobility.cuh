// mobility.cuh -- the hot kernel: matrix-free all-pairs mobility apply, Eq. (1a) deterministic
// part with the tensor of Eq. (3a,3b), fused with the O(N) tail of the
// time step (self term, reduction, integrator update, next force evaluation).
//
// Decomposition ("row owner": no partial sum ever leaves the SM).
//   grid = (n_cta row tiles, B systems), one CTA of NT = 512 threads per SM.
//   The N alpha-spheres of a system are cut into NQ = ceil(N/4) quads; CTA c owns the contiguous
//   quads [c NQ / n_cta, (c+1) NQ / n_cta) -- nq of them, chosen by the host so that
//   B * n_cta fills the 148 SMs in whole waves (N = 4096: 148 CTAs of 6 or 7 quads).
//   Thread t = (ith, jg) = (t % nq, t / nq): it keeps the I = 4 alpha-spheres of quad q0 + ith in
//   registers and belongs to beta-group jg of n_jg = NT / nq.  The split over beta is therefore
//   INSIDE the CTA; it is undone through shared memory in a fixed order (deterministic, no
//   floating-point atomics, no global scratch, no inter-CTA dependency).
//   Every CTA streams ALL beta-spheres of its system through a ring of NS shared-memory slots filled
//   by TMA bulk copies (cp.async.bulk global -> shared, completion on an mbarrier; one elected
//   thread issues them, consumer warps release slots through a second mbarrier).  The beta-stream
//   lives in global memory in the exact shared-memory layout ("units", see pack.cuh): one unit =
//   W beta-spheres = 6 packs = 48 bytes, so a chunk is one contiguous copy.  N = 4096 (FP32: 96 KB,
//   FP64: 192 KB) is resident at once: all copies are issued up front and the loop only waits.
//   Inside a chunk, group jg takes units jg, jg + n_jg, ... (consecutive groups read consecutive
//   48-byte units: conflict-free LDS.128, broadcast within a group); a chunk holds a multiple of
//   n_jg units (the stream is padded with far-away zero-force units), so every thread of the CTA
//   makes the same number of iterations.
//   r = 0 (alpha == beta) is excluded by a guarded rsqrt compiled only into the loop variant used
//   for chunks that intersect the CTA's own rows (CTA-uniform choice).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pack.cuh"

namespace ds {

enum { TENSOR_OSEEN = 0, TENSOR_RPY = 1 };
enum EpiMode { EPI_APPLY = 0, EPI_EULER = 1, EPI_PRED = 2, EPI_CORR = 3 };

constexpr int NT = 512;                  // threads per CTA: 16 warps, one CTA per SM
constexpr int QI = 4;                    // alpha-spheres per thread (one quad)
constexpr int UNIT_BYTES = 48;           // 6 packs of 8 bytes: x y z Fx Fy Fz of W beta-spheres
constexpr int CHU = 512;                 // units per ring slot (24 KB)
constexpr int NS = 8;                    // ring slots (192 KB)
constexpr int RING_BYTES = NS * CHU * UNIT_BYTES;
constexpr int SMEM_BYTES = RING_BYTES + 2 * NS * 8;
constexpr int PAD_UNITS = CHU;           // dummy units appended to every system's stream

struct MobArgs {
    // problem
    int N, B, NQ, U, n_cta;   // spheres, systems, quads = ceil(N/4), units = ceil(N/W), row tiles per system
    long long unit_stride;    // units per system in the streams (>= U + PAD_UNITS)
    const void *src_units;    // beta-stream T[B][unit_stride][6][W] (also the source of the alpha positions)
    // Eq. (3) constants
    double self_mob;  // 1/(6 pi eta a)   Eq. (3a)
    double pre;       // 1/(8 pi eta)     Eq. (3b)
    double c1, c2;    // 2a^2/3, 2a^2     second line of Eq. (3b), see pair body
    // epilogue
    int mode;
    void *out_u;             // EPI_APPLY: u [B][N][3] user precision
    const double *Fd_in;     // state modes: F(X) in double for the self term, [B][N][3]; NULL -> stream's F
    double *X;               // state positions X_n [B][N][3] (read; written by EULER/CORR)
    double *V1;              // Heun: V(X_n, t_n) [B][N][3] (written by PRED, read by CORR)
    void *units_out;         // stream of the new positions / forces, same layout as src_units
    double *Fd_out;          // new forces in double [B][N][3]
    const double *phase;     // [B][S]
    const long long *n_read; // step counter read by this launch
    long long *n_write;      // = *n_read + n_inc, written by block 0 (double-buffered counter)
    long long n_inc;
    double t0, dt, ell, lambda, omega, k0;
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

// Eq. (4), for the sphere with local row il of a tile whose new positions are in
// sx[c * rows + il]:  n = (X_{2s+1} - X_{2s})/d, g = k0 (d - L(t)), F_{2s} = +g n, F_{2s+1} = -g n.
__device__ __forceinline__ void spring_force(const double *sx, int rows, int il, double phi, double t,
                                             const MobArgs &A, double (&F)[3]) {
    const int e = il & ~1, o = e | 1;
    const double s0 = sx[o] - sx[e], s1 = sx[rows + o] - sx[rows + e], s2 = sx[2 * rows + o] - sx[2 * rows + e];
    const double d = sqrt(s0 * s0 + s1 * s1 + s2 * s2);
    const double L = A.ell + A.lambda * sin(A.omega * t + phi);
    const double g = A.k0 * (d - L);
    const double sgn = (il & 1) ? -1.0 : 1.0;
    F[0] = sgn * (g * (s0 / d));
    F[1] = sgn * (g * (s1 / d));
    F[2] = sgn * (g * (s2 / d));
}

// element (sphere i, component c in 0..5 = x y z Fx Fy Fz) of a unit stream
template <typename T> __device__ __forceinline__ size_t unit_index(long long i, int c) {
    constexpr int W = Pack<T>::W;
    return (size_t)(i / W) * (6 * W) + (size_t)c * W + (size_t)(i % W);
}

// ---------------------------------------------------------------------------------------------
template <typename T, int TENSOR>
__global__ void __launch_bounds__(NT, 1) mobility_kernel(const MobArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + RING_BYTES);
    uint64_t *empty = full + NS;

    const int tid = threadIdx.x, lane = tid & 31;
    const int c = blockIdx.x, b = blockIdx.y;

    // rows of this CTA and the (alpha-thread, beta-group) shape
    const int q0 = (int)((long long)c * A.NQ / A.n_cta), q1 = (int)((long long)(c + 1) * A.NQ / A.n_cta);
    const int nq = q1 - q0;                 // 1 .. NT (host guarantees)
    const int n_jg = NT / nq;
    const int ith = tid % nq, jg = tid / nq;
    const bool active = jg < n_jg;
    const int chu = (CHU / n_jg) * n_jg;    // units per chunk: a multiple of n_jg, <= CHU (n_jg <= NT = CHU)
    const int nchunks = (A.U + chu - 1) / chu;
    const T *units = reinterpret_cast<const T *>(A.src_units) + (size_t)b * A.unit_stride * (6 * W);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, NT / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    // chunk ch = units [ch chu, ch chu + cu): cu rounded up to a multiple of n_jg (the pad units exist)
    auto chunk_units = [&](int ch) {
        const int rem = A.U - ch * chu;
        return rem >= chu ? chu : (rem + n_jg - 1) / n_jg * n_jg;
    };
    auto issue = [&](int ch) {
        const int s = ch % NS;
        const uint32_t bytes = (uint32_t)chunk_units(ch) * UNIT_BYTES;
        mbar_expect_tx(full + s, bytes);
        bulk_g2s(smem_raw + (size_t)s * CHU * UNIT_BYTES, units + (size_t)ch * chu * (6 * W), bytes, full + s);
    };
    if (tid == 0) {
        const int n0 = nchunks < NS ? nchunks : NS;
        for (int ch = 0; ch < n0; ++ch) issue(ch);
        if (A.n_write != nullptr && c == 0 && b == 0) *A.n_write = *A.n_read + A.n_inc;
    }

    // alpha-spheres of this thread: rows 4 (q0 + ith) + k
    V xi[QI][3], acc[QI][3];
#pragma unroll
    for (int k = 0; k < QI; ++k) {
        const long long i = 4LL * (q0 + ith) + k;
        T x = T(0), y = T(0), z = T(0);
        if (i < A.N) {
            x = __ldg(units + unit_index<T>(i, 0));
            y = __ldg(units + unit_index<T>(i, 1));
            z = __ldg(units + unit_index<T>(i, 2));
        }
        xi[k][0] = P::bc(x); xi[k][1] = P::bc(y); xi[k][2] = P::bc(z);
        acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
    }
    const V c1 = P::bc((T)A.c1), negc2 = P::bc((T)(-A.c2));
    const int d0 = (4 * q0) / W, d1 = (4 * q1 + W - 1) / W;  // units that hold this CTA's own rows

    for (int ch = 0; ch < nchunks; ++ch) {
        const int s = ch % NS;
        const uint32_t par = (uint32_t)(ch / NS) & 1u;
        mbar_wait(full + s, par);
        if (active) {
            const int u0 = ch * chu, cu = chunk_units(ch);
            const V2<T> *p = reinterpret_cast<const V2<T> *>(smem_raw + (size_t)s * CHU * UNIT_BYTES) + 3 * jg;
            if (u0 < d1 && u0 + cu > d0)
                pair_units<T, TENSOR, true>(p, 3 * n_jg, cu / n_jg, xi, acc, c1, negc2);
            else
                pair_units<T, TENSOR, false>(p, 3 * n_jg, cu / n_jg, xi, acc, c1, negc2);
        }
        if (ch + NS < nchunks) {  // the slot is needed again: release it, and the producer refills it
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (tid == 0) {
                mbar_wait(empty + s, par);
                issue(ch + NS);
            }
        }
    }
    __syncthreads();  // every chunk consumed by every warp: the ring is free and becomes scratch

    // ---- sum over the n_jg beta-groups (fixed order) ----
    double *red = reinterpret_cast<double *>(smem_raw);  // [n_jg][n_out]        <= 12 NT doubles
    double *red2 = red + 12 * NT;                         // [nparts][n_out]      <= 12 NT
    double *usum = red2 + 12 * NT;                        // [n_out]              <= 12 NT
    double *sx = usum + 12 * NT;                          // [3][rows]            <= 12 NT   (4 x 12 NT x 8 = RING_BYTES)
    const int n_out = 12 * nq, rows = 4 * nq;
    if (active) {
#pragma unroll
        for (int k = 0; k < QI; ++k)
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) red[(size_t)jg * n_out + (k * 3 + cc) * nq + ith] = (double)P::hsum(acc[k][cc]);
    }
    __syncthreads();
    int nparts = NT / n_out;
    nparts = nparts < 1 ? 1 : (nparts > n_jg ? n_jg : nparts);
    for (int idx = tid; idx < n_out * nparts; idx += NT) {
        const int o = idx % n_out, part = idx / n_out;
        double sum = 0.0;
        for (int g = part; g < n_jg; g += nparts) sum += red[(size_t)g * n_out + o];
        red2[(size_t)part * n_out + o] = sum;
    }
    __syncthreads();
    for (int o = tid; o < n_out; o += NT) {
        double sum = red2[o];
        for (int part = 1; part < nparts; ++part) sum += red2[(size_t)part * n_out + o];
        usum[o] = sum;
    }
    __syncthreads();

    // ---- epilogue: Eq. (3a) self term, integrator, next force ----
    const long long nstep = (A.n_read != nullptr) ? *A.n_read : 0;
    // t_{n+1} = t0 + (n+1) dt, formed from the step index (never accumulated), no contraction
    const double t1 = __dadd_rn(A.t0, __dmul_rn((double)(nstep + 1), A.dt));
    for (int il = tid; il < rows; il += NT) {
        const long long i = 4LL * q0 + il;
        if (i < A.N) {
            const int ithr = il >> 2, k = il & 3;
            const size_t g3 = ((size_t)b * A.N + i) * 3;
            double Fi[3];
            if (A.Fd_in != nullptr) {
                Fi[0] = A.Fd_in[g3]; Fi[1] = A.Fd_in[g3 + 1]; Fi[2] = A.Fd_in[g3 + 2];
            } else {
                Fi[0] = units[unit_index<T>(i, 3)]; Fi[1] = units[unit_index<T>(i, 4)]; Fi[2] = units[unit_index<T>(i, 5)];
            }
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                const double v = A.self_mob * Fi[cc] + A.pre * usum[(k * 3 + cc) * nq + ithr];
                if (A.mode == EPI_APPLY) {
                    reinterpret_cast<T *>(A.out_u)[g3 + cc] = (T)v;
                } else if (A.mode == EPI_EULER) {
                    const double xn = A.X[g3 + cc] + A.dt * v;
                    A.X[g3 + cc] = xn;
                    sx[cc * rows + il] = xn;
                } else if (A.mode == EPI_PRED) {
                    A.V1[g3 + cc] = v;
                    sx[cc * rows + il] = A.X[g3 + cc] + A.dt * v;
                } else {  // EPI_CORR
                    const double xn = A.X[g3 + cc] + (0.5 * A.dt) * (A.V1[g3 + cc] + v);
                    A.X[g3 + cc] = xn;
                    sx[cc * rows + il] = xn;
                }
            }
        }
    }
    if (A.mode == EPI_APPLY) return;
    __syncthreads();
    T *uo = reinterpret_cast<T *>(A.units_out) + (size_t)b * A.unit_stride * (6 * W);
    for (int il = tid; il < rows; il += NT) {
        const long long i = 4LL * q0 + il;
        if (i < A.N) {
            const size_t g3 = ((size_t)b * A.N + i) * 3;
            double F[3];
            spring_force(sx, rows, il, A.phase[(size_t)b * (A.N / 2) + (i >> 1)], t1, A, F);
            A.Fd_out[g3] = F[0]; A.Fd_out[g3 + 1] = F[1]; A.Fd_out[g3 + 2] = F[2];
            uo[unit_index<T>(i, 0)] = (T)sx[il];
            uo[unit_index<T>(i, 1)] = (T)sx[rows + il];
            uo[unit_index<T>(i, 2)] = (T)sx[2 * rows + il];
            uo[unit_index<T>(i, 3)] = (T)F[0];
            uo[unit_index<T>(i, 4)] = (T)F[1];
            uo[unit_index<T>(i, 5)] = (T)F[2];
        }
    }
}

}  // namespace ds
