// mobility.cuh -- the hot kernel: matrix-free all-pairs mobility apply, Eq. (1a) deterministic
// part with the tensor of Eq. (3a,3b), fused with the O(N) tail of the
// time step (self term, split-j reduction, integrator update, next force evaluation).
//
// Decomposition (one launch = one apply for all B systems):
//   grid = (JS j-splits, n_it i-tiles, B systems); block = 32*WI*WJ threads.
//   An i-tile holds TI = 32*I*WI spheres alpha: lane l of i-warp wi owns alpha = it*TI + wi*32*I + k*32 + l,
//   k < I, in registers (positions broadcast into packs, 3 accumulator packs each).
//   The block's beta-range [js*jchunk, (js+1)*jchunk) is staged through shared memory in stages
//   of <= SJ spheres; inside a stage the WJ j-warp-groups take consecutive sub-ranges.
//   Every inner iteration loads one "unit" (W beta-spheres: 3 x LDS.128, same address for the whole
//   warp = broadcast) and applies it to the I alpha-spheres of the lane.
//   r = 0 (alpha == beta) is excluded by a guarded rsqrt that is only compiled into the loop
//   taken when a warp's alpha-range and beta-sub-range intersect (warp-uniform choice).
//   Tail: the WJ groups are summed through shared memory in fixed order; with JS > 1 the block
//   stores its partial sums, takes a ticket, and the LAST block of the i-tile adds the JS partials
//   in fixed order (deterministic; no floating-point atomics) and runs the epilogue.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pack.cuh"

namespace ds {

enum { TENSOR_OSEEN = 0, TENSOR_RPY = 1 };
enum EpiMode { EPI_APPLY = 0, EPI_EULER = 1, EPI_PRED = 2, EPI_CORR = 3 };

struct MobArgs {
    // problem
    int N, B, Npad, n_it, JS, jchunk;
    // beta/alpha source: user layout T[B][N][3] (src_user = 1) or packed T4[B][Npad]
    const void *src_pos, *src_F;
    // split-j reduction scratch
    double *partial;     // [B][JS][3][Npad]
    unsigned *counters;  // [B][n_it], zero between launches
    // Eq. (3) constants
    double self_mob;  // 1/(6 pi eta a)   Eq. (3a)
    double pre;       // 1/(8 pi eta)     Eq. (3b)
    double c1, c2;    // 2a^2/3, 2a^2     second line of Eq. (3b), see pair body
    // epilogue
    int mode;
    void *out_u;             // EPI_APPLY: u [B][N][3] user precision
    const double *Fd_in;     // state modes: F(X) in double for the self term, [B][N][3]; NULL -> src_F
    double *X;               // state positions X_n [B][N][3] (read; written by EULER/CORR)
    double *V1;              // Heun: V(X_n, t_n) [B][N][3] (written by PRED, read by CORR)
    void *pos4_out, *F4_out; // packed copies of the new positions / forces, T4[B][Npad]
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
// source loaders
template <typename T, bool USER>
__device__ __forceinline__ void load_pos(const MobArgs &A, int b, int j, T &x, T &y, T &z) {
    typedef typename Pack<T>::T4 T4;
    if (j < A.N) {
        if (USER) {
            const T *p = reinterpret_cast<const T *>(A.src_pos) + ((size_t)b * A.N + j) * 3;
            x = p[0]; y = p[1]; z = p[2];
        } else {
            T4 v = reinterpret_cast<const T4 *>(A.src_pos)[(size_t)b * A.Npad + j];
            x = v.x; y = v.y; z = v.z;
        }
    } else {
        x = y = z = Pack<T>::dummy();
    }
}
template <typename T, bool USER>
__device__ __forceinline__ void load_F(const MobArgs &A, int b, int j, T &x, T &y, T &z) {
    typedef typename Pack<T>::T4 T4;
    if (j < A.N) {
        if (USER) {
            const T *p = reinterpret_cast<const T *>(A.src_F) + ((size_t)b * A.N + j) * 3;
            x = p[0]; y = p[1]; z = p[2];
        } else {
            T4 v = reinterpret_cast<const T4 *>(A.src_F)[(size_t)b * A.Npad + j];
            x = v.x; y = v.y; z = v.z;
        }
    } else {
        x = y = z = T(0);
    }
}

// ---------------------------------------------------------------------------------------------
// The pair body.  With r = x_a - x_b, w = 1/r^2, Eq. (3b) contracted with F_b is
//   Oseen: (1/8 pi mu) (1/r) [ F_b + (r.F_b) w r ]
//   RPY  : (1/8 pi mu) { (1/r + c1/r^3) F_b + (r.F_b) (1/r^3) (1 - c2 w) r },  c1 = 2a^2/3, c2 = 2a^2
// (second line of (3b): 2a^2/(24 pi mu r^3) (delta - 3 rr/r^2) = (1/8 pi mu)(1/r^3)[(2a^2/3) delta - 2a^2 rr/r^2]).
// The common factor 1/(8 pi mu) is applied once per alpha in the epilogue.
// FP32-pipe instruction count per pack: 3 sub + 3 (r^2) + 3 (r.F) + 2 + 6 = 17 (Oseen), 21 (RPY).
template <typename T, int TENSOR, int I, bool GUARD, int UNROLL>
__device__ __forceinline__ void pair_units(const V2<T> *__restrict__ sU, int u0, int u1,
                                           const typename Pack<T>::V (&xi)[I][3],
                                           typename Pack<T>::V (&acc)[I][3], typename Pack<T>::V c1,
                                           typename Pack<T>::V negc2) {
    typedef Pack<T> P;
    typedef typename P::V V;
#pragma unroll UNROLL
    for (int u = u0; u < u1; ++u) {
        const V2<T> q0 = sU[3 * u], q1 = sU[3 * u + 1], q2 = sU[3 * u + 2];
        const V xj = q0.a, yj = q0.b, zj = q1.a, fx = q1.b, fy = q2.a, fz = q2.b;
#pragma unroll
        for (int k = 0; k < I; ++k) {
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

// Eq. (4), for the sphere with local index il of a tile whose new positions are in
// sx[c][il]:  n = (X_{2s+1} - X_{2s})/d, g = k0 (d - L(t)), F_{2s} = +g n, F_{2s+1} = -g n.
template <int TI>
__device__ __forceinline__ void spring_force(const double (*sx)[TI], int il, double phi, double t,
                                             const MobArgs &A, double (&F)[3]) {
    const int e = il & ~1, o = e | 1;
    const double s0 = sx[0][o] - sx[0][e], s1 = sx[1][o] - sx[1][e], s2 = sx[2][o] - sx[2][e];
    const double d = sqrt(s0 * s0 + s1 * s1 + s2 * s2);
    const double L = A.ell + A.lambda * sin(A.omega * t + phi);
    const double g = A.k0 * (d - L);
    const double sgn = (il & 1) ? -1.0 : 1.0;
    F[0] = sgn * (g * (s0 / d));
    F[1] = sgn * (g * (s1 / d));
    F[2] = sgn * (g * (s2 / d));
}

template <typename T> struct MakeT4;
template <> struct MakeT4<float> {
    static __device__ __forceinline__ float4 make(double x, double y, double z) {
        return make_float4((float)x, (float)y, (float)z, 0.f);
    }
};
template <> struct MakeT4<double> {
    static __device__ __forceinline__ double4 make(double x, double y, double z) {
        return make_double4(x, y, z, 0.0);
    }
};

template <int I, int WI, int WJ, int SJ> struct MobShape {
    static constexpr int TI = 32 * I * WI;
    static constexpr int NT = 32 * WI * WJ;
    static constexpr size_t stage_bytes = (size_t)SJ * 6 * 8 / 1;  // per j: 6 scalars; sized for T = double
    static constexpr size_t red_bytes = (size_t)WJ * 3 * TI * sizeof(double);
    static constexpr size_t epi_bytes = (size_t)2 * 3 * TI * sizeof(double);
};

template <typename T> __host__ __device__ constexpr size_t stage_bytes_for(int SJ) { return (size_t)SJ * 6 * sizeof(T); }

// ---------------------------------------------------------------------------------------------
template <typename T, int TENSOR, bool USER, int I, int WI, int WJ, int SJ, int UNROLL, int MINB>
__global__ void __launch_bounds__(32 * WI * WJ, MINB) mobility_kernel(const MobArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    typedef typename P::T4 T4;
    constexpr int W = P::W;
    constexpr int TI = 32 * I * WI;
    constexpr int NT = 32 * WI * WJ;
    static_assert(SJ % (W * WJ) == 0, "stage must split evenly over the j-warp-groups");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *sT = reinterpret_cast<T *>(smem_raw);                           // stage: [unit][6][W]
    const V2<T> *sU = reinterpret_cast<const V2<T> *>(smem_raw);
    double(*red)[3][TI] = reinterpret_cast<double(*)[3][TI]>(smem_raw + stage_bytes_for<T>(SJ));
    double(*usum)[TI] = reinterpret_cast<double(*)[TI]>(smem_raw + stage_bytes_for<T>(SJ) +
                                                        (size_t)WJ * 3 * TI * sizeof(double));
    double(*sx)[TI] = usum + 3;
    __shared__ int s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp % WI, wj = warp / WI;
    const int js = blockIdx.x, it = blockIdx.y, b = blockIdx.z;

    if (A.n_write != nullptr && tid == 0 && js == 0 && it == 0 && b == 0) *A.n_write = *A.n_read + A.n_inc;

    // alpha-spheres of this lane
    const int iw0 = it * TI + wi * 32 * I;  // first alpha of this warp
    V xi[I][3], acc[I][3];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        T x, y, z;
        load_pos<T, USER>(A, b, iw0 + k * 32 + lane, x, y, z);
        xi[k][0] = P::bc(x); xi[k][1] = P::bc(y); xi[k][2] = P::bc(z);
        acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
    }
    const V c1 = P::bc((T)A.c1), negc2 = P::bc((T)(-A.c2));

    // beta-range of this block
    const int jbeg = js * A.jchunk;
    const int jend = min(jbeg + A.jchunk, A.N);
    for (int jb = jbeg; jb < jend; jb += SJ) {
        const int nj = min(SJ, jend - jb);
        const int per = (nj + W * WJ - 1) / (W * WJ);  // units per j-warp-group in this stage
        const int njp = per * W * WJ;                  // padded stage length (dummy spheres, F = 0)
        __syncthreads();                               // previous stage fully consumed
        for (int jl = tid; jl < njp; jl += NT) {
            T x, y, z, fx, fy, fz;
            const int j = (jl < nj) ? jb + jl : A.N;   // A.N -> dummy
            load_pos<T, USER>(A, b, j, x, y, z);
            load_F<T, USER>(A, b, j, fx, fy, fz);
            T *d = sT + (size_t)(jl / W) * (6 * W) + (jl % W);
            d[0 * W] = x; d[1 * W] = y; d[2 * W] = z; d[3 * W] = fx; d[4 * W] = fy; d[5 * W] = fz;
        }
        __syncthreads();
        const int u0 = wj * per, u1 = u0 + per;
        const int ja = jb + u0 * W, jz = jb + u1 * W;  // beta sub-range of this warp
        const bool diag = (ja < iw0 + 32 * I) && (iw0 < jz);
        if (diag)
            pair_units<T, TENSOR, I, true, UNROLL>(sU, u0, u1, xi, acc, c1, negc2);
        else
            pair_units<T, TENSOR, I, false, UNROLL>(sU, u0, u1, xi, acc, c1, negc2);
    }

    // ---- sum over the WJ j-warp-groups (fixed order) ----
#pragma unroll
    for (int k = 0; k < I; ++k)
#pragma unroll
        for (int c = 0; c < 3; ++c) red[wj][c][wi * 32 * I + k * 32 + lane] = (double)P::hsum(acc[k][c]);
    __syncthreads();
    const size_t prow = (size_t)A.Npad;
    for (int idx = tid; idx < 3 * TI; idx += NT) {
        const int c = idx / TI, il = idx % TI;
        double s = red[0][c][il];
#pragma unroll
        for (int g = 1; g < WJ; ++g) s += red[g][c][il];
        if (A.JS > 1)
            A.partial[(((size_t)b * A.JS + js) * 3 + c) * prow + (size_t)it * TI + il] = s;
        else
            usum[c][il] = s;
    }

    // ---- split-j: last block of this i-tile reduces the JS partials in fixed order ----
    if (A.JS > 1) {
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const unsigned t = atomicAdd(&A.counters[(size_t)b * A.n_it + it], 1u);
            s_last = (t == (unsigned)(A.JS - 1));
        }
        __syncthreads();
        if (!s_last) return;
        __threadfence();
        if (tid == 0) A.counters[(size_t)b * A.n_it + it] = 0u;  // ready for the next launch
        for (int idx = tid; idx < 3 * TI; idx += NT) {
            const int c = idx / TI, il = idx % TI;
            const double *p = A.partial + ((size_t)b * A.JS * 3 + c) * prow + (size_t)it * TI + il;
            double s = 0.0;
            for (int g = 0; g < A.JS; ++g) s += __ldcg(p + (size_t)g * 3 * prow);
            usum[c][il] = s;
        }
    }
    __syncthreads();

    // ---- epilogue: Eq. (3a) self term, integrator, next force ----
    const long long nstep = (A.n_read != nullptr) ? *A.n_read : 0;
    // t_{n+1} = t0 + (n+1) dt, formed from the step index (never accumulated), no contraction
    const double t1 = __dadd_rn(A.t0, __dmul_rn((double)(nstep + 1), A.dt));
    for (int il = tid; il < TI; il += NT) {
        const int i = it * TI + il;
        if (i < A.N) {
            const size_t g3 = ((size_t)b * A.N + i) * 3;
            double Fi[3];
            if (A.Fd_in != nullptr) {
                Fi[0] = A.Fd_in[g3]; Fi[1] = A.Fd_in[g3 + 1]; Fi[2] = A.Fd_in[g3 + 2];
            } else {
                T fx, fy, fz;
                load_F<T, USER>(A, b, i, fx, fy, fz);
                Fi[0] = fx; Fi[1] = fy; Fi[2] = fz;
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double v = A.self_mob * Fi[c] + A.pre * usum[c][il];
                if (A.mode == EPI_APPLY) {
                    reinterpret_cast<T *>(A.out_u)[g3 + c] = (T)v;
                } else if (A.mode == EPI_EULER) {
                    const double xn = A.X[g3 + c] + A.dt * v;
                    A.X[g3 + c] = xn;
                    sx[c][il] = xn;
                } else if (A.mode == EPI_PRED) {
                    A.V1[g3 + c] = v;
                    sx[c][il] = A.X[g3 + c] + A.dt * v;
                } else {  // EPI_CORR
                    const double xn = A.X[g3 + c] + (0.5 * A.dt) * (A.V1[g3 + c] + v);
                    A.X[g3 + c] = xn;
                    sx[c][il] = xn;
                }
            }
        }
    }
    if (A.mode == EPI_APPLY) return;
    __syncthreads();
    for (int il = tid; il < TI; il += NT) {
        const int i = it * TI + il;
        if (i < A.N) {
            const size_t g3 = ((size_t)b * A.N + i) * 3;
            double F[3];
            spring_force<TI>(sx, il, A.phase[(size_t)b * (A.N / 2) + (i >> 1)], t1, A, F);
            A.Fd_out[g3] = F[0]; A.Fd_out[g3 + 1] = F[1]; A.Fd_out[g3 + 2] = F[2];
            reinterpret_cast<T4 *>(A.pos4_out)[(size_t)b * A.Npad + i] = MakeT4<T>::make(sx[0][il], sx[1][il], sx[2][il]);
            reinterpret_cast<T4 *>(A.F4_out)[(size_t)b * A.Npad + i] = MakeT4<T>::make(F[0], F[1], F[2]);
        }
    }
}

}  // namespace ds
