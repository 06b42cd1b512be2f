// small.cuh -- the step kernel for small systems (S <= 32 dumbbells, N <= 64 spheres; BASELINE.json config 1 is N = 16): the
// same time step as mobility.cuh / pipeline.cuh (Eq. (1a) deterministic part with Eq. (3a,3b), Eq. (4), Heun / Euler of
// PAPER.md:236), ONE WARP per system.  Such a system is pure latency: in run_kernel's one-CTA mode a
// stage costs four block-wide barriers, a block-wide shared-memory reduction and ~500 idle threads (2.5 us per stage at N = 16).
//
// Layout.  P = 32 / S' lanes per dumbbell (S' = S rounded up to a power of two): lane = P * dumbbell + part.  Every lane of a
// dumbbell keeps the FP64 state of its two spheres in registers (all P lanes compute the same O(1) update redundantly, so
// nothing has to be broadcast); part p takes the beta-dumbbells p, p + P, ... of the pair sum, and the P partial sums meet in
// log2(P) xor-shuffle steps (fixed order: bitwise reproducible).  The stage's input (positions and forces rounded to T, in
// the unit format of pack.cuh: one FP32 unit = the two spheres of a dumbbell) sits in a warp-private piece of shared memory;
// loads are broadcasts.  Only __syncwarp between the phases; a CTA is 4 independent warps = 4 systems.
#pragma once
#include "mobility.cuh"

namespace ds {

constexpr int SMALL_MAX_S = 32;
constexpr int SMALL_WARPS = 4;      // systems per CTA

struct SmallArgs {
    int S, B;
    double self_mob, pre, c1, c2;
    float c1f, c2f;
    long long n0, n_steps;
    double *X;                    // state [B][N][3] FP64
    void *xu;                     // the same in user precision
    int from_user;
    const double *phase;
    double t0, dt, ell, lambda, omega, k0, noise_amp;
    unsigned long long seed;
};

template <typename T, int TENSOR, bool HEUN>
__global__ void __launch_bounds__(32 * SMALL_WARPS) small_kernel(const SmallArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;
    constexpr int UPD = 2 / W;                              // units per dumbbell: 1 (FP32 packs) or 2 (FP64)
    __shared__ __align__(16) unsigned char sm[SMALL_WARPS][SMALL_MAX_S * UPD * UNIT_BYTES];
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const int b = blockIdx.x * SMALL_WARPS + wi;
    if (b >= A.B) return;                                   // warps are independent: no block-wide barrier below
    const int S = A.S, N = 2 * S;
    int Sp = 1;
    while (Sp < S) Sp <<= 1;
    const int Pl = 32 / Sp;                                  // lanes per dumbbell
    const int d = lane / Pl, part = lane - d * Pl;
    const bool live = d < S;
    T *const units = reinterpret_cast<T *>(sm[wi]);
    const size_t sys3 = (size_t)b * N * 3;

    // FP64 state of the dumbbell's two spheres: X_n, the stage's positions, V1, the force on the first sphere
    double Xn[6] = {0, 0, 0, 1, 0, 0}, Xc[6], V1[6] = {0, 0, 0, 0, 0, 0}, F0[3] = {0, 0, 0}, phi = 0.0, L1 = 0.0;
    if (live) {
#pragma unroll
        for (int e = 0; e < 6; ++e)
            Xn[e] = A.from_user ? (double)reinterpret_cast<const T *>(A.xu)[sys3 + 6 * d + e] : A.X[sys3 + 6 * d + e];
        phi = A.phase[(size_t)b * S + d];
    }
#pragma unroll
    for (int e = 0; e < 6; ++e) Xc[e] = Xn[e];
    auto force_and_publish = [&](double t_or_L, bool is_time) {
        // Eq. (4) at (Xc, t); the dumbbell's unit(s) of the stage's input
        const double x0[3] = {Xc[0], Xc[1], Xc[2]}, x1[3] = {Xc[3], Xc[4], Xc[5]};
        const double L = is_time ? stroke_length(t_or_L, phi, A.ell, A.lambda, A.omega) : t_or_L;
        dumbbell_force(x0, x1, L, A.k0, F0);
        if (live && part == 0) publish_dumbbell(units, nullptr, 0u, 2 * d, x0, x1, F0);
    };
    force_and_publish(time_of_step(A.t0, A.n0, A.dt), true);
    __syncwarp();

    const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
    const int n_stage = (int)(A.n_steps * (HEUN ? 2 : 1));
    for (int g = 0; g < n_stage; ++g) {
        const bool pred = HEUN && (g & 1) == 0, corr = HEUN && (g & 1) == 1;
        const long long nstep = A.n0 + (HEUN ? (g >> 1) : g);
        if (!HEUN || (g & 1) == 0) L1 = stroke_length(time_of_step(A.t0, nstep + 1, A.dt), phi, A.ell, A.lambda, A.omega);
        // ---- pair sums of the two own spheres over this lane's share of the units (own unit: r = 0 excluded by the guard) ----
        V xi[2][3], acc[2][3];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            // rounded exactly as the stream rounds them
            xi[k][0] = P::bc((T)Xc[3 * k]); xi[k][1] = P::bc((T)Xc[3 * k + 1]); xi[k][2] = P::bc((T)Xc[3 * k + 2]);
            acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
        }
        if (live) {
            const V2<T> *ub = reinterpret_cast<const V2<T> *>(units);
#pragma unroll 1
            for (int u = part; u < UPD * S; u += Pl) pair_unit<T, TENSOR, true, 2>(ub + 3 * u, xi, acc, c1, negc2);
        }
        T sum[6];
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) sum[3 * k + cc] = P::hsum(acc[k][cc]);
        for (int dd = 1; dd < Pl; dd <<= 1) {
#pragma unroll
            for (int e = 0; e < 6; ++e) sum[e] += __shfl_xor_sync(0xffffffffu, sum[e], dd);
        }
        __syncwarp();   // every lane is done reading the stage's units
        // ---- Eq. (3a), the 1/(8 pi mu) factor and the integrator, FP64, redundantly on the P lanes of the dumbbell ----
        const double cdt = corr ? 0.5 * A.dt : A.dt;
#pragma unroll
        for (int e = 0; e < 6; ++e) {
            const double Fe = e < 3 ? F0[e] : -F0[e - 3];
            const double v = A.self_mob * Fe + A.pre * (double)sum[e];
            const double w = corr ? V1[e] + v : v;
            double xn = Xn[e] + cdt * w;
            if (A.noise_amp != 0.0) xn += A.noise_amp * noise_normal(A.seed, nstep, b, 6 * d + e);
            if (pred) V1[e] = v; else Xn[e] = xn;
            Xc[e] = xn;
        }
        if (g + 1 < n_stage) force_and_publish(L1, false);
        __syncwarp();
    }
    if (live && part == 0) {
#pragma unroll
        for (int e = 0; e < 6; ++e) {
            A.X[sys3 + 6 * d + e] = Xn[e];
            reinterpret_cast<T *>(A.xu)[sys3 + 6 * d + e] = (T)Xn[e];
        }
    }
}

}  // namespace ds
