// cluster.cuh -- the step kernel for ensembles of medium systems (BASELINE.json config 5: B = 64 systems of N = 512): the same
// time step as mobility.cuh / pipeline.cuh (Eq. (1a) deterministic part with Eq. (3a,3b), Eq. (4), Heun / Euler of
// PAPER.md:236), one THREAD-BLOCK CLUSTER per system, software-pipelined like pipeline.cuh.
//
// Why.  With B systems on 148 SMs a system gets 148 / B SMs (two at B = 64).  In run_kernel those CTAs hand their rows over
// through global memory: publish, release, arrival counter, poll, copy, four block-wide barriers and a block-wide reduction
// per stage -- 9.7 k of a stage's 35 k cycles at B = 64, N = 512.  The CTAs of a system need nothing from any other system, so
// they can be one cluster and hand over through distributed shared memory; and, as in pipeline.cuh, the tail of a stage can
// run beside the pair loops of the next half stage instead of after them.
//
// How.  grid = (cs, B), cluster = (cs, 1, 1), cs = 2, 4 or 8 CTAs of 640 threads: 16 compute warps + a service warpgroup.
// CTA r owns the contiguous quads [r NQ / cs, (r + 1) NQ / cs) of its system for the whole launch (FP64 state in shared
// memory), cut into two halves A and B of whole quads; a stage is two passes, pass h = (alpha in half h) x (all beta).
// EVERY CTA keeps the whole beta-stream of its system in its own shared memory (positions and forces rounded to T, the unit
// format of pack.cuh), as two regions (region h = the half-h units of all CTAs, in CTA order), twice (stage parity).
//   compute warps   pass h over nq_h quads: nq_h <= 16: 16 / nq_h warps per quad, all lanes of a warp hold the same 4
//                   alpha-spheres; nq_h > 16: QW = 2, 4 or 8 quads per warp, G = 32 / QW lanes per quad.  A lane walks the
//                   units jg, jg + n_jg, ... of region A, then of region B (conflict-free / broadcast LDS.128).  The G lanes
//                   of a quad add their 12 sums with a fixed shuffle tree and leave 12 numbers per (quad, warp) in shared memory.
//   service warps   when the sums of pass h are complete (mbarrier): fixed-order sum over the quad's warps, Eq. (3a),
//                   1/(8 pi mu), integrator (FP64), Eq. (4) at the new positions, and the half's units of the NEXT stage's
//                   stream go into the shared memory of every CTA of the cluster with st.async (16-byte stores through
//                   distributed shared memory, each completing 16 bytes of the destination CTA's "region landed" mbarrier)
//                   -- while the compute warps are in the next pass.
// No block-wide or cluster-wide barrier inside the step loop, no global memory, no counter, no polling of memory.  Pass A
// of stage g + 1 starts on region A, published half a stage earlier by every CTA.  Buffers of parity (g + 1) & 1 are free
// when a CTA publishes into them: it has finished a pass of stage g, which read every CTA's region B of stage g, which each
// CTA sent only after its last read of stage g - 1.  No atomics: bitwise reproducible, independent of how steps are split
// over launches.  Clusters are independent of one another.
#pragma once
#include "pipeline.cuh"

namespace ds {

constexpr int CL_CW = 16;                        // compute warps
constexpr int CL_NT = 32 * (CL_CW + 4);          // + the service warpgroup
constexpr int CL_MAX_CS = 8;                     // portable cluster size (the latency variant also takes 16)
constexpr int CL_MAX_QW = 8;                     // quads per warp (lanes per quad >= 4)
constexpr int CL_BAR_BYTES = 128;                // 8 mbarriers
constexpr int CL_TAB_BYTES = 2 * CL_CW * 2 * 16; // per pass and warp: its place and loop bounds (stage-invariant)
constexpr int CL_PAD_UNITS = 32 * CL_CW;         // far-away units behind a region: an iteration never reads past them

struct ClusterArgs {
    int N, NQ, cs;
    int half_off[2][CL_MAX_CS + 1];   // first unit of CTA r's half h inside region h; [h][cs] = units of region h
    int buf_units[2];                 // capacity of a region buffer in units (region + CL_PAD_UNITS, multiple of 8)
    int rows_max;                     // most rows any CTA owns (state sizing)
    int slots_max;                    // most (quad, warp) sums any pass leaves (scratch sizing)
    double self_mob, pre, c1, c2;     // Eq. (3a), (3b) constants as in RunArgs
    float c1f, c2f;
    long long n0, n_steps;
    double *X;                        // state [B][N][3] FP64
    void *xu;                         // the same in user precision
    int from_user;
    const double *phase;
    double t0, dt, ell, lambda, omega, k0, noise_amp;
    unsigned long long seed;
};

__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// 16 bytes into another CTA's shared memory; completes 16 bytes of the transaction count of that CTA's mbarrier
__device__ __forceinline__ void st_async_16(uint32_t addr, float4 v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(addr),
                 "r"(__float_as_uint(v.x)), "r"(__float_as_uint(v.y)), "r"(__float_as_uint(v.z)), "r"(__float_as_uint(v.w)), "r"(mbar)
                 : "memory");
}
__device__ __forceinline__ void st_async_16(uint32_t addr, double2 v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];" ::"r"(addr),
                 "l"(__double_as_longlong(v.x)), "l"(__double_as_longlong(v.y)), "r"(mbar)
                 : "memory");
}
// wait for a phase completed by other CTAs' st.async
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAITC_%=:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONEC_%=;\n"
        "bra WAITC_%=;\n"
        "DONEC_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// The two spheres of a dumbbell -> their 48 bytes (FP32: one unit) / 96 bytes (FP64: two units) at the shared::cluster
// address `dst` of a CTA's stream buffer.
__device__ __forceinline__ void publish_async(float, uint32_t dst, uint32_t mbar, const double (&x0)[3], const double (&x1)[3],
                                              const double (&F0)[3]) {
    st_async_16(dst, make_float4((float)x0[0], (float)x1[0], (float)x0[1], (float)x1[1]), mbar);
    st_async_16(dst + 16, make_float4((float)x0[2], (float)x1[2], (float)F0[0], (float)(-F0[0])), mbar);
    st_async_16(dst + 32, make_float4((float)F0[1], (float)(-F0[1]), (float)F0[2], (float)(-F0[2])), mbar);
}
__device__ __forceinline__ void publish_async(double, uint32_t dst, uint32_t mbar, const double (&x0)[3], const double (&x1)[3],
                                              const double (&F0)[3]) {
    st_async_16(dst, make_double2(x0[0], x0[1]), mbar);
    st_async_16(dst + 16, make_double2(x0[2], F0[0]), mbar);
    st_async_16(dst + 32, make_double2(F0[1], F0[2]), mbar);
    st_async_16(dst + 48, make_double2(x1[0], x1[1]), mbar);
    st_async_16(dst + 64, make_double2(x1[2], -F0[0]), mbar);
    st_async_16(dst + 80, make_double2(-F0[1], -F0[2]), mbar);
}

// 12 values per lane -> their sums over the G = 4, 8, 16 or 32 lanes of an aligned group, in a fixed order.  After the call
// the lane with bits (G/2, G/4) = (j >> 1, j & 1) and the bits below clear holds in s[0..2] the totals of v[3 j + 0..2].
template <typename T> __device__ __forceinline__ void group_sum12(const T (&v)[12], int lane, int G, T (&s)[3]) {
    const int d1 = G >> 1, d2 = G >> 2;
    const bool up1 = lane & d1, up2 = lane & d2;
    T a[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        const T keep = up1 ? v[6 + i] : v[i], send = up1 ? v[i] : v[6 + i];
        a[i] = keep + __shfl_xor_sync(0xffffffffu, send, d1);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const T keep = up2 ? a[3 + i] : a[i], send = up2 ? a[i] : a[3 + i];
        s[i] = keep + __shfl_xor_sync(0xffffffffu, send, d2);
    }
#pragma unroll 1
    for (int d = d2 >> 1; d >= 1; d >>= 1) {
#pragma unroll
        for (int i = 0; i < 3; ++i) s[i] += __shfl_xor_sync(0xffffffffu, s[i], d);
    }
}

// shape of a pass over nqh quads: quads per warp, warps per quad
__host__ __device__ inline void cluster_pass_shape(int nqh, int &QW, int &m) {
    QW = 1; m = 1;
    if (nqh <= 0) return;
    if (nqh <= CL_CW) { m = CL_CW / nqh; return; }
    while (CL_CW * QW < nqh) QW <<= 1;
}

template <typename T, int TENSOR, bool HEUN>
__global__ void __launch_bounds__(CL_NT, 1) cluster_kernel(const ClusterArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = blockIdx.x, b = blockIdx.y;               // rank in the cluster (cluster = the grid's x extent), system
    const int cs = A.cs;

    const size_t capA_bytes = (size_t)A.buf_units[0] * UNIT_BYTES, par_bytes = capA_bytes + (size_t)A.buf_units[1] * UNIT_BYTES;
    auto region = [&](int par, int h) { return smem_raw + (size_t)par * par_bytes + (h ? capA_bytes : 0); };
    unsigned char *const after = smem_raw + 2 * par_bytes;
    uint64_t *const mb_full = reinterpret_cast<uint64_t *>(after);   // [parity][region]: the region has landed in this CTA
    uint64_t *const mb_part = mb_full + 4;                           // [pass] every compute warp has left its sums of pass h
    uint64_t *const mb_xi = mb_full + 6;                             // [half] the half's rows of the next stage are in XcT
    int4 *const ptab = reinterpret_cast<int4 *>(after + CL_BAR_BYTES);                    // [2][16][2]
    T *const scr = reinterpret_cast<T *>(after + CL_BAR_BYTES + CL_TAB_BYTES);           // [2][slots_max][12]
    double *const st = reinterpret_cast<double *>(after + CL_BAR_BYTES + CL_TAB_BYTES + (size_t)2 * A.slots_max * 12 * 8);

    // rows of this CTA and its two halves (whole quads; a dumbbell never straddles them)
    const int q0 = (int)((long long)r * A.NQ / cs), q1 = (int)((long long)(r + 1) * A.NQ / cs);
    const int nq = q1 - q0;
    const long long r0 = 4LL * q0;
    const int nrows = (int)((A.N - r0) < 4 * nq ? (A.N - r0) : 4 * nq);
    const int nd = nrows >> 1;
    const int nqA = pipe_split(nq);
    const int rowsA = 4 * nqA < nrows ? 4 * nqA : nrows, rowsB = nrows - rowsA;
    const int ownA = A.half_off[0][r], ownB = A.half_off[1][r];      // first own unit inside region 0 / 1
    const int UA = A.half_off[0][cs], UB = A.half_off[1][cs];        // units of region 0 / 1
    const int rows_st = A.rows_max;
    double *const Xs = st, *const Xc = st + 3 * rows_st, *const V1s = st + 6 * rows_st, *const Fs = st + 9 * rows_st;
    double *const Ls = st + 12 * rows_st, *const phs = Ls + (rows_st >> 1);
    T *const XcT = reinterpret_cast<T *>(st + 13 * rows_st);
    const size_t sys3 = (size_t)b * A.N * 3;
    const int n_stage = (int)(A.n_steps * (HEUN ? 2 : 1));

    // dumbbell sl of half h (rows rbase + 2 sl, + 1) -> region h of the stream of parity par in EVERY CTA of the cluster
    auto publish_all = [&](int par, int h, int sl, const double (&x0)[3], const double (&x1)[3], const double (&F0)[3]) {
        const uint32_t dst = smem_u32(region(par, h)) + (uint32_t)((h == 0 ? ownA : ownB) + (2 * sl) / W) * UNIT_BYTES;
        const uint32_t bar = smem_u32(mb_full + 2 * par + h);
        for (int p = 0; p < cs; ++p) publish_async(T(), mapa_u32(dst, (uint32_t)p), mapa_u32(bar, (uint32_t)p), x0, x1, F0);
    };

    // ---- prologue (all warps): state, barriers, pads, F(X_n, t_n), stream 0 ----
    for (int e = tid; e < 3 * nrows; e += CL_NT) {
        const double x = A.from_user ? (double)reinterpret_cast<const T *>(A.xu)[sys3 + 3 * r0 + e] : A.X[sys3 + 3 * r0 + e];
        Xs[e] = x; Xc[e] = x; XcT[e] = (T)x;
    }
    for (int e = 3 * nrows + tid; e < 3 * rows_st; e += CL_NT) XcT[e] = P::dummy();   // rows of a last, partial quad
    for (int sl = tid; sl < nd; sl += CL_NT) phs[sl] = A.phase[(size_t)b * (A.N / 2) + (r0 >> 1) + sl];
    if (tid == 0) {
        for (int k = 0; k < 4; ++k) mbar_init(mb_full + k, 1);
        for (int h = 0; h < 2; ++h) { mbar_init(mb_part + h, CL_CW); mbar_init(mb_xi + h, 1); }
        mbar_fence_init();
        // streams 0 and 1: one pending arrival + the region's bytes each
        for (int par = 0; par < 2; ++par)
            for (int h = 0; h < 2; ++h) mbar_expect_tx(mb_full + 2 * par + h, (uint32_t)(h == 0 ? UA : UB) * UNIT_BYTES);
    }
    if (tid >= 32 && tid < 32 + 2 * CL_CW) {
        // Which warp does what in the two passes (stage-invariant): {first quad or -1, log2 G, n_jg, sub} and the loop bounds
        // {iterations in region 0, in region 1, first / end of the guarded ones (region h only)}.
        const int h = (tid - 32) / CL_CW, w = (tid - 32) % CL_CW;
        const int nqh = h == 0 ? nqA : nq - nqA, rows_h = h == 0 ? rowsA : rowsB;
        int QW, m;
        cluster_pass_shape(nqh, QW, m);
        const int G = 32 / QW, n_jg = G * m, qfirst = (w / m) * QW, sub = w % m;
        int lg = 0;
        while ((1 << lg) < G) ++lg;
        int4 a = make_int4(-1, lg, n_jg, sub), bb = make_int4(0, 0, 0, 0);
        if (qfirst < nqh) {
            a.x = qfirst;
            int itw[2];
            for (int reg = 0; reg < 2; ++reg) {
                const int Ur = reg == 0 ? UA : UB, its = (Ur + n_jg - 1) / n_jg;
                // the last iteration is skipped by warps whose units all lie behind the region
                itw[reg] = its - ((its > 0 && (its - 1) * n_jg + sub * G >= Ur) ? 1 : 0);
            }
            // units of region h that hold rows of this warp's quads (alpha == beta): guarded iterations
            const int own_h = h == 0 ? ownA : ownB;
            const int rl0 = 4 * qfirst, rl1 = 4 * (qfirst + QW) < rows_h ? 4 * (qfirst + QW) : rows_h;
            const int uo0 = own_h + rl0 / W, uo1 = own_h + rl1 / W;
            int g_lo = itw[h], g_hi = itw[h];
            if (uo1 > uo0) {
                g_lo = uo0 / n_jg; g_hi = (uo1 - 1) / n_jg + 1;
                g_lo = g_lo < itw[h] ? g_lo : itw[h]; g_hi = g_hi < itw[h] ? g_hi : itw[h];
            }
            bb = make_int4(itw[0], itw[1], g_lo, g_hi);
        }
        ptab[(h * CL_CW + w) * 2] = a;
        ptab[(h * CL_CW + w) * 2 + 1] = bb;
    }
    for (int k = 0; k < 4; ++k) {   // far-away zero-force pad units behind each region (never overwritten)
        uint4 *bp = reinterpret_cast<uint4 *>(region(k >> 1, k & 1));
        for (int j = 3 * ((k & 1) ? UB : UA) + tid; j < 3 * A.buf_units[k & 1]; j += CL_NT) bp[j] = pad_piece<T>(j % 3);
    }
    cluster_barrier();   // every CTA of the cluster runs and has armed its barriers; own state visible
    {
        const double tn = time_of_step(A.t0, A.n0, A.dt);
        for (int sl = tid; sl < nd; sl += CL_NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xs[6 * sl + cc]; x1[cc] = Xs[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, stroke_length(tn, phs[sl], A.ell, A.lambda, A.omega), A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            const int h = 2 * sl < rowsA ? 0 : 1;
            if (n_stage > 0) publish_all(0, h, sl - (h ? rowsA >> 1 : 0), x0, x1, F0);
        }
    }
    __syncthreads();

    if (warp < CL_CW) {
        // =========================== compute warps ===========================
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_COMPUTE_F64));
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_COMPUTE));
        const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
        for (int g = 0; g < n_stage; ++g) {
            const int par = g & 1;
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int nqh = h == 0 ? nqA : nq - nqA, rbase = h == 0 ? 0 : rowsA;
                const int4 pa = ptab[(h * CL_CW + warp) * 2], pb = ptab[(h * CL_CW + warp) * 2 + 1];
                const int qfirst = pa.x < 0 ? nqh : pa.x, lgG = pa.y, G = 1 << lgG, n_jg = pa.z, sub = pa.w;
                const int quad = qfirst + (lane >> lgG), jg = (sub << lgG) + (lane & (G - 1));
                const bool act = quad < nqh;
                V xi[QI][3], acc[QI][3];
#pragma unroll
                for (int k = 0; k < QI; ++k) acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
                if (qfirst < nqh) {
                    mbar_wait(mb_xi + h, (uint32_t)par);
                    // the quad's 12 coordinates are contiguous and 16-byte aligned (rows beyond the system hold a far-away dummy)
                    T xq[12];
                    const typename P::T4 *xp = reinterpret_cast<const typename P::T4 *>(XcT + 3 * (rbase + 4 * (act ? quad : qfirst)));
#pragma unroll
                    for (int k = 0; k < 3; ++k) { const typename P::T4 q = xp[k]; xq[4 * k] = q.x; xq[4 * k + 1] = q.y; xq[4 * k + 2] = q.z; xq[4 * k + 3] = q.w; }
#pragma unroll
                    for (int k = 0; k < QI; ++k) { xi[k][0] = P::bc(xq[3 * k]); xi[k][1] = P::bc(xq[3 * k + 1]); xi[k][2] = P::bc(xq[3 * k + 2]); }
                }
#pragma unroll 1
                for (int reg = 0; reg < 2; ++reg) {
                    if (h == 0) mbar_wait_cluster(mb_full + 2 * par + reg, (uint32_t)(g >> 1) & 1u);   // pass B need not look again
                    if (act) {
                        const int its_w = reg == 0 ? pb.x : pb.y;
                        const int g_lo = reg == h ? pb.z : its_w, g_hi = reg == h ? pb.w : its_w;
                        const V2<T> *p = reinterpret_cast<const V2<T> *>(region(par, reg)) + 3 * jg;
                        const int stride = 3 * n_jg;
                        int it = 0;
#pragma unroll 1
                        for (; it < g_lo; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
#pragma unroll 1
                        for (; it < g_hi; ++it, p += stride) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
#pragma unroll 1
                        for (; it < its_w; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                    }
                }
                if (qfirst < nqh) {
                    T v[12], s[3];
#pragma unroll
                    for (int k = 0; k < QI; ++k)
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) v[3 * k + cc] = P::hsum(acc[k][cc]);
                    group_sum12<T>(v, lane, G, s);
                    if (act && (lane & ((G >> 2) - 1)) == 0) {
                        const int j = ((lane & (G >> 1)) ? 2 : 0) + ((lane & (G >> 2)) ? 1 : 0);
                        T *dst = scr + ((size_t)(h * A.slots_max + quad * (n_jg >> lgG) + sub)) * 12 + 3 * j;
                        dst[0] = s[0]; dst[1] = s[1]; dst[2] = s[2];
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(mb_part + h);
            }
        }
    } else {
        // all four warps of the service warpgroup
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_SERVICE_F64));
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_SERVICE));
    }
    if (warp >= CL_CW) {
        // =========================== service warpgroup ===========================
        // All 128 threads share the per-element work of a half's tail (one state element per thread) and its per-dumbbell
        // work (Eq. (4), publish); they meet at named barrier 1.  Thread st_id always takes the same dumbbells of a half.
        const int st_id = tid - 32 * CL_CW;      // 0 .. 127
        const bool lead = st_id == 0;
        if (lead) { mbar_arrive(mb_xi + 0); mbar_arrive(mb_xi + 1); }   // stage 0: XcT written by the prologue
        for (int g = 0; g < n_stage; ++g) {
            const uint32_t par = (uint32_t)g & 1u;
            const bool pred = HEUN && (g & 1) == 0, corr = HEUN && (g & 1) == 1;
            const long long nstep = A.n0 + (HEUN ? (g >> 1) : g);
            if (!HEUN || (g & 1) == 0) {   // stroke length at the end of this step, L(t_{n+1}), once per step
                const double t1 = time_of_step(A.t0, nstep + 1, A.dt);
                for (int h = 0; h < 2; ++h) {
                    const int ndh = (h == 0 ? rowsA : rowsB) >> 1, dbase = h == 0 ? 0 : rowsA >> 1;
                    for (int sl = st_id; sl < ndh; sl += 128) Ls[dbase + sl] = stroke_length(t1, phs[dbase + sl], A.ell, A.lambda, A.omega);
                }
            }
            const bool last = g + 1 == n_stage;
            const double cdt = corr ? 0.5 * A.dt : A.dt;
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int nqh = h == 0 ? nqA : nq - nqA, rows_h = h == 0 ? rowsA : rowsB, rbase = h == 0 ? 0 : rowsA;
                int QW, m;
                cluster_pass_shape(nqh, QW, m);
                // the thread's first element: everything that does not depend on the pass's sums is fetched before the wait
                const bool has0 = st_id < 3 * rows_h;
                const int E0 = 3 * rbase + st_id;
                const double f0 = has0 ? Fs[E0] : 0.0, x0s = has0 ? Xs[E0] : 0.0, v10 = (has0 && corr) ? V1s[E0] : 0.0;
                mbar_wait(mb_part + h, par);
                // Eq. (3a), the 1/(8 pi mu) factor and the integrator in FP64, one state element per thread
#pragma unroll 1
                for (int e = st_id; e < 3 * rows_h; e += 128) {
                    const int rl = e / 3, cc = e - 3 * rl, quad = rl >> 2, k = rl & 3;
                    const T *sp = scr + ((size_t)(h * A.slots_max + quad * m)) * 12 + 3 * k + cc;
                    T sacc = T(0);                                  // the m warps of the quad, in order
#pragma unroll 1
                    for (int j = 0; j < m; ++j) sacc += sp[12 * j];
                    const double sum = (double)sacc;
                    const int E = 3 * rbase + e;
                    const bool first = e == st_id;
                    const double v = A.self_mob * (first ? f0 : Fs[E]) + A.pre * sum;
                    const double w = corr ? (first ? v10 : V1s[E]) + v : v;
                    double xn = (first ? x0s : Xs[E]) + cdt * w;
                    if (A.noise_amp != 0.0) xn += A.noise_amp * noise_normal(A.seed, nstep, b, 3 * r0 + E);
                    if (pred) V1s[E] = v; else Xs[E] = xn;
                    Xc[E] = xn;
                    XcT[E] = (T)xn;
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (lead) {
                    mbar_arrive(mb_xi + h);   // the half's rows of stage g + 1 are in XcT, and its sums have been read
                    // Every compute warp of this CTA has passed stage g's "region landed" waits (it has finished pass h, and
                    // pass A waits for both regions): after tail A, arm the two barriers for stage g + 2.
                    if (h == 0 && g + 2 < n_stage) {
                        mbar_expect_tx(mb_full + 2 * par + 0, (uint32_t)UA * UNIT_BYTES);
                        mbar_expect_tx(mb_full + 2 * par + 1, (uint32_t)UB * UNIT_BYTES);
                    }
                }
                // Eq. (4) at the new positions and time; the half's units of the next stage's stream, into every CTA
                for (int sl = st_id; sl < (rows_h >> 1); sl += 128) {
                    const int row = rbase + 2 * sl;
                    double x0[3], x1[3], F0[3];
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xc[3 * row + cc]; x1[cc] = Xc[3 * row + 3 + cc]; }
                    dumbbell_force(x0, x1, Ls[row >> 1], A.k0, F0);
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) { Fs[3 * row + cc] = F0[cc]; Fs[3 * row + 3 + cc] = -F0[cc]; }
                    if (!last) publish_all((g + 1) & 1, h, sl, x0, x1, F0);
                }
            }
        }
    }
    __syncthreads();
    // the state leaves the launch in FP64 and in user precision
    for (int e = tid; e < 3 * nrows; e += CL_NT) {
        const double x = Xs[e];
        A.X[sys3 + 3 * r0 + e] = x;
        reinterpret_cast<T *>(A.xu)[sys3 + 3 * r0 + e] = (T)x;
    }
    cluster_barrier();   // nobody leaves while a peer could still address its shared memory
}

// ---------------------------------------------------------------------------------------------------------------------
// The latency variant for single small systems and small ensembles (BASELINE.json config 2: N = 128): a stage there is not
// arithmetic but the hand-over (3.1 us per stage on run_kernel's 32 CTAs through L2; 1.7 us of pair arithmetic alone on one
// SM).  One cluster of cs = 8 CTAs per system, 512 threads, no service warps and no halves: every warp computes its place
// of the pair sum over the whole stream (natural sphere order), the block finishes its rows (one thread per state
// element, then one per dumbbell) and stores the dumbbells' units of the next stage into the shared memory of all CTAs
// of the cluster with st.async onto the consumers' mbarriers, as above.  Two block barriers per stage, no cluster barrier.
struct ClusterLatArgs {
    int N, NQ, U, cs;
    int buf_units;                // capacity of one stream buffer in units (U + pad, multiple of 8)
    int rows_max, slots_max;
    double self_mob, pre, c1, c2;
    float c1f, c2f;
    long long n0, n_steps;
    double *X;
    void *xu;
    int from_user;
    const double *phase;
    double t0, dt, ell, lambda, omega, k0, noise_amp;
    unsigned long long seed;
};
constexpr int CLL_NT = 512;

template <typename T, int TENSOR, bool HEUN>
__global__ void __launch_bounds__(CLL_NT, 1) cluster_lat_kernel(const ClusterLatArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = blockIdx.x, b = blockIdx.y, cs = A.cs;
    const size_t buf_bytes = (size_t)A.buf_units * UNIT_BYTES;
    unsigned char *const after = smem_raw + 2 * buf_bytes;
    uint64_t *const mb_full = reinterpret_cast<uint64_t *>(after);   // [parity]: the stage's stream has landed in this CTA
    T *const scr = reinterpret_cast<T *>(after + 64);                // [slots_max][12]
    double *const st = reinterpret_cast<double *>(after + 64 + (size_t)A.slots_max * 12 * 8);

    const int q0 = (int)((long long)r * A.NQ / cs), q1 = (int)((long long)(r + 1) * A.NQ / cs);
    const int nq = q1 - q0;
    const long long r0 = 4LL * q0;
    const int nrows = (int)((A.N - r0) < 4 * nq ? (A.N - r0) : 4 * nq);
    const int nd = nrows >> 1;
    const int rows_st = A.rows_max;
    double *const Xs = st, *const Xc = st + 3 * rows_st, *const V1s = st + 6 * rows_st, *const Fs = st + 9 * rows_st;
    double *const Ls = st + 12 * rows_st, *const phs = Ls + (rows_st >> 1);
    T *const XcT = reinterpret_cast<T *>(st + 13 * rows_st);
    const size_t sys3 = (size_t)b * A.N * 3;
    const int n_stage = (int)(A.n_steps * (HEUN ? 2 : 1));
    const uint32_t stream_bytes = (uint32_t)A.U * UNIT_BYTES;

    // this warp's place (stage-invariant): quads per warp / warps per quad as in cluster_kernel, over nq quads
    int QW, m;
    cluster_pass_shape(nq, QW, m);
    int lgG = 0;
    while ((QW << lgG) < 32) ++lgG;
    const int G = 1 << lgG, n_jg = G * m;
    const int qfirst = (warp / m) * QW, sub = warp - (warp / m) * m;
    const int quad = qfirst + (lane >> lgG), jg = (sub << lgG) + (lane & (G - 1));
    const bool act = quad < nq, wact = qfirst < nq;
    const int its = (A.U + n_jg - 1) / n_jg;
    const int its_w = its - ((its > 0 && (its - 1) * n_jg + sub * G >= A.U) ? 1 : 0);
    int g_lo = its_w, g_hi = its_w;
    {   // iterations that may hold rows of this warp's quads (alpha == beta)
        const int rl1 = 4 * (qfirst + QW) < nrows ? 4 * (qfirst + QW) : nrows;
        const int uo0 = (int)((r0 + 4 * qfirst) / W), uo1 = (int)((r0 + rl1 + W - 1) / W);
        if (wact && uo1 > uo0) {
            g_lo = uo0 / n_jg; g_hi = (uo1 - 1) / n_jg + 1;
            g_lo = g_lo < its_w ? g_lo : its_w; g_hi = g_hi < its_w ? g_hi : its_w;
        }
    }
    const int slot = quad * m + sub, stride = 3 * n_jg;

    auto publish_all = [&](int par, int sl, const double (&x0)[3], const double (&x1)[3], const double (&F0)[3]) {
        const uint32_t dst = smem_u32(smem_raw + (size_t)par * buf_bytes) + (uint32_t)((r0 + 2 * sl) / W) * UNIT_BYTES;
        const uint32_t bar = smem_u32(mb_full + par);
        for (int p = 0; p < cs; ++p) publish_async(T(), mapa_u32(dst, (uint32_t)p), mapa_u32(bar, (uint32_t)p), x0, x1, F0);
    };

    // ---- prologue ----
    for (int e = tid; e < 3 * nrows; e += CLL_NT) {
        const double x = A.from_user ? (double)reinterpret_cast<const T *>(A.xu)[sys3 + 3 * r0 + e] : A.X[sys3 + 3 * r0 + e];
        Xs[e] = x; Xc[e] = x; XcT[e] = (T)x;
    }
    for (int e = 3 * nrows + tid; e < 3 * rows_st; e += CLL_NT) XcT[e] = P::dummy();
    for (int sl = tid; sl < nd; sl += CLL_NT) phs[sl] = A.phase[(size_t)b * (A.N / 2) + (r0 >> 1) + sl];
    if (tid == 0) {
        mbar_init(mb_full + 0, 1); mbar_init(mb_full + 1, 1);
        mbar_fence_init();
        mbar_expect_tx(mb_full + 0, stream_bytes); mbar_expect_tx(mb_full + 1, stream_bytes);
    }
    for (int k = 0; k < 2; ++k) {   // far-away zero-force pad units behind the stream (never overwritten)
        uint4 *bp = reinterpret_cast<uint4 *>(smem_raw + (size_t)k * buf_bytes);
        for (int j = 3 * A.U + tid; j < 3 * A.buf_units; j += CLL_NT) bp[j] = pad_piece<T>(j % 3);
    }
    cluster_barrier();
    {
        const double tn = time_of_step(A.t0, A.n0, A.dt);
        for (int sl = tid; sl < nd; sl += CLL_NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xs[6 * sl + cc]; x1[cc] = Xs[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, stroke_length(tn, phs[sl], A.ell, A.lambda, A.omega), A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            if (n_stage > 0) publish_all(0, sl, x0, x1, F0);
        }
    }
    __syncthreads();

    const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
    for (int g = 0; g < n_stage; ++g) {
        const int par = g & 1;
        const bool pred = HEUN && (g & 1) == 0, corr = HEUN && (g & 1) == 1;
        const long long nstep = A.n0 + (HEUN ? (g >> 1) : g);
        // ---- pair sums ----
        V xi[QI][3], acc[QI][3];
#pragma unroll
        for (int k = 0; k < QI; ++k) acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
        if (wact) {
            T xq[12];
            const typename P::T4 *xp = reinterpret_cast<const typename P::T4 *>(XcT + 12 * (act ? quad : qfirst));
#pragma unroll
            for (int k = 0; k < 3; ++k) { const typename P::T4 q = xp[k]; xq[4 * k] = q.x; xq[4 * k + 1] = q.y; xq[4 * k + 2] = q.z; xq[4 * k + 3] = q.w; }
#pragma unroll
            for (int k = 0; k < QI; ++k) { xi[k][0] = P::bc(xq[3 * k]); xi[k][1] = P::bc(xq[3 * k + 1]); xi[k][2] = P::bc(xq[3 * k + 2]); }
        }
        mbar_wait_cluster(mb_full + par, (uint32_t)(g >> 1) & 1u);
        if (act) {
            const V2<T> *p = reinterpret_cast<const V2<T> *>(smem_raw + (size_t)par * buf_bytes) + 3 * jg;
            int it = 0;
#pragma unroll 1
            for (; it < g_lo; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
#pragma unroll 1
            for (; it < g_hi; ++it, p += stride) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
#pragma unroll 1
            for (; it < its_w; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
        }
        if (wact) {
            T v[12], s3[3];
#pragma unroll
            for (int k = 0; k < QI; ++k)
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) v[3 * k + cc] = P::hsum(acc[k][cc]);
            group_sum12<T>(v, lane, G, s3);
            if (act && (lane & ((G >> 2) - 1)) == 0) {
                const int j = ((lane & (G >> 1)) ? 2 : 0) + ((lane & (G >> 2)) ? 1 : 0);
                T *dst = scr + (size_t)slot * 12 + 3 * j;
                dst[0] = s3[0]; dst[1] = s3[1]; dst[2] = s3[2];
            }
        }
        __syncthreads();
        // ---- tail, part 1: one thread per own state element; spare threads take the stroke lengths of the next step ----
        const bool last = g + 1 == n_stage;
        const double cdt = corr ? 0.5 * A.dt : A.dt;
        const int n_item = 3 * nrows + ((!HEUN || (g & 1) == 0) ? nd : 0);
        for (int i = tid; i < n_item; i += CLL_NT) {
            if (i >= 3 * nrows) {   // L(t_{n+1}), once per step
                const int sl = i - 3 * nrows;
                Ls[sl] = stroke_length(time_of_step(A.t0, nstep + 1, A.dt), phs[sl], A.ell, A.lambda, A.omega);
                continue;
            }
            const int E = i, rl = E / 3, cc = E - 3 * rl, qd = rl >> 2, k = rl & 3;
            const T *sp = scr + (size_t)(qd * m) * 12 + 3 * k + cc;
            T sacc = T(0);                                  // the m warps of the quad, in order
#pragma unroll 1
            for (int j = 0; j < m; ++j) sacc += sp[12 * j];
            // Eq. (3a), the 1/(8 pi mu) factor and the integrator in FP64
            const double v = A.self_mob * Fs[E] + A.pre * (double)sacc;
            const double w = corr ? V1s[E] + v : v;
            double xn = Xs[E] + cdt * w;
            if (A.noise_amp != 0.0) xn += A.noise_amp * noise_normal(A.seed, nstep, b, 3 * r0 + E);
            if (pred) V1s[E] = v; else Xs[E] = xn;
            Xc[E] = xn;
            XcT[E] = (T)xn;
        }
        // every warp of this CTA has passed stage g's wait: arm the barrier for stage g + 2 (no peer can send that stream
        // before it has received this CTA's rows of stage g + 1, which leave after the next block barrier)
        if (tid == 0 && g + 2 < n_stage) mbar_expect_tx(mb_full + par, stream_bytes);
        __syncthreads();
        // ---- tail, part 2: Eq. (4) at the new positions and time; the dumbbell's unit of the next stage, into every CTA ----
        for (int sl = tid; sl < nd; sl += CLL_NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xc[6 * sl + cc]; x1[cc] = Xc[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, Ls[sl], A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            if (!last) publish_all((g + 1) & 1, sl, x0, x1, F0);
        }
        // Fs of this stage is read by part 1 of the next stage, behind that stage's first block barrier
    }
    __syncthreads();
    for (int e = tid; e < 3 * nrows; e += CLL_NT) {
        const double x = Xs[e];
        A.X[sys3 + 3 * r0 + e] = x;
        reinterpret_cast<T *>(A.xu)[sys3 + 3 * r0 + e] = (T)x;
    }
    cluster_barrier();   // nobody leaves while a peer could still address its shared memory
}

}  // namespace ds
