// pipeline.cuh -- the step kernel for systems whose pair loop dominates a stage (N of a few thousand spheres on
// all SMs): the same time step as mobility.cuh's run_kernel (Eq. (1a) deterministic part with Eq. (3a,3b), Eq. (4),
// Heun / Euler of PAPER.md:236), reorganised as a software pipeline so that nothing but pair
// arithmetic is left on the critical path.
//
// Why.  In run_kernel a stage ends with: split-beta reduction -> self term -> integrator -> Eq. (4) -> publish rows ->
// inter-CTA hand-over; every CTA does this at the same moment, and all 148 SMs' FMA pipes idle for about 5.5 k of a
// stage's 30 k cycles (N = 4096).  The next stage cannot start earlier, because it needs every row's new position.
//
// How.  The rows of a CTA are cut into two halves A and B (whole quads), and a stage into two passes:
//     pass A: alpha in half A  x  all beta        pass B: alpha in half B  x  all beta
// The beta-stream of a stage is laid out as two regions, region h = the half-h rows of every CTA (a fixed order, so
// sums stay deterministic).  When pass A ends, the sums of the half-A rows are complete: a "service" warpgroup (warps
// 16-19) finishes them (self term, integrator, Eq. (4), publish into region A of the NEXT stage's stream) while the 16
// compute warps are already in pass B.  Likewise the half-B rows are finished during pass A of the next stage, which starts on region A
// of the new stream (published by every CTA half a stage ago) and reaches region B long after it has landed.  The
// lead service warp also prefetches each region into shared memory with one TMA bulk copy as soon as (a) every CTA has
// published it (one arrival counter per region and system, release/acquire at gpu scope) and (b) every compute warp of
// this CTA has finished with the region's previous content (mbarrier).  No block-wide barrier inside the step loop.
//
// Thread shape of a pass over nq quads: m = 16 / nq warps per quad, lanes = 32 m beta-groups; all lanes of a warp hold
// the same 4 alpha-spheres (loads of the alpha rows are broadcasts) and read 32 consecutive units of the stream
// (48-byte stride: conflict-free LDS.128).  At the end of a pass a warp adds its 32 lanes' partial sums with a fixed
// shuffle tree (12 values: 18 SHFL) and leaves 12 numbers in shared memory; the service warpgroup adds the m warps of a
// quad in a fixed order.  No atomics anywhere: results are bitwise reproducible and independent of how the steps are
// split over launches.
#pragma once
#include "mobility.cuh"

namespace ds {

constexpr int PIPE_CW = 16;                      // compute warps
constexpr int PIPE_NT = 32 * (PIPE_CW + 4);      // + the service warp's warpgroup (one warp works; register re-allocation
                                                 // between roles, setmaxnreg, is per warpgroup of 4 warps)
// registers per thread after the role split: 640 x 96 at launch; the service warpgroup gives back 128 x (96 - 64) = 4096,
// the four compute warpgroups take 512 x (104 - 96) = 4096
constexpr int PIPE_REGS_COMPUTE = 104, PIPE_REGS_SERVICE = 64;
// FP64: 128 x (96 - 32) given back, 512 x (112 - 96) taken: the FP64 pair loop is 1.2 % faster with 112 registers (30.3 against 30.7 us
// per stage at N = 4096) although the service warpgroup then spills; the FP32 stage is slower that way (13.62 against 13.55)
constexpr int PIPE_REGS_COMPUTE_F64 = 112, PIPE_REGS_SERVICE_F64 = 32;
constexpr int PIPE_BAR_BYTES = 128;              // 8 mbarriers
constexpr int PIPE_SCR_BYTES = 2 * PIPE_CW * 12 * 8;   // warp sums of the two passes, [2][16][12] T
constexpr int PIPE_TAB_BYTES = 2 * PIPE_CW * 3 * 16;   // per pass and warp: its place in the pass and its loop bounds (stage-invariant)

// quads of a CTA that form half A (the rest is half B)
#ifndef PIPE_SPLIT_EXPR
#define PIPE_SPLIT_EXPR ((nq + 1) >> 1)
#endif
__host__ __device__ inline int pipe_split(int nq) { return PIPE_SPLIT_EXPR; }

struct PipeArgs {
    int N, NQ, n_cta, b0;
    long long unit_stride;        // units per system in the streams
    void *units[2];               // ping-pong streams; stage g reads units[g & 1]: region 0 at unit 0, region 1 at unit reg_units[0]
    const int *half_off;          // device table [2][n_cta + 1]: first unit of CTA c's half inside region 0 / region 1
    int reg_units[2];             // units of region 0 / 1
    int buf_units[2];             // capacity of the two shared-memory region buffers in units (pads included, multiples of 8)
    int rows_max;                 // most rows any CTA owns (state sizing)
    double self_mob, pre, c1, c2; // Eq. (3a), (3b) constants as in RunArgs
    float c1f, c2f;
    long long n0, n_steps;
    double *X;                    // state [B][N][3] FP64
    void *xu;                     // the same in user precision
    int from_user;
    const double *phase;
    double t0, dt, ell, lambda, omega, k0, noise_amp;
    unsigned long long seed;
    unsigned long long *cnt;      // [B][2] arrival counters (one per region), monotonic over launches
    unsigned long long cnt_base;
    const int4 *ptab_g;           // device table [n_cta][2][16][3]: which warp does what in the two passes (pipe_build_table)
    long long *probe;             // dev instrumentation (DS_ENABLE_PROBE builds): PROBE_SLOTS clock samples per CTA, or NULL
};

// 12 values per lane -> their sums over the 32 lanes of the warp, in a fixed order.  After the call lanes 8 j .. 8 j + 7
// all hold the three sums {3 j', ...}: s[0..2] of lane 8 j are the totals of the values v[6 (j >> 1) + 3 (j & 1) + 0..2].
template <typename T> __device__ __forceinline__ void warp_sum12(const T (&v)[12], int lane, T (&s)[3]) {
    const bool up16 = lane & 16, up8 = lane & 8;
    T a[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {   // lanes 0-15 keep values 0-5, lanes 16-31 keep values 6-11
        const T keep = up16 ? v[6 + i] : v[i], send = up16 ? v[i] : v[6 + i];
        a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {   // within a half: lanes with bit 3 clear keep 0-2, set keep 3-5
        const T keep = up8 ? a[3 + i] : a[i], send = up8 ? a[i] : a[3 + i];
        s[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
#pragma unroll
    for (int d = 4; d >= 1; d >>= 1) {
#pragma unroll
        for (int i = 0; i < 3; ++i) s[i] += __shfl_xor_sync(0xffffffffu, s[i], d);
    }
}

// Which warp does what in the two passes of CTA c (stage-invariant; built on the host once per launch shape, 9 k cycles per
// launch when thread 0 of every CTA did it).  The 16 warps of a pass are dealt to its nqp quads, m = 16 / nqp or one more each;
// place (quad, sub), sub < m, walks the units 32 sub + lane + k * 32 m of a region.  Entry [pass][warp] = three int4:
// {active, quad, sub, m}, then per region {iterations of this warp, first / end of the guarded ones, slot of its sums}.
// Places go to the four SM sub-partitions (warp % 4) so that their iteration counts balance over the whole stage;
// sub-partition 0, which also hosts the lead service warp, gets a little less.
inline void pipe_build_table(int N, int NQ, int n_cta, int c, int W, const int *half_off /* [2][n_cta + 1] */, const int reg_units[2],
                             int4 *ptab /* [2][16][3] */) {
    const int q0 = (int)((long long)c * NQ / n_cta), q1 = (int)((long long)(c + 1) * NQ / n_cta);
    const int nq = q1 - q0;
    const long long r0 = 4LL * q0;
    const int nrows = (int)((N - r0) < 4 * nq ? (N - r0) : 4 * nq);
    const int nqA = pipe_split(nq);
    const int rowsA = 4 * nqA < nrows ? 4 * nqA : nrows, rowsB = nrows - rowsA;
    const int ownA = half_off[c], ownB = half_off[(n_cta + 1) + c];
    auto bounds = [&](int h, int cls, int sub, int reg) {   // the place's loop bounds
        const int nqp = h == 0 ? nqA : nq - nqA, rows_h = h == 0 ? rowsA : rowsB;
        const int own0 = h == 0 ? ownA : ownB, own1 = own0 + rows_h / W;
        int4 q = make_int4(0, 0, 0, 0);
        if (nqp > 0) {
            const int m = PIPE_CW / nqp + cls, n_jg = 32 * m;
            const int Ur = reg_units[reg];
            const int its = (Ur + n_jg - 1) / n_jg;
            // the last iteration is skipped by warps whose 32 units all lie behind the region
            const int its_w = its - ((its > 0 && (its - 1) * n_jg + 32 * sub >= Ur) ? 1 : 0);
            int g_lo = its_w, g_hi = its_w;     // iterations that may hold own units (alpha == beta): region h only
            if (reg == h && rows_h > 0) {
                g_lo = own0 / n_jg; g_hi = (own1 - 1) / n_jg + 1;
                g_lo = g_lo < its_w ? g_lo : its_w; g_hi = g_hi < its_w ? g_hi : its_w;
            }
            q = make_int4(its_w, g_lo, g_hi, 0);
        }
        return q;
    };
    int load[4] = {2, 0, 0, 0};
    for (int h = 0; h < 2; ++h) {
        const int nqp = h == 0 ? nqA : nq - nqA;
        int used[4] = {0, 0, 0, 0};
        for (int w = 0; w < PIPE_CW; ++w)
            for (int k = 0; k < 3; ++k) ptab[(h * PIPE_CW + w) * 3 + k] = make_int4(0, 0, 0, 0);
        if (nqp == 0) continue;
        const int mb = PIPE_CW / nqp, mr = PIPE_CW % nqp;          // quad q gets mb + (q < mr) warps
        for (int sub = 0; sub <= mb; ++sub) {                      // heavier places (small sub) first
            for (int quad = 0; quad < nqp; ++quad) {
                const int cls = quad < mr ? 1 : 0, m = mb + cls;
                if (sub >= m) continue;
                int4 qa = bounds(h, cls, sub, 0), qb = bounds(h, cls, sub, 1);
                const int tot = qa.x + qb.x;
                int best = -1;
                for (int k = 3; k >= 0; --k)   // the least loaded sub-partition with a free warp (ties: the higher one)
                    if (used[k] < 4 && (best < 0 || load[k] < load[best])) best = k;
                const int u = used[best]++;
                load[best] += tot;
                int4 *e = ptab + (h * PIPE_CW + best + 4 * u) * 3;
                qa.w = quad * mb + (quad < mr ? quad : mr) + sub;   // slot of this place's sums in scr
                e[0] = make_int4(1, quad, sub, m); e[1] = qa; e[2] = qb;
            }
        }
    }
}

#ifdef DS_ENABLE_PROBE
#define PIPE_PROBE(slot)                                                                                         \
    do {                                                                                                         \
        if (A.probe != nullptr && lane == 0 && (warp == 0 || warp == PIPE_CW) && g == n_stage - 2)               \
            A.probe[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * PROBE_SLOTS + (slot)] = clock64();            \
    } while (0)
#else
#define PIPE_PROBE(slot) do { } while (0)
#endif

template <typename T, int TENSOR, bool HEUN>
__global__ void __launch_bounds__(PIPE_NT, 1) pipe_kernel(const PipeArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x, b = A.b0 + blockIdx.y;

    unsigned char *const buf0 = smem_raw, *const buf1 = smem_raw + (size_t)A.buf_units[0] * UNIT_BYTES;
    unsigned char *const after = buf1 + (size_t)A.buf_units[1] * UNIT_BYTES;
    uint64_t *const mb_full = reinterpret_cast<uint64_t *>(after);   // [2] region landed in shared memory (TMA)
    uint64_t *const mb_empty = mb_full + 2;                          // [2] every compute warp is done with the region (this stage)
    uint64_t *const mb_part = mb_full + 4;                           // [2] every compute warp has left its sums of pass h
    uint64_t *const mb_xi = mb_full + 6;                             // [2] the half's rows of the next stage are in the state arrays
    T *const scr = reinterpret_cast<T *>(after + PIPE_BAR_BYTES);    // [2][16][12], indexed by (pass, quad * m + sub)
    int4 *const ptab = reinterpret_cast<int4 *>(after + PIPE_BAR_BYTES + PIPE_SCR_BYTES);   // [2][16][3]
    double *const st = reinterpret_cast<double *>(after + PIPE_BAR_BYTES + PIPE_SCR_BYTES + PIPE_TAB_BYTES);

    // rows of this CTA and its two halves (whole quads; a dumbbell never straddles them)
    const int q0 = (int)((long long)c * A.NQ / A.n_cta), q1 = (int)((long long)(c + 1) * A.NQ / A.n_cta);
    const int nq = q1 - q0;
    const long long r0 = 4LL * q0;
    const int nrows = (int)((A.N - r0) < 4 * nq ? (A.N - r0) : 4 * nq);
    const int nd = nrows >> 1;
    const int nqA = pipe_split(nq);
    const int rowsA = 4 * nqA < nrows ? 4 * nqA : nrows, rowsB = nrows - rowsA;
    const int *const ho0 = A.half_off, *const ho1 = A.half_off + (A.n_cta + 1);
    const int ownA = ho0[c], ownB = ho1[c];                           // first own unit inside region 0 / 1
    const int rows_st = A.rows_max;
    double *const Xs = st, *const Xc = st + 3 * rows_st, *const V1s = st + 6 * rows_st, *const Fs = st + 9 * rows_st;
    double *const Ls = st + 12 * rows_st, *const phs = Ls + (rows_st >> 1);
    T *const XcT = reinterpret_cast<T *>(st + 13 * rows_st);
    const size_t sys3 = (size_t)b * A.N * 3;
    const int n_stage = (int)(A.n_steps * (HEUN ? 2 : 1));
    unsigned long long *const cnt = A.cnt + 2 * (size_t)b;

    auto stream_of = [&](int g) { return reinterpret_cast<T *>(A.units[g & 1]) + (size_t)b * A.unit_stride * (6 * W); };
    // the CTA's own units of half h inside a stream
    auto own_units = [&](T *stream, int h) { return stream + (size_t)(h == 0 ? ownA : A.reg_units[0] + ownB) * (6 * W); };

    // ---- prologue (all warps): state, F(X_n, t_n), stream 0, pads, barriers ----
    for (int e = tid; e < 3 * nrows; e += PIPE_NT)
        Xs[e] = A.from_user ? (double)reinterpret_cast<const T *>(A.xu)[sys3 + 3 * r0 + e] : A.X[sys3 + 3 * r0 + e];
    for (int sl = tid; sl < nd; sl += PIPE_NT) phs[sl] = A.phase[(size_t)b * (A.N / 2) + (r0 >> 1) + sl];
    if (tid == 0) {
        for (int h = 0; h < 2; ++h) {
            mbar_init(mb_full + h, 1);
            mbar_init(mb_empty + h, PIPE_CW);
            mbar_init(mb_part + h, PIPE_CW);
            mbar_init(mb_xi + h, 1);
        }
        mbar_fence_init();
    }
    // which warp does what in the two passes: the host's table (pipe_build_table)
    for (int i = tid; i < 2 * PIPE_CW * 3; i += PIPE_NT) ptab[i] = A.ptab_g[(size_t)c * (2 * PIPE_CW * 3) + i];
    // far-away zero-force pad units behind each region (never overwritten: the bulk copies bring the real units only)
    for (int h = 0; h < 2; ++h) {
        uint4 *bp = reinterpret_cast<uint4 *>(h == 0 ? buf0 : buf1);
        for (int j = 3 * A.reg_units[h] + tid; j < 3 * A.buf_units[h]; j += PIPE_NT) bp[j] = pad_piece<T>(j % 3);
    }
    __syncthreads();
    {
        const double tn = time_of_step(A.t0, A.n0, A.dt);
        T *s0 = stream_of(0);
        for (int e = tid; e < 3 * nrows; e += PIPE_NT) { Xc[e] = Xs[e]; XcT[e] = (T)Xs[e]; }
        for (int e = 3 * nrows + tid; e < 3 * rows_st; e += PIPE_NT) XcT[e] = P::dummy();   // rows of a last, partial quad
        for (int sl = tid; sl < nd; sl += PIPE_NT) {
            double x0[3], x1[3], F0[3];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xs[6 * sl + cc]; x1[cc] = Xs[6 * sl + 3 + cc]; }
            dumbbell_force(x0, x1, stroke_length(tn, phs[sl], A.ell, A.lambda, A.omega), A.k0, F0);
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) { Fs[6 * sl + cc] = F0[cc]; Fs[6 * sl + 3 + cc] = -F0[cc]; }
            const int row = 2 * sl, h = row < rowsA ? 0 : 1;
            publish_dumbbell(own_units(s0, h), nullptr, 0u, row - (h ? rowsA : 0), x0, x1, F0);
        }
        fence_proxy_async_global();   // the stream is read through the async proxy (TMA)
    }
    __syncthreads();

    if (warp < PIPE_CW) {
        // =========================== compute warps ===========================
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_COMPUTE_F64));
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_COMPUTE));
        const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
        for (int g = 0; g < n_stage; ++g) {
            const uint32_t par = (uint32_t)g & 1u;
            PIPE_PROBE(0);
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int rows_h = h == 0 ? rowsA : rowsB, rbase = h == 0 ? 0 : rowsA;
                const int4 *const tab = ptab + (h * PIPE_CW + warp) * 3;
                const int4 place = tab[0];
                const bool act = place.x != 0;
                const int quad = place.y, sub = place.z, n_jg = 32 * place.w;
                V xi[QI][3], acc[QI][3];
                int slot = 0;
                if (act) {
                    mbar_wait(mb_xi + h, par);
                    // the quad's 12 coordinates are contiguous and 16-byte aligned (rows beyond the system hold a far-away dummy)
                    T xq[12];
                    const typename P::T4 *xp = reinterpret_cast<const typename P::T4 *>(XcT + 3 * (rbase + 4 * quad));
#pragma unroll
                    for (int k = 0; k < 3; ++k) { const typename P::T4 q = xp[k]; xq[4 * k] = q.x; xq[4 * k + 1] = q.y; xq[4 * k + 2] = q.z; xq[4 * k + 3] = q.w; }
#pragma unroll
                    for (int k = 0; k < QI; ++k) {
                        xi[k][0] = P::bc(xq[3 * k]); xi[k][1] = P::bc(xq[3 * k + 1]); xi[k][2] = P::bc(xq[3 * k + 2]);
                        acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
                    }
                }
                PIPE_PROBE(1 + 6 * h);
                const int own0 = h == 0 ? ownA : ownB, own1 = own0 + rows_h / W;
#pragma unroll 1
                for (int reg = 0; reg < 2; ++reg) {
                    if (h == 0) mbar_wait(mb_full + reg, par);   // every warp passes here in pass A: pass B need not look again
                    PIPE_PROBE(2 + 6 * h + 2 * reg);
                    if (act) {
                        const int4 lim = tab[1 + reg];                  // {iterations of this warp, first / end of the guarded ones}
                        if (reg == 0) slot = lim.w;
                        const V2<T> *p = reinterpret_cast<const V2<T> *>(reg == 0 ? buf0 : buf1) + 3 * (32 * sub + lane);
                        const int stride = 3 * n_jg;
                        int it = 0;
#pragma unroll 1
                        for (; it < lim.y; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
#pragma unroll 1
                        for (; it < lim.z; ++it, p += stride) {
                            const int u0 = it * n_jg + 32 * sub;           // this warp's 32 units: [u0, u0 + 32)
                            if (u0 < own1 && u0 + 32 > own0) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
                            else pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                        }
#pragma unroll 1
                        for (; it < lim.x; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
                    }
                    PIPE_PROBE(3 + 6 * h + 2 * reg);
                    if (h == 1) {   // pass B is the last reader of the stage's regions
                        __syncwarp();
                        if (lane == 0) mbar_arrive(mb_empty + reg);
                    }
                }
                if (act) {
                    T v[12], s[3];
#pragma unroll
                    for (int k = 0; k < QI; ++k)
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) v[3 * k + cc] = P::hsum(acc[k][cc]);
                    warp_sum12<T>(v, lane, s);
                    if ((lane & 7) == 0) {
                        const int j = lane >> 3;                       // lanes 0, 8, 16, 24
                        T *dst = scr + (h * PIPE_CW + slot) * 12 + 3 * j;
                        dst[0] = s[0]; dst[1] = s[1]; dst[2] = s[2];
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(mb_part + h);
                PIPE_PROBE(6 + 6 * h);
            }
        }
    } else {
        // all four warps of the service warpgroup
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_SERVICE_F64));
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PIPE_REGS_SERVICE));
    }
    if (warp >= PIPE_CW) {
        // =========================== service warpgroup ===========================
        // All four warps share the per-element work of a half's tail (one state element per thread); warp 16, the lead,
        // also evaluates Eq. (4), publishes, signals and prefetches.  They meet at named barrier 1.
        const int st_id = tid - 32 * PIPE_CW;      // 0 .. 127
        const bool lead = warp == PIPE_CW;
        auto fetch_region = [&](int h, int g) {   // one thread: region h of stream g -> shared memory, once every CTA has published it
            const unsigned long long target = A.cnt_base + (unsigned long long)(g + 1) * (unsigned long long)A.n_cta;
            while (ld_acquire_gpu(cnt + h) < target) {}
            fence_proxy_async();
            const uint32_t bytes = (uint32_t)A.reg_units[h] * UNIT_BYTES;
            if (bytes > 0) {
                mbar_expect_tx(mb_full + h, bytes);
                const T *src = stream_of(g) + (size_t)(h == 0 ? 0 : A.reg_units[0]) * (6 * W);
                bulk_g2s(h == 0 ? buf0 : buf1, src, bytes, mb_full + h);
            } else {
                mbar_arrive(mb_full + h);
            }
        };
        if (lead && lane == 0) {
            // stream 0 is complete once every CTA has arrived once per region
            red_release_gpu(cnt + 0, 1ULL);
            red_release_gpu(cnt + 1, 1ULL);
            mbar_arrive(mb_xi + 0);
            mbar_arrive(mb_xi + 1);
            if (n_stage > 0) { fetch_region(0, 0); fetch_region(1, 0); }
        }
        __syncwarp();
        for (int g = 0; g < n_stage; ++g) {
            const uint32_t par = (uint32_t)g & 1u;
            const bool pred = HEUN && (g & 1) == 0, corr = HEUN && (g & 1) == 1;
            const long long nstep = A.n0 + (HEUN ? (g >> 1) : g);
            if (lead && (!HEUN || (g & 1) == 0)) {   // stroke length at the end of this step, L(t_{n+1}), once per step
                const double t1 = time_of_step(A.t0, nstep + 1, A.dt);
                for (int sl = lane; sl < nd; sl += 32) Ls[sl] = stroke_length(t1, phs[sl], A.ell, A.lambda, A.omega);
            }
            const bool last = g + 1 == n_stage;
            T *const snext = stream_of(g + 1);
            const double cdt = corr ? 0.5 * A.dt : A.dt;
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int nqp = h == 0 ? nqA : nq - nqA, rows_h = h == 0 ? rowsA : rowsB, rbase = h == 0 ? 0 : rowsA;
                const int mb = nqp > 0 ? PIPE_CW / nqp : 0, mr = nqp > 0 ? PIPE_CW % nqp : 0;
                // the thread's first element: everything that does not depend on the pass's sums is fetched before the wait
                const bool has0 = st_id < 3 * rows_h;
                const int E0 = 3 * rbase + st_id;
                const double f0 = has0 ? Fs[E0] : 0.0, x0s = has0 ? Xs[E0] : 0.0, v10 = (has0 && corr) ? V1s[E0] : 0.0;
                mbar_wait(mb_part + h, par);
                PIPE_PROBE(16 + 6 * h);
                // Eq. (3a), the 1/(8 pi mu) factor and the integrator in FP64, one state element per thread
#pragma unroll 1
                for (int e = st_id; e < 3 * rows_h; e += 128) {
                    const int rl = e / 3, cc = e - 3 * rl, quad = rl >> 2, k = rl & 3;
                    const int m = mb + (quad < mr ? 1 : 0);
                    const T *sp = scr + (h * PIPE_CW + quad * mb + (quad < mr ? quad : mr)) * 12 + 3 * k + cc;
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
                PIPE_PROBE(28 + h);
                if (lead) {
                    // Eq. (4) at the new positions and time; publish the half's rows of the next stage's stream
                    for (int sl = lane; sl < (rows_h >> 1); sl += 32) {
                        const int row = rbase + 2 * sl;
                        double x0[3], x1[3], F0[3];
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) { x0[cc] = Xc[3 * row + cc]; x1[cc] = Xc[3 * row + 3 + cc]; }
                        dumbbell_force(x0, x1, Ls[row >> 1], A.k0, F0);
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) { Fs[3 * row + cc] = F0[cc]; Fs[3 * row + 3 + cc] = -F0[cc]; }
                        if (!last) publish_dumbbell(own_units(snext, h), nullptr, 0u, 2 * sl, x0, x1, F0);
                    }
                    PIPE_PROBE(30 + h);
                    if (!last) fence_proxy_async_global();
                    __syncwarp();
                    PIPE_PROBE(17 + 6 * h);
                    if (lane == 0) {
                        if (!last) red_release_gpu(cnt + h, 1ULL);   // this CTA's half of stream g + 1 is out
                        PIPE_PROBE(20 + 6 * h);
                        mbar_arrive(mb_xi + h);                      // ... and its rows of stage g + 1 are in XcT
                        if (!last) {
                            mbar_wait(mb_empty + h, par);            // every compute warp is past the region's old content
                            PIPE_PROBE(18 + 6 * h);
                            fetch_region(h, g + 1);
                            PIPE_PROBE(19 + 6 * h);
                        }
                    }
                    __syncwarp();
                }
            }
        }
    }
    __syncthreads();
    // the state leaves the launch in FP64 and in user precision
    for (int e = tid; e < 3 * nrows; e += PIPE_NT) {
        const double x = Xs[e];
        A.X[sys3 + 3 * r0 + e] = x;
        reinterpret_cast<T *>(A.xu)[sys3 + 3 * r0 + e] = (T)x;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The stateless mobility apply (ds_mobility_apply: Eq. (1a) deterministic part with Eq. (3a,3b)) in the
// thread shape of the pipelined kernel, one pass: the 16 warps of a CTA are dealt to its nq <= 16 quads (16 / nq or one more
// each), all lanes of a warp hold the same 4 alpha-spheres and walk 32 consecutive units of the stream per iteration; the
// split-beta sums meet in the fixed shuffle tree of warp_sum12 and in 12 numbers per warp of shared memory (run_kernel's
// apply mode needs a 24 KB block-wide reduction instead).  Every CTA packs the user's [n][3] arrays into its own stream;
// no inter-CTA dependency: a plain launch with programmatic dependent launch, any number of waves.
struct ApplyArgs {
    int N, NQ, U, n_cta;
    int buf_units;                 // capacity of the stream buffer in units (pads included, multiple of 8)
    double self_mob, pre, c1, c2;
    float c1f, c2f;
    const void *raw_pos, *raw_F;   // user arrays [N][3]
    void *out_u;                   // [N][3]
};

template <typename T, int TENSOR>
__global__ void __launch_bounds__(32 * PIPE_CW, 1) apply_kernel(const ApplyArgs A) {
    typedef Pack<T> P;
    typedef typename P::V V;
    constexpr int W = P::W, NTH = 32 * PIPE_CW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x;
    T *const scr = reinterpret_cast<T *>(smem_raw + (size_t)A.buf_units * UNIT_BYTES);   // [16][12]

    const int q0 = (int)((long long)c * A.NQ / A.n_cta), q1 = (int)((long long)(c + 1) * A.NQ / A.n_cta);
    const int nq = q1 - q0;                                            // 1 .. 16 (host)
    const long long r0 = 4LL * q0;
    const int nrows = (int)((A.N - r0) < 4 * nq ? (A.N - r0) : 4 * nq);
    // this warp's place: quad q gets mb + (q < mr) warps
    const int mb = PIPE_CW / nq, mr = PIPE_CW % nq;
    const int wq = warp < mr * (mb + 1) ? warp / (mb + 1) : mr + (warp - mr * (mb + 1)) / mb;
    const int quad = wq, m = mb + (quad < mr ? 1 : 0);
    const int sub = warp - (quad * mb + (quad < mr ? quad : mr));
    const int n_jg = 32 * m;

    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // the warp's alpha rows, straight from the user's array (in flight while the stream is packed)
    T xq[12];
#pragma unroll
    for (int k = 0; k < QI; ++k) {
        const long long i = r0 + 4 * quad + k;
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) xq[3 * k + cc] = i < A.N ? __ldg(reinterpret_cast<const T *>(A.raw_pos) + 3 * i + cc) : P::dummy();
    }
    {   // every CTA packs the whole stream for itself (units behind the last sphere are far-away zero-force dummies);
        // CTAs start at different units so that they do not read L2 in a convoy
        typedef typename std::conditional<sizeof(T) == 4, float4, double2>::type Q;
        const int up = A.buf_units;
        int u = tid + (int)(((long long)c * up) / A.n_cta);
        for (int k = tid; k < up; k += NTH, u += NTH) {
            u = u >= up ? u - up : u;
            pack_unit(reinterpret_cast<Q *>(smem_raw) + 3 * u, reinterpret_cast<const T *>(A.raw_pos), reinterpret_cast<const T *>(A.raw_F), u, A.N);
        }
    }
    __syncthreads();
    const V c1 = P::bc(sizeof(T) == 4 ? (T)A.c1f : (T)A.c1), negc2 = P::bc(sizeof(T) == 4 ? (T)(-A.c2f) : (T)(-A.c2));
    V xi[QI][3], acc[QI][3];
#pragma unroll
    for (int k = 0; k < QI; ++k) {
        xi[k][0] = P::bc(xq[3 * k]); xi[k][1] = P::bc(xq[3 * k + 1]); xi[k][2] = P::bc(xq[3 * k + 2]);
        acc[k][0] = acc[k][1] = acc[k][2] = P::bc(T(0));
    }
    {
        const int its = (A.U + n_jg - 1) / n_jg;
        const int its_w = its - ((its > 0 && (its - 1) * n_jg + 32 * sub >= A.U) ? 1 : 0);   // all 32 units behind the stream
        const int own0 = (int)(r0 / W), own1 = own0 + (nrows + W - 1) / W;                   // units that hold own rows
        int g_lo = own0 / n_jg, g_hi = (own1 - 1) / n_jg + 1;
        g_lo = g_lo < its_w ? g_lo : its_w; g_hi = g_hi < its_w ? g_hi : its_w;
        const V2<T> *p = reinterpret_cast<const V2<T> *>(smem_raw) + 3 * (32 * sub + lane);
        const int stride = 3 * n_jg;
        int it = 0;
#pragma unroll 1
        for (; it < g_lo; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
#pragma unroll 1
        for (; it < g_hi; ++it, p += stride) {
            const int u0 = it * n_jg + 32 * sub;
            if (u0 < own1 && u0 + 32 > own0) pair_unit<T, TENSOR, true>(p, xi, acc, c1, negc2);
            else pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
        }
#pragma unroll 1
        for (; it < its_w; ++it, p += stride) pair_unit<T, TENSOR, false>(p, xi, acc, c1, negc2);
    }
    {
        T v[12], sm3[3];
#pragma unroll
        for (int k = 0; k < QI; ++k)
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) v[3 * k + cc] = P::hsum(acc[k][cc]);
        warp_sum12<T>(v, lane, sm3);
        if ((lane & 7) == 0) {
            T *dst = scr + warp * 12 + 3 * (lane >> 3);
            dst[0] = sm3[0]; dst[1] = sm3[1]; dst[2] = sm3[2];
        }
    }
    __syncthreads();
    // a2 + a3: the warps of a quad in order, self term Eq. (3a), 1/(8 pi mu); one output element per thread
    for (int e = tid; e < 3 * nrows; e += NTH) {
        const int rl = e / 3, cc = e - 3 * rl, qd = rl >> 2, k = rl & 3;
        const int mq = mb + (qd < mr ? 1 : 0);
        const T *sp = scr + (qd * mb + (qd < mr ? qd : mr)) * 12 + 3 * k + cc;
        T sacc = T(0);
        for (int j = 0; j < mq; ++j) sacc += sp[12 * j];
        const size_t gi = (size_t)3 * r0 + e;
        const double Fi = (double)reinterpret_cast<const T *>(A.raw_F)[gi];
        reinterpret_cast<T *>(A.out_u)[gi] = (T)(A.self_mob * Fi + A.pre * (double)sacc);
    }
}

}  // namespace ds
