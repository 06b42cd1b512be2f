// ds_api.cu -- host runtime behind the C ABI of include/ds.h: parameter validation, device
// buffers, host/device pointer staging, launch-shape choice, kernel-variant dispatch.
// No arithmetic of the method lives here; it is all in mobility.cuh / state.cuh.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "../../include/ds.h"
#include "../../include/ds_dev.h"
#include "mobility.cuh"
#include "pipeline.cuh"
#include "small.cuh"
#include "cluster.cuh"
#include "peak.cuh"
#include "averaged.cuh"
#include "state.cuh"

namespace {

thread_local char g_cuda_err[512] = "";

#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess) {                                                                  \
            snprintf(g_cuda_err, sizeof g_cuda_err, "%s:%d %s -> %s", __FILE__, __LINE__, #expr,  \
                     cudaGetErrorString(e_));                                                     \
            (void)cudaGetLastError();                                                             \
            return DS_ERR_CUDA;                                                                   \
        }                                                                                         \
    } while (0)

#define DS_TRY(expr)            \
    do {                        \
        int r_ = (expr);        \
        if (r_ != DS_OK) return r_; \
    } while (0)

template <typename T> constexpr int pack_w() { return ds::Pack<T>::W; }

// The opt-in to more than 48 KB of dynamic shared memory is a per-device attribute of a kernel: one instance of this
// per kernel variant remembers on which devices it has been set (a mutex makes it safe for concurrent host threads).
struct SmemOptIn {
    std::mutex mu;
    uint64_t done[4] = {0, 0, 0, 0};   // devices 0 .. 255
    int ensure(const void *kern, int device) {
        std::lock_guard<std::mutex> lock(mu);
        if (device >= 0 && device < 256 && (done[device >> 6] >> (device & 63) & 1ULL)) return DS_OK;
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ds::SMEM_MAX));
        if (device >= 0 && device < 256) done[device >> 6] |= 1ULL << (device & 63);
        return DS_OK;
    }
};

struct Buf {
    void *p = nullptr;
    size_t cap = 0;
};

}  // namespace

struct ds_system {
    ds_params P;
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    int N = 0, B = 0, S = 0;
    int W = 1;                  // spheres per unit: 2 (FP32 packs) or 1 (FP64)
    int NQ = 0, U = 0;          // quads = ceil(N/4), units = ceil(N/W)
    long long unit_stride = 0;  // units per system in the streams
    int tune_cta = 0;
    // launch shape of the step modes (ds_step, ds_batch_step, ds_velocity)
    int n_cta = 1;              // row tiles (CTAs) per system
    int sys_per_launch = 1;     // systems advanced by one launch (co-residency: n_cta * sys_per_launch <= SMs)
    int buf_bytes = 0;          // shared-memory stream buffer of the step modes
    int state_smem = 1;         // per-row state in shared memory (else in the global arrays below)
    size_t smem_bytes = 0;
    bool has_state = false;
    double t0 = 0.0;
    long long n_host = 0;       // steps taken since ds_set_state
    int64_t launches = 0;
    // state
    double *X = nullptr, *phase = nullptr;
    double *Rref = nullptr, *msd_part = nullptr, *msd_out = nullptr;   // Eq. (13): reference centres, partial sums, result
    bool has_ref = false;
    void *xu = nullptr;                         // the positions in user precision [B][N][3] (host-buffer fast path)
    bool x_valid = false, xu_valid = false;     // which of X (FP64) / xu holds the current state (at least one does)
    void *units[2] = {nullptr, nullptr};        // beta-streams (mobility.cuh), ping-pong over the stages
    unsigned long long *bar = nullptr;          // [B] arrival counters of the inter-CTA barrier
    unsigned long long bar_base = 0;
    void *ll[2] = {nullptr, nullptr};           // tagged (low-latency) copies of the streams, 96 B per unit
    unsigned int ll_tag = 1;                    // next unused tag (0 = never written)
    double *Xcg = nullptr, *V1g = nullptr, *Fg = nullptr, *Lg = nullptr;  // only when !state_smem
    long long *probe = nullptr;                 // caller's device buffer (ds_set_probe) or NULL
    // pipelined step kernel (pipeline.cuh): used for ds_step / ds_batch_step when the shape allows it and the pair loop
    // dominates a stage
    int pipe_mode = -1;                         // -1 = library heuristic, 0 = never, 1 = whenever the shape allows it
    bool use_pipe = false;
    int cl_cs = 0;                              // > 0: cluster_kernel with this many CTAs per system (cluster.cuh)
    int cl_buf_units[2] = {0, 0}, cl_rows_max = 0, cl_slots_max = 0;
    int cl_half_off[2][ds::CL_MAX_CS + 1] = {};
    int cll_cs = 0, cll_buf_units = 0, cll_rows_max = 0, cll_slots_max = 0;   // > 0: cluster_lat_kernel (cluster.cuh)
    size_t cll_smem = 0;
    size_t cl_smem = 0;
    int *half_off = nullptr;                    // device table [2][n_cta + 1]
    int4 *ptab_g = nullptr;                     // device table [n_cta][2][16][3] (pipe_build_table)
    size_t ptab_cap = 0;
    int half_off_cap = 0;
    int reg_units[2] = {0, 0}, pbuf_units[2] = {0, 0}, rows_max = 0;
    size_t pipe_smem = 0;
    unsigned long long *pcnt = nullptr;         // [B][2] arrival counters of the two stream regions
    unsigned long long pcnt_base = 0;
    // scratch of the stateless apply and of host-pointer staging
    Buf ap_units, st_a, st_b, st_c;
    Buf avg;                                    // FP64 scratch of the stroke-averaged model (Eq. 9)
    Buf avg_sc;                                 // its sin/cos table
    Buf avg_xch;                                // tagged exchange buffers of the device-resident stepping (averaged.cuh)
    unsigned int avg_tag = 1;                   // next unused tag (0 = never written)
    size_t avg_xch_records = 0;
};

namespace {

constexpr long long MAX_STEPS_PER_LAUNCH = 1LL << 16;

int ensure(Buf &b, size_t bytes, bool zero = false) {
    if (b.cap >= bytes) return DS_OK;
    if (b.p) CU_TRY(cudaFree(b.p));
    b.p = nullptr; b.cap = 0;
    size_t want = bytes + bytes / 4 + 256;
    CU_TRY(cudaMalloc(&b.p, want));
    if (zero) CU_TRY(cudaMemset(b.p, 0, want));
    b.cap = want;
    return DS_OK;
}

// 1 = device-accessible pointer, 0 = host pointer
int is_device_ptr(const void *p, int *out) {
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        *out = 0;  // plain malloc'ed memory on old drivers reports an error: host
        return DS_OK;
    }
    *out = (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) ? 1 : 0;
    return DS_OK;
}

size_t elem_size(const ds_system *s) { return s->P.precision == DS_F64 ? sizeof(double) : sizeof(float); }

// Launch shape of the stateless apply: n_cta row tiles (mobility.cuh), any number of waves.  Every CTA
// walks all U units with n_jg = NT / nq beta-groups, i.e. ceil(U / n_jg) iterations of 4 alpha x 1 unit
// per thread, so the modelled time is waves x (iterations + a fixed per-CTA cost, in iterations).
constexpr double ROW_COST = 0.4;   // cost of one more quad of rows in a CTA's tail, in pair-loop iterations
int choose_tiles_apply(const ds_system *s, int NQ, int U) {
    const int lo = (NQ + ds::NT - 1) / ds::NT;  // nq <= NT
    if (s->tune_cta > 0) {
        int t = s->tune_cta < lo ? lo : s->tune_cta;
        return t > NQ ? NQ : t;
    }
    const int hi = NQ < 16 * s->num_sms ? NQ : 16 * s->num_sms;
    double best_cost = 1e300;
    int best = lo;
    for (int n = lo; n <= hi; ++n) {
        const int nq = (NQ + n - 1) / n;
        const int n_jg = ds::NT / nq;
        const long long iters = (U + n_jg - 1) / n_jg;
        const long long waves = ((long long)n + s->num_sms - 1) / s->num_sms;
        const double cost = (double)waves * ((double)iters + 6.0 + ROW_COST * nq);
        if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = n; }
    }
    return best;
}

// Launch shape of the step modes: all CTAs of a launch are co-resident (they meet at the inter-CTA
// barrier every stage), so n_cta <= SMs and floor(SMs / n_cta) systems run per launch; B systems take
// ceil(B / that) launches one after the other.  Same cost model, plus the barrier in the fixed cost.
int choose_shape_step(ds_system *s) {
    const int lo = (s->NQ + ds::NT - 1) / ds::NT;
    if (lo > s->num_sms) return DS_ERR_INVALID_PARAM;
    int hi = s->NQ < s->num_sms ? s->NQ : s->num_sms;
    int best = lo;
    if (s->tune_cta > 0) {
        best = s->tune_cta < lo ? lo : (s->tune_cta > hi ? hi : s->tune_cta);
    } else {
        double best_cost = 1e300;
        for (int n = lo; n <= hi; ++n) {
            const int nq = (s->NQ + n - 1) / n;
            const int n_jg = ds::NT / nq;
            const long long iters = (s->U + n_jg - 1) / n_jg;
            int per = s->num_sms / n;
            per = per < 1 ? 1 : (per > s->B ? s->B : per);
            const long long groups = (s->B + per - 1) / per;
            // a stage's fixed part, in iterations: barrier + hand-over / local, and the tail (reduction, integrator,
            // Eq. (4)), which grows with the rows a CTA owns: at equal iterations more CTAs win (measured, N = 128:
            // 3.0 us per stage on 32 CTAs against 3.9 on 4)
            const double cost = (double)groups * ((double)iters + (n > 1 ? 6.0 : 4.0) + ROW_COST * nq);
            if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = n; }
        }
    }
    s->n_cta = best;
    int per = best > 1 ? s->num_sms / best : s->B;   // n_cta == 1: systems never wait on one another
    s->sys_per_launch = per < 1 ? 1 : (per > s->B ? s->B : per);
    const int rows_max = 4 * ((s->NQ + best - 1) / best);
    const size_t state = (size_t)rows_max * ds::STATE_BYTES_PER_ROW;
    const long long room = ((long long)ds::SMEM_MAX - ds::BAR_BYTES - (long long)state) / 128 * 128;
    if (room >= (long long)ds::NS_MIN * ds::SLOT_BYTES) {
        s->state_smem = 1;
        s->buf_bytes = (int)room;
        s->smem_bytes = (size_t)room + ds::BAR_BYTES + state;
    } else {
        s->state_smem = 0;
        s->buf_bytes = (ds::SMEM_MAX - ds::BAR_BYTES) / 128 * 128;
        s->smem_bytes = (size_t)s->buf_bytes + ds::BAR_BYTES;
    }
    return DS_OK;
}

// The stream of a launch is resident when every CTA's padded stream (iterations x groups x 48 B) fits the buffer;
// CTAs own floor or ceil(NQ / n_cta) quads, hence two shapes to check.
bool stream_resident(int NQ, int U, int n_cta, int buf_bytes) {
    const int nq_lo = NQ / n_cta, nq_hi = (NQ + n_cta - 1) / n_cta;
    for (int nq = nq_lo < 1 ? 1 : nq_lo; nq <= nq_hi; ++nq) {
        const int n_jg = ds::NT / nq < U ? ds::NT / nq : U;
        const long long total_it = (U + n_jg - 1) / n_jg;
        if (total_it * n_jg * ds::UNIT_BYTES > buf_bytes) return false;
    }
    return true;
}

template <typename T, int TENSOR, int MODE, bool RES>
int launch_run_v(ds_system *s, ds::RunArgs &A, dim3 grid, size_t smem, bool coop, cudaStream_t st) {
    auto kern = ds::run_kernel<T, TENSOR, MODE, RES>;
    static SmemOptIn opt_in;
    DS_TRY(opt_in.ensure((const void *)kern, s->P.device));
    if (coop) {
        void *args[] = {(void *)&A};
        CU_TRY(cudaLaunchCooperativeKernel((const void *)kern, grid, dim3(ds::NT), args, smem, st));
    } else if (MODE == ds::KM_APPLY) {
        // programmatic dependent launch: the CTAs of this apply may become resident while the previous kernel of the
        // stream drains; the kernel waits (griddepcontrol.wait) before its first global access
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = grid; cfg.blockDim = dim3(ds::NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        CU_TRY(cudaLaunchKernelEx(&cfg, kern, A));
    } else {
        kern<<<grid, dim3(ds::NT), smem, st>>>(A);
        CU_TRY(cudaGetLastError());
    }
    s->launches += 1;
    return DS_OK;
}

template <typename T, int TENSOR>
int launch_run_t(ds_system *s, ds::RunArgs &A, dim3 grid, size_t smem, bool coop, cudaStream_t st) {
    const int km = A.mode == ds::RUN_APPLY ? ds::KM_APPLY : A.mode == ds::RUN_VELOCITY ? ds::KM_VELOCITY
                 : A.heun ? ds::KM_HEUN : ds::KM_EULER;
    const bool res = stream_resident(A.NQ, A.U, A.n_cta, A.buf_bytes);
#define DS_CASE(M)                                                                      \
    case M: return res ? launch_run_v<T, TENSOR, M, true>(s, A, grid, smem, coop, st)   \
                       : launch_run_v<T, TENSOR, M, false>(s, A, grid, smem, coop, st);
    switch (km) {
        DS_CASE(ds::KM_APPLY)
        DS_CASE(ds::KM_VELOCITY)
        DS_CASE(ds::KM_EULER)
        DS_CASE(ds::KM_HEUN)
    }
#undef DS_CASE
    return DS_ERR_INVALID_PARAM;
}

int launch_run(ds_system *s, ds::RunArgs &A, dim3 grid, size_t smem, bool coop, cudaStream_t st) {
    const bool f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
    if (f64)
        return rpy ? launch_run_t<double, ds::TENSOR_RPY>(s, A, grid, smem, coop, st)
                   : launch_run_t<double, ds::TENSOR_OSEEN>(s, A, grid, smem, coop, st);
    return rpy ? launch_run_t<float, ds::TENSOR_RPY>(s, A, grid, smem, coop, st)
               : launch_run_t<float, ds::TENSOR_OSEEN>(s, A, grid, smem, coop, st);
}

void fill_constants(const ds_system *s, ds::RunArgs &A) {
    const double pi = 3.14159265358979323846264338327950288;
    A.self_mob = 1.0 / (6.0 * pi * s->P.eta * s->P.a);
    A.pre = 1.0 / (8.0 * pi * s->P.eta);
    A.c1 = 2.0 * s->P.a * s->P.a / 3.0;
    A.c2 = 2.0 * s->P.a * s->P.a;
    A.c1f = (float)A.c1; A.c2f = (float)A.c2;
    A.t0 = s->t0; A.dt = s->P.dt; A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
    A.noise_amp = s->P.kT > 0.0 ? sqrt(2.0 * s->P.kT * s->P.dt * A.self_mob) : 0.0;   // Eq. (1a) with 2H ~ 2/(6 pi mu a) = C C^T
    A.seed = s->P.seed;
}


// Pipelined step kernel (pipeline.cuh): every CTA's rows are cut into two halves of whole quads; region h of a stream
// holds the half-h units of all CTAs.  Builds the offset table and decides whether the shape is eligible: both halves
// of every CTA at most 16 quads (one warp per quad at least), everything in shared memory.
int setup_pipe(ds_system *s) {
    s->use_pipe = false;
    if (s->n_cta < 2 || s->pipe_mode == 0) return DS_OK;
    const int n = s->n_cta, W = s->W;
    std::vector<int> off(2 * (size_t)(n + 1), 0);
    int rows_max = 0, nqh_max = 0;
    std::vector<int> shapes;   // distinct beta-group counts n_jg = 32 (16 / nq_h) of all passes
    for (int c = 0; c < n; ++c) {
        const long long q0 = (long long)c * s->NQ / n, q1 = (long long)(c + 1) * s->NQ / n;
        const int nq = (int)(q1 - q0);
        const long long left = (long long)s->N - 4 * q0;
        const int nrows = (int)(left < 4LL * nq ? left : 4LL * nq);
        const int nqA = ds::pipe_split(nq), nqB = nq - nqA;
        const int rowsA = 4 * nqA < nrows ? 4 * nqA : nrows, rowsB = nrows - rowsA;
        off[c + 1] = off[c] + rowsA / W;
        off[(n + 1) + c + 1] = off[(n + 1) + c] + rowsB / W;
        rows_max = nrows > rows_max ? nrows : rows_max;
        nqh_max = nqA > nqh_max ? nqA : nqh_max;
        for (int nqh : {nqA, nqB})
            if (nqh > 0 && nqh <= ds::PIPE_CW) {   // the 16 warps of a pass: 16 / nqh per quad, or one more
                shapes.push_back(32 * (ds::PIPE_CW / nqh));
                if (ds::PIPE_CW % nqh) shapes.push_back(32 * (ds::PIPE_CW / nqh + 1));
            }
    }
    if (nqh_max > ds::PIPE_CW) return DS_OK;
    rows_max = (rows_max + 3) / 4 * 4;
    int bu[2];
    for (int h = 0; h < 2; ++h) {
        const int U = off[(size_t)h * (n + 1) + n];
        int cap = U;
        for (int n_jg : shapes) { const int need = (U + n_jg - 1) / n_jg * n_jg; cap = need > cap ? need : cap; }
        bu[h] = (cap + 7) / 8 * 8;
    }
    const size_t smem = (size_t)(bu[0] + bu[1]) * ds::UNIT_BYTES + ds::PIPE_BAR_BYTES + ds::PIPE_SCR_BYTES + ds::PIPE_TAB_BYTES +
                       (size_t)rows_max * ds::STATE_BYTES_PER_ROW;
    if (smem > (size_t)ds::SMEM_MAX) return DS_OK;
    if (s->pipe_mode < 0) {
        // heuristic: the pipeline hides a stage's fixed cost behind the pair loop of the other half, but its own hand-over chain
        // (tail -> release -> every CTA arrived -> bulk copy, about 7 k cycles, twice per stage through one service warp) bounds a
        // stage from below at about 6.8 us.  Measured per stage, pipelined / one-pass: N = 1024: 6.9 / 4.9 us, 2048: 7.6 / 7.8,
        // 3072: 10.5 / 11.8, 4096: 13.5 / 15.6.  Switch at 8 pair-loop iterations of the one-pass shape (N = 2048 on 128 CTAs).
        const int nq = (s->NQ + n - 1) / n, n_jg = ds::NT / nq;
        if ((s->U + n_jg - 1) / n_jg < 8) return DS_OK;
    }
    if (s->half_off_cap < 2 * (n + 1)) {
        if (s->half_off) CU_TRY(cudaFree(s->half_off));
        s->half_off = nullptr; s->half_off_cap = 0;
        CU_TRY(cudaMalloc((void **)&s->half_off, 2 * (size_t)(n + 1) * sizeof(int)));
        s->half_off_cap = 2 * (n + 1);
    }
    CU_TRY(cudaMemcpy(s->half_off, off.data(), 2 * (size_t)(n + 1) * sizeof(int), cudaMemcpyHostToDevice));
    {   // which warp does what in the two passes of every CTA (pipe_build_table)
        const size_t per = 2 * (size_t)ds::PIPE_CW * 3;
        std::vector<int4> tab((size_t)n * per);
        const int ru[2] = {off[n], off[(size_t)(n + 1) + n]};
        for (int c = 0; c < n; ++c) ds::pipe_build_table(s->N, s->NQ, n, c, W, off.data(), ru, tab.data() + (size_t)c * per);
        if (s->ptab_cap < tab.size()) {
            if (s->ptab_g) CU_TRY(cudaFree(s->ptab_g));
            s->ptab_g = nullptr; s->ptab_cap = 0;
            CU_TRY(cudaMalloc((void **)&s->ptab_g, tab.size() * sizeof(int4)));
            s->ptab_cap = tab.size();
        }
        CU_TRY(cudaMemcpy(s->ptab_g, tab.data(), tab.size() * sizeof(int4), cudaMemcpyHostToDevice));
    }
    s->reg_units[0] = off[n]; s->reg_units[1] = off[(size_t)(n + 1) + n];
    s->pbuf_units[0] = bu[0]; s->pbuf_units[1] = bu[1];
    s->rows_max = rows_max;
    s->pipe_smem = smem;
    s->use_pipe = true;
    return DS_OK;
}

template <typename T, int TENSOR, bool HEUN>
int launch_pipe_v(ds_system *s, ds::PipeArgs &A, dim3 grid) {
    auto kern = ds::pipe_kernel<T, TENSOR, HEUN>;
    static SmemOptIn opt_in;
    DS_TRY(opt_in.ensure((const void *)kern, s->P.device));
    void *args[] = {(void *)&A};
    CU_TRY(cudaLaunchCooperativeKernel((const void *)kern, grid, dim3(ds::PIPE_NT), args, s->pipe_smem, s->stream));
    s->launches += 1;
    return DS_OK;
}

// RUN_STEP through the pipelined kernel: one launch per group of co-resident systems
int launch_pipe_run(ds_system *s, long long n_steps) {
    ds::PipeArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.NQ = s->NQ; A.n_cta = s->n_cta; A.unit_stride = s->unit_stride;
    A.units[0] = s->units[0]; A.units[1] = s->units[1];
    A.half_off = s->half_off;
    A.ptab_g = s->ptab_g;
    A.reg_units[0] = s->reg_units[0]; A.reg_units[1] = s->reg_units[1];
    A.buf_units[0] = s->pbuf_units[0]; A.buf_units[1] = s->pbuf_units[1];
    A.rows_max = s->rows_max;
    ds::RunArgs R;
    memset(&R, 0, sizeof R);
    fill_constants(s, R);
    A.self_mob = R.self_mob; A.pre = R.pre; A.c1 = R.c1; A.c2 = R.c2; A.c1f = R.c1f; A.c2f = R.c2f;
    A.t0 = R.t0; A.dt = R.dt; A.ell = R.ell; A.lambda = R.lambda; A.omega = R.omega; A.k0 = R.k0;
    A.noise_amp = R.noise_amp; A.seed = R.seed;
    A.n0 = s->n_host; A.n_steps = n_steps;
    A.X = s->X; A.xu = s->xu; A.from_user = s->x_valid ? 0 : 1; A.phase = s->phase;
    A.cnt = s->pcnt; A.cnt_base = s->pcnt_base;
    A.probe = s->probe;
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
    const long long n_stage = n_steps * (heun ? 2 : 1);
    for (int b0 = 0; b0 < s->B; b0 += s->sys_per_launch) {
        const int nb = s->B - b0 < s->sys_per_launch ? s->B - b0 : s->sys_per_launch;
        A.b0 = b0;
        const dim3 grid((unsigned)s->n_cta, (unsigned)nb);
#define DS_PIPE(TT, TEN) (heun ? launch_pipe_v<TT, TEN, true>(s, A, grid) : launch_pipe_v<TT, TEN, false>(s, A, grid))
        if (f64) DS_TRY(rpy ? DS_PIPE(double, ds::TENSOR_RPY) : DS_PIPE(double, ds::TENSOR_OSEEN));
        else DS_TRY(rpy ? DS_PIPE(float, ds::TENSOR_RPY) : DS_PIPE(float, ds::TENSOR_OSEEN));
#undef DS_PIPE
    }
    s->pcnt_base += (unsigned long long)s->n_cta * (unsigned long long)n_stage;
    s->x_valid = true; s->xu_valid = true;
    return DS_OK;
}


// ds_mobility_apply through apply_kernel (pipeline.cuh) when every CTA owns at most 16 quads and the stream with its pad
// units fits shared memory; *used says whether it ran.
template <typename T, int TENSOR> int launch_apply_v(ds_system *s, const ds::ApplyArgs &A, size_t smem) {
    auto kern = ds::apply_kernel<T, TENSOR>;
    static SmemOptIn opt_in;
    DS_TRY(opt_in.ensure((const void *)kern, s->P.device));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)A.n_cta); cfg.blockDim = dim3(32 * ds::PIPE_CW); cfg.dynamicSmemBytes = smem; cfg.stream = s->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    CU_TRY(cudaLaunchKernelEx(&cfg, kern, A));
    s->launches += 1;
    return DS_OK;
}

int apply_warp_shape(ds_system *s, const ds::RunArgs &R, const void *dpos, const void *dF, void *du, bool *used) {
    *used = false;
    if (s->pipe_mode == 0) return DS_OK;
    const int nq_hi = (R.NQ + R.n_cta - 1) / R.n_cta, nq_lo = R.NQ / R.n_cta;
    if (nq_hi > ds::PIPE_CW || nq_lo < 1) return DS_OK;
    int cap = R.U;
    for (int nq = nq_lo; nq <= nq_hi; ++nq)
        for (int extra = 0; extra < 2; ++extra) {
            if (extra && ds::PIPE_CW % nq == 0) continue;
            const int n_jg = 32 * (ds::PIPE_CW / nq + extra), need = (R.U + n_jg - 1) / n_jg * n_jg;
            cap = need > cap ? need : cap;
        }
    cap = (cap + 7) / 8 * 8;
    const size_t smem = (size_t)cap * ds::UNIT_BYTES + (size_t)ds::PIPE_CW * 12 * sizeof(double);
    if (smem > (size_t)ds::SMEM_MAX) return DS_OK;
    ds::ApplyArgs A;
    memset(&A, 0, sizeof A);
    A.N = R.N; A.NQ = R.NQ; A.U = R.U; A.n_cta = R.n_cta; A.buf_units = cap;
    A.self_mob = R.self_mob; A.pre = R.pre; A.c1 = R.c1; A.c2 = R.c2; A.c1f = R.c1f; A.c2f = R.c2f;
    A.raw_pos = dpos; A.raw_F = dF; A.out_u = du;
    const bool f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
    int rc;
    if (f64) rc = rpy ? launch_apply_v<double, ds::TENSOR_RPY>(s, A, smem) : launch_apply_v<double, ds::TENSOR_OSEEN>(s, A, smem);
    else rc = rpy ? launch_apply_v<float, ds::TENSOR_RPY>(s, A, smem) : launch_apply_v<float, ds::TENSOR_OSEEN>(s, A, smem);
    DS_TRY(rc);
    *used = true;
    return DS_OK;
}

// the cluster kernel variant a system uses
const void *cluster_kernel_of(const ds_system *s) {
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
#define DS_CLK(TT, TEN) (heun ? (const void *)ds::cluster_kernel<TT, TEN, true> : (const void *)ds::cluster_kernel<TT, TEN, false>)
    if (f64) return rpy ? DS_CLK(double, ds::TENSOR_RPY) : DS_CLK(double, ds::TENSOR_OSEEN);
    return rpy ? DS_CLK(float, ds::TENSOR_RPY) : DS_CLK(float, ds::TENSOR_OSEEN);
#undef DS_CLK
}

// Shared-memory layout of the cluster kernel for cs CTAs per system; false if a half has too many quads or it does not fit.
bool cluster_layout(ds_system *s, int cs) {
    const int W = s->W;
    int rows_max = 0, slots = 1, njg_max = 32;
    s->cl_half_off[0][0] = s->cl_half_off[1][0] = 0;
    for (int c = 0; c < cs; ++c) {
        const long long q0 = (long long)c * s->NQ / cs, q1 = (long long)(c + 1) * s->NQ / cs;
        const int nq = (int)(q1 - q0);
        const long long left = (long long)s->N - 4 * q0;
        const int nrows = (int)(left < 4LL * nq ? left : 4LL * nq);
        const int nqA = ds::pipe_split(nq), nqB = nq - nqA;
        const int rowsA = 4 * nqA < nrows ? 4 * nqA : nrows, rowsB = nrows - rowsA;
        if (nqA > ds::CL_CW * ds::CL_MAX_QW) return false;
        rows_max = rows_max > 4 * nq ? rows_max : 4 * nq;
        for (int h = 0; h < 2; ++h) {
            int QW, m;
            ds::cluster_pass_shape(h == 0 ? nqA : nqB, QW, m);
            const int sl = (h == 0 ? nqA : nqB) * m, njg = (32 / QW) * m;
            slots = slots > sl ? slots : sl;
            njg_max = njg_max > njg ? njg_max : njg;
        }
        s->cl_half_off[0][c + 1] = s->cl_half_off[0][c] + rowsA / W;
        s->cl_half_off[1][c + 1] = s->cl_half_off[1][c] + rowsB / W;
    }
    size_t smem = ds::CL_BAR_BYTES + ds::CL_TAB_BYTES + (size_t)2 * slots * 12 * 8 + (size_t)rows_max * ds::STATE_BYTES_PER_ROW;
    for (int h = 0; h < 2; ++h) {
        s->cl_buf_units[h] = (s->cl_half_off[h][cs] + njg_max + 7) / 8 * 8;
        smem += 2 * (size_t)s->cl_buf_units[h] * ds::UNIT_BYTES;
    }
    if (smem > (size_t)ds::SMEM_MAX) return false;
    s->cl_rows_max = rows_max; s->cl_slots_max = slots; s->cl_smem = smem;
    return true;
}

// Cluster step kernel (cluster.cuh) for ensembles: one thread-block cluster of cs CTAs per system, cs the largest of 8, 4, 2
// for which all B clusters are resident at once (cudaOccupancyMaxActiveClusters: a cluster lives inside one GPC, so this is
// fewer than SMs / cs).  Taken when those clusters fill at least 3/4 of the SMs (B = 64: cs = 2, 128 of 148), a CTA owns at
// least a quad per warp, every half of a CTA has at most 16 * 8 quads, and two copies of the stream plus the state fit
// shared memory.
int setup_cluster(ds_system *s) {
    s->cl_cs = 0;
    const bool forced = s->pipe_mode == 2;   // ds_set_pipeline(2): whenever the layout fits and the clusters are co-resident
    if (s->pipe_mode == 0 || s->tune_cta != 0 || ((s->B < 2 || s->S <= ds::SMALL_MAX_S) && !forced)) return DS_OK;
    const void *kern = cluster_kernel_of(s);
    for (int cs = ds::CL_MAX_CS; cs >= 2; cs >>= 1) {
        if ((long long)s->B * cs > s->num_sms || cs > s->NQ) continue;
        if (!forced && s->NQ / cs < ds::CL_CW) continue;
        if (!forced && 4LL * s->B * cs < 3LL * s->num_sms) break;
        if (!cluster_layout(s, cs)) continue;
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ds::SMEM_MAX));
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3((unsigned)cs, (unsigned)s->B); cfg.blockDim = dim3(ds::CL_NT); cfg.dynamicSmemBytes = s->cl_smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n_active = 0;
        CU_TRY(cudaOccupancyMaxActiveClusters(&n_active, kern, &cfg));
        if (n_active >= s->B) { s->cl_cs = cs; return DS_OK; }
    }
    return DS_OK;
}

template <typename T, int TENSOR, bool HEUN>
int launch_cluster_v(ds_system *s, const ds::ClusterArgs &A) {
    auto kern = ds::cluster_kernel<T, TENSOR, HEUN>;
    static SmemOptIn opt_in;
    DS_TRY(opt_in.ensure((const void *)kern, s->P.device));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)A.cs, (unsigned)s->B); cfg.blockDim = dim3(ds::CL_NT);
    cfg.dynamicSmemBytes = s->cl_smem; cfg.stream = s->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)A.cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    CU_TRY(cudaLaunchKernelEx(&cfg, kern, A));
    s->launches += 1;
    return DS_OK;
}

// RUN_STEP through the cluster kernel: one launch for all B systems
int launch_cluster_run(ds_system *s, long long n_steps) {
    ds::ClusterArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.NQ = s->NQ; A.cs = s->cl_cs;
    memcpy(A.half_off, s->cl_half_off, sizeof A.half_off);
    A.buf_units[0] = s->cl_buf_units[0]; A.buf_units[1] = s->cl_buf_units[1];
    A.rows_max = s->cl_rows_max; A.slots_max = s->cl_slots_max;
    ds::RunArgs R;
    memset(&R, 0, sizeof R);
    fill_constants(s, R);
    A.self_mob = R.self_mob; A.pre = R.pre; A.c1 = R.c1; A.c2 = R.c2; A.c1f = R.c1f; A.c2f = R.c2f;
    A.t0 = R.t0; A.dt = R.dt; A.ell = R.ell; A.lambda = R.lambda; A.omega = R.omega; A.k0 = R.k0;
    A.noise_amp = R.noise_amp; A.seed = R.seed;
    A.n0 = s->n_host; A.n_steps = n_steps;
    A.X = s->X; A.xu = s->xu; A.from_user = s->x_valid ? 0 : 1; A.phase = s->phase;
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
#define DS_CL(TT, TEN) (heun ? launch_cluster_v<TT, TEN, true>(s, A) : launch_cluster_v<TT, TEN, false>(s, A))
    if (f64) DS_TRY(rpy ? DS_CL(double, ds::TENSOR_RPY) : DS_CL(double, ds::TENSOR_OSEEN));
    else DS_TRY(rpy ? DS_CL(float, ds::TENSOR_RPY) : DS_CL(float, ds::TENSOR_OSEEN));
#undef DS_CL
    s->x_valid = true; s->xu_valid = true;
    return DS_OK;
}

// RUN_STEP for small systems (S <= 32): one warp per system (small.cuh), any number of systems per launch
template <typename T, int TENSOR, bool HEUN> int launch_small_v(ds_system *s, const ds::SmallArgs &A) {
    const unsigned grid = (unsigned)((s->B + ds::SMALL_WARPS - 1) / ds::SMALL_WARPS);
    ds::small_kernel<T, TENSOR, HEUN><<<grid, 32 * ds::SMALL_WARPS, 0, s->stream>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

// Warp-per-system kernel or run_kernel for S <= 32?  With 17 ... 32 dumbbells a lane has a whole dumbbell's pair sum to
// itself (64 FP64 units at S = 32) and a stage takes 4.7 - 7.3 us in FP64 (2.4 - 3.6 in FP32) whatever B is; run_kernel on
// several CTAs per system takes 3.2 - 3.5 us (2.8 - 3.0), but only as long as all systems are resident at once (measured,
// B = 1 ... 600: DESIGN.md section 6c).  A forced tiling (ds_set_tuning) keeps small systems on run_kernel (tests).
bool use_small_kernel(const ds_system *s) {
    if (s->S > ds::SMALL_MAX_S || s->tune_cta != 0) return false;
    if (s->S <= 16) return true;
    if (s->P.precision == DS_F64) return (long long)s->B * s->n_cta > s->num_sms;
    return s->S <= 24 || (long long)s->B * s->n_cta > s->num_sms;
}

int launch_small_run(ds_system *s, long long n_steps) {
    ds::SmallArgs A;
    memset(&A, 0, sizeof A);
    A.S = s->S; A.B = s->B;
    ds::RunArgs R;
    memset(&R, 0, sizeof R);
    fill_constants(s, R);
    A.self_mob = R.self_mob; A.pre = R.pre; A.c1 = R.c1; A.c2 = R.c2; A.c1f = R.c1f; A.c2f = R.c2f;
    A.t0 = R.t0; A.dt = R.dt; A.ell = R.ell; A.lambda = R.lambda; A.omega = R.omega; A.k0 = R.k0;
    A.noise_amp = R.noise_amp; A.seed = R.seed;
    A.n0 = s->n_host; A.n_steps = n_steps;
    A.X = s->X; A.xu = s->xu; A.from_user = s->x_valid ? 0 : 1; A.phase = s->phase;
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
#define DS_SMALL(TT, TEN) (heun ? launch_small_v<TT, TEN, true>(s, A) : launch_small_v<TT, TEN, false>(s, A))
    if (f64) DS_TRY(rpy ? DS_SMALL(double, ds::TENSOR_RPY) : DS_SMALL(double, ds::TENSOR_OSEEN));
    else DS_TRY(rpy ? DS_SMALL(float, ds::TENSOR_RPY) : DS_SMALL(float, ds::TENSOR_OSEEN));
#undef DS_SMALL
    s->x_valid = true; s->xu_valid = true;
    return DS_OK;
}

// the latency variant of the cluster kernel a system uses
const void *cluster_lat_kernel_of(const ds_system *s) {
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
#define DS_CLK(TT, TEN) (heun ? (const void *)ds::cluster_lat_kernel<TT, TEN, true> : (const void *)ds::cluster_lat_kernel<TT, TEN, false>)
    if (f64) return rpy ? DS_CLK(double, ds::TENSOR_RPY) : DS_CLK(double, ds::TENSOR_OSEEN);
    return rpy ? DS_CLK(float, ds::TENSOR_RPY) : DS_CLK(float, ds::TENSOR_OSEEN);
#undef DS_CLK
}

// cluster_lat_kernel (cluster.cuh) for single small systems and small ensembles: one cluster of 2 ... 16 CTAs per system when
// all B clusters are resident at once and a stage's pair loops are short (at most LAT_MAX_ITERS iterations per warp: beyond
// that the 148-SM shapes of run_kernel / pipe_kernel win).  ds_set_pipeline(3) forces it for every shape that fits.
// Measured (FP32 / FP64 us per stage, this kernel against the earlier choice): S = 20: 1.6 / 2.0 against 2.5 / 3.3; S = 64
// (C2): 1.8 / 2.3 against 3.1 / 3.5; S = 128: 2.2 / 3.3 against 3.2 / 4.1; S = 192: 2.7 / 4.7 against 3.7 / 4.7; 18 x S = 64:
// 1.8 / 2.8 against 3.2 / 5.2.  S <= 16 stays on the warp-per-system kernel (0.8 - 2.2 us).
// ... and, at 4 iterations per warp: single systems S = 256 FP32 3.7 against 3.6, S = 160 FP64 4.1 against 4.3 (a tie), but ensembles
// 18 x S = 128 FP32 3.3 against 4.4, 16 x S = 128 FP64 6.1 against 7.1 (run_kernel has fewer CTAs per system there).
constexpr int LAT_MAX_ITERS_SINGLE = 3, LAT_MAX_ITERS_ENSEMBLE = 4;
int setup_cluster_lat(ds_system *s) {
    s->cll_cs = 0;
    const bool forced = s->pipe_mode == 3;
    const int LAT_MAX_ITERS = s->B >= 2 ? LAT_MAX_ITERS_ENSEMBLE : LAT_MAX_ITERS_SINGLE;
    if (s->pipe_mode == 0 || s->pipe_mode == 2 || s->tune_cta != 0 || s->cl_cs > 0) return DS_OK;
    if (!forced && (s->pipe_mode == 1 || s->S <= 16)) return DS_OK;
    const void *kern = cluster_lat_kernel_of(s);
    double best_cost = 1e300;
    // Cost of a stage in pair-loop iterations: waves x (iterations per warp + 4 for the tail and the hand-over); the smallest cluster
    // wins a tie (S = 64: 4 CTAs 1.8 us per stage, 8 CTAs 1.9, 16 CTAs 2.0; S = 128: 2.4 on 8, 2.2 on 16; S = 192: 3.6 / 2.7).
    // 16 CTAs per cluster is beyond the portable size (opt-in attribute).
    for (int cs = 1; cs <= 16; cs <<= 1) {
        if (cs > s->NQ || cs > s->num_sms) continue;
        const int nq = (s->NQ + cs - 1) / cs;
        if (nq > ds::CL_CW * ds::CL_MAX_QW) continue;
        int njg = 32, slots = 1, its = 0;
        for (int n = s->NQ / cs; n <= nq; ++n) {   // CTAs own floor or ceil(NQ / cs) quads
            int QW, m;
            ds::cluster_pass_shape(n, QW, m);
            const int j = (32 / QW) * m, i = (s->U + j - 1) / j;
            njg = njg > j ? njg : j; slots = slots > n * m ? slots : n * m; its = its > i ? its : i;
        }
        if (!forced && its > LAT_MAX_ITERS) continue;
        const int buf_units = (s->U + njg + 7) / 8 * 8, rows_max = 4 * nq;
        const size_t smem = 2 * (size_t)buf_units * ds::UNIT_BYTES + 64 + (size_t)slots * 12 * 8 + (size_t)rows_max * ds::STATE_BYTES_PER_ROW;
        if (smem > (size_t)ds::SMEM_MAX) continue;
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ds::SMEM_MAX));
        if (cs > ds::CL_MAX_CS && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
            (void)cudaGetLastError();
            continue;
        }
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3((unsigned)cs, (unsigned)s->B); cfg.blockDim = dim3(ds::CLL_NT); cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n_active = 0;
        if (cudaOccupancyMaxActiveClusters(&n_active, kern, &cfg) != cudaSuccess) { (void)cudaGetLastError(); continue; }
        if (n_active < 1) continue;
        const long long waves = ((long long)s->B + n_active - 1) / n_active;
        // several waves only for one CTA per system and S > 32 (the alternatives there, run_kernel with one CTA per system or the
        // warp-per-system kernel, run in waves too; measured: 600 x S = 64 FP32 15.3 us per stage against 22.4, but 600 x S = 20
        // 7.8 against 3.2 of the warp-per-system kernel, and clusters of 2 or 4 in several waves lose to run_kernel: 40 x S = 100
        // 6.5 against 5.1)
        if (waves > 1 && !(cs == 1 && s->S > ds::SMALL_MAX_S)) continue;
        const double cost = (double)waves * (its + 4.0);
        if (cost >= best_cost * (1.0 - 1e-9)) continue;
        best_cost = cost;
        s->cll_cs = cs; s->cll_buf_units = buf_units; s->cll_rows_max = rows_max; s->cll_slots_max = slots; s->cll_smem = smem;
    }
    return DS_OK;
}

template <typename T, int TENSOR, bool HEUN>
int launch_cluster_lat_v(ds_system *s, const ds::ClusterLatArgs &A) {
    auto kern = ds::cluster_lat_kernel<T, TENSOR, HEUN>;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)A.cs, (unsigned)s->B); cfg.blockDim = dim3(ds::CLL_NT);
    cfg.dynamicSmemBytes = s->cll_smem; cfg.stream = s->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)A.cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    CU_TRY(cudaLaunchKernelEx(&cfg, kern, A));
    s->launches += 1;
    return DS_OK;
}

int launch_cluster_lat_run(ds_system *s, long long n_steps) {
    ds::ClusterLatArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.NQ = s->NQ; A.U = s->U; A.cs = s->cll_cs;
    A.buf_units = s->cll_buf_units; A.rows_max = s->cll_rows_max; A.slots_max = s->cll_slots_max;
    ds::RunArgs R;
    memset(&R, 0, sizeof R);
    fill_constants(s, R);
    A.self_mob = R.self_mob; A.pre = R.pre; A.c1 = R.c1; A.c2 = R.c2; A.c1f = R.c1f; A.c2f = R.c2f;
    A.t0 = R.t0; A.dt = R.dt; A.ell = R.ell; A.lambda = R.lambda; A.omega = R.omega; A.k0 = R.k0;
    A.noise_amp = R.noise_amp; A.seed = R.seed;
    A.n0 = s->n_host; A.n_steps = n_steps;
    A.X = s->X; A.xu = s->xu; A.from_user = s->x_valid ? 0 : 1; A.phase = s->phase;
    const bool heun = s->P.integrator == DS_HEUN, f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
#define DS_CL(TT, TEN) (heun ? launch_cluster_lat_v<TT, TEN, true>(s, A) : launch_cluster_lat_v<TT, TEN, false>(s, A))
    if (f64) DS_TRY(rpy ? DS_CL(double, ds::TENSOR_RPY) : DS_CL(double, ds::TENSOR_OSEEN));
    else DS_TRY(rpy ? DS_CL(float, ds::TENSOR_RPY) : DS_CL(float, ds::TENSOR_OSEEN));
#undef DS_CL
    s->x_valid = true; s->xu_valid = true;
    return DS_OK;
}


// RUN_VELOCITY (n_steps ignored) or RUN_STEP on the system's own state: one launch per group of
// co-resident systems; the barrier counters advance by n_cta per stage.
int launch_state_run(ds_system *s, int mode, long long n_steps, void *out_u) {
    ds::RunArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.NQ = s->NQ; A.U = s->U; A.n_cta = s->n_cta; A.buf_bytes = s->buf_bytes; A.unit_stride = s->unit_stride;
    A.units[0] = s->units[0]; A.units[1] = s->units[1]; A.cur = 0;
    fill_constants(s, A);
    A.mode = mode; A.heun = s->P.integrator == DS_HEUN ? 1 : 0;
    A.n0 = s->n_host; A.n_steps = n_steps; A.out_u = out_u;
    A.X = s->X; A.phase = s->phase; A.xu = s->xu; A.from_user = s->x_valid ? 0 : 1;
    A.bar = s->bar; A.bar_base = s->bar_base;
    // low-latency stage hand-over (tagged stream copy) whenever CTAs meet at a barrier (measured per stage: 147 CTAs -9 %,
    // 16 CTAs -10 %, 4 CTAs -15 %, 2 CTAs -1 %)
    const bool low_latency = s->n_cta > 1;
    A.ll[0] = low_latency ? s->ll[0] : nullptr; A.ll[1] = low_latency ? s->ll[1] : nullptr;
    A.h0_ll = 4;
    A.state_smem = s->state_smem; A.Xcg = s->Xcg; A.V1g = s->V1g; A.Fg = s->Fg; A.Lg = s->Lg;
    A.probe = s->probe;
    const long long n_stage = mode == ds::RUN_STEP ? n_steps * (A.heun ? 2 : 1) : 1;
    // tags ll_tag .. ll_tag + n_stage are used by this call; a tag value is never reused while it may still sit in
    // a buffer: on wrap-around of the 32-bit counter the buffers are cleared
    if ((unsigned long long)s->ll_tag + (unsigned long long)n_stage + 1ULL >= 0xffffffffULL) {
        const size_t ub = (size_t)s->B * (size_t)s->unit_stride * ds::UNIT_BYTES;
        for (int k = 0; k < 2; ++k) CU_TRY(cudaMemsetAsync(s->ll[k], 0, 2 * ub, s->stream));
        s->ll_tag = 1;
    }
    A.ll_tag0 = s->ll_tag;
    for (int b0 = 0; b0 < s->B; b0 += s->sys_per_launch) {
        const int nb = s->B - b0 < s->sys_per_launch ? s->B - b0 : s->sys_per_launch;
        A.b0 = b0;
        DS_TRY(launch_run(s, A, dim3((unsigned)s->n_cta, (unsigned)nb), s->smem_bytes, s->n_cta > 1, s->stream));
    }
    if (s->n_cta > 1) s->bar_base += (unsigned long long)s->n_cta * (unsigned long long)n_stage;
    s->ll_tag += (unsigned int)n_stage + 1u;
    if (mode == ds::RUN_STEP) { s->x_valid = true; s->xu_valid = true; }   // the kernel leaves the state in both forms
    return DS_OK;
}

int set_device(const ds_system *s) {
    CU_TRY(cudaSetDevice(s->P.device));
    return DS_OK;
}

template <typename T> int run_state_init(ds_system *s, const void *dpos) {
    ds::StateArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.user_pos = dpos; A.X = s->X;
    const long long n = (long long)s->B * s->N * 3;
    ds::state_init_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

template <typename T> int run_forces_out(ds_system *s, void *dF) {
    ds::StateArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.user_out = dF; A.X = s->X; A.phase = s->phase;
    A.t = s->t0 + (double)s->n_host * s->P.dt;
    A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
    const long long n = (long long)s->B * s->S;
    ds::forces_out_kernel<T><<<(unsigned)((n + 127) / 128), 128, 0, s->stream>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

template <typename T> int run_pad_init(ds_system *s, void *units) {
    const long long n = (long long)s->B * (s->unit_stride - s->U);
    if (n <= 0) return DS_OK;
    ds::pad_init_kernel<T><<<(unsigned)((n + 127) / 128), 128, 0, s->stream>>>(units, s->U, s->unit_stride, s->B);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

template <typename T> int peak_probe_t(int num_sms, double *flops_per_s) {
    constexpr int CHAINS = 12, THREADS = 256, ITERS = 2048;
    const int blocks = num_sms * 8;
    T *out = nullptr;
    CU_TRY(cudaMalloc((void **)&out, (size_t)blocks * THREADS * sizeof(T)));
    cudaEvent_t e0, e1;
    CU_TRY(cudaEventCreate(&e0));
    CU_TRY(cudaEventCreate(&e1));
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // rep 0 warms up
        CU_TRY(cudaEventRecord(e0, 0));
        ds::fma_chain_kernel<T, CHAINS><<<blocks, THREADS>>>(out, ITERS, (T)0.999, (T)0.001);
        CU_TRY(cudaEventRecord(e1, 0));
        CU_TRY(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    CU_TRY(cudaGetLastError());
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    const double flops = (double)blocks * THREADS * ITERS * 8.0 * CHAINS * ds::Pack<T>::W * 2.0;
    *flops_per_s = flops / (best_ms * 1e-3);
    return DS_OK;
}

bool finite_pos(double x) { return isfinite(x) && x > 0.0; }

ds::AvgConsts avg_consts(const ds_system *s) {
    const double a = s->P.a, ell = s->P.ell, lam = s->P.lambda, w = s->P.omega, ll = lam / ell;
    ds::AvgConsts C;
    C.cj = a * w * (9.0 / 64.0) * ll * ll * ell * ell * ell * ell;
    C.ck = w * (15.0 / 64.0) * (a / ell) * ll * ll * ell * ell * ell * ell * ell;
    return C;
}

// sin/cos of the phases (device pointer) into s->avg_sc
int avg_sincos(ds_system *s, const double *dphi, int S) {
    DS_TRY(ensure(s->avg_sc, (size_t)S * sizeof(double2)));
    ds::avg_sincos_kernel<<<(unsigned)((S + 127) / 128), 128, 0, s->stream>>>(dphi, S, (double2 *)s->avg_sc.p);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

// One evaluation of the right-hand sides of Eq. (9a,b).  The r sum is split into Y <= 8 chunks, one CTA of a cluster
// each (S / 32 blocks alone would leave most SMs idle at the paper's S = 729).
template <typename T, typename IO>
int launch_avg_rhs_t(ds_system *s, const IO *R, const IO *N, int S, IO *dR, IO *dN, const ds::AvgUpdate &U) {
    auto kern = ds::avg_rhs_kernel<T, IO>;
    const int X = (S + ds::AVG_SB - 1) / ds::AVG_SB, slots = 2 * s->num_sms;   // two 512-thread CTAs per SM
    int Y = std::max(1, std::min(std::min(slots / X, ds::AVG_YMAX), (S + ds::AVG_W - 1) / ds::AVG_W));
    int chunk = (S + Y - 1) / Y;
    chunk = (chunk + ds::AVG_W - 1) / ds::AVG_W * ds::AVG_W;
    Y = (S + chunk - 1) / chunk;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)X, (unsigned)Y); cfg.blockDim = dim3(ds::AVG_NT); cfg.stream = s->stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = 1; at[1].val.clusterDim.y = (unsigned)Y; at[1].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = Y > 1 ? 2 : 1;
    CU_TRY(cudaLaunchKernelEx(&cfg, kern, R, N, (const double2 *)s->avg_sc.p, S, chunk, avg_consts(s), dR, dN, U));
    s->launches += 1;
    return DS_OK;
}

// IO = double: the FP64 state of ds_avg_step; IO = the user's type: the stateless ds_avg_rhs on device buffers.
// avg_sincos() must have run on the phases first.
template <typename IO>
int launch_avg_rhs(ds_system *s, const IO *R, const IO *N, int S, IO *dR, IO *dN, const ds::AvgUpdate &U = ds::AvgUpdate{}) {
    if (s->P.precision == DS_F64) return launch_avg_rhs_t<double, IO>(s, R, N, S, dR, dN, U);
    return launch_avg_rhs_t<float, IO>(s, R, N, S, dR, dN, U);
}

// Device-resident Heun stepping of Eq. (9) (averaged.cuh, avg_persist_kernel) when the whole input of a stage fits one
// CTA's shared memory and the grid is co-resident; *used tells the caller whether it ran.
constexpr int AVG_PERSIST_MAX_S = 4096;
template <typename T>
int avg_step_persistent_t(ds_system *s, double *Rd, double *Nd, int S, double dt, long long n_steps, bool *used) {
    *used = false;
    if (S > AVG_PERSIST_MAX_S || n_steps < 1) return DS_OK;
    constexpr int W = ds::Pack<T>::W, PPR = 8 * (int)sizeof(T) / 8;
    int G = S < s->num_sms ? S : s->num_sms;
    const int ns = (S + G - 1) / G;
    G = (S + ns - 1) / ns;
    if (ns > 64) return DS_OK;
    const int nu = (S + W - 1) / W, n_sl = ds::AVG_NT / ns, n_out = 6 * ns;
    const size_t smem = (size_t)nu * 64 + (size_t)n_sl * n_out * sizeof(T) + (size_t)n_out * sizeof(double) + (size_t)ns * 20 * sizeof(double);
    if (smem > (size_t)ds::SMEM_MAX) return DS_OK;
    const size_t rec_bytes = (size_t)PPR * 16, need = 2 * (size_t)S * rec_bytes;
    const long long n_stage = 2 * n_steps;
    if (s->avg_xch.cap < need || (unsigned long long)s->avg_tag + (unsigned long long)n_stage + 2ULL >= 0xffffffffULL) {
        DS_TRY(ensure(s->avg_xch, need));
        CU_TRY(cudaMemsetAsync(s->avg_xch.p, 0, s->avg_xch.cap, s->stream));   // tag 0 = never written
        s->avg_tag = 1;
    }
    auto kern = ds::avg_persist_kernel<T>;
    static SmemOptIn opt_in;
    DS_TRY(opt_in.ensure((const void *)kern, s->P.device));
    long long left = n_steps;
    while (left > 0) {
        const long long k = left < MAX_STEPS_PER_LAUNCH ? left : MAX_STEPS_PER_LAUNCH;
        ds::AvgPersistArgs A;
        memset(&A, 0, sizeof A);
        A.S = S; A.ns = ns; A.R = Rd; A.N = Nd; A.sc = (const double2 *)s->avg_sc.p; A.C = avg_consts(s); A.dt = dt; A.n_steps = k;
        A.xch[0] = (uint4 *)s->avg_xch.p; A.xch[1] = (uint4 *)((char *)s->avg_xch.p + (size_t)S * rec_bytes);
        A.tag0 = s->avg_tag;
        A.probe = s->probe;
        void *args[] = {(void *)&A};
        CU_TRY(cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)G), dim3(ds::AVG_NT), args, smem, s->stream));
        s->launches += 1;
        s->avg_tag += (unsigned int)(2 * k) + 1u;
        left -= k;
    }
    *used = true;
    return DS_OK;
}

int avg_step_persistent(ds_system *s, double *Rd, double *Nd, int S, double dt, long long n_steps, bool *used) {
    if (s->P.precision == DS_F64) return avg_step_persistent_t<double>(s, Rd, Nd, S, dt, n_steps, used);
    return avg_step_persistent_t<float>(s, Rd, Nd, S, dt, n_steps, used);
}

// user buffer (device or host, user precision, n elements) -> FP64 device array dst
int avg_in(ds_system *s, const void *src, double *dst, size_t n, Buf &stage) {
    const size_t nb = n * elem_size(s);
    int dev = 0;
    DS_TRY(is_device_ptr(src, &dev));
    const void *d = src;
    if (!dev) { DS_TRY(ensure(stage, nb)); CU_TRY(cudaMemcpyAsync(stage.p, src, nb, cudaMemcpyHostToDevice, s->stream)); d = stage.p; }
    const unsigned g = (unsigned)((n + 255) / 256);
    if (s->P.precision == DS_F64) ds::widen_kernel<double><<<g, 256, 0, s->stream>>>((const double *)d, dst, (long long)n);
    else ds::widen_kernel<float><<<g, 256, 0, s->stream>>>((const float *)d, dst, (long long)n);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

// FP64 device array -> user buffer; returns whether the caller must synchronise (host destination)
int avg_out(ds_system *s, const double *src, void *dst, size_t n, Buf &stage, bool *host) {
    const size_t nb = n * elem_size(s);
    int dev = 0;
    DS_TRY(is_device_ptr(dst, &dev));
    void *d = dst;
    if (!dev) { DS_TRY(ensure(stage, nb)); d = stage.p; }
    const unsigned g = (unsigned)((n + 255) / 256);
    if (s->P.precision == DS_F64) ds::narrow_kernel<double><<<g, 256, 0, s->stream>>>(src, (double *)d, (long long)n);
    else ds::narrow_kernel<float><<<g, 256, 0, s->stream>>>(src, (float *)d, (long long)n);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    if (!dev) { CU_TRY(cudaMemcpyAsync(dst, d, nb, cudaMemcpyDeviceToHost, s->stream)); *host = true; }
    return DS_OK;
}

// X (FP64) <- xu (user precision) when only the latter is current (ds_set_state with a host buffer)
int materialize_x(ds_system *s) {
    if (s->x_valid) return DS_OK;
    DS_TRY(s->P.precision == DS_F64 ? run_state_init<double>(s, s->xu) : run_state_init<float>(s, s->xu));
    s->x_valid = true;
    return DS_OK;
}

}  // namespace

// =================================================================================================
// ---------------------------------------------------------------------------------------------------------------------
// ds_msd_static: Eq. (13) with no allocation.  The partial sums of msd_partial_kernel live in this file-scope array (one
// copy per GPU that loads the library, until exit).  In host code `msd_static_partials` is only a stand-in for the
// symbol, NOT a device address: the kernels get the pointer cudaGetSymbolAddress returns, looked up once per device with
// that device current.
static __device__ __align__(256) double msd_static_partials[DS_MSD_STATIC_MAX_PARTIALS];

namespace {
constexpr int MSD_STATIC_MAX_DEVICES = 64;
std::mutex msd_static_mu;
double *msd_static_ptr[MSD_STATIC_MAX_DEVICES] = {nullptr};

// device address of msd_static_partials on `device`, which must be current
int msd_static_address(int device, double **out) {
    std::lock_guard<std::mutex> lock(msd_static_mu);
    if (msd_static_ptr[device] == nullptr) {
        double *p = nullptr;
        CU_TRY(cudaGetSymbolAddress((void **)&p, msd_static_partials));
        if (p == nullptr) return DS_ERR_CUDA;
        msd_static_ptr[device] = p;
    }
    *out = msd_static_ptr[device];
    return DS_OK;
}
}  // namespace

extern "C" {

const char *ds_version(void) { return "paper_1004_1932_b200 0.1 (sm_100a)"; }

const char *ds_last_cuda_error(void) { return g_cuda_err; }

const char *ds_strerror(int code) {
    switch (code) {
        case DS_OK: return "ok";
        case DS_ERR_INVALID_PARAM: return "invalid parameter";
        case DS_ERR_NULL: return "null pointer";
        case DS_ERR_CUDA: return "CUDA runtime error";
        case DS_ERR_STATE: return "call not valid in the system's current state";
        case DS_ERR_NO_DEVICE: return "no sm_100-class CUDA device";
        case DS_ERR_ALLOC: return "allocation failed";
        case DS_ERR_TOO_LARGE: return "problem exceeds the fixed capacity of this entry point";
        default: return "unknown error";
    }
}

int ds_create(const ds_params *p, ds_system **out) {
    if (!p || !out) return DS_ERR_NULL;
    *out = nullptr;
    if (p->n_dumbbells < 1 || p->n_batch < 1) return DS_ERR_INVALID_PARAM;
    if ((long long)p->n_dumbbells * 2 > (1LL << 30)) return DS_ERR_INVALID_PARAM;
    if (p->precision != DS_F32 && p->precision != DS_F64) return DS_ERR_INVALID_PARAM;
    if (p->tensor != DS_OSEEN && p->tensor != DS_RPY) return DS_ERR_INVALID_PARAM;
    if (p->integrator != DS_EULER && p->integrator != DS_HEUN) return DS_ERR_INVALID_PARAM;
    if (!finite_pos(p->a) || !finite_pos(p->eta) || !finite_pos(p->k0) || !finite_pos(p->dt) || !finite_pos(p->ell))
        return DS_ERR_INVALID_PARAM;
    if (!isfinite(p->lambda) || !isfinite(p->omega) || p->omega < 0.0) return DS_ERR_INVALID_PARAM;
    if (!(p->ell > 2.0 * p->a + fabs(p->lambda))) return DS_ERR_INVALID_PARAM;
    if (p->n_batch > 65535) return DS_ERR_INVALID_PARAM;
    if (!isfinite(p->kT) || p->kT < 0.0) return DS_ERR_INVALID_PARAM;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return DS_ERR_NO_DEVICE; }
    if (p->device < 0 || p->device >= ndev) return DS_ERR_INVALID_PARAM;
    cudaDeviceProp prop;
    CU_TRY(cudaGetDeviceProperties(&prop, p->device));
    if (prop.major != 10) return DS_ERR_NO_DEVICE;  // the kernels are sm_100a SASS only

    ds_system *s = new (std::nothrow) ds_system();
    if (!s) return DS_ERR_ALLOC;
    s->P = *p;
    s->stream = (cudaStream_t)p->stream;
    s->num_sms = prop.multiProcessorCount;
    s->S = p->n_dumbbells; s->N = 2 * p->n_dumbbells; s->B = p->n_batch;
    const bool f64 = p->precision == DS_F64;
    s->W = f64 ? pack_w<double>() : pack_w<float>();
    s->NQ = (s->N + ds::QI - 1) / ds::QI;
    s->U = (s->N + s->W - 1) / s->W;
    s->unit_stride = (long long)s->U + ds::PAD_UNITS;
    int rc = DS_OK;
    auto fail = [&](int code) { ds_destroy(s); return code; };
    if (set_device(s) != DS_OK) return fail(DS_ERR_CUDA);
    rc = choose_shape_step(s);   // N too large for one co-resident grid: the step modes cannot run
    if (rc != DS_OK) return fail(rc);
    rc = setup_pipe(s);
    if (rc == DS_OK) rc = setup_cluster(s);
    if (rc == DS_OK) rc = setup_cluster_lat(s);
    if (rc != DS_OK) return fail(rc);
    const size_t n3 = (size_t)s->B * s->N * 3;
    const size_t ub = (size_t)s->B * (size_t)s->unit_stride * ds::UNIT_BYTES;
    cudaError_t e = cudaSuccess;
    auto al = [&](void **ptr, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(ptr, bytes); };
    al((void **)&s->X, n3 * 8);
    al(&s->xu, n3 * (f64 ? 8 : 4));
    al((void **)&s->phase, (size_t)s->B * s->S * 8);
    al(&s->units[0], ub); al(&s->units[1], ub);
    al(&s->ll[0], 2 * ub); al(&s->ll[1], 2 * ub);
    al((void **)&s->bar, (size_t)s->B * sizeof(unsigned long long));
    al((void **)&s->pcnt, 2 * (size_t)s->B * sizeof(unsigned long long));
    // global homes of the per-row state, used only by tiles too large for shared memory (any tuning)
    al((void **)&s->Xcg, n3 * 8); al((void **)&s->V1g, n3 * 8); al((void **)&s->Fg, n3 * 8);
    al((void **)&s->Lg, (size_t)s->B * s->S * 8);
    if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof g_cuda_err, "cudaMalloc -> %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return fail(DS_ERR_ALLOC); }
    if (cudaMemsetAsync(s->bar, 0, (size_t)s->B * sizeof(unsigned long long), s->stream) != cudaSuccess) return fail(DS_ERR_CUDA);
    if (cudaMemsetAsync(s->pcnt, 0, 2 * (size_t)s->B * sizeof(unsigned long long), s->stream) != cudaSuccess) return fail(DS_ERR_CUDA);
    for (int k = 0; k < 2; ++k)
        if (cudaMemsetAsync(s->ll[k], 0, 2 * ub, s->stream) != cudaSuccess) return fail(DS_ERR_CUDA);
    for (int k = 0; k < 2 && rc == DS_OK; ++k) rc = f64 ? run_pad_init<double>(s, s->units[k]) : run_pad_init<float>(s, s->units[k]);
    if (rc != DS_OK) return fail(rc);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return fail(DS_ERR_CUDA);
    *out = s;
    return DS_OK;
}

int ds_destroy(ds_system *s) {
    if (!s) return DS_OK;
    cudaSetDevice(s->P.device);
    cudaStreamSynchronize(s->stream);
    void *ptrs[] = {s->X, s->xu, s->Rref, s->msd_part, s->msd_out, s->phase, s->units[0], s->units[1], s->ll[0], s->ll[1], s->bar, s->pcnt, s->half_off, s->ptab_g, s->Xcg, s->V1g, s->Fg, s->Lg,
                    s->ap_units.p, s->st_a.p, s->st_b.p, s->st_c.p, s->avg.p, s->avg_sc.p, s->avg_xch.p};
    for (void *q : ptrs) if (q) cudaFree(q);
    (void)cudaGetLastError();
    delete s;
    return DS_OK;
}

int ds_set_stream(ds_system *s, void *stream) {
    if (!s) return DS_ERR_NULL;
    DS_TRY(set_device(s));
    // work still queued on the old stream touches the system's buffers: the new stream waits for it.  While the old
    // stream is being captured an event cannot order against it; the caller owns the ordering then.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s->stream, &cap) != cudaSuccess) { (void)cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
    if (cap == cudaStreamCaptureStatusNone && (cudaStream_t)stream != s->stream) {
        cudaEvent_t ev;
        CU_TRY(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        CU_TRY(cudaEventRecord(ev, s->stream));
        CU_TRY(cudaStreamWaitEvent((cudaStream_t)stream, ev, 0));
        CU_TRY(cudaEventDestroy(ev));
    }
    s->stream = (cudaStream_t)stream;
    return DS_OK;
}

int ds_set_tuning(ds_system *s, int32_t n_tiles) {
    if (!s) return DS_ERR_NULL;
    if (n_tiles < 0) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    CU_TRY(cudaStreamSynchronize(s->stream));
    s->tune_cta = n_tiles;
    DS_TRY(choose_shape_step(s));
    DS_TRY(setup_pipe(s));
    DS_TRY(setup_cluster(s));
    return setup_cluster_lat(s);
}

int ds_set_pipeline(ds_system *s, int32_t mode) {
    if (!s) return DS_ERR_NULL;
    if (mode < -1 || mode > 3) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    CU_TRY(cudaStreamSynchronize(s->stream));
    s->pipe_mode = mode;
    DS_TRY(setup_pipe(s));
    DS_TRY(setup_cluster(s));
    return setup_cluster_lat(s);
}

int ds_pipeline_active(const ds_system *s) { return !s ? 0 : (s->cl_cs > 0 ? 2 : (s->cll_cs > 0 ? 3 : (s->use_pipe ? 1 : 0))); }

int ds_set_probe(ds_system *s, void *device_buffer) {
    if (!s) return DS_ERR_NULL;
    s->probe = (long long *)device_buffer;
    return DS_OK;
}

int64_t ds_launch_count(const ds_system *s) { return s ? s->launches : 0; }

int ds_set_state(ds_system *s, const void *pos, const void *phase, double t0) {
    if (!s || !pos || !phase) return DS_ERR_NULL;
    if (!isfinite(t0)) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    const size_t es = elem_size(s), nb = (size_t)s->B * s->N * 3 * es, pb = (size_t)s->B * s->S * 8;
    int dev = 0;
    DS_TRY(is_device_ptr(phase, &dev));
    CU_TRY(cudaMemcpyAsync(s->phase, phase, pb, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream));
    DS_TRY(is_device_ptr(pos, &dev));
    s->t0 = t0;
    s->n_host = 0;
    if (!dev) {
        // host buffer: one copy into the user-precision image; the next kernel widens it to FP64 itself
        CU_TRY(cudaMemcpyAsync(s->xu, pos, nb, cudaMemcpyHostToDevice, s->stream));
        s->xu_valid = true; s->x_valid = false;
    } else {
        DS_TRY(s->P.precision == DS_F64 ? run_state_init<double>(s, pos) : run_state_init<float>(s, pos));
        s->x_valid = true; s->xu_valid = false;
    }
    s->has_state = true;
    return DS_OK;
}

int ds_get_state(ds_system *s, void *pos, double *t) {
    if (!s) return DS_ERR_NULL;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    if (t) *t = s->t0 + (double)s->n_host * s->P.dt;
    if (!pos) return DS_OK;
    const size_t es = elem_size(s), nb = (size_t)s->B * s->N * 3 * es;
    int dev = 0;
    DS_TRY(is_device_ptr(pos, &dev));
    if (!s->xu_valid) {   // user-precision image of X
        const long long n3 = (long long)s->B * s->N * 3;
        if (s->P.precision == DS_F64)
            ds::state_out_kernel<double><<<(unsigned)((n3 + 255) / 256), 256, 0, s->stream>>>(s->X, s->xu, n3);
        else
            ds::state_out_kernel<float><<<(unsigned)((n3 + 255) / 256), 256, 0, s->stream>>>(s->X, s->xu, n3);
        CU_TRY(cudaGetLastError());
        s->launches += 1;
        s->xu_valid = true;
    }
    CU_TRY(cudaMemcpyAsync(pos, s->xu, nb, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->stream));
    if (!dev) CU_TRY(cudaStreamSynchronize(s->stream));
    return DS_OK;
}

int ds_forces(ds_system *s, void *F) {
    if (!s || !F) return DS_ERR_NULL;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    const size_t nb = (size_t)s->B * s->N * 3 * elem_size(s);
    int dev = 0;
    DS_TRY(is_device_ptr(F, &dev));
    void *dF = F;
    if (!dev) { DS_TRY(ensure(s->st_c, nb)); dF = s->st_c.p; }
    DS_TRY(materialize_x(s));
    DS_TRY(s->P.precision == DS_F64 ? run_forces_out<double>(s, dF) : run_forces_out<float>(s, dF));
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(F, dF, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
    return DS_OK;
}

int ds_dumbbell_coords(ds_system *s, void *R, void *Nv) {
    if (!s) return DS_ERR_NULL;
    if (!R && !Nv) return DS_ERR_NULL;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    DS_TRY(materialize_x(s));
    const long long n_db = (long long)s->B * s->S;
    const size_t nb = (size_t)n_db * 3 * elem_size(s);
    int rdev = 1, ndev = 1;
    if (R) DS_TRY(is_device_ptr(R, &rdev));
    if (Nv) DS_TRY(is_device_ptr(Nv, &ndev));
    void *dR = R, *dN = Nv;
    if (R && !rdev) { DS_TRY(ensure(s->st_b, nb)); dR = s->st_b.p; }
    if (Nv && !ndev) { DS_TRY(ensure(s->st_c, nb)); dN = s->st_c.p; }
    const unsigned grid = (unsigned)((n_db + 127) / 128);
    if (s->P.precision == DS_F64)
        ds::coords_kernel<double><<<grid, 128, 0, s->stream>>>(s->X, n_db, (double *)dR, (double *)dN, nullptr);
    else
        ds::coords_kernel<float><<<grid, 128, 0, s->stream>>>(s->X, n_db, (float *)dR, (float *)dN, nullptr);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    if (R && !rdev) CU_TRY(cudaMemcpyAsync(R, dR, nb, cudaMemcpyDeviceToHost, s->stream));
    if (Nv && !ndev) CU_TRY(cudaMemcpyAsync(Nv, dN, nb, cudaMemcpyDeviceToHost, s->stream));
    if ((R && !rdev) || (Nv && !ndev)) CU_TRY(cudaStreamSynchronize(s->stream));
    return DS_OK;
}

int ds_msd_set_reference(ds_system *s) {
    if (!s) return DS_ERR_NULL;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    DS_TRY(materialize_x(s));
    const long long n_db = (long long)s->B * s->S;
    if (!s->Rref) {
        const int n_chunk = (s->S + 255) / 256;
        CU_TRY(cudaMalloc((void **)&s->Rref, (size_t)n_db * 3 * sizeof(double)));
        CU_TRY(cudaMalloc((void **)&s->msd_part, (size_t)s->B * n_chunk * sizeof(double)));
        CU_TRY(cudaMalloc((void **)&s->msd_out, sizeof(double)));
    }
    ds::coords_kernel<double><<<(unsigned)((n_db + 127) / 128), 128, 0, s->stream>>>(s->X, n_db, nullptr, nullptr, s->Rref);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    s->has_ref = true;
    return DS_OK;
}

int ds_msd(ds_system *s, double *msd) {
    if (!s || !msd) return DS_ERR_NULL;
    if (!s->has_state || !s->has_ref) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    DS_TRY(materialize_x(s));
    int dev = 0;
    DS_TRY(is_device_ptr(msd, &dev));
    const int n_chunk = (s->S + 255) / 256;
    ds::msd_partial_kernel<<<dim3((unsigned)n_chunk, (unsigned)s->B), 256, 0, s->stream>>>(s->X, s->Rref, s->S, s->msd_part);
    CU_TRY(cudaGetLastError());
    ds::msd_final_kernel<<<1, 256, 0, s->stream>>>(s->msd_part, s->B, s->S, n_chunk, dev ? msd : s->msd_out);
    CU_TRY(cudaGetLastError());
    s->launches += 2;
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(msd, s->msd_out, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
    return DS_OK;
}

int ds_avg_rhs(ds_system *s, const void *R, const void *Nv, const void *phase, void *dR, void *dN, int32_t S) {
    if (!s || !R || !Nv || !phase || !dR || !dN) return DS_ERR_NULL;
    if (S < 1) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    const size_t M = 3 * (size_t)S, nb = M * elem_size(s);
    // host buffers are staged through device scratch in the user's precision; device buffers are used in place
    int dv[5];
    const void *in[3] = {R, Nv, phase};
    void *outp[2] = {dR, dN};
    for (int k = 0; k < 3; ++k) DS_TRY(is_device_ptr(in[k], &dv[k]));
    for (int k = 0; k < 2; ++k) DS_TRY(is_device_ptr(outp[k], &dv[3 + k]));
    DS_TRY(ensure(s->avg, 4 * nb + (size_t)S * sizeof(double) + 64));
    char *scr = (char *)s->avg.p;
    const void *dRin = R, *dNin = Nv;
    const double *dph = (const double *)phase;
    void *dRo = dR, *dNo = dN;
    if (!dv[0]) { CU_TRY(cudaMemcpyAsync(scr, R, nb, cudaMemcpyHostToDevice, s->stream)); dRin = scr; }
    if (!dv[1]) { CU_TRY(cudaMemcpyAsync(scr + nb, Nv, nb, cudaMemcpyHostToDevice, s->stream)); dNin = scr + nb; }
    if (!dv[2]) {
        double *p = (double *)(scr + 4 * nb + ((8 - (4 * nb) % 8) % 8));
        CU_TRY(cudaMemcpyAsync(p, phase, (size_t)S * sizeof(double), cudaMemcpyHostToDevice, s->stream));
        dph = p;
    }
    if (!dv[3]) dRo = scr + 2 * nb;
    if (!dv[4]) dNo = scr + 3 * nb;
    DS_TRY(avg_sincos(s, dph, S));
    if (s->P.precision == DS_F64)
        DS_TRY(launch_avg_rhs<double>(s, (const double *)dRin, (const double *)dNin, S, (double *)dRo, (double *)dNo));
    else
        DS_TRY(launch_avg_rhs<float>(s, (const float *)dRin, (const float *)dNin, S, (float *)dRo, (float *)dNo));
    if (!dv[3]) CU_TRY(cudaMemcpyAsync(dR, dRo, nb, cudaMemcpyDeviceToHost, s->stream));
    if (!dv[4]) CU_TRY(cudaMemcpyAsync(dN, dNo, nb, cudaMemcpyDeviceToHost, s->stream));
    if (!dv[3] || !dv[4]) CU_TRY(cudaStreamSynchronize(s->stream));
    return DS_OK;
}

int ds_avg_step(ds_system *s, void *R, void *Nv, const void *phase, int32_t S, double dt, int64_t n_steps) {
    if (!s || !R || !Nv || !phase) return DS_ERR_NULL;
    if (S < 1 || n_steps < 0 || !isfinite(dt) || dt <= 0.0) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    const size_t M = 3 * (size_t)S;
    DS_TRY(ensure(s->avg, (6 * M + (size_t)S) * sizeof(double)));
    double *Rd = (double *)s->avg.p, *Nd = Rd + M, *Rp = Nd + M, *Np = Rp + M, *dR1 = Np + M, *dN1 = dR1 + M, *phd = dN1 + M;
    int pdev = 0;
    DS_TRY(is_device_ptr(phase, &pdev));
    CU_TRY(cudaMemcpyAsync(phd, phase, (size_t)S * sizeof(double), pdev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream));
    DS_TRY(avg_sincos(s, phd, S));
    DS_TRY(avg_in(s, R, Rd, M, s->st_a));
    DS_TRY(avg_in(s, Nv, Nd, M, s->st_b));
    // Heun.  Sizes of the paper (S up to a few thousand): one cooperative launch runs all steps on the device
    // (avg_persist_kernel).  Larger S: two launches per step, the update of a block of dumbbells done by the CTA that
    // completes its right-hand sides (avg_rhs_kernel).
    bool persistent = false;
    DS_TRY(avg_step_persistent(s, Rd, Nd, S, dt, n_steps, &persistent));
    if (!persistent) {
        ds::AvgUpdate P1{ds::AVG_PRED, dt, Rd, Nd, dR1, dN1, Rp, Np}, P2{ds::AVG_CORR, dt, Rd, Nd, dR1, dN1, Rd, Nd};
        for (int64_t n = 0; n < n_steps; ++n) {
            DS_TRY(launch_avg_rhs<double>(s, Rd, Nd, S, (double *)nullptr, (double *)nullptr, P1));
            DS_TRY(launch_avg_rhs<double>(s, Rp, Np, S, (double *)nullptr, (double *)nullptr, P2));
        }
    }
    bool host = false;
    DS_TRY(avg_out(s, Rd, R, M, s->st_a, &host));
    DS_TRY(avg_out(s, Nd, Nv, M, s->st_b, &host));
    if (host) CU_TRY(cudaStreamSynchronize(s->stream));
    return DS_OK;
}

int ds_velocity(ds_system *s, void *V) {
    if (!s || !V) return DS_ERR_NULL;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    const size_t nb = (size_t)s->B * s->N * 3 * elem_size(s);
    int dev = 0;
    DS_TRY(is_device_ptr(V, &dev));
    void *dV = V;
    if (!dev) { DS_TRY(ensure(s->st_c, nb)); dV = s->st_c.p; }
    DS_TRY(launch_state_run(s, ds::RUN_VELOCITY, 0, dV));
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(V, dV, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
    return DS_OK;
}

int ds_mobility_apply(ds_system *s, const void *pos, const void *F, void *u, int32_t n) {
    if (!s || !pos || !F || !u) return DS_ERR_NULL;
    if (n < 1 || n > DS_MAX_APPLY_N) return DS_ERR_INVALID_PARAM;   // the kernel's piece arithmetic is 32-bit
    DS_TRY(set_device(s));
    const bool f64 = s->P.precision == DS_F64;
    const size_t nb = (size_t)n * 3 * elem_size(s);
    int dpos_dev = 0, dF_dev = 0, du_dev = 0;
    DS_TRY(is_device_ptr(pos, &dpos_dev));
    DS_TRY(is_device_ptr(F, &dF_dev));
    DS_TRY(is_device_ptr(u, &du_dev));
    const void *dpos = pos, *dF = F;
    void *du = u;
    if (!dpos_dev) { DS_TRY(ensure(s->st_a, nb)); CU_TRY(cudaMemcpyAsync(s->st_a.p, pos, nb, cudaMemcpyHostToDevice, s->stream)); dpos = s->st_a.p; }
    if (!dF_dev) { DS_TRY(ensure(s->st_b, nb)); CU_TRY(cudaMemcpyAsync(s->st_b.p, F, nb, cudaMemcpyHostToDevice, s->stream)); dF = s->st_b.p; }
    if (!du_dev) { DS_TRY(ensure(s->st_c, nb)); du = s->st_c.p; }

    // the mobility kernel in RUN_APPLY mode.  A stream that fits one CTA's shared memory is packed by every CTA
    // for itself, straight from the user's arrays; a larger one goes through the pack kernel and a global stream.
    const int U = (n + s->W - 1) / s->W;
    ds::RunArgs A;
    memset(&A, 0, sizeof A);
    A.N = n; A.NQ = (n + ds::QI - 1) / ds::QI; A.U = U;
    A.n_cta = choose_tiles_apply(s, A.NQ, A.U);
    A.buf_bytes = (ds::SMEM_MAX - ds::BAR_BYTES) / 128 * 128;
    fill_constants(s, A);
    A.mode = ds::RUN_APPLY;
    A.out_u = du;
    A.probe = s->probe;
    const bool aligned = (((uintptr_t)dpos | (uintptr_t)dF) & 7u) == 0;   // the in-kernel pack reads 8-byte pairs
    bool warp_shape = false;
    if (aligned && (s->tune_cta == 0 || s->pipe_mode == 1)) DS_TRY(apply_warp_shape(s, A, dpos, dF, du, &warp_shape));
    if (warp_shape) {
        // done: apply_kernel packed the user's arrays itself
    } else if (aligned && stream_resident(A.NQ, A.U, A.n_cta, A.buf_bytes)) {
        A.raw_pos = dpos; A.raw_F = dF;
        A.unit_stride = (long long)U + ds::PAD_UNITS;
    } else {
        const long long n_units = (long long)U + ds::PAD_UNITS;
        DS_TRY(ensure(s->ap_units, (size_t)n_units * ds::UNIT_BYTES));
        const unsigned pg = (unsigned)((n_units + 255) / 256);
        if (f64)
            ds::pack_user_kernel<double><<<pg, 256, 0, s->stream>>>((const double *)dpos, (const double *)dF, (double *)s->ap_units.p, n, n_units);
        else
            ds::pack_user_kernel<float><<<pg, 256, 0, s->stream>>>((const float *)dpos, (const float *)dF, (float *)s->ap_units.p, n, n_units);
        CU_TRY(cudaGetLastError());
        s->launches += 1;
        A.unit_stride = n_units;
        A.units[0] = s->ap_units.p; A.units[1] = s->ap_units.p;
    }
    if (!warp_shape) DS_TRY(launch_run(s, A, dim3((unsigned)A.n_cta, 1), (size_t)A.buf_bytes + ds::BAR_BYTES, false, s->stream));
    if (!du_dev) {
        CU_TRY(cudaMemcpyAsync(u, du, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
    return DS_OK;
}

int ds_batch_step(ds_system *s, int64_t n_steps) {
    if (!s) return DS_ERR_NULL;
    if (n_steps < 0) return DS_ERR_INVALID_PARAM;
    if (!s->has_state) return DS_ERR_STATE;
    DS_TRY(set_device(s));
    int64_t left = n_steps;
    while (left > 0) {   // one launch runs up to MAX_STEPS_PER_LAUNCH steps entirely on the device
        const long long k = left < MAX_STEPS_PER_LAUNCH ? left : MAX_STEPS_PER_LAUNCH;
        // small systems: a warp per system; a forced tiling (ds_set_tuning) keeps them on run_kernel (tests)
        if (s->cl_cs > 0 && s->pipe_mode == 2) DS_TRY(launch_cluster_run(s, k));
        else if (s->cll_cs > 0) DS_TRY(launch_cluster_lat_run(s, k));
        else if (use_small_kernel(s)) DS_TRY(launch_small_run(s, k));
        else if (s->cl_cs > 0) DS_TRY(launch_cluster_run(s, k));
        else DS_TRY(s->use_pipe ? launch_pipe_run(s, k) : launch_state_run(s, ds::RUN_STEP, k, nullptr));
        s->n_host += k; left -= k;
    }
    return DS_OK;
}

int ds_peak_probe(int32_t precision, int32_t device, double *flops_per_s) {
    if (!flops_per_s) return DS_ERR_NULL;
    if (precision != DS_F32 && precision != DS_F64) return DS_ERR_INVALID_PARAM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return DS_ERR_NO_DEVICE; }
    if (device < 0 || device >= ndev) return DS_ERR_INVALID_PARAM;
    cudaDeviceProp prop;
    CU_TRY(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return DS_ERR_NO_DEVICE;
    CU_TRY(cudaSetDevice(device));
    return precision == DS_F64 ? peak_probe_t<double>(prop.multiProcessorCount, flops_per_s)
                               : peak_probe_t<float>(prop.multiProcessorCount, flops_per_s);
}

int ds_step(ds_system *s, int64_t n_steps) {
    if (!s) return DS_ERR_NULL;
    if (s->B != 1) return DS_ERR_STATE;
    return ds_batch_step(s, n_steps);
}

int ds_msd_static(const double *X, const double *Rref, int32_t S, int32_t W, double *msd, void *stream, int32_t device) {
    if (!X || !Rref || !msd) return DS_ERR_NULL;
    if (S < 1 || W < 1) return DS_ERR_INVALID_PARAM;
    const long long n_chunk = ((long long)S + 255) / 256;
    if ((long long)W * n_chunk > DS_MSD_STATIC_MAX_PARTIALS || W > 65535) return DS_ERR_TOO_LARGE;   // W is also a grid y extent
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return DS_ERR_NO_DEVICE; }
    if (device < 0 || device >= ndev || device >= MSD_STATIC_MAX_DEVICES) return DS_ERR_INVALID_PARAM;
    CU_TRY(cudaSetDevice(device));
    double *partial = nullptr;
    DS_TRY(msd_static_address(device, &partial));
    cudaStream_t st = (cudaStream_t)stream;
    // every partial the second kernel reads is written by the first: nothing in the shared array has to start at zero
    ds::msd_partial_kernel<<<dim3((unsigned)n_chunk, (unsigned)W), 256, 0, st>>>(X, Rref, S, partial);
    CU_TRY(cudaGetLastError());
    ds::msd_final_kernel<<<1, 256, 0, st>>>(partial, W, S, (int)n_chunk, msd);
    CU_TRY(cudaGetLastError());
    return DS_OK;
}

}  // extern "C"
