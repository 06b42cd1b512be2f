// ds_api.cu -- host runtime behind the C ABI of include/ds.h: parameter validation, device
// buffers, host/device pointer staging, launch-shape choice, CUDA-graph build and replay.
// No arithmetic of the method lives here; it is all in mobility.cuh / state.cuh.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "../../include/ds.h"
#include "mobility.cuh"
#include "peak.cuh"
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

// ---- kernel shape (compile-time) -------------------------------------------------------------
// FP32: 4 alpha per lane x 2 beta per pack; FP64: 2 alpha per lane.  See DESIGN.md "Kernels".
struct ShapeF32 { static constexpr int I = 4, WI = 2, WJ = 4, SJ = 1024, UNROLL = 2, MINB = 2; };
struct ShapeF64 { static constexpr int I = 2, WI = 4, WJ = 2, SJ = 1024, UNROLL = 2, MINB = 2; };
template <typename T> struct ShapeOf;
template <> struct ShapeOf<float> { typedef ShapeF32 S; };
template <> struct ShapeOf<double> { typedef ShapeF64 S; };

template <typename T> constexpr int tile_i() { return 32 * ShapeOf<T>::S::I * ShapeOf<T>::S::WI; }
template <typename T> constexpr int group_j() { return ds::Pack<T>::W * ShapeOf<T>::S::WJ; }
template <typename T> constexpr size_t smem_bytes() {
    typedef typename ShapeOf<T>::S S;
    return ds::stage_bytes_for<T>(S::SJ) + (size_t)S::WJ * 3 * tile_i<T>() * sizeof(double) +
           (size_t)2 * 3 * tile_i<T>() * sizeof(double);
}

struct Buf {
    void *p = nullptr;
    size_t cap = 0;
};

}  // namespace

struct ds_system {
    ds_params P;
    cudaStream_t stream = nullptr;
    cudaStream_t cap_stream = nullptr;
    int num_sms = 148;
    int N = 0, B = 0, S = 0, Npad = 0, n_it = 0;
    int tune_js = 0;
    bool has_state = false;
    double t0 = 0.0;
    long long n_host = 0;  // mirror of the device step counter
    int64_t launches = 0;
    // state
    double *X = nullptr, *V1 = nullptr, *FdA = nullptr, *FdB = nullptr, *phase = nullptr;
    void *pos4A = nullptr, *F4A = nullptr, *pos4B = nullptr, *F4B = nullptr;
    double *partial = nullptr;
    unsigned *counters = nullptr;
    long long *stepc = nullptr;  // c[0], c[1]
    int JS = 1, jchunk = 0;
    // graphs
    cudaGraphExec_t graphK = nullptr;  // GRAPH_STEPS steps
    int graph_steps = 0;
    int graph_nodes = 0;
    // scratch of the stateless apply and of host-pointer staging
    Buf ap_partial, ap_counters, st_a, st_b, st_c;
    int ap_counters_n = 0;
};

namespace {

constexpr int GRAPH_STEPS = 32;

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

// Launch shape: JS j-splits of jchunk spheres so that B*n_it*JS blocks fill the SMs in whole waves.
void choose_split(const ds_system *s, int N, int B, int n_it, int gj, int resident_per_sm, int *JS, int *jchunk) {
    const int slots = s->num_sms * resident_per_sm;
    const long long tiles = (long long)B * n_it;
    const int min_chunk = 16 * gj;  // at least 16 inner iterations per j-warp-group
    int js_max = (N + min_chunk - 1) / min_chunk;
    if (js_max < 1) js_max = 1;
    int best = 1;
    if (s->tune_js > 0) {
        best = s->tune_js < js_max ? s->tune_js : js_max;
    } else {
        double best_cost = 1e300;
        for (int js = 1; js <= js_max && js <= 4096; ++js) {
            const int ch = ((N + js - 1) / js + gj - 1) / gj * gj;
            const int js_eff = (N + ch - 1) / ch;
            const long long ctas = tiles * js_eff;
            const long long waves = (ctas + slots - 1) / slots;
            // time ~ waves * (chunk + fixed per-block overhead expressed in j-iterations)
            const double cost = (double)waves * ((double)ch + 48.0) + 0.02 * js_eff;
            if (cost < best_cost) { best_cost = cost; best = js_eff; }
        }
    }
    int ch = ((N + best - 1) / best + gj - 1) / gj * gj;
    *jchunk = ch;
    *JS = (N + ch - 1) / ch;
}

template <typename T, int TENSOR, bool USER> int launch_mob_t(ds_system *s, const ds::MobArgs &A, cudaStream_t st) {
    typedef typename ShapeOf<T>::S S;
    auto kern = ds::mobility_kernel<T, TENSOR, USER, S::I, S::WI, S::WJ, S::SJ, S::UNROLL, S::MINB>;
    static bool attr_done = false;
    if (!attr_done) {
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<T>()));
        attr_done = true;
    }
    dim3 grid((unsigned)A.JS, (unsigned)A.n_it, (unsigned)A.B), block(32 * S::WI * S::WJ);
    kern<<<grid, block, smem_bytes<T>(), st>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

int launch_mob(ds_system *s, const ds::MobArgs &A, bool user, cudaStream_t st) {
    const bool f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
    if (f64) {
        if (rpy) return user ? launch_mob_t<double, ds::TENSOR_RPY, true>(s, A, st) : launch_mob_t<double, ds::TENSOR_RPY, false>(s, A, st);
        return user ? launch_mob_t<double, ds::TENSOR_OSEEN, true>(s, A, st) : launch_mob_t<double, ds::TENSOR_OSEEN, false>(s, A, st);
    }
    if (rpy) return user ? launch_mob_t<float, ds::TENSOR_RPY, true>(s, A, st) : launch_mob_t<float, ds::TENSOR_RPY, false>(s, A, st);
    return user ? launch_mob_t<float, ds::TENSOR_OSEEN, true>(s, A, st) : launch_mob_t<float, ds::TENSOR_OSEEN, false>(s, A, st);
}

void fill_constants(const ds_system *s, ds::MobArgs &A) {
    const double pi = 3.14159265358979323846264338327950288;
    A.self_mob = 1.0 / (6.0 * pi * s->P.eta * s->P.a);
    A.pre = 1.0 / (8.0 * pi * s->P.eta);
    A.c1 = 2.0 * s->P.a * s->P.a / 3.0;
    A.c2 = 2.0 * s->P.a * s->P.a;
    A.t0 = s->t0; A.dt = s->P.dt; A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
}

// One stage of the integrator on the system's own state.  set 0: (pos4A,F4A,FdA) -> writes set B
// (predictor) ; set 1: reads B, writes A (corrector).  Euler reads A and writes A... see below.
int launch_state_stage(ds_system *s, int mode, int cr, int cw, long long inc, cudaStream_t st) {
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.Npad = s->Npad; A.n_it = s->n_it; A.JS = s->JS; A.jchunk = s->jchunk;
    A.partial = s->partial; A.counters = s->counters;
    fill_constants(s, A);
    A.mode = mode;
    A.X = s->X; A.V1 = s->V1; A.phase = s->phase;
    A.n_read = s->stepc + cr; A.n_write = s->stepc + cw; A.n_inc = inc;
    const bool fromB = (mode == ds::EPI_CORR);
    A.src_pos = fromB ? s->pos4B : s->pos4A;
    A.src_F = fromB ? s->F4B : s->F4A;
    A.Fd_in = fromB ? s->FdB : s->FdA;
    const bool toB = (mode == ds::EPI_PRED);
    A.pos4_out = toB ? s->pos4B : s->pos4A;
    A.F4_out = toB ? s->F4B : s->F4A;
    A.Fd_out = toB ? s->FdB : s->FdA;
    return launch_mob(s, A, false, st);
}

// One full step.  Heun: PRED (reads c[0], writes c[1] = n) then CORR (reads c[1], writes c[0] = n+1).
// Euler: in place on set A is NOT safe (other blocks still read pos4A), so Euler ping-pongs the
// packed sets: even steps read A write B, odd steps read B write A; the counters ping-pong too.
int launch_one_step(ds_system *s, long long n_index, cudaStream_t st) {
    if (s->P.integrator == DS_HEUN) {
        DS_TRY(launch_state_stage(s, ds::EPI_PRED, 0, 1, 0, st));
        return launch_state_stage(s, ds::EPI_CORR, 1, 0, 1, st);
    }
    const int par = (int)(n_index & 1);
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.Npad = s->Npad; A.n_it = s->n_it; A.JS = s->JS; A.jchunk = s->jchunk;
    A.partial = s->partial; A.counters = s->counters;
    fill_constants(s, A);
    A.mode = ds::EPI_EULER;
    A.X = s->X; A.V1 = s->V1; A.phase = s->phase;
    A.n_read = s->stepc + par; A.n_write = s->stepc + (par ^ 1); A.n_inc = 1;
    A.src_pos = par ? s->pos4B : s->pos4A; A.src_F = par ? s->F4B : s->F4A; A.Fd_in = par ? s->FdB : s->FdA;
    A.pos4_out = par ? s->pos4A : s->pos4B; A.F4_out = par ? s->F4A : s->F4B; A.Fd_out = par ? s->FdA : s->FdB;
    return launch_mob(s, A, false, st);
}

void destroy_graphs(ds_system *s) {
    if (s->graphK) { cudaGraphExecDestroy(s->graphK); s->graphK = nullptr; }
    s->graph_steps = 0;
}

int build_graph(ds_system *s) {
    destroy_graphs(s);
    cudaGraph_t g = nullptr;
    const int64_t before = s->launches;
    CU_TRY(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = DS_OK;
    for (int k = 0; k < GRAPH_STEPS && rc == DS_OK; ++k) rc = launch_one_step(s, k, s->cap_stream);  // parity 0 start
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &g);
    s->graph_nodes = (int)(s->launches - before);
    s->launches = before;
    if (rc != DS_OK) { if (g) cudaGraphDestroy(g); return rc; }
    CU_TRY(e);
    e = cudaGraphInstantiate(&s->graphK, g, 0);
    cudaGraphDestroy(g);
    CU_TRY(e);
    s->graph_steps = GRAPH_STEPS;
    return DS_OK;
}

int set_device(const ds_system *s) {
    CU_TRY(cudaSetDevice(s->P.device));
    return DS_OK;
}

template <typename T> int run_state_init(ds_system *s, const void *dpos) {
    ds::StateArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.Npad = s->Npad; A.user_pos = dpos; A.X = s->X; A.pos4 = s->pos4A; A.F4 = s->F4A;
    A.Fd = s->FdA; A.phase = s->phase; A.counters = s->stepc; A.t = s->t0;
    A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
    const long long n = (long long)s->B * s->S;
    ds::state_init_kernel<T><<<(unsigned)((n + 127) / 128), 128, 0, s->stream>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

template <typename T> int run_forces_out(ds_system *s, void *dF) {
    ds::StateArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.Npad = s->Npad; A.user_out = dF; A.X = s->X; A.phase = s->phase;
    A.t = s->t0 + (double)s->n_host * s->P.dt;
    A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
    const long long n = (long long)s->B * s->S;
    ds::forces_out_kernel<T><<<(unsigned)((n + 127) / 128), 128, 0, s->stream>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

template <typename T> int run_pad_init(ds_system *s, void *p4, void *f4) {
    const long long n = (long long)s->B * (s->Npad - s->N);
    if (n <= 0) return DS_OK;
    ds::pad_init_kernel<T><<<(unsigned)((n + 127) / 128), 128, 0, s->stream>>>(p4, f4, s->N, s->Npad, s->B);
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

}  // namespace

// =================================================================================================
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
    const int TI = f64 ? tile_i<double>() : tile_i<float>();
    s->n_it = (s->N + TI - 1) / TI;
    s->Npad = s->n_it * TI;
    int rc = DS_OK;
    auto fail = [&](int code) { ds_destroy(s); return code; };
    if (set_device(s) != DS_OK) return fail(DS_ERR_CUDA);
    if (cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(DS_ERR_CUDA);
    const size_t n3 = (size_t)s->B * s->N * 3, np = (size_t)s->B * s->Npad;
    const size_t t4 = f64 ? sizeof(double4) : sizeof(float4);
    cudaError_t e = cudaSuccess;
    auto al = [&](void **ptr, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(ptr, bytes); };
    al((void **)&s->X, n3 * 8); al((void **)&s->V1, n3 * 8); al((void **)&s->FdA, n3 * 8); al((void **)&s->FdB, n3 * 8);
    al((void **)&s->phase, (size_t)s->B * s->S * 8);
    al(&s->pos4A, np * t4); al(&s->F4A, np * t4); al(&s->pos4B, np * t4); al(&s->F4B, np * t4);
    al((void **)&s->counters, (size_t)s->B * s->n_it * sizeof(unsigned));
    al((void **)&s->stepc, 2 * sizeof(long long));
    if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof g_cuda_err, "cudaMalloc -> %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return fail(DS_ERR_ALLOC); }
    if (cudaMemset(s->counters, 0, (size_t)s->B * s->n_it * sizeof(unsigned)) != cudaSuccess) return fail(DS_ERR_CUDA);
    if (cudaMemset(s->stepc, 0, 2 * sizeof(long long)) != cudaSuccess) return fail(DS_ERR_CUDA);
    rc = f64 ? run_pad_init<double>(s, s->pos4A, s->F4A) : run_pad_init<float>(s, s->pos4A, s->F4A);
    if (rc == DS_OK) rc = f64 ? run_pad_init<double>(s, s->pos4B, s->F4B) : run_pad_init<float>(s, s->pos4B, s->F4B);
    if (rc != DS_OK) return fail(rc);
    rc = ds_set_tuning(s, 0);
    if (rc != DS_OK) return fail(rc);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return fail(DS_ERR_CUDA);
    *out = s;
    return DS_OK;
}

int ds_destroy(ds_system *s) {
    if (!s) return DS_OK;
    cudaSetDevice(s->P.device);
    cudaStreamSynchronize(s->stream);
    destroy_graphs(s);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    void *ptrs[] = {s->X, s->V1, s->FdA, s->FdB, s->phase, s->pos4A, s->F4A, s->pos4B, s->F4B, s->partial,
                    s->counters, s->stepc, s->ap_partial.p, s->ap_counters.p, s->st_a.p, s->st_b.p, s->st_c.p};
    for (void *q : ptrs) if (q) cudaFree(q);
    (void)cudaGetLastError();
    delete s;
    return DS_OK;
}

int ds_set_stream(ds_system *s, void *stream) {
    if (!s) return DS_ERR_NULL;
    s->stream = (cudaStream_t)stream;
    return DS_OK;
}

int ds_set_tuning(ds_system *s, int32_t j_splits) {
    if (!s) return DS_ERR_NULL;
    if (j_splits < 0) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    CU_TRY(cudaStreamSynchronize(s->stream));
    s->tune_js = j_splits;
    const bool f64 = s->P.precision == DS_F64;
    const int gj = f64 ? group_j<double>() : group_j<float>();
    const int res = f64 ? ShapeF64::MINB : ShapeF32::MINB;
    choose_split(s, s->N, s->B, s->n_it, gj, res, &s->JS, &s->jchunk);
    if (s->partial) { CU_TRY(cudaFree(s->partial)); s->partial = nullptr; }
    CU_TRY(cudaMalloc((void **)&s->partial, (size_t)s->B * s->JS * 3 * s->Npad * sizeof(double)));
    destroy_graphs(s);
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
    const void *dpos = pos;
    if (!dev) {
        DS_TRY(ensure(s->st_a, nb));
        CU_TRY(cudaMemcpyAsync(s->st_a.p, pos, nb, cudaMemcpyHostToDevice, s->stream));
        dpos = s->st_a.p;
    }
    s->t0 = t0;
    s->n_host = 0;
    if (s->graphK) destroy_graphs(s);  // t0 is baked into the graph's kernel arguments
    DS_TRY(s->P.precision == DS_F64 ? run_state_init<double>(s, dpos) : run_state_init<float>(s, dpos));
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
    void *dpos = pos;
    if (!dev) { DS_TRY(ensure(s->st_c, nb)); dpos = s->st_c.p; }
    const long long n3 = (long long)s->B * s->N * 3;
    if (s->P.precision == DS_F64)
        ds::state_out_kernel<double><<<(unsigned)((n3 + 255) / 256), 256, 0, s->stream>>>(s->X, dpos, n3);
    else
        ds::state_out_kernel<float><<<(unsigned)((n3 + 255) / 256), 256, 0, s->stream>>>(s->X, dpos, n3);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(pos, dpos, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
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
    DS_TRY(s->P.precision == DS_F64 ? run_forces_out<double>(s, dF) : run_forces_out<float>(s, dF));
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(F, dF, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
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
    // the packed set that holds the current state: A for Heun; for Euler it ping-pongs with the step parity
    const bool useB = (s->P.integrator == DS_EULER) && (s->n_host & 1);
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    A.N = s->N; A.B = s->B; A.Npad = s->Npad; A.n_it = s->n_it; A.JS = s->JS; A.jchunk = s->jchunk;
    A.partial = s->partial; A.counters = s->counters;
    fill_constants(s, A);
    A.mode = ds::EPI_APPLY;
    A.out_u = dV;
    A.src_pos = useB ? s->pos4B : s->pos4A; A.src_F = useB ? s->F4B : s->F4A; A.Fd_in = useB ? s->FdB : s->FdA;
    DS_TRY(launch_mob(s, A, false, s->stream));
    if (!dev) {
        CU_TRY(cudaMemcpyAsync(V, dV, nb, cudaMemcpyDeviceToHost, s->stream));
        CU_TRY(cudaStreamSynchronize(s->stream));
    }
    return DS_OK;
}

int ds_mobility_apply(ds_system *s, const void *pos, const void *F, void *u, int32_t n) {
    if (!s || !pos || !F || !u) return DS_ERR_NULL;
    if (n < 1) return DS_ERR_INVALID_PARAM;
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

    const int TI = f64 ? tile_i<double>() : tile_i<float>();
    const int gj = f64 ? group_j<double>() : group_j<float>();
    const int res = f64 ? ShapeF64::MINB : ShapeF32::MINB;
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    A.N = n; A.B = 1; A.n_it = (n + TI - 1) / TI; A.Npad = A.n_it * TI;
    choose_split(s, n, 1, A.n_it, gj, res, &A.JS, &A.jchunk);
    if (A.JS > 1) {
        DS_TRY(ensure(s->ap_partial, (size_t)A.JS * 3 * A.Npad * sizeof(double)));
        DS_TRY(ensure(s->ap_counters, (size_t)A.n_it * sizeof(unsigned), true));
    }
    A.partial = (double *)s->ap_partial.p; A.counters = (unsigned *)s->ap_counters.p;
    fill_constants(s, A);
    A.mode = ds::EPI_APPLY;
    A.src_pos = dpos; A.src_F = dF; A.out_u = du;
    DS_TRY(launch_mob(s, A, true, s->stream));
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
    // graphs start at even step parity (Euler ping-pong); GRAPH_STEPS is even
    while (left > 0 && ((s->n_host & 1) != 0 || left < GRAPH_STEPS)) {
        DS_TRY(launch_one_step(s, s->n_host, s->stream));
        s->n_host += 1; left -= 1;
    }
    if (left >= GRAPH_STEPS) {
        if (!s->graphK) DS_TRY(build_graph(s));
        while (left >= GRAPH_STEPS) {
            CU_TRY(cudaGraphLaunch(s->graphK, s->stream));
            s->launches += s->graph_nodes;
            s->n_host += GRAPH_STEPS; left -= GRAPH_STEPS;
        }
    }
    while (left > 0) {
        DS_TRY(launch_one_step(s, s->n_host, s->stream));
        s->n_host += 1; left -= 1;
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

}  // extern "C"
