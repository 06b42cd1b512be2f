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

template <typename T> constexpr int pack_w() { return ds::Pack<T>::W; }

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
    int N = 0, B = 0, S = 0;
    int W = 1;                  // spheres per unit: 2 (FP32 packs) or 1 (FP64)
    int NQ = 0, U = 0;          // quads = ceil(N/4), units = ceil(N/W)
    long long unit_stride = 0;  // units per system in the streams
    int tune_cta = 0, n_cta = 1;
    bool has_state = false;
    double t0 = 0.0;
    long long n_host = 0;  // mirror of the device step counter
    int64_t launches = 0;
    // state
    double *X = nullptr, *V1 = nullptr, *FdA = nullptr, *FdB = nullptr, *phase = nullptr;
    void *unitsA = nullptr, *unitsB = nullptr;  // beta-streams (mobility.cuh), ping-pong
    long long *stepc = nullptr;                 // c[0], c[1]
    // graphs
    cudaGraphExec_t graphK = nullptr;  // GRAPH_STEPS steps
    int graph_steps = 0;
    int graph_nodes = 0;
    // scratch of the stateless apply and of host-pointer staging
    Buf ap_units, st_a, st_b, st_c;
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

// Launch shape: n_cta row tiles per system (mobility.cuh).  Every CTA walks all U units with
// n_jg = NT / nq beta-groups, i.e. ceil(U / n_jg) iterations of 4 alpha x 1 unit per thread, so the
// modelled time of a launch is waves x (iterations + a fixed per-CTA cost, in iterations).
int choose_tiles(const ds_system *s, int NQ, int U, int B) {
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
        const long long waves = ((long long)B * n + s->num_sms - 1) / s->num_sms;
        const double cost = (double)waves * ((double)iters + 6.0);
        if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = n; }
    }
    return best;
}

template <typename T, int TENSOR> int launch_mob_t(ds_system *s, const ds::MobArgs &A, cudaStream_t st) {
    auto kern = ds::mobility_kernel<T, TENSOR>;
    static bool attr_done = false;
    if (!attr_done) {
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ds::SMEM_BYTES));
        attr_done = true;
    }
    dim3 grid((unsigned)A.n_cta, (unsigned)A.B), block(ds::NT);
    kern<<<grid, block, ds::SMEM_BYTES, st>>>(A);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    return DS_OK;
}

int launch_mob(ds_system *s, const ds::MobArgs &A, cudaStream_t st) {
    const bool f64 = s->P.precision == DS_F64, rpy = s->P.tensor == DS_RPY;
    if (f64) return rpy ? launch_mob_t<double, ds::TENSOR_RPY>(s, A, st) : launch_mob_t<double, ds::TENSOR_OSEEN>(s, A, st);
    return rpy ? launch_mob_t<float, ds::TENSOR_RPY>(s, A, st) : launch_mob_t<float, ds::TENSOR_OSEEN>(s, A, st);
}

void fill_shape(const ds_system *s, ds::MobArgs &A) {
    A.N = s->N; A.B = s->B; A.NQ = s->NQ; A.U = s->U; A.n_cta = s->n_cta; A.unit_stride = s->unit_stride;
}

void fill_constants(const ds_system *s, ds::MobArgs &A) {
    const double pi = 3.14159265358979323846264338327950288;
    A.self_mob = 1.0 / (6.0 * pi * s->P.eta * s->P.a);
    A.pre = 1.0 / (8.0 * pi * s->P.eta);
    A.c1 = 2.0 * s->P.a * s->P.a / 3.0;
    A.c2 = 2.0 * s->P.a * s->P.a;
    A.t0 = s->t0; A.dt = s->P.dt; A.ell = s->P.ell; A.lambda = s->P.lambda; A.omega = s->P.omega; A.k0 = s->P.k0;
}

// One stage of the integrator on the system's own state.  set 0: (unitsA,FdA) -> writes set B
// (predictor) ; set 1: reads B, writes A (corrector).  Euler reads A and writes A... see below.
int launch_state_stage(ds_system *s, int mode, int cr, int cw, long long inc, cudaStream_t st) {
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    fill_shape(s, A);
    fill_constants(s, A);
    A.mode = mode;
    A.X = s->X; A.V1 = s->V1; A.phase = s->phase;
    A.n_read = s->stepc + cr; A.n_write = s->stepc + cw; A.n_inc = inc;
    const bool fromB = (mode == ds::EPI_CORR);
    A.src_units = fromB ? s->unitsB : s->unitsA;
    A.Fd_in = fromB ? s->FdB : s->FdA;
    const bool toB = (mode == ds::EPI_PRED);
    A.units_out = toB ? s->unitsB : s->unitsA;
    A.Fd_out = toB ? s->FdB : s->FdA;
    return launch_mob(s, A, st);
}

// One full step.  Heun: PRED (reads c[0], writes c[1] = n) then CORR (reads c[1], writes c[0] = n+1).
// Euler: in place on set A is NOT safe (other blocks still read unitsA), so Euler ping-pongs the
// packed sets: even steps read A write B, odd steps read B write A; the counters ping-pong too.
int launch_one_step(ds_system *s, long long n_index, cudaStream_t st) {
    if (s->P.integrator == DS_HEUN) {
        DS_TRY(launch_state_stage(s, ds::EPI_PRED, 0, 1, 0, st));
        return launch_state_stage(s, ds::EPI_CORR, 1, 0, 1, st);
    }
    const int par = (int)(n_index & 1);
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    fill_shape(s, A);
    fill_constants(s, A);
    A.mode = ds::EPI_EULER;
    A.X = s->X; A.V1 = s->V1; A.phase = s->phase;
    A.n_read = s->stepc + par; A.n_write = s->stepc + (par ^ 1); A.n_inc = 1;
    A.src_units = par ? s->unitsB : s->unitsA; A.Fd_in = par ? s->FdB : s->FdA;
    A.units_out = par ? s->unitsA : s->unitsB; A.Fd_out = par ? s->FdA : s->FdB;
    return launch_mob(s, A, st);
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
    A.N = s->N; A.B = s->B; A.unit_stride = s->unit_stride; A.user_pos = dpos; A.X = s->X; A.units = s->unitsA;
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
    A.N = s->N; A.B = s->B; A.unit_stride = s->unit_stride; A.user_out = dF; A.X = s->X; A.phase = s->phase;
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
    s->W = f64 ? pack_w<double>() : pack_w<float>();
    s->NQ = (s->N + ds::QI - 1) / ds::QI;
    s->U = (s->N + s->W - 1) / s->W;
    s->unit_stride = (long long)s->U + ds::PAD_UNITS;
    int rc = DS_OK;
    auto fail = [&](int code) { ds_destroy(s); return code; };
    if (set_device(s) != DS_OK) return fail(DS_ERR_CUDA);
    if (cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(DS_ERR_CUDA);
    const size_t n3 = (size_t)s->B * s->N * 3;
    const size_t ub = (size_t)s->B * (size_t)s->unit_stride * ds::UNIT_BYTES;
    cudaError_t e = cudaSuccess;
    auto al = [&](void **ptr, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(ptr, bytes); };
    al((void **)&s->X, n3 * 8); al((void **)&s->V1, n3 * 8); al((void **)&s->FdA, n3 * 8); al((void **)&s->FdB, n3 * 8);
    al((void **)&s->phase, (size_t)s->B * s->S * 8);
    al(&s->unitsA, ub); al(&s->unitsB, ub);
    al((void **)&s->stepc, 2 * sizeof(long long));
    if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof g_cuda_err, "cudaMalloc -> %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return fail(DS_ERR_ALLOC); }
    if (cudaMemset(s->stepc, 0, 2 * sizeof(long long)) != cudaSuccess) return fail(DS_ERR_CUDA);
    rc = f64 ? run_pad_init<double>(s, s->unitsA) : run_pad_init<float>(s, s->unitsA);
    if (rc == DS_OK) rc = f64 ? run_pad_init<double>(s, s->unitsB) : run_pad_init<float>(s, s->unitsB);
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
    void *ptrs[] = {s->X, s->V1, s->FdA, s->FdB, s->phase, s->unitsA, s->unitsB, s->stepc,
                    s->ap_units.p, s->st_a.p, s->st_b.p, s->st_c.p};
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

int ds_set_tuning(ds_system *s, int32_t n_tiles) {
    if (!s) return DS_ERR_NULL;
    if (n_tiles < 0) return DS_ERR_INVALID_PARAM;
    DS_TRY(set_device(s));
    CU_TRY(cudaStreamSynchronize(s->stream));
    s->tune_cta = n_tiles;
    s->n_cta = choose_tiles(s, s->NQ, s->U, s->B);
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
    fill_shape(s, A);
    fill_constants(s, A);
    A.mode = ds::EPI_APPLY;
    A.out_u = dV;
    A.src_units = useB ? s->unitsB : s->unitsA; A.Fd_in = useB ? s->FdB : s->FdA;
    DS_TRY(launch_mob(s, A, s->stream));
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

    // user arrays -> one beta-stream (pack kernel), then the mobility kernel in EPI_APPLY mode
    const int U = (n + s->W - 1) / s->W;
    const long long n_units = (long long)U + ds::PAD_UNITS;
    DS_TRY(ensure(s->ap_units, (size_t)n_units * ds::UNIT_BYTES));
    const unsigned pg = (unsigned)((n_units + 255) / 256);
    if (f64)
        ds::pack_user_kernel<double><<<pg, 256, 0, s->stream>>>((const double *)dpos, (const double *)dF, (double *)s->ap_units.p, n, n_units);
    else
        ds::pack_user_kernel<float><<<pg, 256, 0, s->stream>>>((const float *)dpos, (const float *)dF, (float *)s->ap_units.p, n, n_units);
    CU_TRY(cudaGetLastError());
    s->launches += 1;
    ds::MobArgs A;
    memset(&A, 0, sizeof A);
    A.N = n; A.B = 1; A.NQ = (n + ds::QI - 1) / ds::QI; A.U = U; A.unit_stride = n_units;
    A.n_cta = choose_tiles(s, A.NQ, A.U, 1);
    fill_constants(s, A);
    A.mode = ds::EPI_APPLY;
    A.src_units = s->ap_units.p; A.out_u = du;
    DS_TRY(launch_mob(s, A, s->stream));
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
