/*
 * ds.h -- C ABI of the B200-native hot path of arXiv 1004.1932
 * (Putz, Dunkel, Yeomans, "CUDA simulations of active dumbbell suspensions").
 *
 * The library evaluates, on one sm_100a device, the deterministic limit of the paper's
 * equation of motion (Eq. (1a) with T = 0):
 *
 *     dX_(alpha i)/dt = sum_beta H_(alpha i)(beta j) F_(beta j)
 *
 * with H the Rotne-Prager-Yamakawa-Mazur tensor of Eq. (3a,3b) or its Oseen
 * truncation (first line of (3b)), F the spring + stroke force of Eq. (4)
 * and the explicit Euler / one-step Heun predictor-corrector integrator of
 * PAPER.md:236.  Every step runs in hand-written CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   S dumbbells, N = 2S spheres per system.  0-based storage: dumbbell s owns
 *   spheres 2s and 2s+1 (paper, 1-based: alpha = 2s-1, beta = 2s).
 *   Arrays are [system][sphere][xyz] contiguous (the paper's X_(alpha i) index order), element
 *   type float for DS_F32 and double for DS_F64.  `phase` is always double, [system][dumbbell].
 *
 * Pointers
 *   Every data pointer may be a DEVICE pointer (e.g. a torch tensor's data_ptr()) or a HOST
 *   pointer (pageable or pinned); the library asks the CUDA runtime which (cudaPointerGetAttributes)
 *   and stages host buffers through its own device scratch with cudaMemcpyAsync on the system's
 *   stream.  The caller owns all buffers; the library never stores a caller pointer in the system.
 *   Work is enqueued on the system's stream.  Calls with device pointers are asynchronous; calls
 *   that write to a HOST pointer synchronise the stream before returning.  Calls that only READ
 *   host pointers do not synchronise: a pageable input has been staged when the call returns, but
 *   a PINNED host input is read by the copy engine when the stream reaches the copy, so it must
 *   stay unchanged until then (until the next synchronising call on the system, or a
 *   cudaStreamSynchronize of its stream).  ds_create/ds_destroy are synchronous.
 *
 * Errors
 *   Every call returns DS_OK (0) or a negative ds_status; nothing throws across the ABI.
 *   Device-side preconditions that are NOT checked: r_ab > 0 for all alpha != beta (Eq. (3b) is
 *   applied for every r > 0, the paper has no overlap branch; its stated validity range is
 *   r > 2a), and finite inputs.
 *
 * The library keeps no random state: with kT > 0 the Brownian increments are a pure function of (seed, step, system,
 * sphere, component).
 */
#ifndef DS_H_
#define DS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ds_system ds_system; /* opaque; owned by the library, freed by ds_destroy */

#define DS_MAX_APPLY_N (1 << 28)     /* largest n of ds_mobility_apply (the kernel indexes 16-byte pieces of the stream in 32 bits) */

enum { DS_F32 = 0, DS_F64 = 1 };     /* element type of user buffers and of the O(N^2) pair arithmetic */
enum { DS_OSEEN = 0, DS_RPY = 1 };   /* Eq. (3b): first line only / both lines */
enum { DS_EULER = 0, DS_HEUN = 1 };

typedef enum {
    DS_OK = 0,
    DS_ERR_INVALID_PARAM = -1, /* a parameter violates the model's constraints (see ds_create)  */
    DS_ERR_NULL = -2,          /* a required pointer is NULL                                     */
    DS_ERR_CUDA = -3,          /* a CUDA runtime call failed; ds_last_cuda_error() says which    */
    DS_ERR_STATE = -4,         /* call needs a state (ds_set_state) or a different n_batch       */
    DS_ERR_NO_DEVICE = -5,     /* no sm_100-class CUDA device                                    */
    DS_ERR_ALLOC = -6,         /* host or device allocation failed                               */
    DS_ERR_TOO_LARGE = -7      /* the problem exceeds a fixed capacity stated at the call (ds_msd_static) */
} ds_status;

typedef struct {
    int32_t n_dumbbells; /* S per system, >= 1; N = 2S                                           */
    int32_t n_batch;     /* B >= 1 independent systems sharing every scalar below                */
    int32_t precision;   /* DS_F32 | DS_F64                                                      */
    int32_t tensor;      /* DS_OSEEN | DS_RPY                                                    */
    int32_t integrator;  /* DS_EULER | DS_HEUN                                                   */
    int32_t device;      /* CUDA device ordinal                                                  */
    double a;            /* sphere radius               */
    double eta;          /* viscosity (paper: mu)                   */
    double ell;          /* mean dumbbell length                   */
    double lambda;       /* stroke amplitude; ell > 2a + |lambda|                   */
    double omega;        /* driving angular frequency 2 pi / T                   */
    double k0;           /* spring constant                        PAPER.md:65 Eq. (4)           */
    double dt;           /* time step                  */
    void *stream;        /* cudaStream_t the work is enqueued on; NULL = legacy default stream   */
    double kT;           /* thermal energy k_B T of Eq. (1a); 0 = the deterministic limit
                            the paper simulates.  > 0: additive Brownian increments
                            dW = sqrt(2 kT dt / (6 pi eta a)) z per sphere, component and step, the constant-C
                            approximation of PAPER.md:240; z from Philox4x32-10 keyed by `seed`, counter
                            (step, state element, system)                                            */
    uint64_t seed;       /* key of the generator (the library itself keeps no random state)        */
} ds_params;

/* Validate p, allocate the system's device buffers and choose its launch shape.
 * Rejects (DS_ERR_INVALID_PARAM): S < 1, B < 1, unknown enum values, non-positive or non-finite
 * a, eta, k0, dt, ell, negative omega, negative or non-finite kT, and ell <= 2a + |lambda|.               */
int ds_create(const ds_params *p, ds_system **out);

/* Free everything the system owns.  Synchronises the system's stream first.  NULL is a no-op. */
int ds_destroy(ds_system *s);

/* Re-target the system to another cudaStream_t (e.g. one that is being captured).  Work already queued on the old
 * stream is ordered before anything enqueued on the new one (an event); if the OLD stream is being captured at the
 * time of the call, the caller owns that ordering. */
int ds_set_stream(ds_system *s, void *stream);

/* Set the state: sphere positions pos [B][N][3] (user precision), stroke phases phase [B][S]
 * (double), time origin t0; the step counter n is reset to 0, so that t = t0 + n dt
 * (never accumulated).  PAPER.md:36 (state = positions only, inertia neglected).   */
int ds_set_state(ds_system *s, const void *pos, const void *phase, double t0);

/* Read the state back: pos [B][N][3] (user precision; may be NULL) and t = t0 + n dt (may be NULL). */
int ds_get_state(ds_system *s, void *pos, double *t);

/* Eq. (4), at the current state and time: F [B][N][3] (user precision).
 * With n = (X_{2s+1} - X_{2s})/d, d = |X_{2s+1} - X_{2s}|, L = ell + lambda sin(omega t + phi_s):
 * F_{2s} = +k0 (d - L) n, F_{2s+1} = -k0 (d - L) n  (F = -dU/dX).                               */
int ds_forces(ds_system *s, void *F);

/* Stateless mobility apply, Eq. (1a) deterministic part with Eq. (3a,3b), PAPER.md:38, 57-59:
 *   u_a = F_a / (6 pi eta a) + sum_{b != a} T(x_a - x_b) F_b,   a = 0 .. n-1,
 *   Oseen: T(r) = 1/(8 pi eta r) (1 + rr/r^2);  RPY: + 2a^2/(24 pi eta r^3) (1 - 3 rr/r^2).
 * pos, F, u are [n][3] in user precision; 1 <= n <= DS_MAX_APPLY_N is any sphere count (odd allowed,
 * independent of S; DS_ERR_INVALID_PARAM outside that range); a, eta, tensor and precision come from the system.  u must not alias pos or F.
 * Does not touch the system's state.                                                           */
int ds_mobility_apply(ds_system *s, const void *pos, const void *F, void *u, int32_t n);

/* Advance the state by n_steps explicit steps: Heun = predictor X* = X + dt V(X,t_n),
 * corrector X <- X + dt/2 (V(X,t_n) + V(X*,t_n + dt)); Euler = X <- X + dt V(X,t_n);
 * V(X,t) = H(X) F(X,t).  The whole loop runs on the device: one persistent kernel launch per
 * call (per 65536 steps) and per group of co-resident systems, no host round trip per step.
 * ds_step requires n_batch == 1 (DS_ERR_STATE otherwise); ds_batch_step advances all B systems
 * by n_steps each.  n_steps >= 0.                                                               */
int ds_step(ds_system *s, int64_t n_steps);
int ds_batch_step(ds_system *s, int64_t n_steps);

/* Velocities V(X, t) = H(X) F(X, t) at the current state, [B][N][3] in user precision (the
 * right-hand side of Eq. (1a) the integrator uses; exported for tests and observables).        */
int ds_velocity(ds_system *s, void *V);

/* Observables (computed on the device from the FP64 state).
 * ds_dumbbell_coords: direction and geometric centre of every dumbbell, Eq. (6a), (6b):
 *   N^s = (X_{2s+1} - X_{2s}) / |X_{2s+1} - X_{2s}|,  R^s = (X_{2s+1} + X_{2s}) / 2;
 *   R, Nv are [B][S][3] in user precision; either may be NULL.
 * ds_msd_set_reference: R^s(0; w) := the current centres (call it after the discarded first period).
 * ds_msd: mean square displacement per particle averaged over the W = n_batch systems, Eq. (13):
 *   (1/W) sum_w (1/S) sum_s |R^s(t; w) - R^s(0; w)|^2, written as one double to *msd (host or device pointer);
 *   DS_ERR_STATE without a reference.                                                             */
int ds_dumbbell_coords(ds_system *s, void *R, void *Nv);
int ds_msd_set_reference(ds_system *s);
int ds_msd(ds_system *s, double *msd);

/* Eq. (13) for callers that may not allocate: CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  The same two kernels as ds_msd (per-chunk partial sums, then one block adds them in a fixed order), but the
 * partial sums live in a file-scope `static __device__` array of DS_MSD_STATIC_MAX_PARTIALS doubles (128 KB, held by every
 * GPU that loads the library until the process exits) instead of a buffer ds_msd_set_reference allocates.  The call needs
 * no ds_system and calls no cudaMalloc, cudaFree or allocating library routine (its one-time set-up per device is a
 * cudaGetSymbolAddress).
 *   X     device pointer, FP64 sphere positions [W][2 S][3] (spheres 2s, 2s + 1 = dumbbell s, as in ds_set_state)
 *   Rref  device pointer, FP64 reference centres R^s(0; w) [W][S][3]
 *   S, W  dumbbells per system (>= 1), systems (>= 1); W * ceil(S / 256) <= DS_MSD_STATIC_MAX_PARTIALS, else DS_ERR_TOO_LARGE
 *   msd   device pointer to one double, written by the second kernel (read it after the stream has reached that point)
 *   stream  a cudaStream_t of `device` (NULL = default stream); device = CUDA device ordinal, made current by the call
 * Asynchronous.  Inputs are read, *msd is written, nothing else of the caller's is touched.  Every partial sum a call reads
 * it has written itself (nothing has to start at zero, the array keeps the last call's contents otherwise).  ALL calls on a
 * device share the one array: calls that overlap on the GPU (different streams, no ordering between them) race and give
 * wrong sums; calls in one stream, or ordered by events, are safe.
 * DS_ERR_NULL for a NULL X, Rref or msd; DS_ERR_INVALID_PARAM for S < 1, W < 1 or an unknown device; DS_ERR_TOO_LARGE beyond
 * the limit (nothing is launched); DS_ERR_NO_DEVICE / DS_ERR_CUDA as elsewhere.                                         */
#define DS_MSD_STATIC_MAX_PARTIALS 16384
int ds_msd_static(const double *X, const double *Rref, int32_t S, int32_t W, double *msd, void *stream, int32_t device);

/* Stroke-averaged far-field model, Eq. (9a)-(9d): the paper's comparison model, a second O(S^2) pair sum
 * over dumbbells (centres R, unit directions Nv, stroke phases).  Stateless: S is any dumbbell count >= 1; a, ell, lambda,
 * omega and the precision of the pair arithmetic come from the system; R, Nv, dR, dN are [S][3] in user precision, phase
 * [S] double; device or host pointers.
 *   ds_avg_rhs : dR = sum_r J^{sr},  dN = -(1 - N N) sum_r K^{sr}   (right-hand sides of (9a), (9b)).
 *   ds_avg_step: n_steps Heun steps of size dt on R, Nv in place; the state is FP64 inside the call (the
 *                increments are below FP32 resolution) and Nv is renormalised after every stage.
 * Precondition, not checked: distinct centres (Eq. (9) is a far-field expansion, |R^s - R^r| >> ell; a pair at zero
 * distance is skipped like the self term).                                                                        */
int ds_avg_rhs(ds_system *s, const void *R, const void *Nv, const void *phase, void *dR, void *dN, int32_t S);
int ds_avg_step(ds_system *s, void *R, void *Nv, const void *phase, int32_t S, double dt, int64_t n_steps);

const char *ds_strerror(int code);
const char *ds_last_cuda_error(void); /* text of the last failing CUDA call on this thread, or "" */
const char *ds_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DS_H_ */
