/*
 * ds_oracle.c -- CPU ORACLE for the active-dumbbell hot path of arXiv 1004.1932
 * (Putz, Dunkel, Yeomans, "CUDA simulations of active dumbbell suspensions").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, double-precision
 * restatement of the paper's equations, written so that a reader can check every line
 * against the paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or
 * helper with the CUDA library under paper_1004_1932_b200/csrc, and neither includes the
 * other.
 *
 * What it computes (citations are lines of /root/reference/PAPER.md):
 *   or_forces            Eq. (4)   PAPER.md:63-67   spring + stroke force per dumbbell
 *   or_dense_mobility    Eq. (3a,b) PAPER.md:57-59  the full 3N x 3N tensor, entry by entry,
 *                                                   in the paper's own form (the "full
 *                                                   tensor" method of PAPER.md:230)
 *   or_mobility_apply    Eq. (1a) deterministic part, PAPER.md:38, 77:
 *                        u_(alpha i) = sum_beta H_(alpha i)(beta j) F_(beta j), matrix free
 *   or_velocity          forces followed by the mobility apply
 *   or_step              explicit Euler / one-step Heun predictor-corrector
 *   or_noise_normal      Eq. (1a-c), additive approximation of PAPER.md:240: the Gaussian increments (Philox4x32-10)
 *   or_avg_rhs, or_avg_step   Eq. (9a-d) PAPER.md:121-135  the stroke-averaged far-field model and its Heun stepping
 *   or_dumbbell_coords   Eq. (6a,b) PAPER.md:87-91  direction and geometric centre of every dumbbell
 *   or_msd               Eq. (13)  PAPER.md:189     mean square displacement per particle over W realisations
 *
 * Readings of the paper used here:
 *   R2  Heun = explicit trapezoid: X* = X + dt V(X,t); X' = X + dt/2 (V(X,t) + V(X*,t+dt)).
 *   R4  Eq. (3b) is applied for every r > 0; no overlap branch (the paper has none).
 *   R5  the intra-dumbbell pair is an ordinary beta != alpha pair (Eq. A16b).
 *   R6  first sphere of a dumbbell gets +g n, the second -g n, n pointing first -> second,
 *       g = k0 (d - L(t)); this is F = -dU/dX for U of Eq. (4).
 *   R7  t = t0 + n dt formed from the integer step count, never accumulated.
 *   R9  one radius a for all spheres.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py against closed
 * forms, textbook series, published known answers and invariants (P1-P10 of SURVEY.md 8(c),
 * P11-P22 for the functions added since: the table in DESIGN.md section 3 lists them function
 * by function); nothing is "parity unpinned".  (A comment only: no arithmetic changed.)
 *
 * Storage: 0-based; dumbbell s owns spheres 2s and 2s+1 (paper, 1-based: 2s-1 and 2s,
 * PAPER.md:63).  X, F, u are [N][3] row-major doubles, N = 2S.
 *
 * Summation: ascending beta with Neumaier-compensated accumulation per component, so that
 * the oracle is the more exact side of every comparison (R12).  Threads (OpenMP over
 * alpha) do not change any result bit: each alpha is summed by one thread in fixed order.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OR_OSEEN 0
#define OR_RPY 1
#define OR_EULER 0
#define OR_HEUN 1

static const double OR_PI = 3.14159265358979323846264338327950288;

typedef struct {
    double a;      /* sphere radius  */
    double eta;    /* viscosity (paper: mu)  */
    double ell;    /* mean dumbbell length  */
    double lambda; /* stroke amplitude  */
    double omega;  /* driving angular frequency 2 pi / T PAPER.md:67  */
    double k0;     /* spring constant  */
    double dt;     /* time step */
    int32_t tensor;     /* OR_OSEEN: first line of (3b) only; OR_RPY: both */
    int32_t integrator; /* OR_EULER or OR_HEUN                           */
    double kT;          /* thermal energy k_B T of Eq. (1a); 0 = deterministic limit */
    uint64_t seed;      /* key of the counter-based generator behind xi(t)                */
    int32_t system;     /* index w of this realisation in a batch (enters the counter)   */
} or_params;

static int g_threads = 1;

void or_set_threads(int n) { g_threads = n < 1 ? 1 : n; }

int or_get_threads(void) { return g_threads; }

int or_max_threads(void) {
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}

/* Neumaier's compensated sum: s + c is the running total. */
static inline void nsum(double *s, double *c, double x) {
    double t = *s + x;
    if (fabs(*s) >= fabs(x))
        *c += (*s - t) + x;
    else
        *c += (x - t) + *s;
    *s = t;
}

/* Eq. (4).  U^s = (k0/2) [d^s - L^s(t)]^2, L^s(t) = ell + lambda sin(omega t + phi^s),
 * d^s = |X_{2s+1} - X_{2s}|, F = -dU/dX.  With n = (X_{2s+1}-X_{2s})/d:
 *   F_{2s} = +k0 (d-L) n,  F_{2s+1} = -k0 (d-L) n.                                         */
void or_forces(int32_t S, const double *X, const double *phi, double t, const or_params *p, double *F) {
    for (int32_t s = 0; s < S; ++s) {
        const double *x1 = X + 6 * (size_t)s, *x2 = x1 + 3;
        double sv[3] = {x2[0] - x1[0], x2[1] - x1[1], x2[2] - x1[2]};
        double d = sqrt(sv[0] * sv[0] + sv[1] * sv[1] + sv[2] * sv[2]);
        double L = p->ell + p->lambda * sin(p->omega * t + phi[s]);
        double g = p->k0 * (d - L);
        for (int i = 0; i < 3; ++i) {
            double n = sv[i] / d;
            F[6 * (size_t)s + i] = g * n;
            F[6 * (size_t)s + 3 + i] = -(g * n);
        }
    }
}

/* Eq. (3a), (3b), written entry by entry exactly as printed:
 *   H_(a i)(a j) = delta_ij / (6 pi mu a)
 *   H_(a i)(b j) = 1/(8 pi mu r) (delta_ij + r_i r_j / r^2)
 *                + 2 a^2/(24 pi mu r^3) (delta_ij - 3 r_i r_j / r^2),   r = x_a - x_b.
 * Oseen keeps the first line only.  H is [3N][3N] row-major, row 3a+i, column 3b+j. */
void or_dense_mobility(int32_t N, const double *X, double a, double eta, int32_t tensor, double *H) {
    size_t M = 3 * (size_t)N;
    for (int32_t al = 0; al < N; ++al) {
        for (int32_t be = 0; be < N; ++be) {
            for (int i = 0; i < 3; ++i) {
                for (int j = 0; j < 3; ++j) {
                    double dij = (i == j) ? 1.0 : 0.0, h;
                    if (al == be) {
                        h = dij / (6.0 * OR_PI * eta * a);
                    } else {
                        double rv[3] = {X[3 * al] - X[3 * be], X[3 * al + 1] - X[3 * be + 1],
                                        X[3 * al + 2] - X[3 * be + 2]};
                        double r = sqrt(rv[0] * rv[0] + rv[1] * rv[1] + rv[2] * rv[2]);
                        double rr = rv[i] * rv[j] / (r * r);
                        h = 1.0 / (8.0 * OR_PI * eta * r) * (dij + rr);
                        if (tensor == OR_RPY)
                            h += 2.0 * a * a / (24.0 * OR_PI * eta * r * r * r) * (dij - 3.0 * rr);
                    }
                    H[(3 * (size_t)al + i) * M + 3 * (size_t)be + j] = h;
                }
            }
        }
    }
}

/* Deterministic part of Eq. (1a), PAPER.md:38 with T = 0, matrix free:
 *   u_a = F_a/(6 pi mu a) + sum_{b != a} T(r_ab) F_b.
 * With r = x_a - x_b, r2 = r.r, rF = r.F_b, Eq. (3b) contracted with F_b is
 *   Oseen: (1/(8 pi mu)) (1/r) [ F_b + r (rF / r2) ]
 *   RPY  : (1/(8 pi mu)) (1/r) [ (1 + 2a^2/(3 r2)) F_b + (1 - 2a^2/r2) (rF / r2) r ]
 * (the second line of (3b), 2a^2/(24 pi mu r^3) (delta - 3 rr/r2), equals
 *  (1/(8 pi mu r)) [ (2a^2/(3 r2)) delta - (2a^2/r2) rr/r2 ]).                           */
void or_mobility_apply(int32_t N, const double *X, const double *F, double a, double eta, int32_t tensor,
                       double *u) {
    const double self = 1.0 / (6.0 * OR_PI * eta * a);
    const double pre = 1.0 / (8.0 * OR_PI * eta);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(g_threads) if (g_threads > 1)
#endif
    for (int32_t al = 0; al < N; ++al) {
        double s[3] = {0, 0, 0}, c[3] = {0, 0, 0};
        const double *xa = X + 3 * (size_t)al;
        for (int32_t be = 0; be < N; ++be) {
            if (be == al) continue;
            const double *xb = X + 3 * (size_t)be, *fb = F + 3 * (size_t)be;
            double r[3] = {xa[0] - xb[0], xa[1] - xb[1], xa[2] - xb[2]};
            double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            double rinv = 1.0 / sqrt(r2);
            double rF = r[0] * fb[0] + r[1] * fb[1] + r[2] * fb[2];
            double cd = 1.0, cr = rF / r2;
            if (tensor == OR_RPY) {
                cd = 1.0 + 2.0 * a * a / (3.0 * r2);
                cr = (1.0 - 2.0 * a * a / r2) * (rF / r2);
            }
            for (int i = 0; i < 3; ++i) nsum(&s[i], &c[i], (cd * fb[i] + cr * r[i]) * rinv);
        }
        for (int i = 0; i < 3; ++i) u[3 * (size_t)al + i] = self * F[3 * (size_t)al + i] + pre * (s[i] + c[i]);
    }
}

/* V(X, t) = H(X) F(X, t): the right-hand side of Eq. (1a) in the deterministic limit. */
void or_velocity(int32_t S, const double *X, const double *phi, double t, const or_params *p, double *V,
                 double *Fwork) {
    or_forces(S, X, phi, t, p, Fwork);
    or_mobility_apply(2 * S, X, Fwork, p->a, p->eta, p->tensor, V);
}

/* n_steps explicit steps from step index n_done (reading R2).
 * t_n = t0 + n dt (R7).  X is updated in place.  Returns 0, or -1 if out of memory.       */
/* Brownian term, Eq. (1a)-(2) in the additive approximation the paper advocates:
 * "a simple additive noise with a constant matrix C ... as the off-diagonal terms in Eq. (3) are negligible", i.e.
 * 2H = C C^T with H reduced to its diagonal (3a): C = sqrt(2 / (6 pi mu a)) 1.  Integrated over one step the term
 * (k_B T)^(1/2) C xi(t) becomes dW_(alpha i) = sqrt(2 k_B T dt / (6 pi mu a)) z, z ~ N(0,1) independent per sphere,
 * component and step (Eq. 1b, 1c).  z comes from a counter-based generator so that any implementation can draw
 * the same numbers: Philox4x32-10 (Salmon et al., SC'11) with counter (n lo, n hi, 3 alpha + i, w), key (seed lo,
 * seed hi); its first two words u1, u2 -> Box-Muller z = sqrt(-2 ln U1) cos(2 pi U2), U = (u + 0.5) / 2^32.       */
void or_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double or_noise_normal(uint64_t seed, int64_t n, int32_t system, int64_t element) {
    const uint32_t ctr[4] = {(uint32_t)((uint64_t)n & 0xffffffffu), (uint32_t)((uint64_t)n >> 32), (uint32_t)element,
                             (uint32_t)system};
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    uint32_t w[4];
    or_philox4x32_10(ctr, key, w);
    const double U1 = ((double)w[0] + 0.5) / 4294967296.0, U2 = ((double)w[1] + 0.5) / 4294967296.0;
    return sqrt(-2.0 * log(U1)) * cos(6.283185307179586476925286766559 * U2);
}

/* Explicit Euler / one-step Heun predictor-corrector.  With k_B T > 0 the same increment dW enters the
 * predictor and the corrector (stochastic Heun for additive noise: "can easily incorporate additive noise").        */
int or_step(int32_t S, double *X, const double *phi, double t0, int64_t n_done, int64_t n_steps,
            const or_params *p) {
    size_t M = 6 * (size_t)S;
    double *buf = (double *)malloc(5 * M * sizeof(double));
    if (!buf) return -1;
    double *V1 = buf, *V2 = buf + M, *Xp = buf + 2 * M, *Fw = buf + 3 * M, *dW = buf + 4 * M;
    const double pi = 3.14159265358979323846264338327950288;
    const double amp = sqrt(2.0 * p->kT * p->dt / (6.0 * pi * p->eta * p->a));
    for (int64_t n = n_done; n < n_done + n_steps; ++n) {
        double t = t0 + (double)n * p->dt;
        for (size_t k = 0; k < M; ++k) dW[k] = p->kT > 0.0 ? amp * or_noise_normal(p->seed, n, p->system, (int64_t)k) : 0.0;
        or_velocity(S, X, phi, t, p, V1, Fw);
        if (p->integrator == OR_EULER) {
            for (size_t k = 0; k < M; ++k) X[k] = X[k] + p->dt * V1[k] + dW[k];
        } else {
            double t1 = t0 + (double)(n + 1) * p->dt;
            for (size_t k = 0; k < M; ++k) Xp[k] = X[k] + p->dt * V1[k] + dW[k];
            or_velocity(S, Xp, phi, t1, p, V2, Fw);
            for (size_t k = 0; k < M; ++k) X[k] = X[k] + 0.5 * p->dt * (V1[k] + V2[k]) + dW[k];
        }
    }
    free(buf);
    return 0;
}

/* Same as or_step, but also records the positions after every `stride`-th step into
 * traj[(k)][N][3], k = 0 .. n_steps/stride - 1 (used by the observable pins, Eq. 11).     */
int or_step_record(int32_t S, double *X, const double *phi, double t0, int64_t n_done, int64_t n_steps,
                   const or_params *p, int64_t stride, double *traj) {
    size_t M = 6 * (size_t)S;
    int64_t k = 0;
    for (int64_t n = 0; n < n_steps; ++n) {
        int rc = or_step(S, X, phi, t0, n_done + n, 1, p);
        if (rc) return rc;
        if ((n + 1) % stride == 0) {
            memcpy(traj + (size_t)k * M, X, M * sizeof(double));
            ++k;
        }
    }
    return 0;
}

/* Dumbbell coordinates, Eq. (6a), (6b), 0-based (dumbbell s = spheres 2s, 2s+1):
 *   N^s = (X_{2s+1} - X_{2s}) / |X_{2s+1} - X_{2s}|,   R^s = (X_{2s+1} + X_{2s}) / 2.
 * X [2S][3] -> R [S][3], Nv [S][3].                                                          */
void or_dumbbell_coords(int32_t S, const double *X, double *R, double *Nv) {
    for (int32_t s = 0; s < S; ++s) {
        const double *x1 = X + 6 * (size_t)s, *x2 = x1 + 3;
        double d[3], len2 = 0.0;
        for (int c = 0; c < 3; ++c) { d[c] = x2[c] - x1[c]; len2 += d[c] * d[c]; }
        const double len = sqrt(len2);
        for (int c = 0; c < 3; ++c) {
            Nv[3 * (size_t)s + c] = d[c] / len;
            R[3 * (size_t)s + c] = 0.5 * (x2[c] + x1[c]);
        }
    }
}

/* Mean square displacement per particle averaged over W initial conditions, Eq. (13):
 *   <<R(t)^2>> = (1/W) sum_w (1/S) sum_s |R^s(t; w) - R^s(0; w)|^2.
 * Rt, R0 [W][S][3] (geometric centres, Eq. 6b).  Plain nested sums in the order of the formula. */
double or_msd(int32_t W, int32_t S, const double *Rt, const double *R0) {
    double outer = 0.0;
    for (int32_t w = 0; w < W; ++w) {
        double inner = 0.0;
        for (int32_t s = 0; s < S; ++s) {
            const size_t k = 3 * ((size_t)w * S + s);
            double q = 0.0;
            for (int c = 0; c < 3; ++c) { const double d = Rt[k + c] - R0[k + c]; q += d * d; }
            inner += q;
        }
        outer += inner / (double)S;
    }
    return outer / (double)W;
}

/* Stroke-averaged far-field model, Eq. (9a)-(9d), as printed (the numerical comparison with the
 * microscopic model, pin P20, confirms the prefactors 9/64, 15/64 and the sign of (9b)):
 *   dR^s/dt = sum_{r != s} J^{sr},      dN^s/dt = -(1 - N^s N^s) sum_{r != s} K^{sr},
 *   J^{sr} = a w sin(phi^s - phi^r) (9/64) (lam/ell)^2 (ell/|D|)^4 { N^s (2s + 4qr - 10 s r^2)
 *                                  + Dh (1 + 2q^2 - 5s^2 - 5r^2 - 20qsr + 35 s^2 r^2) },
 *   K^{sr} = w sin(phi^s - phi^r) (15/64) (a/ell) (lam/ell)^2 (ell/|D|)^5 Dh (3s + 6rq + 6sq^2 - 7s^3 - 21 s r^2
 *                                  - 42 q s^2 r + 63 s^3 r^2),
 *   D = R^s - R^r, Dh = D/|D|, s = Dh.N^s, r = Dh.N^r, q = N^s.N^r   (9d; its printed indices are slips).
 * R, N [S][3] -> dR, dN [S][3].  Plain double loops in the order of the formulas.                                  */
void or_avg_rhs(int32_t S, const double *R, const double *N, const double *phi, const or_params *p, double *dR,
                double *dN) {
    const double a = p->a, ell = p->ell, lam = p->lambda, w = p->omega;
    for (int32_t s_ = 0; s_ < S; ++s_) {
        double Jsum[3] = {0, 0, 0}, Ksum[3] = {0, 0, 0};
        const double *Ns = N + 3 * (size_t)s_;
        for (int32_t r_ = 0; r_ < S; ++r_) {
            if (r_ == s_) continue;
            const double *Nr = N + 3 * (size_t)r_;
            double D[3], Dn2 = 0.0;
            for (int c = 0; c < 3; ++c) { D[c] = R[3 * (size_t)s_ + c] - R[3 * (size_t)r_ + c]; Dn2 += D[c] * D[c]; }
            const double Dn = sqrt(Dn2);
            double Dh[3], s = 0.0, r = 0.0, q = 0.0;
            for (int c = 0; c < 3; ++c) { Dh[c] = D[c] / Dn; s += Dh[c] * Ns[c]; r += Dh[c] * Nr[c]; q += Ns[c] * Nr[c]; }
            const double sn = sin(phi[s_] - phi[r_]);
            const double lr = ell / Dn, ll = lam / ell;
            const double cj = a * w * sn * (9.0 / 64.0) * ll * ll * lr * lr * lr * lr;
            const double ck = w * sn * (15.0 / 64.0) * (a / ell) * ll * ll * lr * lr * lr * lr * lr;
            const double jn = 2.0 * s + 4.0 * q * r - 10.0 * s * r * r;
            const double jd = 1.0 + 2.0 * q * q - 5.0 * s * s - 5.0 * r * r - 20.0 * q * s * r + 35.0 * s * s * r * r;
            const double kd = 3.0 * s + 6.0 * r * q + 6.0 * s * q * q - 7.0 * s * s * s - 21.0 * s * r * r - 42.0 * q * s * s * r +
                              63.0 * s * s * s * r * r;
            for (int c = 0; c < 3; ++c) {
                Jsum[c] += cj * (Ns[c] * jn + Dh[c] * jd);
                Ksum[c] += ck * Dh[c] * kd;
            }
        }
        const double nk = Ns[0] * Ksum[0] + Ns[1] * Ksum[1] + Ns[2] * Ksum[2];
        for (int c = 0; c < 3; ++c) {
            dR[3 * (size_t)s_ + c] = Jsum[c];
            dN[3 * (size_t)s_ + c] = -(Ksum[c] - Ns[c] * nk);
        }
    }
}

/* n_steps Heun steps of Eq. (9) with step dt (reading R16: the paper does not say how it integrates (9); the
 * predictor-corrector of PAPER.md:236 is used, and N is renormalised after every stage because the projector of (9b)
 * keeps |N| = 1 only to first order in dt).                                                                          */
int or_avg_step(int32_t S, double *R, double *N, const double *phi, double dt, int64_t n_steps, const or_params *p) {
    const size_t M = 3 * (size_t)S;
    double *buf = (double *)malloc(6 * M * sizeof(double));
    if (!buf) return -1;
    double *dR1 = buf, *dN1 = buf + M, *dR2 = buf + 2 * M, *dN2 = buf + 3 * M, *Rp = buf + 4 * M, *Np = buf + 5 * M;
    for (int64_t n = 0; n < n_steps; ++n) {
        or_avg_rhs(S, R, N, phi, p, dR1, dN1);
        for (size_t k = 0; k < M; ++k) { Rp[k] = R[k] + dt * dR1[k]; Np[k] = N[k] + dt * dN1[k]; }
        for (int32_t s = 0; s < S; ++s) {
            double *v = Np + 3 * (size_t)s; const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            v[0] /= len; v[1] /= len; v[2] /= len;
        }
        or_avg_rhs(S, Rp, Np, phi, p, dR2, dN2);
        for (size_t k = 0; k < M; ++k) { R[k] = R[k] + 0.5 * dt * (dR1[k] + dR2[k]); N[k] = N[k] + 0.5 * dt * (dN1[k] + dN2[k]); }
        for (int32_t s = 0; s < S; ++s) {
            double *v = N + 3 * (size_t)s; const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            v[0] /= len; v[1] /= len; v[2] /= len;
        }
    }
    free(buf);
    return 0;
}
