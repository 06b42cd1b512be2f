"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the pin (P1-P10 of SURVEY.md 8(c), plus extras) and the passage it rests on.
None of them re-types the oracle's formula: they use closed forms for special geometries,
textbook series, identities of Stokes flow, invariants, numerical differentiation of the
paper's potential, and brute force through the dense tensor.
"""
import os

import numpy as np
import pytest

import oracle
from oracle import OSEEN, RPY, EULER, HEUN, Params
from paper_1004_1932_b200 import inputs

PI = np.pi
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def two_spheres(r, direction=(1.0, 0.0, 0.0)):
    d = np.asarray(direction, float)
    d = d / np.linalg.norm(d)
    return np.stack([np.zeros(3), r * d])


# ----------------------------------------------------------------------------- P1, P2
@pytest.mark.parametrize("r", [2.5, 7.0, 123.0])
def test_P1_oseen_point_force_closed_form(r):
    """PAPER.md:57-61 / 306-309: a unit force on sphere 2 moves sphere 1 with 1/(4 pi eta r)
    along the line of centres (kappa = (4 pi mu)^-1 in 1d, A6) and 1/(8 pi eta r) normal to it;
    sphere 2 itself moves with 1/(6 pi eta a)."""
    a, eta = 0.7, 1.3
    X = two_spheres(r)
    for comp, expect in [(0, 1 / (4 * PI * eta * r)), (1, 1 / (8 * PI * eta * r)), (2, 1 / (8 * PI * eta * r))]:
        F = np.zeros((2, 3))
        F[1, comp] = 1.0
        u = oracle.mobility_apply(X, F, a, eta, OSEEN)
        want = np.zeros((2, 3))
        want[0, comp] = expect
        want[1, comp] = 1 / (6 * PI * eta * a)
        np.testing.assert_allclose(u, want, rtol=1e-14, atol=1e-18)


def _series():
    c = {}
    for line in open(os.path.join(GOLD, "two_sphere_series.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, c1, c3 = line.split()
        c[k] = (float(c1), float(c3))
    return c


@pytest.mark.parametrize("rho", [2.0, 3.5, 10.0, 50.0])
def test_P2_two_sphere_sedimentation_series(rho):
    """tests/golden/two_sphere_series.txt: equal forces on two equal spheres.  RPY gives
    U/U0 = 1 + c1/rho + c3/rho^3 exactly, Oseen 1 + c1/rho (textbook reflections series)."""
    a, eta = 1.0, 1.0
    c = _series()
    U0 = 1 / (6 * PI * eta * a)
    X = two_spheres(rho * a, direction=(0.0, 0.0, 1.0))
    for comp, key in [(2, "parallel"), (0, "perpendicular"), (1, "perpendicular")]:
        F = np.zeros((2, 3))
        F[:, comp] = 1.0
        c1, c3 = c[key]
        u = oracle.mobility_apply(X, F, a, eta, RPY)
        np.testing.assert_allclose(u[:, comp] / U0, 1 + c1 / rho + c3 / rho ** 3, rtol=1e-14)
        u = oracle.mobility_apply(X, F, a, eta, OSEEN)
        np.testing.assert_allclose(u[:, comp] / U0, 1 + c1 / rho, rtol=1e-14)
        other = [k for k in range(3) if k != comp]
        assert np.abs(u[:, other]).max() < 1e-17


def test_rpy_is_oseen_plus_a2_over_3_laplacian():
    """Finite-size correction of two equal spheres = (a^2/6 + a^2/6) Laplacian of the Stokeslet
    (Faxen; Rotne & Prager ref. [26]).  The Laplacian is taken numerically from the oracle's own
    Oseen tensor, so the second line of Eq. (3b) (coefficient 2a^2/24, the -3, the r^-3) is pinned
    by the first line, not by re-typing it."""
    a, eta = 1.3, 0.9
    r0 = np.array([3.1, -2.2, 4.5])
    h = 1e-3

    def block(r, tensor):
        return oracle.dense_mobility(np.stack([r, np.zeros(3)]), a, eta, tensor)[0:3, 3:6]

    lap = -6 * block(r0, OSEEN)
    for k in range(3):
        e = np.zeros(3)
        e[k] = h
        lap = lap + block(r0 + e, OSEEN) + block(r0 - e, OSEEN)
    lap /= h * h
    diff = block(r0, RPY) - block(r0, OSEEN)
    np.testing.assert_allclose(diff, a * a / 3 * lap, rtol=2e-6, atol=1e-9 * np.abs(diff).max())


def test_tensor_is_divergence_free():
    """d/dx_(beta j) H_(alpha i)(beta j) = 0 (incompressibility), both tensors."""
    a, eta, h = 1.0, 1.0, 1e-4
    rng = np.random.default_rng(5)
    X = np.stack([np.zeros(3), rng.uniform(3, 6, 3)])
    for tensor in (OSEEN, RPY):
        div = np.zeros(3)
        for j in range(3):
            Xp, Xm = X.copy(), X.copy()
            Xp[1, j] += h
            Xm[1, j] -= h
            Hp = oracle.dense_mobility(Xp, a, eta, tensor)[0:3, 3:6]
            Hm = oracle.dense_mobility(Xm, a, eta, tensor)[0:3, 3:6]
            div += (Hp[:, j] - Hm[:, j]) / (2 * h)
        scale = np.abs(oracle.dense_mobility(X, a, eta, tensor)[0:3, 3:6]).max() / np.linalg.norm(X[1])
        assert np.abs(div).max() < 1e-6 * scale


# ----------------------------------------------------------------------------- P3, P4, P6
@pytest.mark.parametrize("tensor", [OSEEN, RPY])
def test_P3_symmetry(tensor):
    """Eq. (3) is symmetric in (alpha i)(beta j) (needed by Eq. (2)): G.MF = F.MG."""
    X, F = inputs.apply_case(200, 11, 12)
    G = np.random.default_rng(13).standard_normal(F.shape)
    lhs = np.sum(G * oracle.mobility_apply(X, F, 1.0, 1.0, tensor))
    rhs = np.sum(F * oracle.mobility_apply(X, G, 1.0, 1.0, tensor))
    assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), abs(rhs), 1.0)
    H = oracle.dense_mobility(X[:40], 1.0, 1.0, tensor)
    assert np.array_equal(H, H.T) or np.abs(H - H.T).max() < 1e-17


def test_P4_rpy_positive_definite_beyond_contact():
    """H positive definite for r > 2a, so the Cholesky factor of Eq. (2) exists."""
    w = inputs.config2()
    H = oracle.dense_mobility(w.pos[0], 1.0, 1.0, RPY)
    np.linalg.cholesky(H)
    X = two_spheres(2.0 + 1e-9)
    ev = np.linalg.eigvalsh(oracle.dense_mobility(X, 1.0, 1.0, RPY))
    assert ev.min() > 0
    F = np.random.default_rng(3).standard_normal((w.N, 3))
    assert np.sum(F * oracle.mobility_apply(w.pos[0], F, 1.0, 1.0, RPY)) > 0
    # the Oseen truncation is not: the relative mode of two spheres goes negative at r < 1.5 a
    ev = np.linalg.eigvalsh(oracle.dense_mobility(two_spheres(1.4), 1.0, 1.0, OSEEN))
    assert ev.min() < 0


@pytest.mark.parametrize("tensor", [OSEEN, RPY])
@pytest.mark.parametrize("N", [1, 2, 3, 17, 64])
def test_P6_dense_tensor_brute_force(N, tensor):
    """the paper's own 'full tensor' method, H built entry by entry in the printed
    form of Eq. (3), times F, equals the matrix-free sum (which uses the contracted form)."""
    X, F = inputs.ragged_case(N, 100 + N)
    a, eta = 0.8, 1.7
    u = oracle.mobility_apply(X, F, a, eta, tensor)
    H = oracle.dense_mobility(X, a, eta, tensor)
    np.testing.assert_allclose(u.ravel(), H @ F.ravel(), rtol=0, atol=2e-15 * np.abs(u).max())


@pytest.mark.parametrize("tensor", [OSEEN, RPY])
def test_translation_rotation_permutation(tensor):
    """The tensor depends on x_alpha - x_beta only; it is an isotropic tensor function (rotating
    positions and forces rotates velocities); relabelling spheres relabels velocities."""
    X, F = inputs.ragged_case(33, 7)
    u = oracle.mobility_apply(X, F, 1.0, 1.0, tensor)
    s = np.abs(u).max()
    u_t = oracle.mobility_apply(X + np.array([3.0, -40.0, 7.5]), F, 1.0, 1.0, tensor)
    assert np.abs(u_t - u).max() < 1e-12 * s
    Q, _ = np.linalg.qr(np.random.default_rng(1).standard_normal((3, 3)))
    u_r = oracle.mobility_apply(X @ Q.T, F @ Q.T, 1.0, 1.0, tensor)
    assert np.abs(u_r - u @ Q.T).max() < 1e-13 * s
    perm = np.random.default_rng(2).permutation(33)
    u_p = oracle.mobility_apply(X[perm], F[perm], 1.0, 1.0, tensor)
    assert np.abs(u_p - u[perm]).max() < 1e-14 * s
    # linear in F; scales as 1/eta
    u2 = oracle.mobility_apply(X, 2.5 * F, 1.0, 2.0, tensor)
    assert np.abs(u2 - 1.25 * u).max() < 1e-14 * s


# ----------------------------------------------------------------------------- P5
def test_P5_forces_are_minus_grad_U_force_free_torque_free():
    """Eq. (4): F = -dU/dX with U = sum (k0/2)(d - L(t))^2, checked by central
    differences of U; Eq. (A22)-(A24) PAPER.md:445-460: each dumbbell is force free (bitwise) and
    torque free (F parallel to n)."""
    w = inputs.config2()
    p = Params(k0=37.0)
    t = 0.3731
    rng = np.random.default_rng(9)
    X = w.pos[0] + rng.uniform(-0.7, 0.7, w.pos[0].shape)   # off the minima
    phi = w.phase[0]

    def U(Xq):
        d = np.linalg.norm(Xq[1::2] - Xq[0::2], axis=1)
        L = p.ell + p.lam * np.sin(p.omega * t + phi)
        return 0.5 * p.k0 * np.sum((d - L) ** 2)

    F = oracle.forces(X, phi, t, p)
    h = 1e-6
    for (al, i) in [(0, 0), (1, 2), (50, 1), (127, 0), (64, 2)]:
        Xp, Xm = X.copy(), X.copy()
        Xp[al, i] += h
        Xm[al, i] -= h
        assert abs(F[al, i] + (U(Xp) - U(Xm)) / (2 * h)) < 1e-6 * np.abs(F).max()
    assert np.array_equal(F[0::2], -F[1::2])
    n = X[1::2] - X[0::2]
    assert np.abs(np.cross(n, F[0::2])).max() < 1e-12 * np.abs(F).max() * np.abs(n).max()
    # sign (reading R6): a stretched spring (d > L) pulls sphere 1 towards sphere 2
    Xs = np.array([[0.0, 0, 0], [15.0, 0, 0]])
    Fs = oracle.forces(Xs, np.array([0.0]), 0.0, Params())
    assert Fs[0, 0] > 0 and Fs[1, 0] < 0 and abs(Fs[0, 0] - 1000.0 * 5.0) < 1e-9
    # at the potential minima (input recipe) the force vanishes at t = 0
    F0 = oracle.forces(w.pos[0], phi, 0.0, Params())
    assert np.abs(F0).max() < 1e-9


# ----------------------------------------------------------------------------- P7, P8
def test_P7_isolated_dumbbell_does_not_translate():
    """I^sigma = 0, Eq. (A44); scallop theorem PAPER.md:22; the authors' acceptance
    check 'single dumbbells did not translate'."""
    n = np.array([1.0, 2.0, -0.5])
    n /= np.linalg.norm(n)
    phi = np.array([0.9])
    R0 = np.array([[3.0, -1.0, 2.0]])
    X0 = inputs.place_spheres(R0, n[None], phi)
    for tensor in (OSEEN, RPY):
        p = Params(tensor=tensor)
        V = oracle.velocity(X0 + np.array([[0.3, 0, 0], [0, 0, 0]]), phi, 0.1, p)
        assert np.abs(V[0] + V[1]).max() <= 1e-15 * np.abs(V).max()
        X = oracle.step(X0, phi, 0.0, 0, 3000, p)
        assert np.abs(0.5 * (X[0] + X[1]) - R0[0]).max() < 1e-12
        nn = (X[1] - X[0]) / np.linalg.norm(X[1] - X[0])
        assert np.abs(nn - n).max() < 1e-12          # and does not rotate
        assert abs(np.linalg.norm(X[1] - X[0]) - 10.0) < 2.5   # still a dumbbell of length ~ ell


def test_P8_isolated_dumbbell_length_relaxation_A37():
    """Eq. (A29a), (A36), (A37) PAPER.md:484-535 with the Oseen tensor: for one dumbbell
    d(d)/dt = b f1, b = (4 kappa / d)(1 - 2d/(3a)), kappa = 1/(8 pi mu), f1 = force on sphere 1
    along n.  Pins self mobility, the factor 2 of the parallel Oseen mode and the force sign."""
    a, eta, k0 = 1.0, 1.0, 1000.0
    p = Params(a=a, eta=eta, k0=k0, tensor=OSEEN)
    phi = np.array([0.4])
    t = 0.17
    for d in (8.3, 10.0, 11.9):
        X = np.array([[0.0, 0, 0], [0.0, d, 0]])
        V = oracle.velocity(X, phi, t, p)
        ddot = V[1, 1] - V[0, 1]
        L = p.ell + p.lam * np.sin(p.omega * t + phi[0])
        f1 = k0 * (d - L)                         # on sphere 1, along n = +y (R6)
        kappa = 1 / (8 * PI * eta)
        b = 4 * kappa / d * (1 - 2 * d / (3 * a))
        assert abs(ddot - b * f1) <= 1e-13 * abs(b * f1)


def test_P8_lag_amplitude_and_stroke_frequency():
    """Linear response of d - L to L(t) = ell + lam sin(omega t + phi) with relaxation
    rate Gamma = -k0 b(ell) from (A37): amplitude lam omega / sqrt(Gamma^2 + omega^2); the lag is
    the 'sphere positions lag very slightly behind the potentials' of PAPER.md:238.  Pins the
    time dependence of the rest length and the integrator's time argument."""
    lam = 0.05
    p = Params(lam=lam, tensor=OSEEN, dt=5e-4)
    phi = np.array([1.1])
    X0 = inputs.place_spheres(np.zeros((1, 3)), np.array([[0.0, 0, 1.0]]), phi, lam=lam)
    nsteps = 6000
    _, traj = oracle.step_record(X0, phi, 0.0, 0, nsteps, p, 1)
    tt = p.dt * np.arange(1, nsteps + 1)
    d = np.linalg.norm(traj[:, 1] - traj[:, 0], axis=1)
    dev = (d - (p.ell + lam * np.sin(p.omega * tt + phi[0])))[-2000:]     # last period
    kappa = 1 / (8 * PI * p.eta)
    Gamma = -p.k0 * 4 * kappa / p.ell * (1 - 2 * p.ell / (3 * p.a))
    want = lam * p.omega / np.hypot(Gamma, p.omega)
    got = 0.5 * (dev.max() - dev.min())
    assert abs(got - want) < 0.01 * want
    # d itself oscillates with the stroke period T = 1 about ell with amplitude ~ lam
    dl = d[-2000:]
    assert abs(0.5 * (dl.max() - dl.min()) - lam * Gamma / np.hypot(Gamma, p.omega)) < 0.01 * lam
    assert abs(dl.mean() - p.ell) < 1e-3 * lam


# ----------------------------------------------------------------------------- P9
def _pair_drift(a, ell, lam, D, dphi, tensor=RPY, k0=None, steps_per_period=1000):
    """Displacement of both centres over the second stroke period (first discarded,
    PAPER.md:238) for two dumbbells aligned on the x axis, centres D apart."""
    if k0 is None:
        # same integrator loading Gamma dt ~ 0.09 as the paper's Fig. 1 (reading R1)
        k0 = 90.2 / (2 * (1 / (6 * PI * a) - 1 / (4 * PI * ell)))
    p = Params(a=a, ell=ell, lam=lam, k0=k0, dt=1.0 / steps_per_period, tensor=tensor)
    phi = np.array([0.3, 0.3 + dphi])
    R = np.array([[0.0, 0, 0], [D, 0, 0]])
    n = np.array([[1.0, 0, 0], [1.0, 0, 0]])
    X0 = inputs.place_spheres(R, n, phi, ell=ell, lam=lam)
    X1 = oracle.step(X0, phi, 0.0, 0, steps_per_period, p)
    X2 = oracle.step(X1, phi, 0.0, steps_per_period, steps_per_period, p)
    c1 = 0.5 * (X1[0::2] + X1[1::2])
    c2 = 0.5 * (X2[0::2] + X2[1::2])
    return (c2 - c1)[:, 0], np.abs((c2 - c1)[:, 1:]).max()


def _eq10(a, ell, lam, D, dphi, omega=2 * PI, T=1.0):
    """Eq. (10) PAPER.md:147 for S = 2 over one period: both centres move by
    (9/16) a omega sin(phi2 - phi1) (lam/ell)^2 (ell/D)^4 T along +x."""
    return 9.0 / 16.0 * a * omega * np.sin(dphi) * (lam / ell) ** 2 * (ell / D) ** 4 * T


def test_P9_aligned_pair_vs_stroke_averaged_eq10():
    """PAPER.md:147 Eq. (10), 160-162, Fig. 1: symmetric aligned dumbbells move in the same
    direction with identical speeds, direction set by phi2 - phi1, no motion for phase differences
    that are multiples of pi, displacement per stroke ~ D^-4, and the ratio to Eq. (10) tends to 1
    as a/ell -> 0 at constant lam (Fig. 1c)."""
    a, lam = 1.0, 1.0
    dx, off = _pair_drift(a, 10.0, lam, 100.0, PI / 2)
    assert off < 1e-15
    assert dx[0] > 0 and dx[1] > 0 and abs(dx[0] - dx[1]) < 2e-3 * abs(dx[0])
    ref = _eq10(a, 10.0, lam, 100.0, PI / 2)
    assert 1.0 < dx.mean() / ref < 1.3            # a/ell = 0.1: above Eq. (10), Fig. 1(c)
    dxm, _ = _pair_drift(a, 10.0, lam, 100.0, -PI / 2)
    assert abs(dxm.mean() + dx.mean()) < 0.02 * dx.mean()      # reversed phase lag reverses the motion
    for dphi in (0.0, PI):
        d0, _ = _pair_drift(a, 10.0, lam, 100.0, dphi)
        assert np.abs(d0).max() < 1e-3 * dx.mean()
    dhalf, _ = _pair_drift(a, 10.0, lam, 100.0, PI / 6)        # sin(pi/6) = 1/2
    assert abs(dhalf.mean() / dx.mean() - 0.5) < 0.02
    dnear, _ = _pair_drift(a, 10.0, lam, 50.0, PI / 2)
    assert abs(dnear.mean() / dx.mean() - 16.0) < 1.0          # D^-4
    ratios = []
    for ell in (5.0, 10.0, 20.0, 40.0):                        # a/ell = 0.2 ... 0.025, D = 10 ell
        d, _ = _pair_drift(a, ell, lam, 10 * ell, PI / 2)
        ratios.append(d.mean() / _eq10(a, ell, lam, 10 * ell, PI / 2))
    assert all(r1 > r2 for r1, r2 in zip(ratios, ratios[1:])), ratios
    assert 1.2 < ratios[0] < 1.5 and abs(ratios[-1] - 1.0) < 0.07, ratios
    # Oseen and RPY agree to a few per cent in the dilute, slender regime
    do, _ = _pair_drift(a, 10.0, lam, 100.0, PI / 2, tensor=OSEEN)
    assert abs(do.mean() / dx.mean() - 1.0) < 0.05


# ----------------------------------------------------------------------------- P10
def test_P10_integrator_order():
    """one-step Heun predictor-corrector is 2nd order, Euler 1st."""
    X0, phase = inputs.random_suspension(3, 77, side=40.0)
    T_end = 0.064
    errs = {}
    for integ in (EULER, HEUN):
        pref = Params(integrator=HEUN, dt=T_end / 4096, k0=200.0)
        Xref = oracle.step(X0, phase, 0.0, 0, 4096, pref)
        e = []
        for n in (64, 128, 256):
            p = Params(integrator=integ, dt=T_end / n, k0=200.0)
            e.append(np.abs(oracle.step(X0, phase, 0.0, 0, n, p) - Xref).max())
        errs[integ] = e
    rh = [errs[HEUN][i] / errs[HEUN][i + 1] for i in range(2)]
    re = [errs[EULER][i] / errs[EULER][i + 1] for i in range(2)]
    assert all(3.5 < r < 4.6 for r in rh), rh
    assert all(1.8 < r < 2.3 for r in re), re


def test_step_bookkeeping_time_from_step_index():
    """Reading R7: t_n = t0 + n dt from the integer step count, so n steps in one call equal the
    same n steps split over several calls, bit for bit; t0 shifts the stroke phase."""
    w = inputs.config1()
    p = Params()
    Xa = oracle.step(w.pos[0], w.phase[0], 0.25, 0, 40, p)
    Xb = oracle.step(w.pos[0], w.phase[0], 0.25, 0, 15, p)
    Xb = oracle.step(Xb, w.phase[0], 0.25, 15, 25, p)
    assert np.array_equal(Xa, Xb)
    # omega t0 = 2 pi * 1.0 is a full period: same forces as t0 = 0 up to rounding of the argument
    F0 = oracle.forces(w.pos[0] * 1.01, w.phase[0], 0.0, p)
    F1 = oracle.forces(w.pos[0] * 1.01, w.phase[0], 1.0, p)
    assert np.abs(F0 - F1).max() < 1e-9 * np.abs(F0).max()
    # threads do not change a bit
    X, F = inputs.apply_case(300, 5, 6)
    oracle.set_threads(1)
    u1 = oracle.mobility_apply(X, F, 1.0, 1.0, RPY)
    oracle.set_threads(4)
    u4 = oracle.mobility_apply(X, F, 1.0, 1.0, RPY)
    oracle.set_threads(1)
    assert np.array_equal(u1, u4)


# --------------------------------------------------------------------------------- observables, Eq. (6a,b), (13)
def test_P11_dumbbell_coordinates_closed_forms():
    """PAPER.md:87-91 Eq. (6a), (6b).  A dumbbell placed at centre R along unit vector n with length L has exactly
    that centre and direction (the input generator places spheres at R -/+ (L/2) n); swapping the two
    spheres flips N and keeps R; translating by d shifts R by d and keeps N; N has unit length."""
    rng = np.random.default_rng(11)
    S = 7
    Rc = rng.uniform(-50, 50, (S, 3))
    n = rng.standard_normal((S, 3)); n /= np.linalg.norm(n, axis=1, keepdims=True)
    L = rng.uniform(8, 12, S)
    X = np.empty((2 * S, 3)); X[0::2] = Rc - 0.5 * L[:, None] * n; X[1::2] = Rc + 0.5 * L[:, None] * n
    R, N = oracle.dumbbell_coords(X)
    np.testing.assert_allclose(R, Rc, rtol=0, atol=1e-13)
    np.testing.assert_allclose(N, n, rtol=0, atol=1e-14)
    np.testing.assert_allclose(np.linalg.norm(N, axis=1), 1.0, rtol=0, atol=1e-15)
    Xs = X.copy(); Xs[0::2], Xs[1::2] = X[1::2], X[0::2]
    R2, N2 = oracle.dumbbell_coords(Xs)
    assert np.array_equal(R2, R) and np.array_equal(N2, -N)
    d = np.array([3.0, -4.0, 12.0])
    R3, N3 = oracle.dumbbell_coords(X + d)
    np.testing.assert_allclose(R3 - R, np.broadcast_to(d, R.shape), rtol=0, atol=1e-13)
    np.testing.assert_allclose(N3, N, rtol=0, atol=1e-14)


def test_P12_msd_closed_forms():
    """PAPER.md:189 Eq. (13).  (i) zero displacement -> 0; (ii) every centre moved by the same vector d -> |d|^2
    (3-4-12 triangle: 169 exactly); (iii) W realisations moved by different d_w -> the mean of |d_w|^2;
    (iv) one dumbbell of S moved by d -> |d|^2 / S; (v) brute force with numpy on random data."""
    rng = np.random.default_rng(12)
    W, S = 5, 9
    R0 = rng.uniform(-30, 30, (W, S, 3))
    assert oracle.msd(R0, R0) == 0.0
    assert oracle.msd(R0 + np.array([3.0, 4.0, 12.0]), R0) == pytest.approx(169.0, rel=1e-14)
    dw = rng.standard_normal((W, 1, 3))
    assert oracle.msd(R0 + dw, R0) == pytest.approx(float(np.mean(np.sum(dw ** 2, axis=-1))), rel=1e-13)
    Rt = R0.copy(); Rt[2, 4] += np.array([1.0, 2.0, 2.0])
    assert oracle.msd(Rt, R0) == pytest.approx(9.0 / (S * W), rel=1e-13)
    Rt = R0 + rng.standard_normal(R0.shape)
    assert oracle.msd(Rt, R0) == pytest.approx(float(np.mean(np.sum((Rt - R0) ** 2, axis=-1))), rel=1e-13)


def test_P13_isolated_dumbbell_has_no_msd():
    """Scallop theorem / I^sigma = 0: the centre of an isolated deterministic dumbbell does not
    move, so Eq. (13) of a one-dumbbell system stays at rounding level over a period, while its direction is constant."""
    p = oracle.Params()
    phi = np.array([0.7])
    n = np.array([[0.3, -0.5, 0.8]]); n /= np.linalg.norm(n)
    X0 = inputs.place_spheres(np.array([[1.0, 2.0, 3.0]]), n, phi)
    R0, N0 = oracle.dumbbell_coords(X0)
    X = oracle.step(X0, phi, 0.0, 0, 1000, p)
    R, N = oracle.dumbbell_coords(X)
    assert oracle.msd(R[None], R0[None]) < 1e-24
    np.testing.assert_allclose(N, N0, rtol=0, atol=1e-12)


# --------------------------------------------------------------------------------- Brownian term, additive approximation
def test_P14_philox_known_answers():
    """The generator is Philox4x32-10 as published: tests/golden/philox4x32_10_kat.txt (Salmon et al., SC'11)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_P15_increments_are_standard_normal_and_independent():
    """Eq. (1b), (1c): <xi> = 0, <xi xi'> = delta: unit variance, no correlation between steps, spheres /
    components, realisations or seeds (counter-based draws: sample moments within 4 standard errors)."""
    n = 40000
    z = np.array([oracle.noise_normal(7, k, 0, 0) for k in range(n)])
    ze = np.array([oracle.noise_normal(7, 0, 0, k) for k in range(n)])
    zs = np.array([oracle.noise_normal(7, 0, k, 0) for k in range(n)])
    z2 = np.array([oracle.noise_normal(8, k, 0, 0) for k in range(n)])
    for v in (z, ze, zs, z2):
        assert abs(v.mean()) < 4 / np.sqrt(n)
        assert abs(v.var() - 1.0) < 4 * np.sqrt(2.0 / n)
        assert abs(np.mean(v ** 4) - 3.0) < 4 * np.sqrt(96.0 / n)
        assert abs(np.mean(v[1:] * v[:-1])) < 4 / np.sqrt(n)
    for a, b in ((z, ze), (z, zs), (z, z2), (ze, zs)):
        assert abs(np.mean(a * b)) < 4 / np.sqrt(n)
    assert oracle.noise_normal(7, 5, 2, 11) == oracle.noise_normal(7, 5, 2, 11)      # a pure function of its counter


def test_P16_isolated_dumbbell_centre_is_the_sum_of_its_increments():
    """Additive noise, with the shared-increment Heun step: for an isolated dumbbell the
    deterministic velocities of the two spheres cancel (I^sigma = 0), so the centre moves by exactly
    (dW_1 + dW_2)/2 per step, dW = sqrt(2 kT dt / (6 pi eta a)) z.  Checked against the generator's own draws, and the
    ensemble mean square displacement against 6 D_R t with D_R = kT / (12 pi eta a)."""
    kT, seed, nst = 0.05, 99, 60
    p = oracle.Params(kT=kT, seed=seed, system=3)
    phi = np.array([1.1])
    n = np.array([[0.2, 0.9, -0.4]]); n /= np.linalg.norm(n)
    X0 = inputs.place_spheres(np.array([[0.0, 0.0, 0.0]]), n, phi)
    X = oracle.step(X0, phi, 0.0, 0, nst, p)
    amp = np.sqrt(2 * kT * p.dt / (6 * np.pi * p.eta * p.a))
    expect = np.zeros(3)
    for m in range(nst):
        for c in range(3):
            expect[c] += 0.5 * amp * (oracle.noise_normal(seed, m, 3, c) + oracle.noise_normal(seed, m, 3, 3 + c))
    R0, _ = oracle.dumbbell_coords(X0); R, _ = oracle.dumbbell_coords(X)
    np.testing.assert_allclose((R - R0)[0], expect, rtol=0, atol=1e-13)
    # ensemble: W realisations (system index w), MSD of the centre = 3 * (2 D_R) t = kT t / (2 pi eta a)
    W = 400
    disp2 = []
    for w_ in range(W):
        Xw = oracle.step(X0, phi, 0.0, 0, nst, oracle.Params(kT=kT, seed=seed, system=w_))
        disp2.append(np.sum((oracle.dumbbell_coords(Xw)[0] - R0) ** 2))
    theory = kT * nst * p.dt / (2 * np.pi * p.eta * p.a)
    assert abs(np.mean(disp2) / theory - 1.0) < 4 * np.sqrt(2.0 / (3 * W))


def test_P17_zero_temperature_is_the_deterministic_path():
    """kT = 0 is the deterministic limit: bit-identical to a run that never heard of the noise term; a
    different seed changes nothing then, and at kT > 0 Euler's first step is X + dt V + dW exactly."""
    w = inputs.config1()
    a = oracle.step(w.pos[0], w.phase[0], 0.0, 0, 50, oracle.Params())
    b = oracle.step(w.pos[0], w.phase[0], 0.0, 0, 50, oracle.Params(kT=0.0, seed=1234, system=9))
    assert np.array_equal(a, b)
    pe = oracle.Params(integrator=oracle.EULER, kT=0.3, seed=5)
    V = oracle.velocity(w.pos[0], w.phase[0], 0.0, pe)
    amp = np.sqrt(2 * pe.kT * pe.dt / (6 * np.pi))
    dW = amp * np.array([oracle.noise_normal(5, 0, 0, k) for k in range(w.N * 3)]).reshape(w.N, 3)
    X1 = oracle.step(w.pos[0], w.phase[0], 0.0, 0, 1, pe)
    np.testing.assert_allclose(X1, w.pos[0] + pe.dt * V + dW, rtol=0, atol=1e-13)


# --------------------------------------------------------------------------------- stroke-averaged model, Eq. (9)
def _random_RN(rng, S, side=400.0):
    R = rng.uniform(-side / 2, side / 2, (S, 3))
    N = rng.standard_normal((S, 3)); N /= np.linalg.norm(N, axis=1, keepdims=True)
    return R, N, rng.uniform(0, 2 * np.pi, S)


def test_P18_aligned_dumbbells_reduce_to_eq10():
    """PAPER.md:147 Eq. (10): for aligned dumbbells (all N along the common axis, either sign) Eq. (9a) reduces to
    dR^s/dt = (9/16) a w sum_r sin(phi^s - phi^r) (lam/ell)^2 (ell/|D|)^4 Dh, and the orientations do not change."""
    rng = np.random.default_rng(18)
    p = oracle.Params(a=0.7, ell=9.0, lam=1.5, omega=5.0)
    S = 6
    axis = np.array([2.0, -1.0, 0.5]); axis /= np.linalg.norm(axis)
    pos = np.cumsum(rng.uniform(30, 80, S))
    R = pos[:, None] * axis
    sign = np.array([1, -1, 1, 1, -1, 1])[:, None]
    N = sign * axis
    phi = rng.uniform(0, 2 * np.pi, S)
    dR, dN = oracle.avg_rhs(R, N, phi, p)
    expect = np.zeros((S, 3))
    for s in range(S):
        for r in range(S):
            if r != s:
                D = R[s] - R[r]; Dn = np.linalg.norm(D)
                expect[s] += 9 / 16 * p.a * p.omega * np.sin(phi[s] - phi[r]) * (p.lam / p.ell) ** 2 * (p.ell / Dn) ** 4 * D / Dn
    np.testing.assert_allclose(dR, expect, rtol=1e-12, atol=1e-18)
    assert np.abs(dN).max() < 1e-17


def test_P19_structure_of_the_averaged_interactions():
    """J ~ |D|^-4, K ~ |D|^-5, both vanish when the phases differ by multiples of pi; (9b) keeps N on the
    unit sphere (N . dN/dt = 0); the equations are covariant under rotations; relabelling the two identical spheres of a
    dumbbell (N -> -N, same stroke phase) changes nothing physical (dR equal, that dumbbell's dN flips with its N)."""
    rng = np.random.default_rng(19)
    p = oracle.Params()
    S = 9
    R, N, phi = _random_RN(rng, S)
    dR, dN = oracle.avg_rhs(R, N, phi, p)
    assert np.abs(np.sum(N * dN, axis=1)).max() < 1e-20 + 1e-12 * np.abs(dN).max()
    dR2, dN2 = oracle.avg_rhs(3.0 * R, N, phi, p)
    np.testing.assert_allclose(dR2, dR / 3.0 ** 4, rtol=1e-12)
    np.testing.assert_allclose(dN2, dN / 3.0 ** 5, rtol=1e-12)
    for shift in (0.0, np.pi):
        phis = np.full(S, 0.3) + shift * (np.arange(S) % 2)
        a, b = oracle.avg_rhs(R, N, phis, p)
        assert np.abs(a).max() < 1e-18 and np.abs(b).max() < 1e-20
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    dRq, dNq = oracle.avg_rhs(R @ Q.T, N @ Q.T, phi, p)
    np.testing.assert_allclose(dRq, dR @ Q.T, rtol=1e-11, atol=1e-20)
    np.testing.assert_allclose(dNq, dN @ Q.T, rtol=1e-11, atol=1e-22)
    Nf = N.copy()
    Nf[2] *= -1
    dRf, dNf = oracle.avg_rhs(R, Nf, phi, p)
    np.testing.assert_allclose(dRf, dR, rtol=1e-11, atol=1e-20)
    np.testing.assert_allclose(dNf[2], -dN[2], rtol=1e-11, atol=1e-22)
    np.testing.assert_allclose(np.delete(dNf, 2, 0), np.delete(dN, 2, 0), rtol=1e-11, atol=1e-22)


def test_P20_averaged_model_matches_the_microscopic_one_in_the_far_field():
    """for slender, distant dumbbells the stroke-averaged equations reproduce the microscopic
    (spring-based) dynamics.  Two non-aligned dumbbells, a/ell = 0.0125, lam/ell = 0.05, D = 6 ell, Oseen tensor (the
    tensor the averaged model is derived from): per-period drift of the centre within 4 % and per-period rotation of
    the direction within 8 % of Eq. (9) with the printed prefactors 9/64, 15/64 and the minus sign of (9b) (this fixes
    the reading of the garbled (9c), R14; a factor 2 or a sign error in K fails here)."""
    a, ell, lam, Dsep, dt, periods = 0.125, 10.0, 0.5, 60.0, 1e-3, 6
    b = 2 * (1 / (6 * np.pi * a) - 1 / (4 * np.pi * ell))
    p = oracle.Params(a=a, ell=ell, lam=lam, k0=0.09 / dt / b, dt=dt, tensor=oracle.OSEEN)
    phi = np.array([0.0, np.pi / 2])
    Nn = np.array([[1.0, 0.6, 0.0], [0.3, 1.0, 0.2]]); Nn /= np.linalg.norm(Nn, axis=1, keepdims=True)
    X0 = inputs.place_spheres(np.array([[0.0, 0, 0], [Dsep, 0, 0]]), Nn, phi, ell=ell, lam=lam)
    nper = int(round(1 / dt))
    X1 = oracle.step(X0, phi, 0.0, 0, nper, p)                       # the first period is discarded
    X2 = oracle.step(X1, phi, 0.0, nper, nper * periods, p)
    Ra, Na = oracle.dumbbell_coords(X1); Rb, Nb = oracle.dumbbell_coords(X2)
    dR_micro, dN_micro = (Rb - Ra) / periods, (Nb - Na) / periods     # per period T = 1
    dR_avg, dN_avg = oracle.avg_rhs(Ra, Na, phi, p)
    for s in (0, 1):
        assert np.linalg.norm(dR_micro[s] - dR_avg[s]) <= 0.04 * np.linalg.norm(dR_avg[s])
    # dumbbell 0 is the one whose leading-order rotation does not vanish by geometry
    assert np.linalg.norm(dN_micro[0] - dN_avg[0]) <= 0.08 * np.linalg.norm(dN_avg[0])
    # stepping the averaged model over the same 6 periods lands on the microscopic centres / directions likewise
    Rs, Ns = oracle.avg_step(Ra, Na, phi, 0.5, 2 * periods, p)
    assert np.linalg.norm((Rs - Ra)[0] - (Rb - Ra)[0]) <= 0.04 * np.linalg.norm((Rb - Ra)[0])
    np.testing.assert_allclose(np.linalg.norm(Ns, axis=1), 1.0, rtol=0, atol=1e-15)


# --------------------------------------------------------------------------------- P21, P22: the two integrators
def _avg_case():
    """Three non-aligned dumbbells two to three lengths apart: the directions turn by tens of degrees over the test."""
    R = np.array([[0.0, 0.0, 0.0], [22.0, 3.0, -2.0], [5.0, 24.0, 6.0]])
    N = np.array([[1.0, 0.6, 0.0], [0.3, 1.0, 0.2], [-0.5, 0.2, 1.0]])
    N /= np.linalg.norm(N, axis=1, keepdims=True)
    return R, N, np.array([0.0, np.pi / 2, 2.2])


def test_P21_averaged_model_integrator_is_second_order_heun():
    """PAPER.md:236 and reading R16: Eq. (9) is stepped with the one-step Heun predictor-corrector, N
    renormalised after the predictor and after the corrector.  (a) Order: against a reference at dt/256 the error at
    dt, dt/2, dt/4, dt/8 falls by about 4 per halving (a plain-Euler corrector gives about 2 and fails).  (b) One step
    rebuilt from the already pinned right-hand side (P18-P20): R + dt/2 (f(R, N) + f(R*, N*/|N*|)), N likewise and
    normalised, equals avg_step to rounding; leaving out either renormalisation, or the corrector, is far outside."""
    p = oracle.Params()
    R, N, phi = _avg_case()
    T_end = 4000.0
    Rr, Nr = oracle.avg_step(R, N, phi, T_end / 4096, 4096, p)
    turn = np.degrees(np.arccos(np.clip(np.sum(N * Nr, axis=1), -1, 1)))
    assert turn.max() > 30.0                       # N turns visibly: the (9b) part of the integrator is exercised
    eR, eN = [], []
    for n in (16, 32, 64, 128):
        Rn, Nn = oracle.avg_step(R, N, phi, T_end / n, n, p)
        eR.append(np.abs(Rn - Rr).max()); eN.append(np.abs(Nn - Nr).max())
    for e in (eR, eN):
        ratios = [e[i] / e[i + 1] for i in range(3)]
        assert all(3.6 < r < 4.4 for r in ratios), ratios
    # (b) one large step from pinned parts
    dt = 250.0
    unit = lambda v: v / np.linalg.norm(v, axis=1, keepdims=True)

    def one_step(renorm_pred=True, renorm_end=True, corrector=True):
        dR1, dN1 = oracle.avg_rhs(R, N, phi, p)
        Rp, Np = R + dt * dR1, N + dt * dN1
        if renorm_pred:
            Np = unit(Np)
        if not corrector:
            return Rp, unit(Np)
        dR2, dN2 = oracle.avg_rhs(Rp, Np, phi, p)
        R1, N1 = R + 0.5 * dt * (dR1 + dR2), N + 0.5 * dt * (dN1 + dN2)
        return R1, (unit(N1) if renorm_end else N1)

    Ro, No = oracle.avg_step(R, N, phi, dt, 1, p)
    Ra, Na = one_step()
    np.testing.assert_allclose(Ra, Ro, rtol=0, atol=1e-13)
    np.testing.assert_allclose(Na, No, rtol=0, atol=1e-15)
    np.testing.assert_allclose(np.linalg.norm(No, axis=1), 1.0, rtol=0, atol=1e-15)
    for kw in (dict(renorm_pred=False), dict(renorm_end=False), dict(corrector=False)):
        Rb, Nb = one_step(**kw)
        assert max(np.abs(Rb - Ro).max(), np.abs(Nb - No).max()) > 1e-6, kw      # the pin tells these readings apart
    # two steps in one call = two calls of one step (no hidden state)
    R2, N2 = oracle.avg_step(R, N, phi, dt, 2, p)
    R2b, N2b = oracle.avg_step(Ro, No, phi, dt, 1, p)
    assert np.array_equal(R2, R2b) and np.array_equal(N2, N2b)


@pytest.mark.parametrize("tensor", [OSEEN, RPY])
def test_P22_heun_with_additive_noise_shares_the_increment(tensor):
    """PAPER.md:236 ("can easily incorporate additive noise"), reading R15: with k_B T > 0 one increment
    dW per step enters the predictor AND the corrector:
        X* = X + dt V(X, t_n) + dW,   X_{n+1} = X + dt/2 (V(X, t_n) + V(X*, t_{n+1})) + dW.
    Three steps rebuilt from the pinned parts (oracle.velocity: P1-P8; oracle.noise_normal: P14, P15) equal oracle.step
    to rounding; a predictor without dW, a corrector evaluated at t_n, or increments drawn with the wrong step index
    are far outside (the increments are ~ 2e-3, the readings differ by ~ 1e-4)."""
    kT, seed, system, t0 = 0.05, 11, 2, 0.3
    p = oracle.Params(kT=kT, seed=seed, system=system, tensor=tensor)
    X0, phase = inputs.random_suspension(2, 5, side=30.0)
    dt = p.dt
    amp = np.sqrt(2 * kT * dt / (6 * np.pi * p.eta * p.a))

    def rebuild(pred_noise=True, t_corr_shift=1, index_shift=0):
        X = X0.copy()
        for n in range(3):
            dW = amp * np.array([oracle.noise_normal(seed, n + index_shift, system, k) for k in range(X.size)]).reshape(X.shape)
            V1 = oracle.velocity(X, phase, t0 + n * dt, p)
            Xp = X + dt * V1 + (dW if pred_noise else 0.0)
            V2 = oracle.velocity(Xp, phase, t0 + (n + t_corr_shift) * dt, p)
            X = X + 0.5 * dt * (V1 + V2) + dW
        return X

    Xo = oracle.step(X0, phase, t0, 0, 3, p)
    np.testing.assert_allclose(rebuild(), Xo, rtol=0, atol=1e-13)
    assert np.abs(rebuild(pred_noise=False) - Xo).max() > 1e-5
    assert np.abs(rebuild(t_corr_shift=0) - Xo).max() > 1e-7
    assert np.abs(rebuild(index_shift=1) - Xo).max() > 1e-4
    # steps 1..2 of a run that starts at n_done = 1 use the increments of steps 1 and 2 (counter = absolute step index)
    X1 = oracle.step(X0, phase, t0, 0, 1, p)
    assert np.array_equal(oracle.step(X1, phase, t0, 1, 2, p), Xo)
