"""Seeded synthetic inputs shaped like the workloads of arXiv 1004.1932.

This module serves both the CPU oracle's tests and the CUDA path's tests/bench; it holds
none of the method's arithmetic (no mobility tensor, no force law, no integrator) and imports
neither of them.  It only places dumbbells: centres, orientations, phases, and the spheres at
the spring's potential minima at t = 0 ("we initially placed the spheres
centred at the potential minima", i.e. X = R -/+ (1/2) L(0) n with L(0) = ell + lambda sin(phi),
PAPER.md:67, A14c PAPER.md:382).

The paper uses no public dataset; its workloads are 1d aligned lines and
3d lattices / arrays with orientations uniform on the sphere and phases uniform in [0, 2 pi)
(PAPER.md:187-200).  The recipes below restate BASELINE.json's five configs (DESIGN.md
"Input recipe").  Units: a = eta = T = 1.

Draw order (fixed, so a seed names one input): centres first (all dumbbells), then
orientations (3 Gaussians each, normalised), then phases.
"""
from dataclasses import dataclass, field

import numpy as np

A, ELL, LAM, OMEGA, K0, DT = 1.0, 10.0, 2.0, 2.0 * np.pi, 1000.0, 1e-3
HARD_CORE = 2.5 * A           # BASELINE.json config 3: "hard-core rejection at 2.5a"
SPACING_RANDOM = 4.0 * ELL    # number density 1/(4L)^3


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # [B][N][3] float64 (B = 1 for single systems)
    phase: np.ndarray          # [B][S]    float64
    scalars: dict = field(default_factory=lambda: dict(a=A, eta=1.0, ell=ELL, lam=LAM, omega=OMEGA, k0=K0, dt=DT))
    n_steps: int = 0
    seed: int = 0

    @property
    def S(self):
        return self.phase.shape[-1]

    @property
    def N(self):
        return 2 * self.S

    @property
    def B(self):
        return self.pos.shape[0]


def place_spheres(R, n, phase, ell=ELL, lam=LAM):
    """Spheres of dumbbell s at R_s -/+ (1/2)(ell + lam sin(phase_s)) n_s -> [2S][3]."""
    L0 = ell + lam * np.sin(phase)
    X = np.empty((2 * R.shape[0], 3), dtype=np.float64)
    X[0::2] = R - 0.5 * L0[:, None] * n
    X[1::2] = R + 0.5 * L0[:, None] * n
    return X


def _unit_vectors(rng, S):
    g = rng.standard_normal((S, 3))
    return g / np.linalg.norm(g, axis=1, keepdims=True)


def _min_cross_distance_violations(X, hard_core):
    """Indices of dumbbells that own a sphere closer than hard_core to a sphere of another
    dumbbell (the higher-numbered dumbbell of each offending pair)."""
    from scipy.spatial import cKDTree
    pairs = cKDTree(X).query_pairs(hard_core, output_type="ndarray")
    if pairs.size == 0:
        return np.empty(0, dtype=np.int64)
    d = pairs // 2
    cross = d[:, 0] != d[:, 1]
    return np.unique(np.maximum(d[cross, 0], d[cross, 1]))


def random_suspension(S, seed, side=None, hard_core=HARD_CORE):
    """S dumbbells with centres uniform in a cube of the given side centred on the origin
    (default: density 1/(4 ell)^3), orientations uniform on the sphere, phases uniform in
    [0, 2 pi).  Dumbbells owning a sphere within hard_core of another dumbbell's sphere are
    redrawn (centre, orientation; phase kept) until none is left."""
    rng = np.random.default_rng(seed)
    if side is None:
        side = SPACING_RANDOM * S ** (1.0 / 3.0)
    R = rng.uniform(-0.5 * side, 0.5 * side, size=(S, 3))
    n = _unit_vectors(rng, S)
    phase = rng.uniform(0.0, 2.0 * np.pi, size=S)
    for _ in range(1000):
        X = place_spheres(R, n, phase)
        bad = _min_cross_distance_violations(X, hard_core)
        if bad.size == 0:
            return X, phase
        R[bad] = rng.uniform(-0.5 * side, 0.5 * side, size=(bad.size, 3))
        n[bad] = _unit_vectors(rng, bad.size)
    raise RuntimeError("hard-core rejection did not converge")


def config1(seed=1001):
    """C1: 1d line of S = 8 dumbbells on the x axis, spaced D = 5 ell, all along +x, phases
    uniform in [0, 2 pi).  FP64, dt = 1e-3, 10^4 steps."""
    S = 8
    rng = np.random.default_rng(seed)
    R = np.zeros((S, 3))
    R[:, 0] = 5.0 * ELL * np.arange(S)
    n = np.tile(np.array([1.0, 0.0, 0.0]), (S, 1))
    phase = rng.uniform(0.0, 2.0 * np.pi, size=S)
    return Workload("C1_line_S8", place_spheres(R, n, phase)[None], phase[None], n_steps=10_000, seed=seed)


def config2(seed=1002):
    """C2: 4x4x4 cubic array, spacing 3 ell, centres jittered +/- 0.1 ell per component,
    orientations uniform on the sphere.  FP32 and FP64, 10^4 steps."""
    rng = np.random.default_rng(seed)
    g = np.arange(4) - 1.5
    R = 3.0 * ELL * np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    S = R.shape[0]
    R = R + rng.uniform(-0.1 * ELL, 0.1 * ELL, size=(S, 3))
    n = _unit_vectors(rng, S)
    phase = rng.uniform(0.0, 2.0 * np.pi, size=S)
    return Workload("C2_lattice_S64", place_spheres(R, n, phase)[None], phase[None], n_steps=10_000, seed=seed)


def config3(seed=1003):
    """C3: S = 512 random suspension, density 1/(4 ell)^3, hard core 2.5a.  FP32, 10^5 steps."""
    X, phase = random_suspension(512, seed)
    return Workload("C3_random_S512", X[None], phase[None], n_steps=100_000, seed=seed)


def config4(seed=1004):
    """C4: S = 2048 (N = 4096) random suspension, same density.  FP32 and FP64."""
    X, phase = random_suspension(2048, seed)
    return Workload("C4_random_S2048", X[None], phase[None], n_steps=1000, seed=seed)


def config5(B=64, S=256, seed=1005):
    """C5: B = 64 independent systems of S = 256 dumbbells, seeds seed + b.  FP32, 10^4 steps."""
    Xs, ps = zip(*(random_suspension(S, seed + b) for b in range(B)))
    return Workload(f"C5_batch_B{B}_S{S}", np.stack(Xs), np.stack(ps), n_steps=10_000, seed=seed)


def apply_case(N, seed_pos, seed_force):
    """Standalone mobility-apply input: N spheres of a random suspension of N/2 dumbbells at
    density 1/(4 ell)^3, forces i.i.d. N(0,1) per component (BASELINE.json config 4/5).
    Returns pos [N][3], F [N][3] (float64)."""
    assert N % 2 == 0
    X, _ = random_suspension(N // 2, seed_pos)
    F = np.random.default_rng(seed_force).standard_normal((N, 3))
    return X, F


def sweep_case(log2N):
    """Scaling-sweep member N = 2^log2N: positions seed 3000 + log2N, forces seed 4000 + log2N."""
    return apply_case(1 << log2N, 3000 + log2N, 4000 + log2N)


def ragged_case(N, seed):
    """Arbitrary N >= 1 spheres (odd allowed): uniform in a cube at the same sphere density,
    min separation 2.5a by redraw, forces N(0,1).  For edge-case parity of the stateless apply."""
    rng = np.random.default_rng(seed)
    side = SPACING_RANDOM * max(N / 2.0, 1.0) ** (1.0 / 3.0)
    X = rng.uniform(-0.5 * side, 0.5 * side, size=(N, 3))
    from scipy.spatial import cKDTree
    for _ in range(1000):
        pairs = cKDTree(X).query_pairs(HARD_CORE, output_type="ndarray")
        if pairs.size == 0:
            break
        bad = np.unique(pairs[:, 1])
        X[bad] = rng.uniform(-0.5 * side, 0.5 * side, size=(bad.size, 3))
    F = rng.standard_normal((N, 3))
    return X, F
