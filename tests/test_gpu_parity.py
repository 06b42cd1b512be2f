"""Parity of the CUDA path (through the C ABI, include/ds.h) with the CPU oracle, element by element
on the same seeded inputs.  Run on the B200 box: pytest -m gpu.

Tolerances (BASELINE.json north_star; error norms SURVEY.md 8(c) R13):
  mobility apply  FP64: ||u - u_or||_2 / ||u_or||_2 <= 1e-12     FP32: <= 1e-5
  trajectory      FP32: max |X - X_or| <= 1e-4 ell after 1000 steps
FP32 runs feed the oracle the SAME float32-rounded inputs (widened to double).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1004_1932_b200 import ds, inputs

pytestmark = pytest.mark.gpu

TOL = {ds.F32: 1e-5, ds.F64: 1e-12}
NPDT = {ds.F32: np.float32, ds.F64: np.float64}
TDT = {ds.F32: torch.float32, ds.F64: torch.float64}
ELL = inputs.ELL


@pytest.fixture(scope="module", autouse=True)
def _device():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    assert torch.cuda.get_device_capability(0)[0] == 10, "sm_100 device required"
    oracle.set_threads(oracle.max_threads())   # bit-identical at any thread count
    yield
    oracle.set_threads(1)


def rel_l2(u, ref):
    return float(np.linalg.norm((u - ref).ravel()) / np.linalg.norm(ref.ravel()))


def dev(x, precision):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=NPDT[precision]), device="cuda")


def gpu_apply(X, F, precision, tensor, a=1.0, eta=1.0, n_tiles=0, host=False, pipeline=None):
    n = X.shape[0]
    with ds.System(1, precision=precision, tensor=tensor, a=a, eta=eta) as s:
        if n_tiles:
            s.set_tuning(n_tiles)
        if pipeline is not None:
            s.set_pipeline(pipeline)
        if host:
            Xh = np.ascontiguousarray(X, dtype=NPDT[precision])
            Fh = np.ascontiguousarray(F, dtype=NPDT[precision])
            uh = np.full((n, 3), np.nan, dtype=NPDT[precision])
            s.mobility_apply(Xh, Fh, uh, n)
            return uh.astype(np.float64)
        Xd, Fd = dev(X, precision), dev(F, precision)
        ud = torch.full((n, 3), float("nan"), dtype=TDT[precision], device="cuda")
        s.mobility_apply(Xd, Fd, ud, n)
        torch.cuda.synchronize()
        return ud.cpu().numpy().astype(np.float64)


def oracle_apply(X, F, precision, tensor, a=1.0, eta=1.0):
    Xr = np.asarray(X, dtype=NPDT[precision]).astype(np.float64)
    Fr = np.asarray(F, dtype=NPDT[precision]).astype(np.float64)
    return oracle.mobility_apply(Xr, Fr, a, eta, tensor)


# --------------------------------------------------------------------------------- mobility apply
@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
@pytest.mark.parametrize("N", [1, 2, 3, 17, 64, 255, 256, 257, 1000, 1027, 2048])
def test_apply_parity_sizes(N, tensor, precision):
    """Sizes below one tile, exactly one tile, ragged tails, several tiles and splits."""
    X, F = inputs.ragged_case(N, 500 + N)
    u = gpu_apply(X, F, precision, tensor, a=0.9, eta=1.3)
    ref = oracle_apply(X, F, precision, tensor, a=0.9, eta=1.3)
    assert np.isfinite(u).all()
    assert rel_l2(u, ref) <= TOL[precision]
    # per row: no single sphere is off by more than a few tolerances of the typical |u|
    assert np.abs(u - ref).max() <= 20 * TOL[precision] * np.sqrt(np.mean(ref ** 2))


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_apply_parity_config4_full_size(tensor, precision):
    """BASELINE.json config 4: N = 4096 random suspension, forces N(0,1): the headline apply, in the
    launch configuration bench.py times (library heuristic)."""
    X, F = inputs.apply_case(4096, 1004, 2004)
    u = gpu_apply(X, F, precision, tensor)
    ref = oracle_apply(X, F, precision, tensor)
    assert rel_l2(u, ref) <= TOL[precision]
    # per-sphere check too: no single row is off by more than a few tolerances of the typical |u|
    scale = np.sqrt(np.mean(ref ** 2))
    assert np.abs(u - ref).max() <= 20 * TOL[precision] * scale


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
@pytest.mark.parametrize("n_tiles", [1, 2, 5, 16, 100, 384])
def test_apply_parity_forced_tiles(n_tiles, precision):
    """Every (alpha-thread, beta-group) shape of the CTA gives the same answer: 1 tile = 384 quads x 1
    beta-group ... 384 tiles = 1 quad x 512 beta-groups."""
    X, F = inputs.apply_case(1536, 21, 22)
    u = gpu_apply(X, F, precision, ds.RPY, n_tiles=n_tiles)
    assert rel_l2(u, oracle_apply(X, F, precision, ds.RPY)) <= TOL[precision]


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
@pytest.mark.parametrize("N,n_tiles", [(1536, 24), (1536, 35), (1536, 100), (1536, 384), (1537, 97), (130, 33), (6, 1), (1, 1), (4096, 0), (8192, 0)])
def test_apply_warp_shaped_kernel(N, n_tiles, tensor, precision):
    """apply_kernel (the stateless apply in the thread shape of the pipelined kernel) under forced tilings: 16 ... 1 quads per
    CTA (1 ... 16 warps per quad, uneven deals like 11 quads on 16 warps), odd N (a half-filled last unit that holds an own
    sphere), tiny N, and the library's own shapes at N = 4096 and 8192; per row against the oracle; the one-pass run_kernel on
    the same tiling agrees within the tolerance; bitwise reproducible."""
    X, F = inputs.ragged_case(N, 900 + N)
    ref = oracle_apply(X, F, precision, tensor)
    u = gpu_apply(X, F, precision, tensor, n_tiles=n_tiles, pipeline=1)
    assert np.isfinite(u).all()
    assert rel_l2(u, ref) <= TOL[precision]
    assert np.abs(u - ref).max() <= 20 * TOL[precision] * np.sqrt(np.mean(ref ** 2))
    u1 = gpu_apply(X, F, precision, tensor, n_tiles=n_tiles, pipeline=0)
    assert rel_l2(u1, ref) <= TOL[precision]
    assert np.array_equal(u, gpu_apply(X, F, precision, tensor, n_tiles=n_tiles, pipeline=1))


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
def test_apply_host_pointers_and_determinism(precision):
    X, F = inputs.apply_case(700, 31, 32)
    u_host = gpu_apply(X, F, precision, ds.RPY, host=True)
    u_dev = gpu_apply(X, F, precision, ds.RPY)
    u_dev2 = gpu_apply(X, F, precision, ds.RPY)
    assert np.array_equal(u_host, u_dev)          # same kernels either way
    assert np.array_equal(u_dev, u_dev2)          # fixed summation order: bitwise reproducible
    assert rel_l2(u_dev, oracle_apply(X, F, precision, ds.RPY)) <= TOL[precision]


@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_apply_scaling_sweep_16384(tensor):
    """BASELINE.json config 5 sweep member N = 16384 (FP32), full parity."""
    X, F = inputs.sweep_case(14)
    u = gpu_apply(X, F, ds.F32, tensor)
    assert rel_l2(u, oracle_apply(X, F, ds.F32, tensor)) <= TOL[ds.F32]


def test_apply_two_sphere_closed_form_on_gpu():
    """the GPU path itself reproduces the two-sphere Oseen closed form."""
    r, a, eta = 7.0, 0.7, 1.3
    X = np.array([[0.0, 0, 0], [r, 0, 0]])
    F = np.array([[0.0, 0, 0], [1.0, 0, 0]])
    u = gpu_apply(X, F, ds.F64, ds.OSEEN, a=a, eta=eta)
    np.testing.assert_allclose(u[0, 0], 1 / (4 * np.pi * eta * r), rtol=1e-14)
    np.testing.assert_allclose(u[1, 0], 1 / (6 * np.pi * eta * a), rtol=1e-14)


# --------------------------------------------------------------------------------- forces / velocity
def make_system(w, precision, tensor=ds.RPY, integrator=ds.HEUN, **kw):
    sc = dict(w.scalars)
    sc.update(kw)
    s = ds.System(w.S, n_batch=w.B, precision=precision, tensor=tensor, integrator=integrator, a=sc["a"],
                  eta=sc["eta"], ell=sc["ell"], lam=sc["lam"], omega=sc["omega"], k0=sc["k0"], dt=sc["dt"],
                  kT=sc.get("kT", 0.0), seed=sc.get("seed", 0))
    return s, oracle.Params(a=sc["a"], eta=sc["eta"], ell=sc["ell"], lam=sc["lam"], omega=sc["omega"], k0=sc["k0"],
                            dt=sc["dt"], tensor=tensor, integrator=integrator, kT=sc.get("kT", 0.0), seed=sc.get("seed", 0))


def rounded(w, precision):
    return np.asarray(w.pos, dtype=NPDT[precision]).astype(np.float64)


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
def test_forces_and_velocity_parity(precision):
    w = inputs.config2()
    X0 = rounded(w, precision)
    X0 = X0 + np.random.default_rng(4).uniform(-0.3, 0.3, X0.shape).astype(NPDT[precision]).astype(np.float64)
    X0 = X0.astype(NPDT[precision]).astype(np.float64)
    s, p = make_system(w, precision)
    with s:
        s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"), t0=0.37)
        F = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
        V = torch.empty_like(F)
        s.forces(F)
        s.velocity(V)
        torch.cuda.synchronize()
        Fo = oracle.forces(X0[0], w.phase[0], 0.37, p)
        Vo = oracle.velocity(X0[0], w.phase[0], 0.37, p)
        assert rel_l2(F.cpu().numpy()[0].astype(np.float64), Fo) <= (1e-14 if precision == ds.F64 else 1e-7)
        assert rel_l2(V.cpu().numpy()[0].astype(np.float64), Vo) <= TOL[precision]
        Xb = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
        assert s.get_state(Xb) == pytest.approx(0.37)
        assert np.array_equal(Xb.cpu().numpy().astype(np.float64), X0)


# --------------------------------------------------------------------------------- stepping
def gpu_steps(w, precision, n_steps, tensor=ds.RPY, integrator=ds.HEUN, t0=0.0, chunks=None, **kw):
    s, p = make_system(w, precision, tensor, integrator, **kw)
    with s:
        X0 = rounded(w, precision)
        s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"), t0=t0)
        for c in (chunks or [n_steps]):
            s.batch_step(c) if w.B > 1 else s.step(c)
        out = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
        t = s.get_state(out)
        torch.cuda.synchronize()
        assert t == pytest.approx(t0 + n_steps * p.dt, rel=1e-12)
        return out.cpu().numpy().astype(np.float64), X0, p


def test_step_config1_fp64_full_run():
    """C1: 1d line, S = 8, FP64, all 10^4 steps (10 stroke periods)."""
    w = inputs.config1()
    Xg, X0, p = gpu_steps(w, ds.F64, w.n_steps)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, w.n_steps, p)
    assert np.abs(Xg[0] - Xo).max() <= 1e-9 * ELL
    assert np.abs(Xg[0, :, 1:]).max() == 0.0           # stays on the x axis exactly


@pytest.mark.parametrize("precision,n_steps,tol", [(ds.F64, 10_000, 1e-8), (ds.F32, 1000, 1e-4), (ds.F32, 10_000, 1e-4)])
def test_step_config2(precision, n_steps, tol):
    """C2: 4x4x4 lattice; FP32 within 1e-4 ell after 1000 steps (north_star), FP64 over the full 10^4."""
    w = inputs.config2()
    Xg, X0, p = gpu_steps(w, precision, n_steps)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, n_steps, p)
    assert np.abs(Xg[0] - Xo).max() <= tol * ELL


def test_step_config3_fp32_1000_steps():
    """C3: S = 512 random suspension, FP32, first 1000 steps."""
    w = inputs.config3()
    Xg, X0, p = gpu_steps(w, ds.F32, 1000)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 1000, p)
    assert np.abs(Xg[0] - Xo).max() <= 1e-4 * ELL


@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
def test_step_config4_200_steps(precision, tol):
    """C4: S = 2048 (N = 4096), the split-j + fused-epilogue path at full size."""
    w = inputs.config4()
    Xg, X0, p = gpu_steps(w, precision, 200)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 200, p)
    assert np.abs(Xg[0] - Xo).max() <= tol * ELL


def test_batch_step_config5_three_systems():
    """C5: B = 64 systems of S = 256, FP32; parity on 3 of the 64 over 1000 steps."""
    w = inputs.config5()
    Xg, X0, p = gpu_steps(w, ds.F32, 1000)
    for b in (0, 31, 63):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 1000, p)
        assert np.abs(Xg[b] - Xo).max() <= 1e-4 * ELL


@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_step_integrators_tensors_chunking_t0(integrator, tensor):
    """Euler and Heun, both tensors, t0 != 0, odd step counts; the result does not depend on how the
    steps are split over calls (one persistent launch vs several), bit for bit."""
    w = inputs.config2()
    Xa, X0, p = gpu_steps(w, ds.F64, 101, tensor, integrator, t0=0.25)
    Xb, _, _ = gpu_steps(w, ds.F64, 101, tensor, integrator, t0=0.25, chunks=[1, 33, 3, 64])
    assert np.array_equal(Xa, Xb)
    Xo = oracle.step(X0[0], w.phase[0], 0.25, 0, 101, p)
    assert np.abs(Xa[0] - Xo).max() <= 1e-10 * ELL


def test_step_zero_steps_and_state_errors():
    w = inputs.config1()
    s, _ = make_system(w, ds.F64)
    with s:
        buf = torch.empty((1, w.N, 3), dtype=torch.float64, device="cuda")
        with pytest.raises(ds.DsError) as e:
            s.step(1)
        assert e.value.code == ds.ERR_STATE
        with pytest.raises(ds.DsError):
            s.get_state(buf)
        s.set_state(dev(w.pos, ds.F64), torch.as_tensor(w.phase, device="cuda"))
        s.step(0)
        assert s.get_state(buf) == 0.0
        assert np.array_equal(buf.cpu().numpy(), w.pos)
        with pytest.raises(ds.DsError):
            s.step(-1)
    w5 = inputs.config5(B=2, S=4)
    s, _ = make_system(w5, ds.F32)
    with s:
        s.set_state(dev(w5.pos, ds.F32), torch.as_tensor(w5.phase, device="cuda"))
        with pytest.raises(ds.DsError) as e:
            s.step(1)                      # ds_step requires n_batch == 1
        assert e.value.code == ds.ERR_STATE
        s.batch_step(2)


def test_isolated_dumbbell_does_not_translate_on_gpu():
    """PAPER.md:236 'single dumbbells did not translate' -- the authors' own acceptance check."""
    phi = np.array([[0.9]])
    n = np.array([[1.0, 2.0, -0.5]])
    n /= np.linalg.norm(n)
    X0 = inputs.place_spheres(np.array([[3.0, -1.0, 2.0]]), n, phi[0])[None]
    w = inputs.Workload("single", X0, phi)
    Xg, _, _ = gpu_steps(w, ds.F64, 3000)
    assert np.abs(0.5 * (Xg[0, 0] + Xg[0, 1]) - np.array([3.0, -1.0, 2.0])).max() < 1e-12


# --------------------------------------------------------------------------------- launch shapes of the step kernel
@pytest.mark.parametrize("n_tiles", [1, 3, 17, 40, 96])
def test_step_forced_tiles_cover_every_hand_over_mode(n_tiles):
    """The persistent kernel under forced row tilings of one S = 192 system (N = 384): 1 CTA (no barrier),
    3 CTAs (blocking barrier), 17+ CTAs (low-latency hand-over: tagged stream copy for the first granule, barrier
    passed inside the stage), including shapes whose whole stream is the first granule."""
    w = inputs.config5(B=1, S=192)
    s, p = make_system(w, ds.F64)
    with s:
        s.set_tuning(n_tiles)
        X0 = rounded(w, ds.F64)
        s.set_state(dev(X0, ds.F64), torch.as_tensor(w.phase, device="cuda"), t0=0.1)
        for c in (7, 1, 42):
            s.step(c)
        out = torch.empty((1, w.N, 3), dtype=torch.float64, device="cuda")
        s.get_state(out)
        V = torch.empty_like(out)
        s.velocity(V)
        torch.cuda.synchronize()
    Xo = oracle.step(X0[0], w.phase[0], 0.1, 0, 50, p)
    assert np.abs(out.cpu().numpy()[0] - Xo).max() <= 1e-10 * ELL
    Vo = oracle.velocity(Xo, w.phase[0], 0.1 + 50 * p.dt, p)
    assert rel_l2(V.cpu().numpy()[0], Vo) <= 1e-9


def test_step_fp32_forced_tiles_low_latency():
    w = inputs.config5(B=1, S=192)
    Xg = {}
    for n_tiles in (2, 48):
        s, p = make_system(w, ds.F32)
        with s:
            s.set_tuning(n_tiles)
            X0 = rounded(w, ds.F32)
            s.set_state(dev(X0, ds.F32), torch.as_tensor(w.phase, device="cuda"))
            s.step(300)
            out = torch.empty((1, w.N, 3), dtype=torch.float32, device="cuda")
            s.get_state(out)
            torch.cuda.synchronize()
            Xg[n_tiles] = out.cpu().numpy()[0].astype(np.float64)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 300, p)
    for n_tiles in Xg:
        assert np.abs(Xg[n_tiles] - Xo).max() <= 1e-4 * ELL


def test_step_stream_larger_than_shared_memory():
    """N = 16384 (FP32): the stage input (384 KB) does not fit a CTA's shared memory, so the step kernel streams it
    through the TMA ring and keeps the blocking barrier; 2 Heun steps against the oracle."""
    w = inputs.config5(B=1, S=8192)
    s, p = make_system(w, ds.F32)
    X0 = rounded(w, ds.F32)
    with s:
        s.set_state(dev(X0, ds.F32), torch.as_tensor(w.phase, device="cuda"), t0=0.13)
        out = torch.empty((1, w.N, 3), dtype=torch.float32, device="cuda")
        V = torch.empty_like(out)
        s.velocity(V)            # at the state just set: the FP64 state is exactly the float32 input widened
        s.step(2)
        s.get_state(out)
        torch.cuda.synchronize()
    assert rel_l2(V.cpu().numpy()[0].astype(np.float64), oracle.velocity(X0[0], w.phase[0], 0.13, p)) <= TOL[ds.F32]
    Xo = oracle.step(X0[0], w.phase[0], 0.13, 0, 2, p)
    assert np.abs(out.cpu().numpy()[0].astype(np.float64) - Xo).max() <= 1e-4 * ELL


def test_batch_more_systems_than_sms():
    """B = 200 systems of S = 8: one CTA per system, any number of systems per launch."""
    w = inputs.config5(B=200, S=8)
    Xg, X0, p = gpu_steps(w, ds.F64, 100)
    for b in (0, 77, 199):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 100, p)
        assert np.abs(Xg[b] - Xo).max() <= 1e-10 * ELL


def test_step_config4_fp32_1000_steps():
    """north_star: FP32 trajectory within 1e-4 ell after 1000 steps, at the headline size (N = 4096)."""
    w = inputs.config4()
    Xg, X0, p = gpu_steps(w, ds.F32, 1000)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 1000, p)
    assert np.abs(Xg[0] - Xo).max() <= 1e-4 * ELL


def test_apply_scaling_sweep_65536_full_size():
    """BASELINE.json config 5, the largest sweep member N = 65536 (FP32, RPY), in the launch configuration bench.py
    times (pack kernel + TMA ring, several waves): every output against the oracle (4.3e9 pair evaluations)."""
    X, F = inputs.sweep_case(16)
    u = gpu_apply(X, F, ds.F32, ds.RPY)
    ref = oracle_apply(X, F, ds.F32, ds.RPY)
    assert rel_l2(u, ref) <= TOL[ds.F32]
    scale = np.sqrt(np.mean(ref ** 2))
    assert np.abs(u - ref).max() <= 20 * TOL[ds.F32] * scale


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
def test_host_buffers_state_path_matches_device_buffers(precision):
    """ds_set_state / ds_get_state / ds_forces / ds_velocity with HOST buffers (the library keeps a user-precision image
    of the state; the next kernel widens it) give bit-identical results to the device-buffer path, in any call order."""
    w = inputs.config2()
    X0 = np.ascontiguousarray(rounded(w, precision), dtype=NPDT[precision])
    ph = np.ascontiguousarray(w.phase)
    res = {}
    for host in (False, True):
        s, p = make_system(w, precision)
        with s:
            def buf():
                return np.empty((w.B, w.N, 3), dtype=NPDT[precision]) if host else \
                    torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")

            def val(b):
                torch.cuda.synchronize()
                return np.array(b if host else b.cpu().numpy(), dtype=np.float64)
            s.set_state(X0 if host else dev(X0, precision), ph if host else torch.as_tensor(ph, device="cuda"), t0=0.2)
            g0 = buf(); s.get_state(g0)                       # before any kernel touched the state
            v0 = buf(); s.velocity(v0)
            f0 = buf(); s.forces(f0)
            s.step(25)
            f1 = buf(); s.forces(f1)
            g1 = buf(); t = s.get_state(g1)
            s.set_state(X0 if host else dev(X0, precision), ph if host else torch.as_tensor(ph, device="cuda"), t0=0.2)
            s.step(25)                                        # straight from set_state into the step kernel
            g2 = buf(); s.get_state(g2)
            res[host] = [val(x) for x in (g0, v0, f0, f1, g1, g2)]
            assert t == pytest.approx(0.2 + 25 * p.dt)
    for a, b_ in zip(res[False], res[True]):
        assert np.array_equal(a, b_)
    assert np.array_equal(res[True][0], X0.astype(np.float64))
    assert np.array_equal(res[True][4], res[True][5])
    Xo = oracle.step(X0[0].astype(np.float64), ph[0], 0.2, 0, 25, p)
    assert np.abs(res[True][4][0] - Xo).max() <= (1e-4 if precision == ds.F32 else 1e-10) * ELL


# --------------------------------------------------------------------------------- observables, Eq. (6a,b), (13)
@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
def test_observables_parity_batch(precision):
    """Dumbbell coordinates Eq. (6a,b) and the mean square displacement Eq. (13) over W = B systems, computed on the
    device from the FP64 state, against the oracle run on the same systems; reference set after 60 steps (the paper
    discards the settling transient), host and device output buffers."""
    w = inputs.config5(B=5, S=300)          # S spans two 256-dumbbell chunks of the reduction
    s, p = make_system(w, precision)
    X0 = rounded(w, precision)
    with s:
        with pytest.raises(ds.DsError):
            s.msd_set_reference()                        # no state yet
        s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"))
        with pytest.raises(ds.DsError) as e:
            s.msd()
        assert e.value.code == ds.ERR_STATE               # no reference yet
        s.batch_step(60)
        s.msd_set_reference()
        assert s.msd() == 0.0
        s.batch_step(240)
        msd_gpu = s.msd()
        R = torch.empty((w.B, w.S, 3), dtype=TDT[precision], device="cuda")
        Nh = np.empty((w.B, w.S, 3), dtype=NPDT[precision])
        s.dumbbell_coords(R, Nh)
        torch.cuda.synchronize()
    Rref, Rt, Nt = [], [], []
    for b in range(w.B):
        Xa = oracle.step(X0[b], w.phase[b], 0.0, 0, 60, p)
        Xb = oracle.step(Xa, w.phase[b], 0.0, 60, 240, p)
        Rref.append(oracle.dumbbell_coords(Xa)[0])
        r, n = oracle.dumbbell_coords(Xb)
        Rt.append(r); Nt.append(n)
    msd_or = oracle.msd(np.stack(Rt), np.stack(Rref))
    tol_x = (1e-4 if precision == ds.F32 else 1e-10) * ELL
    assert np.abs(R.cpu().numpy().astype(np.float64) - np.stack(Rt)).max() <= tol_x
    assert np.abs(Nh.astype(np.float64) - np.stack(Nt)).max() <= tol_x / ELL * 10
    # the displacements themselves are ~1e-2 a over 0.24 T: compare Eq. (13) through the per-dumbbell error bound
    disp = np.sqrt(msd_or)
    assert abs(np.sqrt(msd_gpu) - disp) <= (2e-5 if precision == ds.F32 else 1e-9)
    assert msd_gpu > 0.0


def test_msd_closed_form_on_gpu():
    """Eq. (13) on the device against its closed form: every system translated rigidly by its own vector d_w gives
    the mean of |d_w|^2 (no dynamics involved: set_state, reference, set_state again)."""
    w = inputs.config5(B=3, S=40)
    dw = np.array([[3.0, 4.0, 12.0], [1.0, 2.0, 2.0], [0.0, 0.0, 0.5]])
    s, _ = make_system(w, ds.F64)
    with s:
        s.set_state(dev(w.pos, ds.F64), torch.as_tensor(w.phase, device="cuda"))
        s.msd_set_reference()
        s.set_state(dev(w.pos + dw[:, None, :], ds.F64), torch.as_tensor(w.phase, device="cuda"))
        np.testing.assert_allclose(s.msd(), np.mean(np.sum(dw ** 2, axis=1)), rtol=1e-12)


@pytest.mark.parametrize("n_tiles", [1, 2])
def test_step_state_in_global_memory(n_tiles):
    """Row tiles too large for the shared-memory state (here forced: N = 1600 in 1 or 2 CTAs, 800+ rows each): the
    per-row state lives in the library's global arrays instead; same results."""
    w = inputs.config5(B=1, S=800)
    s, p = make_system(w, ds.F64)
    X0 = rounded(w, ds.F64)
    with s:
        s.set_tuning(n_tiles)
        s.set_state(np.ascontiguousarray(X0), np.ascontiguousarray(w.phase), t0=0.05)     # host buffers: starts from the user-precision image
        s.step(12)
        out = torch.empty((1, w.N, 3), dtype=torch.float64, device="cuda")
        s.get_state(out)
        V = torch.empty_like(out)
        s.velocity(V)
        torch.cuda.synchronize()
    Xo = oracle.step(X0[0], w.phase[0], 0.05, 0, 12, p)
    assert np.abs(out.cpu().numpy()[0] - Xo).max() <= 1e-10 * ELL
    assert rel_l2(V.cpu().numpy()[0], oracle.velocity(Xo, w.phase[0], 0.05 + 12 * p.dt, p)) <= 1e-9


@pytest.mark.parametrize("n_tiles", [0, 100])
def test_batch_in_several_launch_groups(n_tiles):
    """B = 5 systems of N = 1024: with the library's shape all five share one launch (29 CTAs each); with 100 CTAs per
    system only one system is co-resident at a time, so the call runs five launches one after the other."""
    w = inputs.config5(B=5, S=512)
    s, p = make_system(w, ds.F64)
    X0 = rounded(w, ds.F64)
    with s:
        s.set_tuning(n_tiles)
        s.set_state(dev(X0, ds.F64), torch.as_tensor(w.phase, device="cuda"))
        l0 = s.launch_count()
        s.batch_step(40)
        n_launch = s.launch_count() - l0
        out = torch.empty((w.B, w.N, 3), dtype=torch.float64, device="cuda")
        s.get_state(out)
        torch.cuda.synchronize()
    assert n_launch == (5 if n_tiles == 100 else 1)
    for b in (0, 3, 4):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 40, p)
        assert np.abs(out.cpu().numpy()[b] - Xo).max() <= 1e-10 * ELL


# --------------------------------------------------------------------------------- Brownian term (additive approximation)
@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("precision,tol", [(ds.F64, 1e-9), (ds.F32, 1e-4)])
def test_step_with_additive_noise_matches_oracle(precision, tol, integrator):
    """kT > 0 (Eq. (1a) in the constant-C approximation of PAPER.md:240): the device draws the same
    Philox4x32-10 increments as the oracle (counter = step, element, system), so trajectories agree like the
    deterministic ones do; 3 systems = 3 realisations w, several launch shapes, steps split over calls."""
    import dataclasses
    w = inputs.config5(B=3, S=96)
    X0 = rounded(w, precision)
    for n_tiles in (1, 6):
        s, p = make_system(w, precision, integrator=integrator, kT=0.02, seed=0x1234567ABCDEF)
        with s:
            s.set_tuning(n_tiles)
            s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"))
            s.batch_step(37)
            s.batch_step(63)
            out = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
            s.get_state(out)
            torch.cuda.synchronize()
        for b in range(w.B):
            Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 100, dataclasses.replace(p, system=b))
            assert np.abs(out.cpu().numpy()[b].astype(np.float64) - Xo).max() <= tol * ELL
        # the noise did move the spheres: far more than the tolerance
        Xdet = oracle.step(X0[0], w.phase[0], 0.0, 0, 100, dataclasses.replace(p, kT=0.0))
        assert np.abs(Xo * 0 + out.cpu().numpy()[0].astype(np.float64) - Xdet).max() > 1e-2


def test_noise_at_headline_size_low_latency_path():
    """N = 4096, FP32, 147 CTAs (tagged hand-over): 50 noisy Heun steps against the oracle."""
    import dataclasses
    w = inputs.config4()
    Xg, X0, p = gpu_steps(w, ds.F32, 50, kT=0.01, seed=77)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 50, p)
    assert np.abs(Xg[0] - Xo).max() <= 1e-4 * ELL


# --------------------------------------------------------------------------------- stroke-averaged model, Eq. (9)
def _avg_case(S, seed, side):
    rng = np.random.default_rng(seed)
    R = rng.uniform(-side / 2, side / 2, (S, 3))
    N = rng.standard_normal((S, 3)); N /= np.linalg.norm(N, axis=1, keepdims=True)
    return R, N, rng.uniform(0, 2 * np.pi, S)


@pytest.mark.parametrize("precision", [ds.F32, ds.F64])
@pytest.mark.parametrize("S", [1, 2, 9, 33, 300, 729, 2500, 9600])
def test_avg_rhs_parity(S, precision):
    """Eq. (9a)-(9d) on the device against the oracle: S below one block, a cluster whose last CTA holds one dumbbell
    (9), ragged chunks, the paper's largest lattice 9^3 = 729, chunks of more than one shared-memory
    tile (2500) and the single-CTA-per-block grid of large S (9600); device and host buffers."""
    R, N, phi = _avg_case(S, 900 + S, 60.0 * max(S, 2) ** (1 / 3))
    Rr, Nr = R.astype(NPDT[precision]), N.astype(NPDT[precision])
    p = oracle.Params(a=0.8, ell=9.0, lam=1.7, omega=5.5)
    dRo, dNo = oracle.avg_rhs(Rr.astype(np.float64), Nr.astype(np.float64), phi, p)
    with ds.System(1, precision=precision, a=p.a, ell=p.ell, lam=p.lam, omega=p.omega) as s:
        dR = torch.empty((S, 3), dtype=TDT[precision], device="cuda")
        dN = np.empty((S, 3), dtype=NPDT[precision])
        s.avg_rhs(dev(Rr, precision), np.ascontiguousarray(Nr), torch.as_tensor(phi, device="cuda"), dR, dN, S)
        torch.cuda.synchronize()
    if S == 1:
        assert np.all(dR.cpu().numpy() == 0) and np.all(dN == 0)
        return
    tol = 2e-5 if precision == ds.F32 else 1e-12
    assert rel_l2(dR.cpu().numpy().astype(np.float64), dRo) <= tol
    assert rel_l2(dN.astype(np.float64), dNo) <= tol


@pytest.mark.parametrize("precision,tol", [(ds.F64, 1e-12), (ds.F32, 1e-5)])
def test_avg_step_parity_lattice(precision, tol):
    """5 x 5 x 5 lattice of the paper's Fig. 3, random directions and phases: 40 Heun steps of half a
    period each of the averaged model on the device against the oracle; the FP64 state keeps the tiny increments even
    when the pair arithmetic is FP32, and N stays on the unit sphere."""
    g = np.arange(5) * 30.0
    R = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    _, N, phi = _avg_case(125, 5, 1.0)
    p = oracle.Params()
    Ro, No = oracle.avg_step(R, N, phi, 0.5, 40, p)
    with ds.System(1, precision=precision) as s:
        Rd = dev(R, precision); Nd = dev(N, precision)
        s.avg_step(Rd, Nd, torch.as_tensor(phi, device="cuda"), 125, 0.5, 40)
        torch.cuda.synchronize()
    Rg, Ng = Rd.cpu().numpy().astype(np.float64), Nd.cpu().numpy().astype(np.float64)
    disp = np.abs(Ro - R).max()
    if precision == ds.F64:
        assert np.abs(Rg - Ro).max() <= tol * 120 and np.abs(Ng - No).max() <= tol
        assert np.abs(Rg - R).max() > 0.5 * disp > 0
    else:   # the output buffers are float32: the comparison is limited by their rounding, not by the stepping
        assert np.abs(Rg - Ro).max() <= 120 * 6e-8 * 2 and np.abs(Ng - No).max() <= tol
    np.testing.assert_allclose(np.linalg.norm(Ng, axis=1), 1.0, rtol=0, atol=3e-7 if precision == ds.F32 else 1e-15)


@pytest.mark.parametrize("precision", [ds.F64, ds.F32])
def test_avg_step_parity_729(precision):
    """The paper's largest lattice, 9 x 9 x 9, sites displaced by up to 5 (no close pairs: Eq. (9) is a
    far-field model), random directions and phases: 6 Heun steps from the state as rounded to the working precision;
    the device-resident kernel: 5 dumbbells per CTA, all steps in one launch."""
    S = 729
    g = np.arange(9) * 30.0
    jit, N, phi = _avg_case(S, 31, 10.0)
    R = (np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) + jit).astype(NPDT[precision]).astype(np.float64)
    N = N.astype(NPDT[precision]).astype(np.float64)
    p = oracle.Params()
    Ro, No = oracle.avg_step(R, N, phi, 0.5, 6, p)
    with ds.System(1, precision=precision) as s:
        Rd = torch.as_tensor(R, device="cuda").to(TDT[precision]); Nd = torch.as_tensor(N, device="cuda").to(TDT[precision])
        s.avg_step(Rd, Nd, phi, S, 0.5, 6)
        torch.cuda.synchronize()
    Rg, Ng = Rd.cpu().numpy().astype(np.float64), Nd.cpu().numpy().astype(np.float64)
    assert np.abs(Ro - R).max() > 0
    if precision == ds.F64:
        assert np.abs(Rg - Ro).max() <= 1e-12 * 250 and np.abs(Ng - No).max() <= 1e-12
    else:   # float32 output buffers: half an ulp of 250 is 1.5e-5
        assert np.abs(Rg - Ro).max() <= 2e-5 and np.abs(Ng - No).max() <= 1e-5


@pytest.mark.parametrize("precision", [ds.F64, ds.F32])
@pytest.mark.parametrize("S", [1, 2, 7, 147, 149, 301, 2500, 4097])
def test_avg_step_device_resident_and_two_launch_paths(S, precision):
    """ds_avg_step over its launch shapes: one dumbbell (no pair at all), fewer dumbbells than SMs (one per CTA), one more
    than the SM count (two per CTA, a last CTA with one), odd S (an odd lane in the last FP32 pack), many dumbbells per CTA
    (S = 2500: 17), and S = 4097, above the limit of the device-resident kernel (two launches per step through
    avg_rhs_kernel).  5 Heun steps; a second call continues from the first (tags of the exchange buffers advance)."""
    m = int(np.ceil(S ** (1 / 3)))
    g_ = np.arange(m) * 30.0                      # jittered lattice as in Fig. 3 / 4: no close pairs (Eq. (9) is a far-field model)
    jit, N, phi = _avg_case(S, 700 + S, 10.0)
    R = np.stack(np.meshgrid(g_, g_, g_, indexing="ij"), -1).reshape(-1, 3)[:S] + jit
    R = R.astype(NPDT[precision]).astype(np.float64); N = N.astype(NPDT[precision]).astype(np.float64)
    p = oracle.Params(a=0.8, ell=9.0, lam=1.7, omega=5.5)
    Ro, No = oracle.avg_step(R, N, phi, 40.0, 5, p)
    with ds.System(1, precision=precision, a=p.a, ell=p.ell, lam=p.lam, omega=p.omega) as s:
        Rd = torch.as_tensor(R, device="cuda").to(TDT[precision]); Nd = torch.as_tensor(N, device="cuda").to(TDT[precision])
        l0 = s.launch_count()
        s.avg_step(Rd, Nd, torch.as_tensor(phi, device="cuda"), S, 40.0, 5)
        n_launch = s.launch_count() - l0
        torch.cuda.synchronize()
        Rg, Ng = Rd.cpu().numpy().astype(np.float64), Nd.cpu().numpy().astype(np.float64)
        if precision == ds.F64:
            s.avg_step(Rd, Nd, torch.as_tensor(phi, device="cuda"), S, 40.0, 3)     # 5 + 3 steps = 8 steps
            torch.cuda.synchronize()
            R8, N8 = oracle.avg_step(R, N, phi, 40.0, 8, p)
            assert np.abs(Rd.cpu().numpy() - R8).max() <= 1e-11 * np.abs(R).max() + 1e-13
            assert np.abs(Nd.cpu().numpy() - N8).max() <= 1e-12
    # launches: sin/cos table + 2 widen + (1 resident | 2 per step) + 2 narrow
    assert n_launch == (6 if S <= 4096 else 5 + 2 * 5)
    scale = np.abs(R).max() + 1.0
    if precision == ds.F64:
        assert np.abs(Rg - Ro).max() <= 1e-12 * scale and np.abs(Ng - No).max() <= 1e-12
    else:   # FP32 pair arithmetic (2e-5 of the right-hand sides) and float32 output buffers
        assert np.abs(Rg - Ro).max() <= 1e-4 * np.abs(Ro - R).max() + 1.2e-7 * scale
        assert np.abs(Ng - No).max() <= 1e-4 * np.abs(No - N).max() + 3e-7


# --------------------------------------------------------------------------------- pipelined step kernel (pipeline.cuh)
def pipe_steps(w, precision, chunks, n_tiles=0, tensor=ds.RPY, integrator=ds.HEUN, t0=0.0, pipeline=1, host=False, **kw):
    """Steps through the two-pass pipelined kernel (forced on; `pipeline=0` forces the one-pass kernel)."""
    s, p = make_system(w, precision, tensor, integrator, **kw)
    with s:
        if n_tiles:
            s.set_tuning(n_tiles)
        s.set_pipeline(pipeline)
        assert s.pipeline_active() == bool(pipeline), (w.N, n_tiles)
        X0 = rounded(w, precision)
        if host:
            s.set_state(np.ascontiguousarray(X0, dtype=NPDT[precision]), np.ascontiguousarray(w.phase), t0=t0)
        else:
            s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"), t0=t0)
        for c in chunks:
            s.batch_step(c) if w.B > 1 else s.step(c)
        out = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
        s.get_state(out)
        torch.cuda.synchronize()
        return out.cpu().numpy().astype(np.float64), X0, p


@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
@pytest.mark.parametrize("S,n_tiles", [(192, 3), (192, 17), (192, 48), (191, 5), (97, 2), (333, 31), (600, 148), (1024, 0)])
def test_pipeline_parity_shapes(S, n_tiles, precision, tol):
    """The pipelined kernel under forced row tilings: halves of 1 ... 16 quads (16 ... 1 warps per quad), CTAs with an
    empty second half (48 tiles of N = 384: one quad each), odd S (a last quad of two rows), regions that end inside a
    warp's 32 units, the library's own tiling (S = 1024: 128 CTAs).  50 Heun steps split over three launches, t0 != 0,
    element by element against the oracle."""
    w = inputs.config5(B=1, S=S)
    Xg, X0, p = pipe_steps(w, precision, [7, 1, 42], n_tiles=n_tiles, t0=0.1)
    Xo = oracle.step(X0[0], w.phase[0], 0.1, 0, 50, p)
    assert np.abs(Xg[0] - Xo).max() <= tol * ELL


@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_pipeline_integrators_tensors_chunking_determinism(integrator, tensor):
    """Euler and Heun, both tensors: the result does not depend on how the steps are split over launches and is bitwise
    reproducible run to run (fixed summation trees, no atomics); host-buffer start equals device-buffer start."""
    w = inputs.config5(B=1, S=300)
    Xa, X0, p = pipe_steps(w, ds.F64, [101], n_tiles=20, tensor=tensor, integrator=integrator, t0=0.25)
    Xb, _, _ = pipe_steps(w, ds.F64, [1, 33, 3, 64], n_tiles=20, tensor=tensor, integrator=integrator, t0=0.25)
    Xc, _, _ = pipe_steps(w, ds.F64, [101], n_tiles=20, tensor=tensor, integrator=integrator, t0=0.25, host=True)
    assert np.array_equal(Xa, Xb)
    assert np.array_equal(Xa, Xc)
    Xo = oracle.step(X0[0], w.phase[0], 0.25, 0, 101, p)
    assert np.abs(Xa[0] - Xo).max() <= 1e-10 * ELL
    # the one-pass kernel integrates the same equations (its sums are ordered differently: last bits only)
    Xd, _, _ = pipe_steps(w, ds.F64, [101], n_tiles=20, tensor=tensor, integrator=integrator, t0=0.25, pipeline=0)
    assert np.abs(Xa - Xd).max() <= 1e-11 * ELL


@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
def test_pipeline_config4_headline_shape(precision, tol):
    """C4 (N = 4096) in the launch configuration bench.py times: the library picks the pipelined kernel by itself (147
    CTAs of 7 / 6 quads: halves of 4 + 3 and 3 + 3 quads); 200 steps against the oracle."""
    w = inputs.config4()
    s, p = make_system(w, precision)
    with s:
        assert s.pipeline_active()
        X0 = rounded(w, precision)
        s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"))
        s.step(200)
        out = torch.empty((1, w.N, 3), dtype=TDT[precision], device="cuda")
        s.get_state(out)
        V = torch.empty_like(out)
        s.velocity(V)            # the one-pass kernel on the state the pipelined one left
        torch.cuda.synchronize()
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 200, p)
    assert np.abs(out.cpu().numpy()[0].astype(np.float64) - Xo).max() <= tol * ELL
    if precision == ds.F64:   # (in FP32 mode get_state rounds the FP64 state; the stiff spring amplifies that in V)
        Vo = oracle.velocity(out.cpu().numpy()[0], w.phase[0], 200 * p.dt, p)
        assert rel_l2(V.cpu().numpy()[0], Vo) <= 1e-9


def test_pipeline_batch_and_noise():
    """B = 5 systems of N = 600 in one launch (29 CTAs each) with k_B T > 0: per-system arrival counters, Philox
    increments drawn by the service warp, steps split over calls."""
    import dataclasses
    w = inputs.config5(B=5, S=300)
    Xg, X0, p = pipe_steps(w, ds.F64, [37, 63], n_tiles=29, kT=0.02, seed=0x1234567ABCDEF)
    for b in range(w.B):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 100, dataclasses.replace(p, system=b))
        assert np.abs(Xg[b] - Xo).max() <= 1e-9 * ELL


# --------------------------------------------------------------------------------- variants no other test reaches
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
@pytest.mark.parametrize("N", [8192, 16384])
def test_apply_fp64_ring_mode(N, tensor):
    """FP64 applies whose stream (48 B per sphere) exceeds shared memory: pack_user_kernel<double> + the TMA ring
    (run_kernel<double, *, APPLY, false>), element by element."""
    X, F = inputs.sweep_case(13 if N == 8192 else 14)
    u = gpu_apply(X, F, ds.F64, tensor)
    ref = oracle_apply(X, F, ds.F64, tensor)
    assert rel_l2(u, ref) <= TOL[ds.F64]
    assert np.abs(u - ref).max() <= 20 * TOL[ds.F64] * np.sqrt(np.mean(ref ** 2))


@pytest.mark.parametrize("N", [8192, 8194])
def test_apply_fp32_resident_ring_boundary(N):
    """FP32 applies on both sides of the resident / ring boundary of the stream (N = 8192 is the last resident size)."""
    X, F = inputs.apply_case(N, 81, 82)
    u = gpu_apply(X, F, ds.F32, ds.RPY)
    ref = oracle_apply(X, F, ds.F32, ds.RPY)
    assert rel_l2(u, ref) <= TOL[ds.F32]
    assert np.abs(u - ref).max() <= 20 * TOL[ds.F32] * np.sqrt(np.mean(ref ** 2))


@pytest.mark.parametrize("integrator,n_steps", [(ds.HEUN, 2), (ds.EULER, 3)])
def test_step_fp64_ring_mode(integrator, n_steps):
    """N = 8192 in FP64: the stage input (384 KB) streams through the TMA ring with the blocking barrier
    (run_kernel<double, *, VELOCITY / EULER / HEUN, false>)."""
    w = inputs.config5(B=1, S=4096)
    s, p = make_system(w, ds.F64, integrator=integrator)
    X0 = rounded(w, ds.F64)
    with s:
        s.set_state(dev(X0, ds.F64), torch.as_tensor(w.phase, device="cuda"), t0=0.13)
        out = torch.empty((1, w.N, 3), dtype=torch.float64, device="cuda")
        V = torch.empty_like(out)
        s.velocity(V)
        s.step(n_steps)
        s.get_state(out)
        torch.cuda.synchronize()
    assert rel_l2(V.cpu().numpy()[0], oracle.velocity(X0[0], w.phase[0], 0.13, p)) <= 1e-12
    Xo = oracle.step(X0[0], w.phase[0], 0.13, 0, n_steps, p)
    assert np.abs(out.cpu().numpy()[0] - Xo).max() <= 1e-10 * ELL


def test_step_fp32_euler_ring_mode():
    """N = 16384, FP32, Euler through the ring (run_kernel<float, *, EULER, false>)."""
    w = inputs.config5(B=1, S=8192)
    Xg, X0, p = gpu_steps(w, ds.F32, 3, integrator=ds.EULER)
    Xo = oracle.step(X0[0], w.phase[0], 0.0, 0, 3, p)
    assert np.abs(Xg[0] - Xo).max() <= 1e-4 * ELL


def test_step_state_in_global_memory_odd_S_batch():
    """The global-memory home of the per-row state with an odd number of dumbbells and two systems: the last quad of a
    system has two rows, and the integrator must not touch the first spheres of the next system (S = 1051, 1 tile)."""
    w = inputs.config5(B=2, S=1051)
    s, p = make_system(w, ds.F64)
    X0 = rounded(w, ds.F64)
    with s:
        s.set_tuning(1)
        s.set_pipeline(0)
        s.set_state(dev(X0, ds.F64), torch.as_tensor(w.phase, device="cuda"))
        s.batch_step(6)
        out = torch.empty((w.B, w.N, 3), dtype=torch.float64, device="cuda")
        s.get_state(out)
        torch.cuda.synchronize()
    for b in range(w.B):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 6, p)
        assert np.abs(out.cpu().numpy()[b] - Xo).max() <= 1e-10 * ELL


# --------------------------------------------------------------------------------- small systems: one warp per system (small.cuh)
@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
@pytest.mark.parametrize("S,B", [(1, 1), (2, 3), (3, 1), (5, 7), (8, 1), (17, 5), (32, 9), (17, 160), (32, 160)])
def test_small_system_kernel_shapes(S, B, precision, tol):
    """S <= 32 dumbbells run one warp per system: 32, 16, 8, 4, 2, 1 lanes per dumbbell (S = 1 ... 32, powers of two and
    not), several systems per CTA and a ragged last CTA; with 17 ... 32 dumbbells the warp-per-system kernel serves ensembles
    too large to be resident on run_kernel at once (B = 160) and run_kernel the small ones.  60 Heun steps over three calls, t0 != 0, against the oracle;
    the same steps through run_kernel's one-CTA mode (forced tiling) agree to rounding."""
    w = inputs.config5(B=B, S=S)
    Xg, X0, p = gpu_steps(w, precision, 60, t0=0.1, chunks=[7, 1, 52])
    for b in range(B):
        Xo = oracle.step(X0[b], w.phase[b], 0.1, 0, 60, p)
        assert np.abs(Xg[b] - Xo).max() <= tol * ELL
    Xr, _, _ = pipe_steps(w, precision, [60], n_tiles=1, t0=0.1, pipeline=0)       # run_kernel, one CTA per system
    assert np.abs(Xg - Xr).max() <= (1e-5 if precision == ds.F32 else 1e-11) * ELL


@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_small_system_kernel_integrators_tensors_noise(integrator, tensor):
    """Euler / Heun, Oseen / RPY, k_B T > 0 (Philox increments drawn per lane), chunking invariance bit for bit, host-buffer
    start."""
    import dataclasses
    w = inputs.config5(B=3, S=12)
    Xa, X0, p = gpu_steps(w, ds.F64, 101, tensor, integrator, t0=0.25, kT=0.02, seed=0xABCDEF12345)
    Xb, _, _ = gpu_steps(w, ds.F64, 101, tensor, integrator, t0=0.25, chunks=[1, 33, 3, 64], kT=0.02, seed=0xABCDEF12345)
    assert np.array_equal(Xa, Xb)
    for b in range(w.B):
        Xo = oracle.step(X0[b], w.phase[b], 0.25, 0, 101, dataclasses.replace(p, system=b))
        assert np.abs(Xa[b] - Xo).max() <= 1e-9 * ELL


# --------------------------------------------------------------------------------- ensembles: one cluster per system (cluster.cuh)
def cluster_steps(w, precision, chunks, tensor=ds.RPY, integrator=ds.HEUN, t0=0.0, host=False, expect=2, pipeline=-1, **kw):
    """Steps of an ensemble through the library's own choice of kernel, which must be the cluster kernel (`expect` = 2;
    `pipeline=0`, `expect=0` forces the one-pass kernel instead)."""
    s, p = make_system(w, precision, tensor, integrator, **kw)
    with s:
        s.set_pipeline(pipeline)
        assert s.pipeline_active() == expect, (w.B, w.S)
        X0 = rounded(w, precision)
        if host:
            s.set_state(np.ascontiguousarray(X0, dtype=NPDT[precision]), np.ascontiguousarray(w.phase), t0=t0)
        else:
            s.set_state(dev(X0, precision), torch.as_tensor(w.phase, device="cuda"), t0=t0)
        for c in chunks:
            s.batch_step(c)
        out = torch.empty((w.B, w.N, 3), dtype=TDT[precision], device="cuda")
        s.get_state(out)
        torch.cuda.synchronize()
        return out.cpu().numpy().astype(np.float64), X0, p


@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
@pytest.mark.parametrize("B,S,check", [(64, 256, (0, 17, 63)), (32, 256, (0, 31)), (74, 64, (0, 36, 73)), (70, 100, (0, 69)),
                                       (70, 99, (0, 35, 69)), (14, 512, (3, 13)), (14, 700, (7,))])
def test_cluster_kernel_shapes(B, S, check, precision, tol):
    """Ensembles that get one thread-block cluster per system: 2 CTAs (B = 64, 74, 70), 4 (B = 32) and 8 (B = 14) per
    system; halves of 32 quads (2 quads per warp, 16 lanes per quad), 16 (a warp per quad), 8 (2 warps per quad), 13 + 12
    (idle warps), 22 + 22 and 22 + 21 (S = 700: idle warps and a warp whose second quad does not exist) and, with S = 99, a last quad of two rows; C5's own shape first.  Heun, t0 != 0, 9 steps over three calls,
    against the oracle on a sample of the systems."""
    w = inputs.config5(B=B, S=S)
    Xg, X0, p = cluster_steps(w, precision, [4, 1, 4], t0=0.3)
    for b in check:
        Xo = oracle.step(X0[b], w.phase[b], 0.3, 0, 9, p)
        assert np.abs(Xg[b] - Xo).max() <= tol * ELL, b


@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_cluster_kernel_integrators_tensors_chunking_determinism(integrator, tensor):
    """Euler / Heun and both tensors through the cluster kernel (B = 32, S = 128: 4 CTAs per system); host buffers;
    the result is bit-identical however the steps are split over launches and from run to run, and agrees with the one-pass
    kernel to rounding."""
    w = inputs.config5(B=32, S=128)
    Xa, X0, p = cluster_steps(w, ds.F64, [31], tensor, integrator, t0=0.25)
    Xb, _, _ = cluster_steps(w, ds.F64, [1, 13, 2, 15], tensor, integrator, t0=0.25, host=True)
    assert np.array_equal(Xa, Xb)
    Xc, _, _ = cluster_steps(w, ds.F64, [31], tensor, integrator, t0=0.25, pipeline=0, expect=0)
    assert np.abs(Xa - Xc).max() <= 1e-10 * ELL
    for b in (0, 31):
        Xo = oracle.step(X0[b], w.phase[b], 0.25, 0, 31, p)
        assert np.abs(Xa[b] - Xo).max() <= 1e-10 * ELL


def test_cluster_kernel_with_additive_noise():
    """k_B T > 0 through the cluster kernel: Philox increments drawn by the service warps, per system and sphere, steps
    split over calls (B = 64, S = 64: 2 CTAs per system, FP64)."""
    import dataclasses
    w = inputs.config5(B=64, S=64)
    Xg, X0, p = cluster_steps(w, ds.F64, [7, 13], kT=0.02, seed=0x1234567ABCDEF)
    for b in (0, 40, 63):
        Xo = oracle.step(X0[b], w.phase[b], 0.0, 0, 20, dataclasses.replace(p, system=b))
        assert np.abs(Xg[b] - Xo).max() <= 1e-9 * ELL


def test_cluster_kernel_not_taken_when_clusters_do_not_fit():
    """Shapes the heuristic must leave to the other kernels: too few systems to fill 3/4 of the SMs (B = 48 x 2 CTAs),
    more clusters than are resident at once (B = 37 x 4 CTAs in FP32), less than a quad per warp (S = 40), one system."""
    for (B, S, precision) in ((48, 256, ds.F32), (37, 500, ds.F32), (64, 40, ds.F32), (1, 256, ds.F64)):
        w = inputs.config5(B=B, S=S)
        s, _ = make_system(w, precision)
        with s:
            assert s.pipeline_active() in (0, 1, 3), (B, S)   # 3: the latency variant (short pair loops), tested below


# --------------------------------------------------------------------------------- small systems: a cluster of CTAs, no pipeline (cluster_lat_kernel)
@pytest.mark.parametrize("precision,tol", [(ds.F32, 1e-4), (ds.F64, 1e-10)])
@pytest.mark.parametrize("B,S", [(1, 17), (1, 33), (3, 40), (1, 64), (2, 99), (1, 128), (12, 128), (18, 64), (64, 40), (37, 64), (300, 64)])
def test_cluster_lat_kernel_shapes(B, S, precision, tol):
    """Systems with short pair loops on one cluster each (cluster_lat_kernel), the cluster size the library picks: 2 CTAs per
    system (S = 17; the ensembles of 64 and 37), 4 (S = 33, 40, 64 = C2's shape; 18 x S = 64), 8 (12 x S = 128), 16 (S = 99, 128),
    one CTA per system in three waves (300 x S = 64: 2 quads per warp);
    1 - 16 quads per CTA (16 ... 1 warps per quad, idle warps, CTAs of uneven quad counts; S = 99: a last quad of two rows).
    40 Heun steps over three calls, t0 != 0, against the oracle on every system (a sample for the big ensembles)."""
    w = inputs.config5(B=B, S=S)
    Xg, X0, p = cluster_steps(w, precision, [7, 1, 32], t0=0.1, expect=3, pipeline=3)   # forced: the heuristic is tested below
    for b in sorted({0, B // 2, B - 1}):
        Xo = oracle.step(X0[b], w.phase[b], 0.1, 0, 40, p)
        assert np.abs(Xg[b] - Xo).max() <= tol * ELL, b


@pytest.mark.parametrize("integrator", [ds.EULER, ds.HEUN])
@pytest.mark.parametrize("tensor", [ds.OSEEN, ds.RPY])
def test_cluster_lat_kernel_integrators_tensors_noise_chunking(integrator, tensor):
    """Euler / Heun, Oseen / RPY, k_B T > 0 through cluster_lat_kernel (C2's lattice, B = 1 and an ensemble of 5): bit-identical
    however the steps are split over launches, from host buffers too; against the oracle; forced on a shape the heuristic
    leaves to run_kernel (S = 300: 10 iterations per warp) it still agrees."""
    import dataclasses
    w = inputs.config2()
    Xa, X0, p = cluster_steps(w, ds.F64, [101], tensor, integrator, t0=0.25, expect=3, kT=0.02, seed=0xABCDEF12345)
    Xb, _, _ = cluster_steps(w, ds.F64, [1, 33, 3, 64], tensor, integrator, t0=0.25, expect=3, host=True, kT=0.02, seed=0xABCDEF12345)
    assert np.array_equal(Xa, Xb)
    Xo = oracle.step(X0[0], w.phase[0], 0.25, 0, 101, p)
    assert np.abs(Xa[0] - Xo).max() <= 1e-9 * ELL
    w5 = inputs.config5(B=5, S=48)
    Xc, X05, p5 = cluster_steps(w5, ds.F32, [20, 21], tensor, integrator, expect=3, kT=0.01, seed=77)
    for b in range(w5.B):
        Xo = oracle.step(X05[b], w5.phase[b], 0.0, 0, 41, dataclasses.replace(p5, system=b))
        assert np.abs(Xc[b] - Xo).max() <= 1e-4 * ELL
    w3 = inputs.config5(B=2, S=300)
    Xd, X03, p3 = cluster_steps(w3, ds.F64, [9], tensor, integrator, expect=3, pipeline=3)
    for b in range(w3.B):
        Xo = oracle.step(X03[b], w3.phase[b], 0.0, 0, 9, p3)
        assert np.abs(Xd[b] - Xo).max() <= 1e-10 * ELL


def test_cluster_lat_kernel_heuristic():
    """Which shapes the library sends to cluster_lat_kernel by itself: short pair loops only (C2 yes, S = 300 no), never S <= 16
    (warp-per-system kernel), clusters of 2 or more CTAs only when all are resident at once (40 x S = 100: no), one CTA per
    system also in waves but not for S <= 32 (600 x S = 64 yes, 600 x S = 20 no)."""
    for (B, S, precision, want) in ((1, 64, ds.F32, 3), (1, 64, ds.F64, 3), (18, 64, ds.F32, 3), (1, 20, ds.F64, 3), (1, 8, ds.F64, 0),
                                    (1, 16, ds.F32, 0), (1, 300, ds.F64, 0), (100, 33, ds.F32, 3), (40, 100, ds.F32, 0),
                                    (600, 64, ds.F32, 3), (600, 20, ds.F32, 0), (64, 256, ds.F32, 2)):
        w = inputs.config5(B=B, S=S)
        s, _ = make_system(w, precision)
        with s:
            assert s.pipeline_active() == want, (B, S, precision)
