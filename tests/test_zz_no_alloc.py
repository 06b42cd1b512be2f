"""ds_msd_static (include/ds.h): Eq. (13), through the entry point that allocates nothing (partial sums in a
static device array) against the existing ds_msd path and the oracle, two calls in a row.  Collected last on purpose."""
import numpy as np
import pytest
import torch

import oracle
from paper_1004_1932_b200 import ds, inputs


def _centres(X):
    return 0.5 * (X[:, 0::2, :] + X[:, 1::2, :])


@pytest.mark.gpu
def test_msd_static_matches_ds_msd_two_calls_in_a_row():
    B, S = 5, 300                                   # two chunks of 256 dumbbells per system, a ragged second one
    Xs, ps = zip(*(inputs.random_suspension(S, 4100 + b) for b in range(B)))
    X0, phase = np.stack(Xs), np.stack(ps)
    stream = torch.cuda.current_stream().cuda_stream
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    with ds.System(S, n_batch=B, precision=ds.F64, tensor=ds.RPY, integrator=ds.HEUN, dt=1e-3, stream=stream) as s:
        s.set_state(torch.as_tensor(X0, device="cuda"), torch.as_tensor(phase, device="cuda"), 0.0)
        s.msd_set_reference()
        Rref = torch.empty((B, S, 3), dtype=torch.float64, device="cuda")   # R^s(0; w) as a caller gets them: Eq. (6b) on the device
        s.dumbbell_coords(Rref, None)
        for call, n_steps in enumerate((40, 25)):   # second call: other data, the array still holds the first call's sums
            s.batch_step(n_steps)
            X = torch.empty((B, 2 * S, 3), dtype=torch.float64, device="cuda")
            s.get_state(X)
            want = s.msd()                           # existing path (allocated scratch)
            ds.msd_static(X, Rref, S, B, out[call:], stream=stream)
            torch.cuda.synchronize()
            got = float(out[call].item())
            assert want > 0.0
            # same kernels, same order of additions
            assert abs(got - want) <= 1e-12 * want, (call, got, want)
            ref = oracle.msd(_centres(X.cpu().numpy()), _centres(X0))
            assert abs(got - ref) <= 1e-12 * ref, (call, got, ref)
    assert float(out[0].item()) != float(out[1].item())


@pytest.mark.gpu
def test_msd_static_small_then_large_and_limit():
    """A large call after a small one (stale partials beyond the small call's range), and the capacity check."""
    rng = np.random.default_rng(7)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for (W, S) in ((1, 3), (64, 1000), (2, 257)):
        X = rng.normal(size=(W, 2 * S, 3))
        R0 = rng.normal(size=(W, S, 3))
        ds.msd_static(torch.as_tensor(X, device="cuda"), torch.as_tensor(R0, device="cuda"), S, W, out)
        torch.cuda.synchronize()
        want = np.mean(np.sum((_centres(X) - R0) ** 2, axis=2))
        assert abs(float(out.item()) - want) <= 1e-12 * want, (W, S)
    x = torch.zeros(6, dtype=torch.float64, device="cuda")
    with pytest.raises(ds.DsError) as e:             # 16385 systems of one chunk: one partial too many; nothing is launched
        ds.msd_static(x, x, 1, ds.MSD_STATIC_MAX_PARTIALS + 1, out)
    assert e.value.code == ds.ERR_TOO_LARGE


def test_msd_static_argument_checks_without_device():
    """Host-side validation runs before any CUDA call."""
    L = ds.lib()
    assert L.ds_msd_static(None, None, 1, 1, None, None, 0) == ds.ERR_NULL
    one = np.zeros(8)
    p = one.ctypes.data
    assert L.ds_msd_static(p, p, 0, 1, p, None, 0) == ds.ERR_INVALID_PARAM
    assert L.ds_msd_static(p, p, 1, 0, p, None, 0) == ds.ERR_INVALID_PARAM
    assert L.ds_msd_static(p, p, 256 * ds.MSD_STATIC_MAX_PARTIALS + 1, 1, p, None, 0) == ds.ERR_TOO_LARGE
