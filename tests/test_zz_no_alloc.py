"""ra_mppi_weights_update_static: weights (17) and update (4) for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not an option: a controller that has given all of its device memory
to a fixed pool at start-up, a plug-in living inside a host process whose allocator it must leave alone, a real-time
thread for which an allocation (a device-wide synchronisation plus a driver call of unbounded length) costs the deadline.
A context is out of reach for them too, because creating one allocates.  The static entry point takes the caller's
input and output buffers and keeps the kernel's own scratch (per-range partial sums and a ticket counter) in an array
compiled into the library, so it needs neither.

What is checked here, through the C ABI: the static entry point gives the same v+ as the context-based
ra_mppi_weights_update on the same inputs, to the tolerance the parity tests use for v+ (parity_utils.TOL_V_ABS); on
two calls in a row with different sizes and inputs, so the second call runs on whatever the first left in the shared
array; sizes beyond the array's limit are refused with a message instead of overrunning it.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this extra must not hide
the parity tests.  It passes alone in a fresh process (its first call does the per-device set-up) and after the others.
"""
import numpy as np
import pytest

from paper_2209_12842_b200 import binding as B
from paper_2209_12842_b200 import workloads as W

from parity_utils import TOL_V_ABS


def _inputs(K, T, seed, lam):
    """Soft weights (about a tenth of the samples carry weight, so every range of samples contributes to v+) and
    controls correlated with the cost, so that the weighted mean sits well away from the plain mean and the clamps."""
    rng = np.random.default_rng(seed)
    z = rng.standard_normal(K)
    S = (40.0 + 1.5 * lam * z).astype(np.float32)
    u = rng.standard_normal((K, T, 2)) * np.array([0.1, 0.8]) + z[:, None, None] * np.array([0.05, 0.3])
    return S, u.astype(np.float32)


@pytest.mark.gpu
def test_static_update_matches_context_update_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2209_12842_b200 import build
    from paper_2209_12842_b200.controller import RaMppi
    build.build()
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    # (K, T): 5 ranges with a ragged last one; then fewer ranges and a shorter horizon, so stale partial sums of the
    # first call sit right behind the entries the second call uses; then one range (no exchange); then the limits
    cases = [(9000, 50), (4097, 30), (1000, 20), (B.RA_STATIC_MAX_K, 128)]
    worst = 0.0
    for i, (K, T) in enumerate(cases):
        p = W.small(W.config1(), K=K, M=16, T=T)
        ctl = RaMppi(p, device=0)
        S, u = _inputs(K, T, 100 + i, p.lam)
        d_S, d_u = ctl.tensor(S), ctl.tensor(u)
        ref = ctl.weights_update(d_S, d_u)["v_plus"]
        out = torch.full((T, 2), float("nan"), device=ctl.device, dtype=torch.float32)
        for call in range(2):   # the same inputs twice as well: the re-armed ticket and the kept partial sums
            out.fill_(float("nan"))
            B.ra_mppi_weights_update_static(K, T, p.lam, p.u_min, p.u_max, d_S.data_ptr(), d_u.data_ptr(),
                                            out.data_ptr(), stream)
            torch.cuda.synchronize()
            err = float((out - ref).abs().max())
            assert np.isfinite(err) and err < TOL_V_ABS, f"K={K} T={T} call {call}: |v+ - context v+| = {err:.3e}"
            worst = max(worst, err)
        # the comparison is not vacuous: the weighted mean is away from the clamps and differs from a plain mean
        r = ref.cpu().numpy()
        assert np.abs(r - u.mean(axis=0)).max() > 10 * TOL_V_ABS
        assert (r > np.asarray(p.u_min)).all() and (r < np.asarray(p.u_max)).all()
        ctl.close()
    print(f"static update vs context update: max |dv+| = {worst:.2e}")


def test_static_update_refuses_what_does_not_fit():
    """No GPU needed: the sizes are checked before any CUDA call, and the reason can be read back."""
    from paper_2209_12842_b200 import build
    build.build()
    lo, hi = [-1.0, -0.5], [1.0, 0.5]
    fake = 256   # never dereferenced: the call is refused first
    for K, T, status, word in ((B.RA_STATIC_MAX_K + 1, 50, B.RA_EUNSUPPORTED, "static scratch"),
                               (1024, 129, B.RA_EUNSUPPORTED, "static scratch"),
                               (0, 50, B.RA_EINVAL, "at least 1")):
        with pytest.raises(B.RaMppiError) as e:
            B.ra_mppi_weights_update_static(K, T, 1.0, lo, hi, fake, fake, fake)
        assert e.value.status == status and word in str(e.value), str(e.value)
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_weights_update_static(1024, 50, 0.0, lo, hi, fake, fake, fake)
    assert e.value.status == B.RA_EINVAL and "lambda" in str(e.value)
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_weights_update_static(1024, 50, 1.0, hi, lo, fake, fake, fake)
    assert e.value.status == B.RA_EINVAL
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_weights_update_static(1024, 50, 1.0, lo, hi, None, fake, fake)
    assert e.value.status == B.RA_EINVAL and "null" in str(e.value)
