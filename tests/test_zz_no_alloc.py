"""gcamb_los_interp_sources_noalloc: InterpolateSources (reading R26) for callers that cannot
allocate device memory: the scratch of the two kernels is a file-scope `static __device__` array of the library
(at most 2^20 doubles), not a caller buffer.

The new entry point is compared with the existing path (gcamb_los_interp_sources with caller-owned scratch) on
two calls in a row with DIFFERENT inputs, so that what the first call leaves in the shared array cannot pass
for the second call's result; the existing path itself is checked against the long-double oracle in
tests/test_gpu_tensor.py, and once more here at the bar that file uses (1e-13 of the largest coarse value).

This file sorts last on purpose (the suite runs with `pytest -x`); it needs nothing from the other tests and
passes alone in a fresh process as well as after them.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_25110_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-13          # of max|S_coarse|: the bar of tests/test_gpu_tensor.py::test_interp_sources_against_the_oracle
TAU0 = 14000.0
STATIC_SCRATCH_DOUBLES = 1 << 20


@pytest.fixture(scope="module")
def los():
    from paper_2509_25110_b200 import los as _los
    _los.load_library()
    assert torch.cuda.is_available()
    return _los


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def coarse_sources(kc, n_tau, n_series, seed):
    rng = np.random.default_rng(seed)
    base = np.cos(30.0 * kc[:, None] * (1.0 + np.arange(n_tau)[None, :] / n_tau)) * np.exp(-(kc[:, None] / 0.3) ** 2)
    return base * (1.0 + 0.01 * rng.standard_normal((n_series,) + base.shape))


@pytest.mark.parametrize("shape", [
    # (n_kc, n_k, n_tau, n_series)
    (300, 3000, 1200, 2),      # the bench workload: T and E of config 1, 300 -> 3000 wavenumbers (720000 doubles of scratch)
    (41, 257, 181, 3),         # ragged sizes, shared-memory solve with 32 threads
    (2, 17, 40, 1),            # two knots: straight lines, all second derivatives zero
])
def test_noalloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row(los, shape):
    n_kc, n_k, n_tau, n_series = shape
    assert n_series * n_kc * n_tau <= STATIC_SCRATCH_DOUBLES
    kc = synth.k_grid(n_kc, 1e-5, 0.6)
    k = synth.k_grid(n_k, 1e-5, 0.6)
    tau = np.linspace(100.0, 13900.0, n_tau)
    plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, tau, TAU0)
    si = los.SourceInterp(plan, kc)
    outs = []
    for call, seed in enumerate((11, 12)):                     # two calls in a row, different sources
        S_c = coarse_sources(kc, n_tau, n_series, seed)
        d_S = dev(S_c)
        ref = si.gcamb_los_interp_sources(d_S)                 # existing path: caller-owned scratch
        out = torch.full((n_series, n_k, n_tau), float("nan"), dtype=torch.float64, device="cuda")
        free_before = torch.cuda.mem_get_info()[0]
        si.gcamb_los_interp_sources_noalloc(d_S, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before     # the call took no device memory
        got, want = out.cpu().numpy(), ref.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got - want)) <= TOL * np.max(np.abs(S_c))
        assert np.array_equal(got, want)                       # same kernels, same order: bit for bit
        if call == 1 and n_kc <= 41:                           # and the oracle, at the bar of the existing test
            for s in range(n_series):
                o = oracle.interp_sources(kc, k, S_c[s], real="f80")
                assert np.max(np.abs(got[s] - o)) <= TOL * np.max(np.abs(S_c[s]))
        outs.append(got)
    assert not np.array_equal(outs[0], outs[1])                # the second call did not return the first one's result
    si.close()
    plan.close()


def test_noalloc_entry_point_rejects_sizes_beyond_the_static_scratch(los):
    n_kc, n_tau = 300, 1200
    kc = synth.k_grid(n_kc, 1e-5, 0.6)
    k = synth.k_grid(50, 1e-5, 0.6)
    plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, np.linspace(100.0, 13900.0, n_tau), TAU0)
    si = los.SourceInterp(plan, kc)
    n_series = 3                                               # 1080000 doubles > 1048576
    assert n_series * n_kc * n_tau > STATIC_SCRATCH_DOUBLES
    S = torch.zeros(n_series, n_kc, n_tau, dtype=torch.float64, device="cuda")
    out = torch.full((n_series, 50, n_tau), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(los.GcambError) as e:
        si.gcamb_los_interp_sources_noalloc(S, out)
    assert e.value.status == 1 and "1080000" in str(e.value) and "1048576" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())                        # nothing was launched
    si.gcamb_los_interp_sources(S, out=out)                    # the existing path takes the same sizes
    torch.cuda.synchronize()
    assert bool((out == 0).all())
    si.close()
    plan.close()
