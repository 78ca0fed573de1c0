"""The allocation-free entry point mcrt_traj_math_device_static against the allocating path it is a variant of.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1203_2941_b200 import binding
    binding.load_library()
    return binding


def _values(seed, n):
    rng = np.random.default_rng(seed)
    z = rng.random(n)
    z = (2.0 * np.floor(z * 2.0 ** 52) + 1.0) * 2.0 ** -53          # the generator's uniforms: strictly inside (0, 1)
    edge = [2.0 ** -53, 1.0 - 2.0 ** -53, 0.25, 0.5]
    z[:min(4, n)] = edge[:min(4, n)]
    return z


def test_static_scratch_entry_point_matches_allocating_path_twice(B):
    """Two calls in a row share the static device array: a full-size call, then a shorter one with other values whose
    results must not show anything the first call left behind.  Bit-equal to mcrt_traj_math_device (the tolerance of
    the parity tests for these functions: none)."""
    for seed, n in ((101, B.MCRT_STATIC_MAX_N), (202, 1000), (303, 1)):
        z = _values(seed, n)
        ref = B.mcrt_traj_math_device(z)
        got = B.mcrt_traj_math_device_static(z)
        for name, a, b in zip(("ln", "sin", "cos"), ref, got):
            assert a.shape == b.shape == (n,)
            assert np.array_equal(a.view(np.uint64), b.view(np.uint64)), (seed, name)
        assert np.all(got[0] < 0.0) and np.all(np.abs(got[1] ** 2 + got[2] ** 2 - 1.0) < 1e-15)


def test_static_scratch_entry_point_rejects_sizes_beyond_its_array(B):
    with pytest.raises(Exception) as ei:
        B.mcrt_traj_math_device_static(_values(1, B.MCRT_STATIC_MAX_N + 1))
    assert "MCRT_STATIC_MAX_N" in str(ei.value) or "65536" in str(ei.value)
    # the entry point still works afterwards
    z = _values(2, 257)
    assert np.array_equal(B.mcrt_traj_math_device(z)[0], B.mcrt_traj_math_device_static(z)[0])
