"""ea_c4_vectors_static: the full-vector C_4 (Eq. 3) without any allocation in the library -- its job list
and counters sit in a file-scope device array instead of cudaMalloc buffers (include/ea.h).  Checked against the existing
ea_c4_vectors path, bit for bit (integer sums), on two calls in a row: the array keeps the last call's contents, so the
second call -- other vectors, other spins, fewer vectors than the first -- would show anything that was not cleared.

Collected last on purpose (the suite runs with pytest -x).  Runs alone in a fresh process as well as after the others."""
import numpy as np
import pytest

from paper_1411_5512_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu


def _vectors(L, n, seed):
    rng = np.random.default_rng(seed)
    v = rng.integers(-2 * L, 2 * L, size=(n, 3)).astype(np.int32)
    run = min(40, n)
    v[:run] = [(k - 3, 1, -2) for k in range(run)]   # a run of consecutive dx: jobs of several vectors
    v[-1] = (0, 0, 0)                                # B = N exactly
    return v


@pytest.mark.parametrize("L", [8, 16, 64])           # L < 16: the transposed field sits in the static array as well
def test_static_scratch_entry_point_matches_the_allocating_path_twice_in_a_row(L):
    g = binding.Sim(L, 0.6, 0.8, n_replicas=2, seed=wl.seed_for(3, L), n_slots=0)
    g.sweep(5)
    first = _vectors(L, binding.C4_STATIC_MAX_VECTORS, 11)
    want = g.c4_vectors(first)
    got = g.c4_vectors_static(first)
    assert got.dtype == np.int64 and got.shape == want.shape
    assert np.array_equal(got, want)
    assert np.all(got[-1] == L ** 3)
    g.sweep(3)                                       # other spins, other and fewer vectors: stale counters would show
    second = _vectors(L, 137, 12)
    want2 = g.c4_vectors(second)
    got2 = g.c4_vectors_static(second)
    assert np.array_equal(got2, want2)
    assert not np.array_equal(got2[:40], got[:40])
    assert np.array_equal(g.c4_vectors_static(second), want2)   # and once more on the same input
    g.close()


def test_static_scratch_entry_point_rejects_what_does_not_fit():
    g = binding.Sim(16, 0.5, 0.8, n_replicas=2, seed=1, n_slots=0)
    assert g.c4_vectors_static(np.zeros((0, 3), dtype=np.int32)).shape == (0, 32)
    with pytest.raises(binding.EAError) as e:
        g.c4_vectors_static(np.zeros((binding.C4_STATIC_MAX_VECTORS + 1, 3), dtype=np.int32))
    assert "exceeds" in str(e.value) and str(binding.C4_STATIC_MAX_VECTORS) in str(e.value)
    g.close()
    one = binding.Sim(16, 0.5, 0.8, n_replicas=1, seed=1, n_slots=0)
    with pytest.raises(binding.EAError):
        one.c4_vectors_static([(1, 0, 0)])
    one.close()
