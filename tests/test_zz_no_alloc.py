"""liets_s2_static, the entry point that allocates nothing (pair counters in a file-scope device array), against liets_s2:
the same integers, on calls in a row that share the array.  Collected last (pytest -x stops at the
first failure)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def liets():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2602_11734_b200 as m
    m.lib()
    return m


def grown(liets, dims, boundary, storage, target=0.5, seed=5):
    L = liets.Liets(*dims, boundary, storage)
    L.set_growth(0.08, 0.03, 0.01, liets.LAW_EQ1)
    L.seed(0.02, 2, rng_seed=seed)
    L.generate(target)
    return L


def same(a, b):
    return a[0].dtype == b[0].dtype and (a[0] == b[0]).all() and (a[1] == b[1]).all()


@pytest.mark.parametrize("storage", [1, 2])
@pytest.mark.parametrize("boundary", [0, 1, 2])
def test_static_scratch_equals_allocating_path_on_calls_in_a_row(liets, storage, boundary):
    """Two (and more) calls in a row, the second with fewer lags on another axis of another grid: the array still holds
    the first call's counts when the second starts, and nothing of them may show."""
    A = grown(liets, (150, 37, 29), boundary, storage)
    B = grown(liets, (70, 45, 33), boundary, storage, target=0.3, seed=9)
    first = A.s2_static(0, 2 * 150 + 3)                       # lags beyond the grid included
    assert same(first, A.s2(0, 2 * 150 + 3))
    assert first[0][0] > 0 and first[0][1] > 0                # the counters were really used
    second = B.s2_static(2, 20)
    assert same(second, B.s2(2, 20))
    for axis in range(3):                                     # and on: every axis of both grids, alternating
        for L, rmax in ((A, 64), (B, 7), (A, 0)):
            assert same(L.s2_static(axis, rmax), L.s2(axis, rmax)), (axis, rmax)
    assert same(A.s2_static(0, 2 * 150 + 3), first)           # the same call again gives the same counts


def test_static_scratch_equals_oracle(liets, oracle_mod):
    """One case against the oracle's triple loop as well (the other path's parity is in test_gpu_parity.py)."""
    L = grown(liets, (130, 9, 17), 0, 1)
    for axis in range(3):
        p, v = L.s2_static(axis, 140)
        po, vo = oracle_mod.s2(L.grid(), False, axis, 140)
        assert (p == po).all() and (v == vo).all(), axis


def test_static_scratch_limits(liets):
    L = grown(liets, (64, 64, 8), 0, 1)
    top = liets.S2_STATIC_MAX_LAGS - 1
    assert same(L.s2_static(1, top), L.s2(1, top))            # the whole array
    with pytest.raises(liets.LietsError) as e:
        L.s2_static(1, top + 1)
    assert e.value.code == liets.E_CAPACITY and "4096" in str(e.value)
    with pytest.raises(liets.LietsError) as e:
        L.s2_static(3, 4)
    assert e.value.code == liets.E_ARG
    assert same(L.s2_static(0, 5), L.s2(0, 5))                # still usable after the refusals
    U = grown(liets, (20, 10, 5), 0, 0)
    with pytest.raises(liets.LietsError) as e:
        U.s2_static(0, 4)
    assert e.value.code == liets.E_ARG and "bit-row" in str(e.value)
    fresh = liets.Liets(8, 8, 8, 0, 1)
    with pytest.raises(liets.LietsError) as e:
        fresh.s2_static(0, 4)
    assert e.value.code == liets.E_STATE


def test_static_scratch_call_allocates_no_device_memory(liets):
    """The driver's free-memory figure does not move across calls (liets_s2's cudaMalloc / cudaFree pairs would not show
    here either; this catches a leak or a lazily created buffer)."""
    import torch
    L = grown(liets, (150, 37, 29), 0, 1)
    L.s2_static(0, 100)                                       # module load and symbol lookup happen at the first call
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        L.s2_static(1, 300)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == before
