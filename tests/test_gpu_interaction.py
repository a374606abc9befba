"""GPU parity of interacting phases (PAPER.md:40 step 4; R20): the growing phase also grows at its interface with
the earlier phases, with the phase-interaction probabilities I -- against the oracle, bit for bit."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def liets():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2602_11734_b200 as m
    m.lib()
    return m


def first_phase(dims, boundary, seed=4):
    a = oracle.Oracle(*dims, boundary)
    a.set_growth(0.2, 0.1, 0.05, 0)
    a.seed(0.01, 0, seed)
    for _ in range(3):
        a.step()
    return a.grid().ravel().copy()


@pytest.mark.parametrize("storage", [1, 2])
@pytest.mark.parametrize("boundary", [0, 1, 2])
@pytest.mark.parametrize("dims", [(70, 45, 33), (130, 9, 17), (5, 4, 3), (64, 64, 8), (191, 3, 2), (150, 97, 1)])
def test_second_phase_with_interaction_equals_oracle(liets, storage, boundary, dims):
    m = first_phase(dims, boundary)
    o = oracle.Oracle(*dims, boundary)
    o.set_growth(0.08, 0.03, 0.01, 1)
    o.set_blocked(m)
    o.set_interaction(0.2, 0.07, 0.004)
    L = liets.Liets(*dims, boundary, storage)
    L.set_growth(0.08, 0.03, 0.01, liets.LAW_EQ1)
    L.set_blocked(m)
    L.set_interaction(0.2, 0.07, 0.004)
    assert L.seed(0.004, 3, 21) == o.seed(0.004, 3, 21)
    o.set_target(0.35)
    L.set_target(0.35)
    for _ in range(3):                                       # step by step first
        o.step()
        n_solid, _ = L.step()
        assert n_solid == o.n_solid
        assert (L.grid() == o.grid()).all()
    rc_o, steps_o = o.generate(0.35)
    rc, steps, n_solid = L.generate(0.35)
    assert (rc, steps, n_solid) == (rc_o, steps_o, o.n_solid)
    g = L.grid()
    assert (g == o.grid()).all()
    assert not (g.ravel() & m).any()                         # the earlier phase keeps its cells
    # and without interaction the same context gives the independent phase again
    L.set_interaction(0.0, 0.0, 0.0)
    o.set_interaction(0.0, 0.0, 0.0)
    assert L.seed(0.004, 3, 21) == o.seed(0.004, 3, 21)
    o.generate(0.2)
    L.generate(0.2)
    assert (L.grid() == o.grid()).all()


@pytest.mark.parametrize("storage", [1, 2])
@pytest.mark.parametrize("boundary", [0, 1])
def test_interaction_with_probability_one_coats_the_earlier_phase_on_the_device(liets, storage, boundary):
    """No seeds, G = 0, I = 1: one step gives exactly the unassigned cells that touch the earlier phase; a second step
    adds nothing.  (The closed form is pinned for the oracle in tests/test_oracle_pins.py.)"""
    dims = (140, 21, 19)
    m = np.zeros(dims[::-1], np.uint8)
    m[3:9, 4:15, 60:70] = 1
    m[0, 0, 0] = 1
    m[18, 20, 139] = 1
    o = oracle.Oracle(*dims, boundary)
    o.set_growth(0.0, 0.0, 0.0, 0)
    o.set_blocked(m)
    o.set_interaction(1.0, 1.0, 1.0)
    o.seed_explicit([], 3)
    L = liets.Liets(*dims, boundary, storage)
    L.set_growth(0.0, 0.0, 0.0, liets.LAW_CONSTANT)
    L.set_blocked(m)
    L.set_interaction(1.0, 1.0, 1.0)
    L.seed_explicit([], 3)
    for _ in range(2):
        o.step()
        n_solid, _ = L.step()
        assert n_solid == o.n_solid and (L.grid() == o.grid()).all()
    assert o.n_solid > 0


def test_interaction_arguments(liets):
    U = liets.Liets(16, 16, 16, 0, 0)
    with pytest.raises(liets.LietsError) as e:
        U.set_interaction(0.1, 0.0, 0.0)
    assert e.value.code == liets.E_ARG
    U.set_interaction(0.0, 0.0, 0.0)                         # switching it off is fine everywhere
    T = liets.Liets(16, 16, 16, 0, 1)
    with pytest.raises(liets.LietsError):
        T.set_interaction(1.5, 0.0, 0.0)
    T.set_growth(0.1, 0.1, 0.1, liets.LAW_CONSTANT)
    T.seed(0.01, 0, 1)
    T.set_interaction(0.1, 0.0, 0.0)
    with pytest.raises(liets.LietsError) as e:
        T.step()                                             # seed again first
    assert e.value.code == liets.E_STATE
    T.seed(0.01, 0, 1)                                       # no earlier phase: nothing interacts, a plain run
    P = liets.Liets(16, 16, 16, 0, 1)
    P.set_growth(0.1, 0.1, 0.1, liets.LAW_CONSTANT)
    P.seed(0.01, 0, 1)
    for _ in range(3):
        assert T.step()[0] == P.step()[0]
    assert (T.grid() == P.grid()).all()
