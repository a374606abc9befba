"""GPU parity of the spacing variants: the keyed acceptance order (R19) and the dense diamond
dilation against the oracle, seeds and grown grids bit for bit."""
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


def both(liets, dims, boundary, storage, core, s, seed, order, method):
    o = oracle.Oracle(*dims, boundary)
    o.set_spacing_order(order)
    o.set_growth(0.08, 0.03, 0.01, 1)
    n_o = o.seed(core, s, seed)
    L = liets.Liets(*dims, boundary, storage)
    L.set_spacing(order, method)
    L.set_growth(0.08, 0.03, 0.01, liets.LAW_EQ1)
    n_g = L.seed(core, s, seed)
    return o, L, n_o, n_g


@pytest.mark.parametrize("storage", [0, 1, 2])
@pytest.mark.parametrize("boundary", [0, 1, 2])
@pytest.mark.parametrize("dims,core,s", [((70, 45, 33), 0.02, 5), ((130, 9, 17), 0.05, 3), ((5, 4, 3), 0.5, 2),
                                         ((64, 64, 8), 0.01, 12), ((191, 3, 2), 0.2, 4), ((40, 40, 40), 0.3, 2)])
def test_keyed_order_seeds_and_growth_equal_oracle(liets, storage, boundary, dims, core, s):
    o, L, n_o, n_g = both(liets, dims, boundary, storage, core, s, 17, 1, 0)
    assert n_g == n_o
    assert (L.grid() == o.grid()).all()
    assert L.spacing_rounds() >= 1
    rc_o = o.generate(0.4)
    rc_g = L.generate(0.4)
    assert rc_g[0] == rc_o[0] and rc_g[2] == o.n_solid
    assert (L.grid() == o.grid()).all()


def test_keyed_order_differs_from_index_order_and_needs_few_rounds(liets):
    """Same candidates, another maximal set; the dependency chains are short (4-5 rounds against a sweep
    through the grid)."""
    dims = (128, 128, 128)
    a = liets.Liets(*dims, 0, 1)
    a.seed(0.002, 10, 3)
    b = liets.Liets(*dims, 0, 1)
    b.set_spacing(liets.ORDER_KEYED, liets.SPACING_SPARSE)
    b.seed(0.002, 10, 3)
    ga, gb = a.grid(), b.grid()
    assert (ga != gb).any() and a.seed_info()[0] == b.seed_info()[0]
    assert 1 <= b.spacing_rounds() <= 12
    o = oracle.Oracle(*dims, 0)
    o.set_spacing_order(1)
    o.seed(0.002, 10, 3)
    assert (gb == o.grid()).all()
    b.set_spacing(liets.ORDER_INDEX, liets.SPACING_SPARSE)          # and back: the default order again
    b.seed(0.002, 10, 3)
    assert (b.grid() == ga).all() and b.spacing_rounds() == 0


@pytest.mark.parametrize("storage", [0, 1, 2])
@pytest.mark.parametrize("dims,core,s", [((70, 45, 33), 0.02, 5), ((130, 9, 17), 0.05, 3), ((66, 5, 4), 0.2, 2), ((64, 1, 9), 0.3, 3),
                                         ((64, 64, 8), 0.01, 12), ((191, 3, 2), 0.2, 4), ((40, 40, 40), 0.3, 2),
                                         ((100, 100, 100), 0.002, 10)])
def test_dense_dilation_gives_the_seeds_of_the_index_order(liets, storage, dims, core, s):
    o, L, n_o, n_g = both(liets, dims, 0, storage, core, s, 23, 0, 1)
    assert n_g == n_o
    assert (L.grid() == o.grid()).all()
    assert L.spacing_rounds() >= 1
    S = liets.Liets(*dims, 0, storage)                                # and of the default (sparse) path
    S.set_growth(0.08, 0.03, 0.01, liets.LAW_EQ1)
    assert S.seed(core, s, 23) == n_g and (S.grid() == L.grid()).all()
    L.generate(0.3)
    o.generate(0.3)
    assert (L.grid() == o.grid()).all()


def test_spacing_variant_arguments(liets):
    L = liets.Liets(16, 16, 16, 1, 1)
    with pytest.raises(liets.LietsError) as e:
        L.set_spacing(liets.ORDER_INDEX, liets.SPACING_DENSE)         # periodic grid
    assert e.value.code == liets.E_ARG
    W = liets.Liets(16, 16, 16, 0, 1)
    with pytest.raises(liets.LietsError) as e:
        W.set_spacing(liets.ORDER_KEYED, liets.SPACING_DENSE)
    assert e.value.code == liets.E_ARG
    with pytest.raises(liets.LietsError):
        W.set_spacing(2, 0)
    T = liets.Liets(1, 64, 64, 0, 1)                                  # one cell per 8-byte row word: the planes do not fit
    T.set_spacing(liets.ORDER_INDEX, liets.SPACING_DENSE)
    with pytest.raises(liets.LietsError) as e:
        T.seed(0.1, 3, 1)
    assert e.value.code == liets.E_CAPACITY


def test_spacing_variants_and_interaction_inside_a_batch(liets):
    """The generators of a batch take the spacing variants like any other; a grid with phase interaction is refused."""
    dims = (96, 40, 24)
    B = liets.LietsBatch(3, *dims)
    singles = []
    for i, (order, method) in enumerate(((0, 0), (1, 0), (0, 1))):
        for L in (B[i], liets.Liets(*dims, 0, 1)):
            L.set_spacing(order, method)
            L.set_growth(0.08, 0.03, 0.01, liets.LAW_EQ1)
            n = L.seed(0.01, 5, 40 + i)
        singles.append(L)
        assert B[i].seed_info()[0] == L.seed_info()[0] and n > 0
    res = B.generate(0.4)
    for i, L in enumerate(singles):
        rc, steps, n_solid = L.generate(0.4)
        assert (rc, steps, n_solid) == tuple(res[i]) and (B[i].grid() == L.grid()).all()
    m = singles[0].grid().ravel()
    B[1].set_blocked(m)
    B[1].set_interaction(0.1, 0.0, 0.0)
    B[1].seed(0.01, 5, 41)
    with pytest.raises(liets.LietsError) as e:
        B.generate(0.4)
    assert e.value.code == liets.E_ARG
