"""Pins of the oracle's composition initial state (S10) and of Eq. 8's normalisation at unequal
concentrations: exact counts, agreement with a position-dictionary recount of the pair statistics, and
alpha = 0 within sampling error for a random solid solution of the paper's Fe29Co29Ni28Al7Ti7 proportions
(PAPER.md:141, 159-163).  A normalisation by the wrong species' concentration fails the last one."""
import numpy as np
import pytest

import oracle
from smcx_inputs import composition_counts, cooling_stages, make_accept_table, make_epi


def test_composition_counts_recipe():
    assert composition_counts(100, (29, 29, 28, 7, 7)) == [29, 29, 28, 7, 7]
    c = composition_counts(8 * 8 * 8 * 4, (29, 29, 28, 7, 7))
    assert sum(c) == 2048 and c == [594, 594, 574, 143, 143]
    assert composition_counts(10, (1, 1, 1)) == [4, 3, 3]
    assert cooling_stages(1720, 860, 5) == [1720, 1505, 1290, 1075, 860] and cooling_stages(700, 100, 1) == [700]


def _oracle(dims=(8, 8, 8), n_sp=5, seed=77):
    epi = make_epi(3, n_sp, 400, 3)
    return oracle.Oracle(1, dims, n_sp, 3, epi, 4, make_accept_table(690), seed, init=False), epi


def test_exact_counts_and_rejections():
    o, _ = _oracle()
    counts = composition_counts(o.n_sites, (29, 29, 28, 7, 7))
    o.init_composition(counts)
    s = o.species()
    assert np.bincount(s, minlength=5).tolist() == counts
    # a species may be absent; the others still get their exact counts
    o.init_composition([0, 2048, 0, 0, 0])
    assert (o.species() == 1).all()
    for bad in ([1, 1, 1, 1, 1], [-1, 2049, 0, 0, 0]):
        with pytest.raises(ValueError):
            o.init_composition(bad)
    # the placement is the permutation of S6: site i holds the species whose range contains pi(i)
    o.init_composition(counts)
    cum = np.cumsum(counts)
    s = o.species()
    for i in (0, 1, 17, 1000, 2047):
        assert s[i] == int(np.searchsorted(cum, o.init_permutation(i), side="right"))


def test_random_solid_solution_has_zero_sro_at_unequal_concentrations():
    """alpha_s^{p'p} = 1 - P(p|p') / c_p: for independent placement P(p|p') = (n_p - [p = p']) / (N - 1), so
    alpha = O(1/N) + noise.  With c_p' in the denominator instead (the transposed normalisation) the
    Fe/Al entries would be 1 - 0.07/0.29 = 0.76 or 1 - 0.29/0.07 = -3.1."""
    o, _ = _oracle(dims=(16, 16, 16), seed=5)
    counts = composition_counts(o.n_sites, (29, 29, 28, 7, 7))
    o.init_composition(counts)
    alpha, pairs = o.sro()
    N = o.n_sites
    Z = [12, 6, 24]
    for s in range(3):
        for a in range(5):
            assert pairs[s, a].sum() == Z[s] * counts[a]                 # sum rule of Eq. 8's counts
            for b in range(5):
                expect = Z[s] * counts[a] * counts[b] / N                 # ordered pairs of a random solution
                sigma = np.sqrt(expect)
                assert abs(pairs[s, a, b] - expect) < 6 * sigma + Z[s], (s, a, b)
                assert abs(alpha[s, a, b]) < 6 * sigma / expect + 2e-3, (s, a, b, alpha[s, a, b])
    assert (pairs == pairs.transpose(0, 2, 1)).all()


def test_energy_bookkeeping_after_sweeps_from_a_composition_state():
    o, _ = _oracle()
    o.init_composition(composition_counts(o.n_sites, (29, 29, 28, 7, 7)))
    e0 = o.energy()
    o.sweep(3)
    assert o.energy() == o.running_energy() and o.energy_trace()[-1] == o.energy() and o.energy() != e0
    assert np.bincount(o.species(), minlength=5).tolist() == composition_counts(o.n_sites, (29, 29, 28, 7, 7))
