"""Pins for the oracle's random-number layer (CPU only).

What is fixed from outside the oracle: the published Philox4x32-10 known answers, the C++26 value,
the worked visiting-order example of PAPER.md L112, exact-representability properties of the variates,
and the bijection/uniformity properties of Fisher-Yates (ref [35]).
"""
import itertools
import math
import os

import numpy as np
from scipy import stats

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]


def test_philox_known_answers(oracle_mod):
    for row in _rows("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row.split()]
        assert oracle_mod.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_philox_cxx26_10000th_value(oracle_mod):
    k0, k1, block, word, value = [int(x) for x in _rows("philox_cxx26.txt")[0].split()]
    assert oracle_mod.philox4x32_10([block, 0, 0, 0], [k0, k1])[word] == value


def test_philox_counter_and_key_words_all_matter(oracle_mod):
    base = oracle_mod.philox4x32_10([1, 2, 3, 4], [5, 6])
    seen = {tuple(base)}
    for pos in range(6):
        v = [1, 2, 3, 4, 5, 6]
        v[pos] ^= 0x10000
        out = tuple(oracle_mod.philox4x32_10(v[:4], v[4:]))
        assert out not in seen
        seen.add(out)


def test_visit_order_paper_example(oracle_mod):
    for row in _rows("visit_order_L112.txt"):
        n_m, perm, seq = [p.split() for p in row.split("|")]
        got = oracle_mod.visit_sequence([int(x) for x in perm], int(n_m[0]))
        assert got == [int(x) for x in seq]


def test_fisher_yates_is_a_bijection_on_index_choices(oracle_mod):
    # word w gives j = floor(w * bound / 2^32); ceil(j 2^32 / bound) is the smallest word for a given j.
    for n in (2, 3, 4):
        perms = set()
        choices = [range(i + 1) for i in range(n - 1, 0, -1)]     # j for i = n-1 .. 1
        for js in itertools.product(*choices):
            words = [-((-j << 32) // (i + 1)) for j, i in zip(js, range(n - 1, 0, -1))]
            p = oracle_mod.fisher_yates(list(range(n)), words)
            # independent restatement of Durstenfeld's algorithm
            ref = list(range(n))
            for j, i in zip(js, range(n - 1, 0, -1)):
                ref[i], ref[j] = ref[j], ref[i]
            assert p == ref
            perms.add(tuple(p))
        assert len(perms) == math.factorial(n)


def test_fisher_yates_single_element_untouched(oracle_mod):
    assert oracle_mod.fisher_yates([7], [123]) == [7]


def test_sweep_draws_uniform(oracle_mod):
    T = 24000
    perm_count = {}
    dirs = np.zeros(4)
    words = np.zeros(T)
    for t in range(T):
        order, d, w = oracle_mod.sweep_draws(12345, t)
        assert sorted(order) == [0, 1, 2, 3]
        perm_count[tuple(order)] = perm_count.get(tuple(order), 0) + 1
        dirs[d] += 1
        words[t] = w / 2.0 ** 32
    assert len(perm_count) == 24
    assert stats.chisquare(list(perm_count.values())).pvalue > 1e-3
    assert stats.chisquare(dirs).pvalue > 1e-3
    assert stats.kstest(words, "uniform").pvalue > 1e-3
    # a different seed or sweep index gives different draws
    assert oracle_mod.sweep_draws(12345, 0) != oracle_mod.sweep_draws(12346, 0)
    assert oracle_mod.sweep_draws(12345, 1 << 32) != oracle_mod.sweep_draws(12345, 0)


def test_variates_exact_symmetric_never_zero(oracle_mod):
    L = oracle_mod.lib()
    for R in (0, 1, 255, 256, 0x7FFFFFFF, 0x80000000, 0xFFFFFF00, 0xFFFFFFFF, 0x12345678):
        u32 = float(L.oracle_variate_sym_f32(R))
        u64 = float(L.oracle_variate_sym_f64(R))
        # closed forms in exact rational arithmetic
        assert u32 == ((2 * (R >> 8) + 1) - 2 ** 24) / 2.0 ** 24
        assert u64 == ((2 * R + 1) - 2 ** 32) / 2.0 ** 32
        assert u32 != 0.0 and u64 != 0.0 and abs(u32) < 1.0 and abs(u64) < 1.0
        # mirror word gives the mirror variate
        assert float(L.oracle_variate_sym_f32(0xFFFFFFFF - R)) == -u32
        assert float(L.oracle_variate_sym_f64(0xFFFFFFFF - R)) == -u64
        assert float(L.oracle_variate_unit_f32(R)) == (R >> 8) / 2.0 ** 24
        assert float(L.oracle_variate_unit_f64(R)) == R / 2.0 ** 32
    assert float(L.oracle_variate_unit_f32(0xFFFFFFFF)) < 1.0
    assert float(L.oracle_variate_unit_f64(0xFFFFFFFF)) < 1.0


def test_variate_moments(oracle_mod):
    L = oracle_mod.lib()
    rng = np.random.default_rng(0)
    R = rng.integers(0, 2 ** 32, size=20000, dtype=np.uint64)
    u = np.array([L.oracle_variate_sym_f64(int(r)) for r in R])
    assert abs(u.mean()) < 4 / math.sqrt(3 * len(u))
    assert abs((u ** 2).mean() - 1 / 3) < 0.01
    assert abs(np.abs(u).mean() - 0.5) < 0.01
