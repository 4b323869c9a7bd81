"""Pins for the oracle's order-k combination (O5), none of which re-types its formula.

P2/P3: recurrence == brute-force k-subset enumeration of the paper's explicit eqs. (2),(4),(5),(6)
        == the paper's printed closed forms (3),(7),(8),(9).
P4:    constant RF gives C(N,k)*a (golden/binomial_constant_rf.txt).
P5:    fewer than k non-zero channels gives exactly 0.
A1:    eq. (9) as extracted is NOT e5; the repaired term is (golden/newton_e5_terms.txt).
"""
import itertools
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _py_brute(s, k):
    """Independent python enumeration: signed k-th root of every k-subset product."""
    tot = 0.0
    for sub in itertools.combinations(range(len(s)), k):
        p = 1.0
        for i in sub:
            p *= s[i]
        tot += math.copysign(abs(p) ** (1.0 / k), p)
    return tot


@pytest.mark.parametrize("n", [5, 7, 9, 12])
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_routes_agree_random(orc, n, k):
    rng = np.random.default_rng(100 * n + k)
    for trial in range(4):
        s = rng.standard_normal(n) * 10.0 ** rng.uniform(-2, 2)
        a = orc.combine(s, k, orc.ROUTE_BRUTE)
        b = orc.combine(s, k, orc.ROUTE_RECUR)
        c = orc.combine(s, k, orc.ROUTE_CLOSED)
        scale = np.sum(np.abs(s)) ** 1.0 * math.comb(n, k) / n   # magnitude of the subset sum
        assert abs(a - b) <= 1e-12 * scale, (a, b)
        assert abs(a - c) <= 1e-11 * scale, (a, c)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_brute_matches_python_enumeration(orc, k):
    rng = np.random.default_rng(7 + k)
    s = rng.standard_normal(8)
    assert orc.combine(s, k, orc.ROUTE_BRUTE) == pytest.approx(_py_brute(s, k), rel=1e-13, abs=1e-13)


def test_order2_is_explicit_pairwise_signed_sqrt(orc):
    """eq. (2) PAPER.md:39 written as the double loop it prints."""
    rng = np.random.default_rng(2)
    s = rng.standard_normal(11)
    ref = 0.0
    for i in range(10):
        for j in range(i + 1, 11):
            p = s[i] * s[j]
            ref += np.sign(p) * math.sqrt(abs(p))
    assert orc.combine(s, 2, orc.ROUTE_RECUR) == pytest.approx(ref, rel=1e-13)
    assert orc.combine(s, 2, orc.ROUTE_CLOSED) == pytest.approx(ref, rel=1e-12)


def test_constant_rf_binomial_golden(orc):
    rows = [l.split() for l in open(os.path.join(GOLD, "binomial_constant_rf.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) >= 10
    for n, a, k, exp in rows:
        n, k, a, exp = int(n), int(k), float(a), float(exp)
        # the fixture itself is C(N,k)*a with the sign rule of PAPER.md:41/:62
        assert exp == math.comb(n, k) * (a if k % 2 else abs(a))
        s = np.full(n, a)
        for route in (orc.ROUTE_BRUTE, orc.ROUTE_RECUR, orc.ROUTE_CLOSED):
            if route == orc.ROUTE_BRUTE and math.comb(n, k) > 20000:
                continue
            assert orc.combine(s, k, route) == pytest.approx(exp, rel=1e-12), (n, a, k, route)


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_fewer_than_k_nonzero_is_exact_zero(orc, k):
    s = np.zeros(10)
    s[[1, 4, 6, 9][: k - 1]] = [3.0, -2.0, 0.5, 7.0][: k - 1]
    assert orc.combine(s, k, orc.ROUTE_BRUTE) == 0.0
    assert orc.combine(s, k, orc.ROUTE_RECUR) == 0.0
    # the Newton closed form only cancels to rounding
    assert abs(orc.combine(s, k, orc.ROUTE_CLOSED)) < 1e-10


def test_zero_channels_drop_out(orc):
    """A6: an out-of-record (zero) sample drops out of every subset; N is not reduced."""
    rng = np.random.default_rng(3)
    s = rng.standard_normal(9)
    s0 = np.concatenate([s[:4], [0.0, 0.0], s[4:]])
    for k in range(1, 6):
        assert orc.combine(s0, k) == pytest.approx(orc.combine(s, k), rel=1e-13, abs=1e-13)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_homogeneity_and_permutation(orc, k):
    """P6: degree-1 homogeneous; alpha<0 flips sign only for odd k."""
    rng = np.random.default_rng(40 + k)
    s = rng.standard_normal(10)
    base = orc.combine(s, k)
    for alpha in (2.5, -0.75):
        exp = base * (alpha if k % 2 else abs(alpha))
        # negative alpha with even k: sgn(prod of k negated samples) is unchanged
        assert orc.combine(alpha * s, k) == pytest.approx(exp, rel=1e-12)
    assert orc.combine(s[rng.permutation(10)], k) == pytest.approx(base, rel=1e-12, abs=1e-13)


def test_eq9_as_extracted_is_not_e5_and_repair_is(orc):
    """Reading A1: PAPER.md:79 lost a square.  golden/newton_e5_terms.txt is Newton's identity."""
    rng = np.random.default_rng(9)
    s = rng.standard_normal(9)
    brute = orc.combine(s, 5, orc.ROUTE_BRUTE)
    assert orc.combine(s, 5, orc.ROUTE_CLOSED, repaired=True) == pytest.approx(brute, rel=1e-10)
    assert abs(orc.combine(s, 5, orc.ROUTE_CLOSED, repaired=False) - brute) > 1e-3 * abs(brute)
    # evaluate the golden monomial table directly on the power sums of the signed fifth roots
    u = np.sign(s) * np.abs(s) ** 0.2
    p = [None] + [np.sum(u ** m) for m in range(1, 6)]
    tot = 0.0
    coeff_sum = 0
    for line in open(os.path.join(GOLD, "newton_e5_terms.txt")):
        if not line.strip() or line[0] == "#":
            continue
        c, *a = [int(v) for v in line.split()]
        assert sum(m * am for m, am in zip(range(1, 6), a)) == 5   # every monomial has weight 5
        coeff_sum += c
        tot += c * np.prod([p[m] ** am for m, am in zip(range(1, 6), a)])
    assert coeff_sum == 0  # e5(1,0,0,...) = 0: all p_m = 1
    assert tot / 120.0 == pytest.approx(brute, rel=1e-10)
