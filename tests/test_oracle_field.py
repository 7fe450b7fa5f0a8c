"""Pins for the oracle's field arithmetic, challenge generator, eq tables, MLEs and interpolation.

Every expected value here comes from Python big-int arithmetic on the *definition*, a published
known-answer vector, or a mathematical identity — never from the CUDA path.
"""
import random

import numpy as np
import pytest

import oracle
from oracle import gkr_def as D

P = (1 << 61) - 1
EDGE = [0, 1, 2, P - 1, P - 2, 1 << 60, (1 << 60) + 1, (1 << 61) - 2, 1 << 32, (1 << 32) - 1, 3]


def test_p_is_mersenne_61():
    # PAPER.md:197 (§6.1): "the finite field F_p with p = 2^61 - 1"
    assert oracle.lib().orc_p() == 2305843009213693951 == 2 ** 61 - 1


def test_field_ops_match_python_bigints():
    L = oracle.lib()
    rnd = random.Random(7)
    vals = EDGE + [rnd.randrange(P) for _ in range(200)]
    for a in vals:
        for b in EDGE + [rnd.randrange(P) for _ in range(5)]:
            assert L.orc_add(a, b) == (a + b) % P
            assert L.orc_sub(a, b) == (a - b) % P
            assert L.orc_mul(a, b) == (a * b) % P


def test_half_and_fermat():
    L = oracle.lib()
    assert L.orc_mul(2, 1 << 60) == 1          # 2^60 = 1/2 mod p
    rnd = random.Random(11)
    for a in [1, 2, P - 1] + [rnd.randrange(1, P) for _ in range(20)]:
        assert L.orc_pow(a, P - 1) == 1        # a^(p-1) = 1 iff a != 0
        assert L.orc_mul(a, L.orc_inv(a)) == 1
    assert L.orc_pow(0, P - 1) == 0


def test_splitmix64_known_answers():
    # Published splitmix64 test vectors (Vigna's splitmix64.c): first outputs for seeds 0 and 1234567.
    assert [oracle.mix(0, k) for k in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    assert [oracle.mix(1234567, k) for k in range(2)] == [6457827717110365317, 3203168211198807973]


def test_draw_is_low_61_bits_and_canonical():
    for seed in (0, 5, 2002):
        for k in range(50):
            v = oracle.mix(seed, k) & P
            assert oracle.draw(seed, k) == (0 if v == P else v)
            assert oracle.draw(seed, k) < P


@pytest.mark.parametrize("s", [0, 1, 2, 3, 4])
def test_eq_table_matches_product_definition(s):
    rnd = random.Random(100 + s)
    x = [rnd.randrange(P) for _ in range(s)]
    T = oracle.eq_table(x)
    assert T.size == 1 << s
    for u in range(1 << s):
        assert int(T[u]) == D.eq(u, x)
    assert sum(int(t) for t in T) % P == 1       # sum_g beta(z,g) = 1 for every z


def test_eq_table_boolean_point_is_indicator():
    s = 4
    for g in (0, 5, 15):
        T = oracle.eq_table(D.bits(g, s))
        assert [int(t) for t in T] == [1 if u == g else 0 for u in range(1 << s)]


@pytest.mark.parametrize("s", [0, 1, 2, 3, 4])
def test_mle_matches_definition_and_interpolates(s):
    rnd = random.Random(200 + s)
    V = [rnd.randrange(P) for _ in range(1 << s)]
    x = [rnd.randrange(P) for _ in range(s)]
    assert oracle.mle(V, x + [0]) == D.mle(V, x)
    for u in range(1 << s):                      # at Boolean points the MLE returns V[u]
        assert oracle.mle(V, D.bits(u, s) + [0]) == V[u]


def test_mle_of_linear_function_is_that_function():
    # V[u] = c0 + sum_k c_k u_k is multilinear already, so V~(x) = c0 + sum_k c_k x_k: closed form.
    s = 5
    rnd = random.Random(9)
    c = [rnd.randrange(P) for _ in range(s + 1)]
    V = [(c[0] + sum(c[k + 1] * ((u >> k) & 1) for k in range(s))) % P for u in range(1 << s)]
    x = [rnd.randrange(P) for _ in range(s)]
    assert oracle.mle(V, x) == (c[0] + sum(c[k + 1] * x[k] for k in range(s))) % P


def test_interp2_and_lagrange_against_known_polynomials():
    rnd = random.Random(3)
    for deg in (0, 1, 2, 5, 20):
        coef = [rnd.randrange(P) for _ in range(deg + 1)]
        poly = lambda t: sum(c * pow(t, k, P) for k, c in enumerate(coef)) % P  # noqa: E731
        q = [poly(t) for t in range(deg + 1)]
        for tau in (0, 1, deg, deg + 1, rnd.randrange(P)):
            assert oracle.lagrange(q, tau) == poly(tau)
    G = [5, 11, 21]                               # t^2*2 + 4t + 5 at 0,1,2
    for r in (0, 1, 2, 3, 10 ** 9):
        assert oracle.interp2(G, r) == (2 * r * r + 4 * r + 5) % P
    # interp2 = G0 (r-1)(r-2) 2^60 - G1 r (r-2) + G2 r (r-1) 2^60
    r = rnd.randrange(P)
    G = [rnd.randrange(P) for _ in range(3)]
    half = 1 << 60
    assert oracle.interp2(G, r) == (G[0] * (r - 1) * (r - 2) * half - G[1] * r * (r - 2) + G[2] * r * (r - 1) * half) % P
    assert oracle.interp2(G, r) == D.interp2(G, r)
