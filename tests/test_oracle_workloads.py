"""The five BASELINE.json circuits: shape pins and oracle evaluation vs the directly computed answer.

PAPER.md:205-208 (§6.2): F2 = sum a_i^2; F0 = #{i: a_i != 0}; PM = number of occurrences of the
pattern; MATMULT = AB.  Direct values are computed with numpy / Python on the raw inputs, not with
any circuit code.
"""
import numpy as np
import pytest

import oracle
import vc_workloads as W

P = (1 << 61) - 1

# d, gates, input words, widest layer (log2), rounds, gate-rounds
SHAPES = {
    1: (11, 2_047, 1 << 10, 10, 130, 38_914),
    2: (21, 2_097_151, 1 << 20, 20, 460, 81_788_930),
    3: (135, 15_597_567, 1 << 16, 17, 4_316, 529_793_026),
    4: (8, 4_177_920, 1 << 15, 21, 282, 146_374_656),
    5: (142, 68_419_583, 1 << 19, 21, 5_062, 2_611_478_530),
}


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_config_shapes(k):
    c = W.config(k)
    d, gates, n_in, widest, rounds, gr = SHAPES[k]
    assert (c.d, c.gates, 1 << c.log_input, max(L.log_size for L in c.layers), c.rounds, c.gate_rounds) == \
        (d, gates, n_in, widest, rounds, gr)
    for i, L in enumerate(c.layers):
        nb = 1 << c.log_below(i)
        assert L.type.size == L.in1.size == L.in2.size == 1 << L.log_size
        assert int(L.in1.max()) < nb and int(L.in2.max()) < nb and int(L.type.max()) <= 3
        assert c.log_below(i) >= 1
        rel = L.type == W.RELAY
        assert np.array_equal(L.in1[rel], L.in2[rel])       # reading c-3: RELAY has in2 := in1
    assert int(c.input.max()) < P


def test_f2_node_count_matches_table2():
    # Table 2: 8.4 M inputs -> 25.2 M gates = 3n (n inputs + n squarers + n-1 adders)
    c = W.f2_circuit(6, 1)
    n = 64
    assert c.gates + n == 3 * n - 1
    assert round(3 * 8.4e6 / 1e6, 1) == 25.2


def test_tree_wiring_is_2g_2g1():
    c = W.config(1)
    for L in c.layers[:-1]:
        g = np.arange(1 << L.log_size, dtype=np.uint32)
        assert np.array_equal(L.in1, 2 * g) and np.array_equal(L.in2, 2 * g + 1)
        assert np.all(L.type == W.ADD)
    assert np.all(c.layers[-1].type == W.MULT)


def test_fermat_exponent_bits():
    # reading c-8: p-1 = 2^61-2 has bits 60..1 set and bit 0 clear -> 59 x (square, multiply) + 1 square
    e = P - 1
    assert [(e >> b) & 1 for b in range(61)] == [0] + [1] * 60
    x = 1                                                   # exponent reached by the chain, in the integers
    for _ in range(59):
        x = 2 * x + 1
    assert 2 * x == e


@pytest.mark.parametrize("k", [1, 2])
def test_f2_output_is_sum_of_squares(k):
    c = W.config(k)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    direct = sum(int(a) * int(a) for a in c.input)
    assert direct < 1 << 61                                 # no wrap-around at these sizes
    assert V[0].size == 1 and int(V[0][0]) == direct


def test_f0_output_is_number_of_nonzeros():
    c = W.config(3)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    assert int(V[0][0]) == int(np.count_nonzero(c.input))
    ind = V[16]                                             # layer just above the chain: a^(p-1) in {0,1}
    assert np.array_equal(ind, (c.input != 0).astype(np.uint64))
    frac = np.count_nonzero(c.input) / c.input.size
    assert 0.45 < frac < 0.55


def test_matmul_outputs_are_the_product():
    c = W.config(4)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    A = c.meta["A"].astype(object)
    B = c.meta["B"].astype(object)
    Cd = A.dot(B)                                           # exact Python ints; entries < 2^27
    assert np.array_equal(V[0].reshape(128, 128), np.array(Cd % P, dtype=np.uint64))
    assert np.array_equal(c.input[:128 * 128].reshape(128, 128), c.meta["A"])


@pytest.mark.parametrize("wrong", [0, 1, 7])
def test_matmul_equality_circuit_has_one_output_that_counts_wrong_entries(wrong):
    """a single output gate, zero iff C = AB (the F0 circuit counts the non-zero entries of AB - C)."""
    c = W.matmul_eq_circuit(3, 21, wrong)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    assert V[0].size == 1 and int(V[0][0]) == wrong
    A, B, Cc = (c.meta[k].astype(object) for k in "ABC")
    diff = (A.dot(B) - Cc) % P                               # exact Python ints
    lay = c.d - 1 - 4                                       # below it: the product layer and the 3 + 1 tree layers over the 2m terms
    assert np.array_equal(V[lay].reshape(8, 8), np.array(diff, dtype=np.uint64))
    assert int(np.count_nonzero(diff)) == wrong and c.meta["wrong"].size == wrong
    assert c.input.size == 4 * 64 and not c.input[3 * 64:].any()


@pytest.mark.slow
def test_pm_output_counts_nonmatching_cyclic_offsets():
    c = W.config(5)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    text, pat = c.meta["text"], c.meta["pattern"]
    T, Q = text.size, pat.size
    match = np.ones(T, dtype=bool)
    for j in range(Q):
        match &= np.roll(text, -j) == pat[j]                # text[(i+j) mod T] == pat[j]
    assert int(V[0][0]) == T - int(match.sum())
    assert int(match.sum()) >= 1 and all(match[o] for o in c.meta["planted_offsets"])


def test_small_pm_and_f0_against_direct():
    c = W.pm_circuit(5, 2, 3, planted=3)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    text, pat = c.meta["text"], c.meta["pattern"]
    cnt = sum(all(text[(i + j) % 32] == pat[j] for j in range(4)) for i in range(32))
    assert int(V[0][0]) == 32 - cnt
    c = W.f0_circuit(4, 8)
    V = oracle.OracleCircuit(c).evaluate(c.input)
    assert int(V[0][0]) == int(np.count_nonzero(c.input))
