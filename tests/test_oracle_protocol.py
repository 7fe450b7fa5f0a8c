"""Pins for the oracle prover/verifier (oracle/gkr_oracle.c) against the definitions and invariants.

Sources of truth: oracle/gkr_def.py (exponential-size sums written from SURVEY.md §8(c) "O-def",
PAPER.md:121 "a large sum over roughly S^3 terms"), the sum-check invariant g(0)+g(1) = claim
(BASELINE.json north_star), direct MLEs, and PAPER.md:47,67 (honest prover accepted, any single
changed word rejected).
"""
import random

import numpy as np
import pytest

import oracle
import vc_workloads as W
from oracle import gkr_def as D

P = (1 << 61) - 1


def _layers_def(c):
    return [(L.type, L.in1, L.in2) for L in c.layers]


def _run_layers(c, seed):
    """Drive the C oracle layer by layer, returning per-layer records for the checks."""
    oc = oracle.OracleCircuit(c)
    V = oc.evaluate(c.input)
    z, claim, ctr = oc.start(V[0], seed)
    recs = []
    for i in range(c.d):
        s = oc.log_below(i)
        tr, z2, claim2, ctr2, dbg = oc.prove_layer(i, V[i + 1], seed, ctr, z, claim)
        recs.append(dict(i=i, s=s, z=[int(v) for v in z[:c.layers[i].log_size]], claim=claim, ctr=ctr, tr=tr,
                         z_out=[int(v) for v in z2[:s]], claim_out=claim2, dbg=dbg))
        z, claim, ctr = z2, claim2, ctr2
    return oc, V, recs, (z, claim, ctr)


TINY = [
    ([0, 1], 1, 1), ([1, 2, 1], 2, 2), ([2, 2], 2, 3), ([0, 2, 3], 2, 4), ([3, 1, 2], 3, 5), ([1, 3], 2, 6),
]


@pytest.mark.parametrize("log_sizes,log_input,seed", TINY)
def test_round_messages_equal_the_exponential_sum(log_sizes, log_input, seed):
    """Per-gate single pass == brute force of the definition, every round, every t."""
    c = W.random_circuit(log_sizes, log_input, seed)
    oc, V, recs, _ = _run_layers(c, 77 + seed)
    Vd = D.evaluate(_layers_def(c), c.input)
    for i in range(c.d):
        assert [int(v) for v in V[i]] == Vd[i]
    for rec in recs:
        i, s = rec["i"], rec["s"]
        if 2 * s > 6:
            continue  # keep the brute force below ~2^5 suffixes x gates
        chal = [oracle.draw(77 + seed, rec["ctr"] + m) for m in range(2 * s)]
        for m in range(2 * s):
            want = D.round_message(_layers_def(c)[i], Vd[i + 1], rec["z"], chal[:m], s)
            got = [int(v) for v in rec["tr"][3 * m:3 * m + 3]]
            assert got == want, (i, m)


def _check_invariants(c, seed):
    oc, V, recs, (zf, claimf, ctrf) = _run_layers(c, seed)
    L = oracle.lib()
    for rec in recs:
        i, s, tr, dbg = rec["i"], rec["s"], rec["tr"], rec["dbg"]
        lay = c.layers[i]
        # first claim of the layer = V~_i(z) by direct MLE
        assert rec["claim"] == oracle.mle(V[i], rec["z"] + [0])
        claim = rec["claim"]
        chal = []
        for m in range(2 * s):
            G = [int(v) for v in tr[3 * m:3 * m + 3]]
            assert (G[0] + G[1]) % P == claim, (i, m)      # north_star: g_j(0)+g_j(1) = previous claim
            r = oracle.draw(seed, rec["ctr"] + m)
            chal.append(r)
            claim = D.interp2(G, r)
        r1, r2 = chal[:s], chal[s:]
        assert [int(v) for v in dbg.r1[:s]] == r1 and [int(v) for v in dbg.r2[:s]] == r2
        # end of phase 1 / 2: A[0] = V~(r1), B[0] = V~(r2)
        assert int(dbg.v1) == oracle.mle(V[i + 1], r1 + [0])
        assert int(dbg.v2) == oracle.mle(V[i + 1], r2 + [0])
        # final weights per type = wiring sums from their definition (eq tables built independently here)
        Tz, T1, T2 = oracle.eq_table(rec["z"]), oracle.eq_table(r1), oracle.eq_table(r2)
        Wdef = [0, 0, 0, 0]
        for g in range(1 << lay.log_size):
            Wdef[int(lay.type[g])] += int(Tz[g]) * int(T1[int(lay.in1[g])]) % P * int(T2[int(lay.in2[g])])
        Wdef = [w % P for w in Wdef]
        assert [int(w) for w in dbg.Wsum] == Wdef
        # last-round claim = sum_tau W_tau f_tau(v1,v2)
        assert claim == sum(Wdef[t] * D.gate_f(t, int(dbg.v1), int(dbg.v2)) for t in range(4)) % P
        # line reduction
        q = [int(v) for v in tr[6 * s:7 * s + 1]]
        assert q[0] == int(dbg.v1) and q[1] == int(dbg.v2)
        extra = oracle.mle(V[i + 1], D.line(r1, r2, s + 1) + [0])       # an (s+2)-th evaluation
        assert D.lagrange_eval(q, s + 1) == extra                        # q has degree <= s
        tau = oracle.draw(seed, rec["ctr"] + 2 * s)
        assert int(dbg.tau) == tau
        assert rec["z_out"] == D.line(r1, r2, tau)
        assert rec["claim_out"] == oracle.mle(V[i + 1], rec["z_out"] + [0])
    # whole proof: final claim = V~_d(z_d) of the input
    assert claimf == oracle.mle(c.input, [int(v) for v in zf[:c.log_input]] + [0])
    return oc, V, recs


@pytest.mark.parametrize("log_sizes,log_input,seed", TINY + [([0, 1, 2, 3, 4, 5], 6, 9), ([4, 6, 5], 7, 10), ([6, 3], 5, 12)])
def test_invariants_random_circuits(log_sizes, log_input, seed):
    _check_invariants(W.random_circuit(log_sizes, log_input, seed), 4242 + seed)


def test_invariants_config1_f2():
    c = W.config(1)
    _check_invariants(c, W.challenge_seed(1))


def test_invariants_small_structured():
    _check_invariants(W.f0_circuit(2, 5), 31)
    _check_invariants(W.matmul_circuit(2, 6), 32)
    _check_invariants(W.pm_circuit(4, 1, 7, planted=2), 33)


def test_wiring_sums_definition_tiny():
    c = W.random_circuit([2, 2], 2, 21)
    oc, V, recs, _ = _run_layers(c, 5)
    for rec in recs:
        s = rec["s"]
        r1 = [int(v) for v in rec["dbg"].r1[:s]]
        r2 = [int(v) for v in rec["dbg"].r2[:s]]
        assert [int(w) for w in rec["dbg"].Wsum] == D.wiring_sums(_layers_def(c)[rec["i"]], rec["z"], r1, r2)


def test_whole_prover_equals_layerwise_and_verifier_accepts():
    for c, seed in [(W.random_circuit([1, 3, 2, 4], 3, 40), 99), (W.config(1), W.challenge_seed(1))]:
        oc, V, recs, (zf, claimf, _) = _run_layers(c, seed)
        out, tr, fz, fc = oc.prove(c.input, seed)
        assert np.array_equal(tr, np.concatenate([r["tr"] for r in recs]))
        assert np.array_equal(out, V[0]) and fc == claimf
        assert tr.size == c.total_transcript_words == oc.transcript_words()
        assert oc.verify(c.input, out, seed, tr) == (True, 0, 0)


def test_layer_entry_in_isolation_matches_the_chain():
    c = W.random_circuit([2, 3, 1, 4, 2], 3, 55)
    seed = 1234
    oc, V, recs, _ = _run_layers(c, seed)
    for rec in recs:
        z, claim, ctr = oc.layer_entry(rec["i"], seed, V[rec["i"]])
        assert [int(v) for v in z[:len(rec["z"])]] == rec["z"]
        assert (claim, ctr) == (rec["claim"], rec["ctr"])


def test_tamper_every_word_is_rejected_where_predicted():
    """deviation in 'even a single bit of a single message' is caught."""
    c = W.random_circuit([1, 2, 3, 2], 3, 61)
    seed = 808
    oc = oracle.OracleCircuit(c)
    out, tr, _, _ = oc.prove(c.input, seed)
    assert oc.verify(c.input, out, seed, tr)[0]
    w = 0
    for i in range(c.d):
        s = oc.log_below(i)
        for m in range(2 * s):
            for t in range(3):
                bad = tr.copy()
                bad[w + 3 * m + t] = (int(bad[w + 3 * m + t]) + 1) % P
                acc, fl, fr = oc.verify(c.input, out, seed, bad)
                assert not acc
                if t < 2:                      # breaks G0+G1 = claim in this very round
                    assert (fl, fr) == (i, m)
                else:                          # G2 only enters the next claim
                    assert (fl, fr) == ((i, m + 1) if m + 1 < 2 * s else (i, 2 * s))
        for t in range(s + 1):
            bad = tr.copy()
            bad[w + 6 * s + t] = (int(bad[w + 6 * s + t]) ^ 1)
            acc, fl, fr = oc.verify(c.input, out, seed, bad)
            assert not acc
            if t < 2:                          # v1 / v2 enter the wiring check of this layer
                assert (fl, fr) == (i, 2 * s)
            else:                              # q[t>=2] only enters the next layer's first claim
                assert (fl, fr) == (i + 1, 0)
        w += 7 * s + 1
    for k in range(out.size):                  # wrong output -> layer 0, round 0
        bad = out.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert oc.verify(c.input, bad, seed, tr) == (False, 0, 0)
    for k in range(c.input.size):              # wrong input -> closing check
        bad = c.input.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert oc.verify(bad, out, seed, tr) == (False, c.d, 0)


def test_boolean_claim_point_reduces_to_one_gate():
    """z = bits of gate g*: beta is an indicator, the first claim is V_i[g*], and round 0 is one gate's term."""
    c = W.random_circuit([3, 3], 3, 71)
    oc = oracle.OracleCircuit(c)
    V = oc.evaluate(c.input)
    lay = c.layers[0]
    for gstar in (0, 5, 7):
        z = np.zeros(64, dtype=np.uint64); z[:3] = D.bits(gstar, 3)
        claim = int(V[0][gstar])
        tr, *_ = oc.prove_layer(0, V[1], 17, 0, z, claim)
        G = [int(v) for v in tr[:3]]
        a, b, typ = int(lay.in1[gstar]), int(lay.in2[gstar]), int(lay.type[gstar])
        bit, u = a & 1, a >> 1
        lo, hi, w = int(V[1][2 * u]), int(V[1][2 * u + 1]), int(V[1][b])
        want = [D.chi(bit, t) * D.gate_f(typ, (lo + t * (hi - lo)) % P, w) % P for t in (0, 1, 2)]
        assert G == want
        assert (G[0] + G[1]) % P == claim


# ------------------------------------------------------------------ the sum gate of large fan-in at the output (c-19)
@pytest.mark.parametrize("s,seed", [(1, 3), (3, 4), (5, 5)])
def test_sum_gate_rounds_equal_the_definition(s, seed):
    """Every message of orc_prove_sum_layer against the exponential sum of gkr_def.sum_gate_round_message on a random table
    of F_p words; the messages are linear in t (two words suffice); the claim chain; the point and the counter."""
    rng = random.Random(seed)
    Vb = np.array([rng.randrange(P) for _ in range(1 << s)], dtype=np.uint64)
    typ = np.array([W.SUM], np.uint8); z0 = np.zeros(1, np.uint32)
    c = W.Circuit([W.Layer(0, typ, z0, z0)], s, Vb, "sum gate alone")
    oc = oracle.OracleCircuit(c)
    assert oc.sum_output and c.sum_output and c.total_transcript_words == 2 * s == oc.transcript_words()
    y = sum(int(v) for v in Vb) % P
    assert int(oc.evaluate(Vb)[0][0]) == y == D.evaluate([(typ, z0, z0)], Vb)[0][0]
    tr, z, claim, ctr, _ = oc.prove_layer(0, Vb, 500 + seed, 0, np.zeros(64, np.uint64), y)
    chal = [oracle.draw(500 + seed, k) for k in range(s)]
    assert ctr == s and [int(v) for v in z[:s]] == chal            # z' = r: one point, no line restriction, no tau
    cur = y
    for m in range(s):
        want = D.sum_gate_round_message([int(v) for v in Vb], chal[:m], s)
        G = [int(v) for v in tr[2 * m:2 * m + 2]]
        assert G == want[:2], m
        assert want[2] == (2 * want[1] - want[0]) % P            # degree 1 in t
        assert (G[0] + G[1]) % P == cur
        cur = (G[0] + chal[m] * (G[1] - G[0])) % P
    assert claim == cur == D.mle([int(v) for v in Vb], chal) == oracle.mle(Vb, z)


def test_sum_gate_circuits_chain_verify_and_reject_tampering():
    """F2 and F0 as the paper draws them (one sum gate over the squares / over the ^(p-1) chain): outputs against the direct
    values, whole prover == layer-wise chain, layer_entry in isolation, honest transcript accepted, every word of the sum
    gate's rounds and the words of the layer below rejected where predicted."""
    for c, seed in [(W.f2_sum_circuit(4, 11), 91), (W.f0_sum_circuit(3, 12), 92)]:
        oc, V, recs, (zf, claimf, _) = _run_layers(c, seed)
        direct = sum(int(a) * int(a) for a in c.input) % P if c.name.startswith("F2") else int(np.count_nonzero(c.input))
        assert V[0].size == 1 and int(V[0][0]) == direct
        out, tr, fz, fc = oc.prove(c.input, seed)
        assert np.array_equal(tr, np.concatenate([r["tr"] for r in recs])) and fc == claimf
        assert tr.size == c.total_transcript_words == oc.transcript_words()
        for rec in recs:
            z, claim, ctr = oc.layer_entry(rec["i"], seed, V[rec["i"]])
            assert [int(v) for v in z[:len(rec["z"])]] == rec["z"] and (claim, ctr) == (rec["claim"], rec["ctr"])
        assert oc.verify(c.input, out, seed, tr) == (True, 0, 0)
        s = oc.log_below(0)
        for w in range(2 * s):                                      # G0 or G1 of round w // 2 breaks that round's sum
            bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
            assert oc.verify(c.input, out, seed, bad) == (False, 0, w // 2)
        bad = tr.copy(); bad[2 * s] = (int(bad[2 * s]) + 1) % P     # first word of layer 1
        assert oc.verify(c.input, out, seed, bad) == (False, 1, 0)
        assert oc.verify(c.input, (out + np.uint64(1)) % np.uint64(P), seed, tr) == (False, 0, 0)
        bad_in = c.input.copy(); bad_in[1] = (int(bad_in[1]) + 1) % P
        assert oc.verify(bad_in, out, seed, tr) == (False, c.d, 0)


def test_sum_gate_and_add_tree_reach_the_same_output():
    """The sum gate replaces the binary add tree of BASELINE.json's configs: same value, fewer layers."""
    a, b = W.f2_circuit(6, 9), W.f2_sum_circuit(6, 9)
    assert np.array_equal(a.input, b.input) and (a.d, b.d) == (7, 2)
    assert oracle.OracleCircuit(a).evaluate(a.input)[0][0] == oracle.OracleCircuit(b).evaluate(b.input)[0][0]
    a, b = W.f0_circuit(4, 9), W.f0_sum_circuit(4, 9)
    assert (a.d, b.d) == (123, 120)
    assert oracle.OracleCircuit(a).evaluate(a.input)[0][0] == oracle.OracleCircuit(b).evaluate(b.input)[0][0]
