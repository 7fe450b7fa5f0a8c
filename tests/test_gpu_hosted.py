"""the copy-every-message approach (§5.1.3) against the oracle, word for word.

A circuit loaded with vc_circuit_load_hosted keeps records and weights in pinned host memory and streams every layer
through two device slots for EVERY message.  The transcript must not depend on where the gates live or on the piece size:
the expected words are the oracle's (and, at config 2's size, the oracle-written golden digests).
"""
import hashlib
import os

import numpy as np
import pytest

import oracle
import vc_workloads as W

pytestmark = pytest.mark.gpu

P = (1 << 61) - 1


@pytest.fixture(scope="module")
def vc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1202_1350_b200 as v
    v.lib()
    return v


def _prove_hosted(vc, c, seed, chunk_log, layerwise=False, swap=False):
    gc = vc.Circuit(c, hosted_chunk_log=chunk_log)
    gc.set_hosted_weights(swap)
    gc.set_input(c.input)
    gc.evaluate()
    ev_bytes = gc.hosted_bytes()
    if layerwise:
        gc.prove_layerwise(seed)
    else:
        gc.prove(seed)
    out, tr = gc.outputs().copy(), gc.transcript().copy()
    assert gc.flags() == 0
    return gc, out, tr, ev_bytes


CASES = [
    # (circuit, seed, chunk logs): pieces smaller than, equal to and larger than the layers; ragged last piece never occurs
    # (layers and pieces are powers of two) but single-piece and many-piece layers mix inside one proof
    (lambda: W.random_circuit([3, 9, 12, 11, 10], 10, 301), 71, (8, 10, 14)),
    (lambda: W.random_circuit([0, 13], 12, 302), 72, (8, 12)),                 # one output gate over a 2^13 layer
    (lambda: W.f0_circuit(9, 303), 73, (8, 9)),                               # two-lane chain layers, 1 and 4 pieces
    (lambda: W.matmul_circuit(4, 304), 74, (9,)),                             # 2^12 product gates in 8 pieces
    (lambda: W.pm_circuit(9, 3, 305, planted=3), 75, (10,)),
    (lambda: W.f2_sum_circuit(12, 306), 76, (8,)),                            # the sum gate on top of streamed squares
]


@pytest.mark.parametrize("make,seed,chunk_logs", CASES)
def test_hosted_circuit_transcript_is_the_oracles(vc, make, seed, chunk_logs):
    c = make()
    oc = oracle.OracleCircuit(c)
    want_out, want_tr, want_z, want_claim = oc.prove(c.input, seed)
    V = oc.evaluate(c.input)
    for chunk_log in chunk_logs:
        for layerwise, swap in ((False, False), (True, False), (False, True), (True, True)):
            gc, out, tr, ev_bytes = _prove_hosted(vc, c, seed, chunk_log, layerwise, swap)
            for i in range(c.d + 1):
                assert np.array_equal(gc.values(i), V[i]), (c.name, chunk_log, i)
            assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), (c.name, chunk_log, layerwise, swap)
            z, claim, ctr = gc.state()
            assert claim == want_claim and np.array_equal(z[:c.log_input], want_z[:c.log_input])
            assert gc.verify(c.input, out, seed, tr) == (True, 0, 0)
            # traffic: evaluation streams each record once; the proof streams, per message, 9 B of records per gate - and,
            # when the weights are swapped through the host, 8 B of weights each way on top (round 0 of a layer computes
            # them instead of reading them); recomputed weights never cross the link
            first = 1 if c.sum_output else 0
            gates = [1 << c.layers[i].log_size for i in range(first, c.d)]
            rounds = [2 * c.log_below(i) for i in range(first, c.d)]
            assert ev_bytes == (9 * sum(gates), 0)
            h2d, d2h = gc.hosted_bytes()
            ch = 1 << chunk_log                      # a layer that fits one slot is copied once (copy-once-per-layer)
            big = [(n, r) for n, r in zip(gates, rounds) if n > ch]
            small = sum(9 * n for n in gates if n <= ch)
            if swap:
                assert h2d == small + sum(n * (17 * r - 8) for n, r in big)
                assert d2h == sum(n * 8 * r for n, r in big)
            else:
                assert h2d == small + sum(n * 9 * r for n, r in big) and d2h == 0
            gc.close()


def test_hosted_matches_golden_digest_at_config_2_size(vc):
    """BASELINE.json config 2 (F2, n = 2^20) with every message streamed in pieces of 2^17 gates: the oracle's golden digests."""
    c = W.config(2)
    seed = W.challenge_seed(2)
    for swap in (False, True):
        _check_config2(vc, c, seed, swap)


def _check_config2(vc, c, seed, swap):
    gc, out, tr, _ = _prove_hosted(vc, c, seed, 17, swap=swap)
    g = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config2.txt")) as f:
        for line in f:
            if not line.startswith("#") and not line.startswith("layer"):
                k, v = line.split()
                g[k] = v
    sha = lambda a: hashlib.sha256(np.ascontiguousarray(a, dtype="<u8").tobytes()).hexdigest()
    assert sha(out) == g["outputs_sha256"] and sha(tr) == g["transcript_sha256"]
    assert gc.state()[1] == int(g["final_claim"])
    gc.close()


def test_hosted_handle_rules(vc):
    """Schedule 2 belongs to hosted handles and only to them; the device verifier needs resident records; chunk_log range."""
    c = W.random_circuit([2, 9], 9, 5)
    gc = vc.Circuit(c, hosted_chunk_log=8)
    for sched, code in ((0, 3), (1, 3)):
        with pytest.raises(vc.VCError) as e:
            gc.set_schedule(sched)
        assert e.value.code == code
    gc.set_schedule(2)
    gc.set_input(c.input); gc.evaluate(); gc.prove(9)
    with pytest.raises(vc.VCError) as e:
        gc.verify_device(9)
    assert e.value.code == 3
    gc.close()
    gr = vc.Circuit(c)
    with pytest.raises(vc.VCError) as e:
        gr.set_schedule(2)
    assert e.value.code == 3
    with pytest.raises(vc.VCError) as e:
        gr.hosted_bytes()
    assert e.value.code == 3
    with pytest.raises(vc.VCError) as e:
        gr.set_hosted_weights(True)
    assert e.value.code == 3
    gr.close()
    for bad in (7, 29):
        with pytest.raises(vc.VCError) as e:
            vc.Circuit(c, hosted_chunk_log=bad)
        assert e.value.code == 1
