"""GPU parity for vc_verify_transcript_device: the verifier's O(S) sums on the device.

Expected values come from oracle/ only: the start claim and the closing input extension are the oracle's MLE, the
per-type wiring sums are the ones the oracle prover reports per layer (pinned against their definition in
tests/test_oracle_protocol.py), accept/reject and the failure coordinates are the oracle verifier's.
"""
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


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint64).view(np.int64)).cuda()


def _oracle_sums(c, seed):
    """[start claim, 4 wiring sums per layer ..., V~_d(z_d)] from the oracle prover, plus its transcript."""
    oc = oracle.OracleCircuit(c)
    V = oc.evaluate(c.input)
    z, claim, ctr = oc.start(V[0], seed)
    sums, tr = [claim], []
    for i in range(c.d):
        t, z, claim, ctr, dbg = oc.prove_layer(i, V[i + 1], seed, ctr, z, claim)
        tr.append(t)
        sums += [int(w) for w in dbg.Wsum]
    sums.append(oracle.mle(c.input, z[:c.log_input]))
    return np.array(sums, dtype=np.uint64), np.concatenate(tr), V[0]


@pytest.mark.parametrize("log_sizes,log_input,seed", [
    ([1, 2, 3, 2], 3, 61), ([0, 1, 1], 1, 5), ([2, 4, 6, 8, 10, 12], 11, 77), ([0, 11, 12], 13, 21)])
def test_device_sums_and_verdict_match_oracle(vc, log_sizes, log_input, seed):
    c = W.random_circuit(log_sizes, log_input, seed)
    want, tr, out = _oracle_sums(c, 900 + seed)
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(900 + seed)
    assert np.array_equal(gc.transcript(), tr)
    assert gc.verify_device(900 + seed) == (True, 0, 0)
    assert np.array_equal(gc.verifier_sums(), want)                       # every device sum, word for word
    # the verifier is independent of the prover's buffers: feed it the oracle's transcript and outputs
    assert gc.verify_device(900 + seed, d_outputs=_dev(out), d_transcript=_dev(tr)) == (True, 0, 0)
    gc.close()


def test_device_verifier_rejects_tampering_like_the_oracle(vc):
    c = W.random_circuit([1, 2, 3, 2], 3, 61)
    seed = 808
    oc = oracle.OracleCircuit(c)
    out, tr, _, _ = oc.prove(c.input, seed)
    gc = vc.Circuit(c)
    d_in, d_out, d_tr = _dev(c.input), _dev(out), _dev(tr)
    assert gc.verify_device(seed, d_in, d_out, d_tr) == (True, 0, 0)
    for w in range(tr.size):
        bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
        got = gc.verify_device(seed, d_in, d_out, _dev(bad))
        assert got == oc.verify(c.input, out, seed, bad) and not got[0], w
    for k in range(out.size):
        bad = out.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert gc.verify_device(seed, d_in, _dev(bad), d_tr) == oc.verify(c.input, bad, seed, tr) == (False, 0, 0)
    for k in range(c.input.size):
        bad = c.input.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert gc.verify_device(seed, _dev(bad), d_out, d_tr) == oc.verify(bad, out, seed, tr) == (False, c.d, 0)
    # a wrong seed changes every challenge: the first round check already fails (or, by chance, a later one)
    assert not gc.verify_device(seed + 1, d_in, d_out, d_tr)[0]
    gc.close()


def test_device_verifier_argument_errors(vc):
    c = W.random_circuit([1, 2], 2, 3)
    oc = oracle.OracleCircuit(c)
    out, tr, _, _ = oc.prove(c.input, 11)
    gc = vc.Circuit(c)
    d_in, d_out, d_tr = _dev(c.input), _dev(out), _dev(tr)
    with pytest.raises(vc.VCError) as e:
        gc.verify_device(11, d_in, d_out, _dev(tr[:-1]))
    assert e.value.code == vc.VC_ERR_ARG
    for which in range(3):                       # a non-canonical word anywhere is an argument error, as on the host
        bufs = [c.input.copy(), out.copy(), tr.copy()]
        bufs[which][0] = P
        with pytest.raises(vc.VCError) as e:
            gc.verify_device(11, *(_dev(b) for b in bufs))
        assert e.value.code == vc.VC_ERR_ARG
    assert gc.verify_device(11, d_in, d_out, d_tr) == (True, 0, 0)
    gc.close()


@pytest.mark.parametrize("k", [1, 2, 4])
def test_device_verifier_on_configs(vc, k):
    """Full-size configs in the bench's launch configuration: the honest GPU transcript is accepted, the sums the
    oracle can compute one by one agree (start claim, closing extension, the widest layer's wiring sums), and a single
    flipped word is rejected where the host verifier of the library rejects it."""
    c = W.config(k)
    seed = W.challenge_seed(k)
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(seed)
    assert gc.verify_device(seed) == (True, 0, 0)
    sums = gc.verifier_sums()
    out, tr = gc.outputs().copy(), gc.transcript().copy()
    logs = [l.log_size for l in c.layers] + [c.log_input]
    z0 = [oracle.draw(seed, j) for j in range(logs[0])]
    assert int(sums[0]) == (oracle.mle(out, z0) if logs[0] else int(out[0]))
    z, _, _ = gc.state()
    assert int(sums[-1]) == oracle.mle(c.input, z[:c.log_input])
    # wiring sums of the widest layer from the oracle's eq tables (Python integers)
    i = max(range(c.d), key=lambda j: logs[j])
    zz, _, ctr = oracle.OracleCircuit(c).layer_entry(i, seed, np.zeros(1 << logs[i], dtype=np.uint64))
    s = logs[i + 1]
    r1 = [oracle.draw(seed, ctr + j) for j in range(s)]
    r2 = [oracle.draw(seed, ctr + s + j) for j in range(s)]
    Tz = oracle.eq_table(zz[:logs[i]]).astype(object)
    T1 = oracle.eq_table(np.array(r1, dtype=np.uint64)).astype(object)
    T2 = oracle.eq_table(np.array(r2, dtype=np.uint64)).astype(object)
    L = c.layers[i]
    terms = Tz * T1[L.in1] % P * T2[L.in2] % P
    for t in range(4):
        assert int(sums[1 + 4 * i + t]) == int(terms[L.type == t].sum() % P), (i, t)
    rng = np.random.default_rng(k)
    for w in rng.integers(0, tr.size, size=3):
        bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
        got = gc.verify_device(seed, d_transcript=_dev(bad))
        assert got == gc.verify(c.input, out, seed, bad) and not got[0]
    gc.close()


def _check_against_paper_golden(kind, n, c, out, tr, claim):
    """Word-for-word parity with the oracle at a paper-scale size: tests/golden/paper_<kind>_<n>.txt holds the per-layer
    SHA-256 digests of the ORACLE's transcript (tests/golden/make_golden.py <kind>:<n>, oracle/ only), same seeds as here."""
    import hashlib
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"paper_{kind}_{n}.txt")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated (python tests/golden/make_golden.py {kind}:{n})")
    sha = lambda a: hashlib.sha256(np.ascontiguousarray(a, dtype="<u8").tobytes()).hexdigest()
    g, layers = {}, {}
    for line in open(path):
        if line.startswith("#"):
            continue
        p_ = line.split()
        if p_[0] == "layer":
            layers[int(p_[1])] = (p_[3], int(p_[4]), int(p_[5]))
        else:
            g[p_[0]] = p_[1]
    assert int(g["gates"]) == c.gates and int(g["transcript_words"]) == tr.size
    assert sha(out) == g["outputs_sha256"] and int(out[0]) == int(g["output0"])
    w = 0
    for i in range(c.d):
        nw = c.transcript_words(i)
        seg = tr[w:w + nw]
        digest, first, last = layers[i]
        assert (int(seg[0]), int(seg[-1])) == (first, last), f"{kind}:{n} layer {i}"
        assert sha(seg) == digest, f"{kind}:{n} layer {i}"
        w += nw
    assert sha(tr) == g["transcript_sha256"] and claim == int(g["final_claim"])


def test_f2_2_22_tree_layers_on_global_state_match_the_oracle(vc):
    """F2 at n = 2^22: its 2^21-gate ADD-tree layer is the implicit-TREE wiring with NON-resident gate state (global scratch),
    a kernel branch no BASELINE.json config reaches.  Oracle digests: tests/golden/paper_f2_22.txt."""
    from vc_workloads import circuits
    c = circuits.f2_circuit(22, 7)
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(31337)
    assert gc.flags() == 0
    _check_against_paper_golden("f2", 22, c, gc.outputs().copy(), gc.transcript().copy(), gc.state()[1])
    gc.close()


def test_paper_scale_f2_runs_and_verifies(vc):
    """the F2 construction at the paper's largest size, n = 2^23 (25.2 M nodes with the inputs,
    Table 2).  The transcript is compared layer by layer with the oracle's digests
    (tests/golden/paper_f2_23.txt, written by the oracle alone in ~2 min); on top of that properties that hold at any
    size: the output is the directly computed sum of squares, the device verifier accepts and rejects flipped words."""
    from vc_workloads import circuits
    c = circuits.f2_circuit(23, 7)
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(31337)
    assert gc.flags() == 0
    out, tr = gc.outputs().copy(), gc.transcript().copy()
    assert int(out[0]) == int((c.input.astype(np.uint64) ** 2).sum(dtype=np.uint64)) % P     # < 2^63: no wrap
    _check_against_paper_golden("f2", 23, c, out, tr, gc.state()[1])                          # the oracle's transcript, layer by layer
    assert gc.verify_device(31337) == (True, 0, 0)
    # round invariant on the whole transcript's first layer and a late one (g(0) + g(1) = claim chain is what V checks)
    rng = np.random.default_rng(5)
    for w in rng.integers(0, tr.size, size=4):
        bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
        ok, fl, fr = gc.verify_device(31337, d_transcript=_dev(bad))
        assert not ok
    bad_in = c.input.copy(); bad_in[12345] = (int(bad_in[12345]) + 1) % P
    assert gc.verify_device(31337, d_input=_dev(bad_in)) == (False, c.d, 0)
    gc.close()


@pytest.mark.parametrize("kind,n", [("matmul", 8), ("matmuleq", 8), ("pm", 19), ("f0", 20), ("f0", 21)])
def test_paper_scale_other_constructions(vc, kind, n):
    """MATMULT 256 x 256 — both the multi-output circuit of BASELINE.json's config 4 and the paper's
    single-output circuit (AB - C entry by entry, then the F0 circuit; three entries of C are wrong here, so
    the output is 3) —, PM with 2^19 text symbols and F0 at 2^20 and 2^21 (Table 2's sizes).
    Transcripts are compared with the oracle's per-layer digests
    (tests/golden/paper_<kind>_<n>.txt); also: outputs equal the directly computed values, the device verifier accepts,
    a flipped word is rejected."""
    from vc_workloads import circuits
    c = {"matmul": lambda: circuits.matmul_circuit(n, 4), "pm": lambda: circuits.pm_circuit(n, 3, 5),
         "f0": lambda: circuits.f0_circuit(n, 3), "matmuleq": lambda: circuits.matmul_eq_circuit(n, 4, wrong=3)}[kind]()
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(4242)
    assert gc.flags() == 0
    out, tr = gc.outputs().copy(), gc.transcript().copy()
    if kind == "matmul":
        assert np.array_equal(out.reshape(c.meta["A"].shape), c.meta["A"] @ c.meta["B"])          # entries < 2^28: no wrap
    elif kind == "matmuleq":
        assert out.size == 1 and int(out[0]) == 3 == int(np.count_nonzero(c.meta["A"] @ c.meta["B"] != c.meta["C"]))
    elif kind == "pm":
        T, Q = c.meta["text"].size, c.meta["pattern"].size
        idx = (np.arange(T)[:, None] + np.arange(Q)[None, :]) % T
        match = (c.meta["text"][idx] == c.meta["pattern"][None, :]).all(axis=1)
        assert int(out[0]) == int(T - match.sum())                                              # reading c-13: non-matching cyclic offsets
    else:
        assert int(out[0]) == int(np.count_nonzero(c.input))
    _check_against_paper_golden(kind, n, c, out, tr, gc.state()[1])   # the oracle's transcript, layer by layer (skips if the digest file is absent)
    assert gc.verify_device(4242) == (True, 0, 0)
    rng = np.random.default_rng(n)
    for w in rng.integers(0, tr.size, size=2):
        bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
        assert not gc.verify_device(4242, d_transcript=_dev(bad))[0]
    gc.close()
