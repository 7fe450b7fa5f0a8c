"""GPU parity: the CUDA path (through the C ABI of libvc.so) vs the CPU oracle, word for word.

All arithmetic is integer, so the bar is bit-exact (BASELINE.json north_star).  Inputs come from
vc_workloads (seeded); expected values come from oracle/ or from tests/golden/*.txt, which
tests/golden/make_golden.py wrote from the oracle alone.
"""
import hashlib
import os
import random

import numpy as np
import pytest

import oracle
import vc_workloads as W

pytestmark = pytest.mark.gpu

P = (1 << 61) - 1
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def vc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1202_1350_b200 as v
    v.lib()                       # fails loudly if libvc.so is missing
    return v


def _sha(a):
    return hashlib.sha256(np.ascontiguousarray(a, dtype="<u8").tobytes()).hexdigest()


def _golden(k):
    g = {"layers": {}}
    with open(os.path.join(GOLDEN, f"config{k}.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            p = line.split()
            if p[0] == "layer":
                g["layers"][int(p[1])] = (int(p[2]), p[3], int(p[4]), int(p[5]))
            else:
                g[p[0]] = p[1]
    return g


def _gpu_prove(vc, c, seed, schedule=0, layerwise=False):
    gc = vc.Circuit(c)
    gc.set_schedule(schedule)
    gc.set_input(c.input)
    gc.evaluate()
    if layerwise:
        gc.prove_layerwise(seed)
    else:
        gc.prove(seed)
    out, tr = gc.outputs().copy(), gc.transcript().copy()
    assert gc.flags() == 0
    return gc, out, tr


# ------------------------------------------------------------------ field arithmetic on the device
def test_device_field_ops_and_draws(vc):
    import torch
    rnd = random.Random(1)
    edge = [0, 1, 2, P - 1, P - 2, 1 << 60, (1 << 60) + 1, (1 << 32) - 1, 1 << 32, 12345678901234567]
    a = edge * len(edge) + [rnd.randrange(P) for _ in range(5000)]
    b = [y for y in edge for _ in edge] + [rnd.randrange(P) for _ in range(5000)]
    ta = torch.from_numpy(np.array(a, dtype=np.uint64).view(np.int64)).cuda()
    tb = torch.from_numpy(np.array(b, dtype=np.uint64).view(np.int64)).cuda()
    to = torch.empty_like(ta)
    L = vc.lib()
    for op, fn in [(0, lambda x, y: (x + y) % P), (1, lambda x, y: (x - y) % P), (2, lambda x, y: x * y % P),
                   (4, lambda x, y: 64 * x * y % P)]:
        assert L.vc_debug_fieldop(op, ta.data_ptr(), tb.data_ptr(), to.data_ptr(), ta.numel(), 0) == 0
        got = to.cpu().numpy().view(np.uint64)
        assert [int(v) for v in got] == [fn(x, y) for x, y in zip(a, b)], op
    seeds = np.array([0, 0, 0, 1234567, 2002, 2002], dtype=np.uint64)
    ctrs = np.array([0, 1, 2, 0, 5, 999], dtype=np.uint64)
    ts, tc = (torch.from_numpy(x.view(np.int64)).cuda() for x in (seeds, ctrs))
    tt = torch.empty_like(ts)
    assert L.vc_debug_fieldop(3, ts.data_ptr(), tc.data_ptr(), tt.data_ptr(), ts.numel(), 0) == 0
    got = [int(v) for v in tt.cpu().numpy().view(np.uint64)]
    assert got == [oracle.draw(int(s), int(k)) for s, k in zip(seeds, ctrs)]
    assert got[0] == 0xE220A8397B1DCDAF & P        # published splitmix64 vector, low 61 bits


# ------------------------------------------------------------------ element-by-element on small/medium circuits
RANDOM_CASES = [
    ([0, 1], 1, 1), ([1, 2, 1], 2, 2), ([0, 2, 3], 2, 4), ([3, 1, 2], 3, 5),
    ([0, 1, 2, 3, 4, 5], 6, 9), ([4, 6, 5], 7, 10), ([6, 3], 5, 12),
    ([9, 12, 10, 13], 11, 13),          # several tiles of every kernel + ragged sizes between layers
    ([14, 11, 15], 13, 14),
    ([12, 17, 8], 9, 15),               # 2^12 gates wired at random into a 2^17 table: tables materialised in L2 (F_MODE_GLOBAL)
    ([21, 17], 10, 16),                 # 2^21 gates: state in global scratch (non-resident) + F_MODE_GLOBAL
]


@pytest.mark.parametrize("schedule", [1, 0])
@pytest.mark.parametrize("log_sizes,log_input,seed", RANDOM_CASES)
def test_random_circuits_bit_exact(vc, log_sizes, log_input, seed, schedule):
    c = W.random_circuit(log_sizes, log_input, seed)
    oc = oracle.OracleCircuit(c)
    want_out, want_tr, want_z, want_claim = oc.prove(c.input, 500 + seed)
    gc, out, tr = _gpu_prove(vc, c, 500 + seed, schedule)
    V = oc.evaluate(c.input)
    for i in range(c.d + 1):
        assert np.array_equal(gc.values(i), V[i]), f"value table {i}"
    assert np.array_equal(out, want_out)
    bad = np.nonzero(tr != want_tr)[0]
    assert bad.size == 0, f"first mismatch at word {bad[:5]} of {tr.size}"
    z, claim, ctr = gc.state()
    assert claim == want_claim and np.array_equal(z[:c.log_input], want_z[:c.log_input])
    assert ctr == c.layers[0].log_size + sum(2 * c.log_below(i) + 1 for i in range(c.d))
    assert gc.verify(c.input, out, 500 + seed, tr) == (True, 0, 0)
    gc.close()


@pytest.mark.parametrize("schedule", [1, 0])
def test_structured_small_circuits_bit_exact(vc, schedule):
    for c, seed in [(W.f0_circuit(5, 5), 31), (W.matmul_circuit(3, 6), 32), (W.pm_circuit(6, 2, 7, planted=3), 33),
                    (W.config(1), W.challenge_seed(1))]:
        oc = oracle.OracleCircuit(c)
        want_out, want_tr, _, want_claim = oc.prove(c.input, seed)
        gc, out, tr = _gpu_prove(vc, c, seed, schedule, layerwise=True)
        assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), c.name
        assert gc.state()[1] == want_claim
        gc.close()


def test_all_kinds_kernel_matches_the_split_launches(vc, monkeypatch):
    """The proof runs either as one launch of the all-kinds kernel or as one launch per run of layer kinds (narrow / thin /
    wide); VC_SINGLE_KERNEL=1 at load forces the former.  Both must give the oracle's transcript word for word: a circuit
    whose kinds alternate (more runs than the split allows: all-kinds kernel by itself) and config 2 forced either way."""
    c = W.random_circuit([3, 12, 5, 13, 2, 12, 6, 11], 9, 99)        # narrow / thin alternating: 8 runs
    want_out, want_tr, _, _ = oracle.OracleCircuit(c).prove(c.input, 606)
    for force in ("0", "1"):
        monkeypatch.setenv("VC_SINGLE_KERNEL", force)
        gc, out, tr = _gpu_prove(vc, c, 606)
        assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), force
        gc.close()
    c2 = W.config(2)
    g = _golden(2)
    monkeypatch.setenv("VC_SINGLE_KERNEL", "1")
    gc, out, tr = _gpu_prove(vc, c2, W.challenge_seed(2))
    monkeypatch.setenv("VC_SINGLE_KERNEL", "0")
    gc2, out2, tr2 = _gpu_prove(vc, c2, W.challenge_seed(2))
    assert np.array_equal(tr, tr2) and np.array_equal(out, out2)
    assert _sha(out) == g["outputs_sha256"] and _sha(tr) == g["transcript_sha256"]
    gc.close(); gc2.close()


# ------------------------------------------------------------------ full sizes: golden digests written by the oracle
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_configs_match_oracle_golden(vc, k):
    path = os.path.join(GOLDEN, f"config{k}.txt")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet (python tests/golden/make_golden.py {k})")
    g = _golden(k)
    c = W.config(k)
    seed = W.challenge_seed(k)
    gc, out, tr = _gpu_prove(vc, c, seed)      # the launch configuration bench.py times (schedule 0)
    assert int(g["gates"]) == c.gates and int(g["transcript_words"]) == tr.size
    assert _sha(out) == g["outputs_sha256"] and int(out[0]) == int(g["output0"])
    w = 0
    for i in range(c.d):
        n = c.transcript_words(i)
        s, digest, first, last = g["layers"][i]
        seg = tr[w:w + n]
        assert (int(seg[0]), int(seg[-1])) == (first, last), f"config {k} layer {i}"
        assert _sha(seg) == digest, f"config {k} layer {i}"
        w += n
    assert _sha(tr) == g["transcript_sha256"]
    assert gc.state()[1] == int(g["final_claim"])
    # properties that hold at any size: both verifiers accept the GPU transcript
    assert gc.verify(c.input, out, seed, tr) == (True, 0, 0)
    if k in (1, 2, 4):
        assert oracle.OracleCircuit(c).verify(c.input, out, seed, tr) == (True, 0, 0)
    gc.close()


def test_sampled_layers_of_config2_against_oracle_in_isolation(vc):
    """Full-size config 2 in the bench launch configuration; the oracle re-proves sampled layers one by one."""
    c = W.config(2)
    seed = W.challenge_seed(2)
    gc, out, tr = _gpu_prove(vc, c, seed)
    oc = oracle.OracleCircuit(c)
    V = oc.evaluate(c.input)
    offs = np.cumsum([0] + [c.transcript_words(i) for i in range(c.d)])
    for i in (0, 7, 13, 17):
        z, claim, ctr = oc.layer_entry(i, seed, V[i])
        want, *_ = oc.prove_layer(i, V[i + 1], seed, ctr, z, claim, debug=False)
        assert np.array_equal(tr[offs[i]:offs[i + 1]], want), f"layer {i}"
    gc.close()


# ------------------------------------------------------------------ verifier of the library: tamper = fault injection
def test_library_verifier_rejects_tampering(vc):
    c = W.random_circuit([1, 2, 3, 2], 3, 61)
    seed = 808
    gc, out, tr = _gpu_prove(vc, c, seed)
    oc = oracle.OracleCircuit(c)
    assert gc.verify(c.input, out, seed, tr) == (True, 0, 0)
    for w in range(tr.size):
        bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
        got = gc.verify(c.input, out, seed, bad)
        assert got == oc.verify(c.input, out, seed, bad) and not got[0], w
    for k in range(out.size):
        bad = out.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert gc.verify(c.input, bad, seed, tr) == (False, 0, 0)
    for k in range(c.input.size):
        bad = c.input.copy(); bad[k] = (int(bad[k]) + 1) % P
        assert gc.verify(bad, out, seed, tr) == (False, c.d, 0)
    gc.close()


# ------------------------------------------------------------------ boundary behaviour
def test_call_order_and_argument_errors(vc):
    import torch
    c = W.random_circuit([1, 2], 2, 3)
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    with pytest.raises(vc.VCError) as e:
        vc.vc_prove_layer(gc.handle, 0, 1, gc.d_transcript)      # before vc_evaluate
    assert e.value.code == vc.VC_ERR_STATE
    gc.evaluate()
    with pytest.raises(vc.VCError) as e:
        vc.vc_prove_layer(gc.handle, 1, 1, gc.d_transcript)      # out of order
    assert e.value.code == vc.VC_ERR_STATE
    small = torch.zeros(3, dtype=torch.int64, device="cuda")
    with pytest.raises(vc.VCError) as e:
        vc.vc_prove_layer(gc.handle, 0, 1, small)                # capacity
    assert e.value.code == vc.VC_ERR_ARG
    vc.vc_prove_layer(gc.handle, 0, 1, gc.d_transcript)
    with pytest.raises(vc.VCError) as e:
        vc.vc_prove_layer(gc.handle, 1, 2, gc.d_transcript)      # seed changed mid-proof
    assert e.value.code == vc.VC_ERR_STATE
    gc.close()
    bad = W.random_circuit([1, 2], 2, 3)
    bad.layers[0].in1[0] = 99
    with pytest.raises(vc.VCError) as e:
        vc.Circuit(bad)
    assert e.value.code == vc.VC_ERR_SHAPE
    bad = W.random_circuit([1, 0], 2, 3)                          # a layer below of size 1
    with pytest.raises(vc.VCError) as e:
        vc.Circuit(bad)
    assert e.value.code == vc.VC_ERR_SHAPE


def test_non_canonical_input_is_flagged(vc):
    c = W.random_circuit([1, 2], 2, 3)
    gc = vc.Circuit(c)
    x = c.input.copy(); x[1] = np.uint64(P)
    gc.set_input(x)
    gc.evaluate()
    assert gc.flags() & 1
    gc.close()


def test_non_canonical_input_through_run_host_and_flag_is_per_evaluation(vc):
    """include/vc.h (vc_evaluate, vc_run_host; SURVEY.md §8(b) "Errors"): a word >= p is detected on the device, reported by
    vc_run_host as VC_ERR_ARG, and the status bit describes the LAST evaluation only: a valid input afterwards runs clean."""
    import torch
    c = W.random_circuit([2, 3, 5], 4, 8)
    seed = 99
    want_out, want_tr, _, _ = oracle.OracleCircuit(c).prove(c.input, seed)
    gc = vc.Circuit(c)
    bad = c.input.copy(); bad[3] = np.uint64(P + 5)
    h_out = torch.zeros(gc.n_out, dtype=torch.int64).pin_memory()
    h_tr = torch.zeros(gc.words, dtype=torch.int64).pin_memory()
    with pytest.raises(vc.VCError) as e:
        vc.vc_run_host(gc.handle, torch.from_numpy(bad.view(np.int64)).pin_memory(), seed, h_out, h_tr)
    assert e.value.code == vc.VC_ERR_ARG
    assert gc.flags() & 1
    vc.vc_run_host(gc.handle, torch.from_numpy(c.input.view(np.int64)).pin_memory(), seed, h_out, h_tr)   # same handle, valid input
    assert gc.flags() == 0
    assert np.array_equal(h_out.numpy().view(np.uint64), want_out) and np.array_equal(h_tr.numpy().view(np.uint64), want_tr)
    gc.close()


def test_default_schedule_is_the_fused_one_not_a_silent_fallback(vc):
    """The streaming schedule is always available and gives the same words, so a broken fused plan would pass every parity
    test unnoticed: check that schedule 0 really runs the persistent kernels (a handful of launches per proof, a kernel kind
    for every layer) and that config 2's layers go where the plan says (cluster engine up to 2^12 gates, grid above)."""
    c = W.config(2)
    gc = vc.Circuit(c)
    kinds = gc.layer_kinds()                      # raises VC_ERR_STATE if the circuit has no fused plan
    K = vc.lib()
    assert list(kinds[:13]) == [9] * 13           # VC_K_CLUSTER
    assert set(int(x) for x in kinds[13:]) <= {6, 8}   # VC_K_FUSED_WIDE / VC_K_FUSED_THIN
    gc.set_input(c.input)
    n0 = K.vc_launch_count()
    gc.evaluate(); gc.prove(W.challenge_seed(2))
    assert K.vc_launch_count() - n0 <= 6          # evaluation + one launch per run of layer kinds
    gc.close()


# ------------------------------------------------------------------ the cluster engine (layers of at most 2^12 gates)
CLUSTER_CASES = [
    ([10, 11, 12, 11, 10], 11, 41),     # 1 -> 8 -> 16 -> 8 -> 1... active CTAs grow and shrink: state hand-over to CTAs that join
    ([12, 4, 12, 3], 9, 42),            # a wide cluster layer after a single-CTA one, twice; tables of 2^4 .. 2^12 words
    ([11, 14, 9], 12, 43),              # irregular wiring into a 2^14 table: every CTA holds the whole table (no slices)
    ([0, 12], 12, 44),                  # one output reading a 2^12 layer: start claim on one gate, line restriction in blocks
]


@pytest.mark.parametrize("log_sizes,log_input,seed", CLUSTER_CASES)
def test_cluster_engine_random_circuits_bit_exact(vc, log_sizes, log_input, seed):
    c = W.random_circuit(log_sizes, log_input, seed)
    want_out, want_tr, want_z, want_claim = oracle.OracleCircuit(c).prove(c.input, 900 + seed)
    for layerwise in (False, True):      # one launch for the run of layers, or one launch per layer (state through DevState)
        gc, out, tr = _gpu_prove(vc, c, 900 + seed, 0, layerwise=layerwise)
        assert np.array_equal(out, want_out)
        bad = np.nonzero(tr != want_tr)[0]
        assert bad.size == 0, f"layerwise={layerwise}: first mismatch at word {bad[:5]} of {tr.size}"
        z, claim, _ = gc.state()
        assert claim == want_claim and np.array_equal(z[:c.log_input], want_z[:c.log_input])
        gc.close()


def test_cluster_engine_and_grid_kernels_give_the_same_transcript(vc, monkeypatch):
    """VC_NO_CLUSTER=1 at load keeps every layer on the grid-wide kernels: both routes must give the oracle's words (the
    structured circuits put tree, self and two-lane chain wiring through the cluster engine's sliced tables)."""
    for c, seed in [(W.f0_circuit(9, 5), 51), (W.matmul_circuit(4, 6), 52), (W.pm_circuit(9, 3, 7, planted=3), 53)]:
        want_out, want_tr, _, want_claim = oracle.OracleCircuit(c).prove(c.input, seed)
        for off in ("0", "1"):
            monkeypatch.setenv("VC_NO_CLUSTER", off)
            gc, out, tr = _gpu_prove(vc, c, seed)
            assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), (c.name, off)
            assert gc.state()[1] == want_claim
            gc.close()
    monkeypatch.delenv("VC_NO_CLUSTER")


def test_computed_wiring_covers_the_paper_circuits_and_changes_no_word(vc, monkeypatch):
    """SURVEY.md §8f NEXT-4 (§5.1.4: indices computed, no record loads).  vc_load fits tree / self / bit-field
    rules to the records; every layer of the four paper circuits gets a computed mode, a random circuit gets none, and with the
    rule switched off (VC_NO_WIRE_RULE=1: those layers read their records) both schedules give the oracle's words either way.
    Sizes put the rule through the cluster engine, the thin and the wide kernels (the product layer is 2^15 gates, the
    sliding-window layer 2^14, the chain lanes 2^14)."""
    cases = [(W.f0_circuit(13, 5), 61), (W.matmul_circuit(5, 6), 62), (W.pm_circuit(11, 3, 7, planted=3), 63),
             (W.f2_circuit(12, 8), 64)]
    for c, seed in cases:
        want_out, want_tr, _, want_claim = oracle.OracleCircuit(c).prove(c.input, seed)
        for off in ("", "1"):
            if off:
                monkeypatch.setenv("VC_NO_WIRE_RULE", off)
            else:
                monkeypatch.delenv("VC_NO_WIRE_RULE", raising=False)
            for schedule in (0, 1):
                gc, out, tr = _gpu_prove(vc, c, seed, schedule=schedule)
                modes = gc.layer_wiring()
                if off:
                    assert not (modes == 3).any(), c.name
                else:
                    assert (modes != 0).all(), (c.name, modes)
                    assert c.name.startswith("F2") or (modes == 3).any(), (c.name, modes)
                assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), (c.name, off, schedule)
                assert gc.state()[1] == want_claim
                gc.close()
    monkeypatch.delenv("VC_NO_WIRE_RULE", raising=False)
    c = W.random_circuit([3, 9, 12, 11], 10, 65)
    gc = vc.Circuit(c)
    assert (gc.layer_wiring() == 0).all()
    gc.close()


@pytest.mark.parametrize("log_m,wrong", [(3, 0), (4, 2), (5, 1)])
def test_matmul_equality_circuit_single_output_bit_exact(vc, log_m, wrong):
    """The paper's single-output MATMULT circuit, element by element against the
    oracle on both schedules: mixed MULT / SUB product layer with irregular wiring (records are read), log m + 1 tree
    layers, the ^(p-1) chain, the counting tree.  The output is the number of wrong entries of C (0 iff C = AB)."""
    c = W.matmul_eq_circuit(log_m, 30 + log_m, wrong)
    seed = 70 + log_m
    want_out, want_tr, _, want_claim = oracle.OracleCircuit(c).prove(c.input, seed)
    assert want_out.size == 1 and int(want_out[0]) == wrong
    for schedule in (0, 1):
        gc, out, tr = _gpu_prove(vc, c, seed, schedule=schedule)
        assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), (log_m, schedule)
        assert gc.state()[1] == want_claim
        assert gc.verify(c.input, out, seed, tr) == (True, 0, 0)
        gc.close()


SUM_GATE_CASES = [
    ("f2", 1), ("f2", 5), ("f2", 11), ("f2", 12), ("f2", 17),     # table = tail only; tail boundary (2^11) and one, six folds before it
    ("f0", 4), ("f0", 13),                                       # 119 chain layers under the sum gate
    ("alone", 9), ("alone", 14),                                  # d = 1: the sum gate reads the input directly, random F_p words
]


@pytest.mark.parametrize("kind,log_n", SUM_GATE_CASES)
def test_sum_gate_of_large_fan_in_bit_exact(vc, kind, log_n):
    """SURVEY.md §8f NEXT-4 / PAPER.md:220, :222 (reading c-19): the paper's own F2 and F0 circuits end in ONE sum gate
    over all of layer 1 (VC_SUM).  Outputs, every transcript word and the final state against the oracle, on the fused and
    the streaming schedule, whole proof and layer by layer; both verifiers accept; a flipped word of the sum gate's rounds
    is rejected at its round by both."""
    import torch
    if kind == "alone":
        rng = random.Random(log_n)
        x = np.array([rng.randrange(P) for _ in range(1 << log_n)], dtype=np.uint64)
        z0 = np.zeros(1, np.uint32)
        c = W.Circuit([W.Layer(0, np.array([W.SUM], np.uint8), z0, z0)], log_n, x, "sum gate alone")
    else:
        c = (W.f2_sum_circuit if kind == "f2" else W.f0_sum_circuit)(log_n, 80 + log_n)
    seed = 300 + log_n
    oc = oracle.OracleCircuit(c)
    want_out, want_tr, want_z, want_claim = oc.prove(c.input, seed)
    for schedule, layerwise in ((0, False), (1, False), (0, True)):
        gc, out, tr = _gpu_prove(vc, c, seed, schedule=schedule, layerwise=layerwise)
        assert gc.words == want_tr.size == c.total_transcript_words
        assert np.array_equal(out, want_out) and np.array_equal(tr, want_tr), (kind, log_n, schedule, layerwise)
        z, claim, ctr = gc.state()[:3]
        assert claim == want_claim and np.array_equal(z[:c.log_input], want_z[:c.log_input])
        assert gc.verify(c.input, out, seed, tr) == (True, 0, 0) and gc.verify_device(seed) == (True, 0, 0)
        s = c.log_below(0)
        for w in sorted({0, 2 * s - 1, s}):
            bad = tr.copy(); bad[w] = (int(bad[w]) + 1) % P
            want = oc.verify(c.input, out, seed, bad)
            assert want == (False, 0, w // 2)
            assert gc.verify(c.input, out, seed, bad) == want
            assert gc.verify_device(seed, d_transcript=torch.from_numpy(bad.view(np.int64)).cuda()) == want
        gc.close()


def test_sum_gate_only_as_the_single_gate_of_layer_0(vc):
    """VC_SUM anywhere else is a shape error at load (include/vc.h)."""
    c = W.f2_sum_circuit(4, 1)
    c.layers[1].type[3] = W.SUM
    with pytest.raises(vc.VCError) as e:
        vc.Circuit(c)
    assert e.value.code == 2
    c = W.f2_circuit(3, 1)
    c.layers[1].type[:] = W.SUM            # a two-gate layer of SUM gates
    with pytest.raises(vc.VCError) as e:
        vc.Circuit(c)
    assert e.value.code == 2


@pytest.mark.parametrize("log_n", [13, 14, 17])
def test_block_local_evaluation_gives_every_layer_value(vc, monkeypatch, log_n):
    """k_eval_all runs tree / self layers block by block in shared memory when the circuit starts with such layers (F2:
    squares, then the add tree) and meets the grid once instead of once per layer: every V_i against the oracle, with the
    local run and without it (VC_NO_EVAL_LOCAL=1 at load), also under a sum gate, also with a non-canonical input word."""
    import torch
    for c in (W.f2_circuit(log_n, 40 + log_n), W.f2_sum_circuit(log_n, 50 + log_n)):
        V = oracle.OracleCircuit(c).evaluate(c.input)
        for off in ("", "1"):
            if off:
                monkeypatch.setenv("VC_NO_EVAL_LOCAL", off)
            else:
                monkeypatch.delenv("VC_NO_EVAL_LOCAL", raising=False)
            gc = vc.Circuit(c)
            gc.set_input(c.input)
            gc.evaluate()
            assert gc.flags() == 0
            for i in range(c.d + 1):
                assert np.array_equal(gc.values(i), V[i]), (c.name, off, i)
            assert np.array_equal(gc.outputs(), V[0])
            bad = c.input.copy(); bad[(1 << log_n) - 3] = P          # in the last block
            gc.set_input(bad); gc.evaluate()
            torch.cuda.synchronize()
            assert gc.flags() == 1
            gc.close()
    monkeypatch.delenv("VC_NO_EVAL_LOCAL", raising=False)


def test_run_host_end_to_end_matches(vc):
    import torch
    c = W.config(1)
    seed = W.challenge_seed(1)
    want_out, want_tr, _, _ = oracle.OracleCircuit(c).prove(c.input, seed)
    gc = vc.Circuit(c)
    h_in = torch.from_numpy(c.input.view(np.int64)).pin_memory()
    h_out = torch.zeros(gc.n_out, dtype=torch.int64).pin_memory()
    h_tr = torch.zeros(gc.words, dtype=torch.int64).pin_memory()
    for _ in range(4):           # the handle is reusable
        h_out.zero_(); h_tr.zero_()
        vc.vc_run_host(gc.handle, h_in, seed, h_out, h_tr)
        assert np.array_equal(h_out.numpy().view(np.uint64), want_out)
        assert np.array_equal(h_tr.numpy().view(np.uint64), want_tr)
    # same buffers, other contents
    x2 = c.input.copy(); x2[::7] = (x2[::7] + np.uint64(5)) % np.uint64(P)
    want_out2, want_tr2, _, _ = oracle.OracleCircuit(c).prove(x2, seed)
    h_in.copy_(torch.from_numpy(x2.view(np.int64)))
    vc.vc_run_host(gc.handle, h_in, seed, h_out, h_tr)
    assert np.array_equal(h_out.numpy().view(np.uint64), want_out2) and np.array_equal(h_tr.numpy().view(np.uint64), want_tr2)
    assert not np.array_equal(want_tr2, want_tr)
    # another seed; then a non-canonical word is reported by this call and not by the next one
    want_out3, want_tr3, _, _ = oracle.OracleCircuit(c).prove(x2, seed + 1)
    for _ in range(3):
        vc.vc_run_host(gc.handle, h_in, seed + 1, h_out, h_tr)
        assert np.array_equal(h_tr.numpy().view(np.uint64), want_tr3)
    h_in[3] = -1                 # 2^64 - 1 >= p
    with pytest.raises(vc.VCError) as e:
        vc.vc_run_host(gc.handle, h_in, seed + 1, h_out, h_tr)
    assert e.value.code == 1
    h_in.copy_(torch.from_numpy(x2.view(np.int64)))
    vc.vc_run_host(gc.handle, h_in, seed + 1, h_out, h_tr)
    assert np.array_equal(h_tr.numpy().view(np.uint64), want_tr3)
    gc.close()
