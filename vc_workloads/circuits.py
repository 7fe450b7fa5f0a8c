"""Layered fan-in-2 circuits shaped like the paper's benchmarks, plus seeded inputs.

Conventions (reading c-1): layer 0 = outputs, layer d = inputs; layer i has
exactly 2**log_size gates; gate g of layer i reads entries in1[g], in2[g] of layer i+1.
Gate type codes (reading c-3): 0 ADD (L+R), 1 MULT (L*R), 2 SUB (L-R), 3 RELAY (L; in2 := in1).

The paper's workloads are "randomly generated" frequency vectors / text / matrices
(§6.2.4); circuits follow PAPER.md:216-230 (§6.2.1) with the changes
BASELINE.json's configs ask for (binary add-trees instead of one large-fan-in sum gate,
a 119-layer square-and-multiply chain for a^(p-1), multi-output MATMUL).

Nothing here does field arithmetic: only index patterns and numpy random draws.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np

ADD, MULT, SUB, RELAY = 0, 1, 2, 3
SUM = 4     # the single sum gate of very large fan-in at the output; only as layer 0, log_size 0

CONFIG_NAMES = {
    1: "F2 n=2^10",
    2: "F2 n=2^20",
    3: "F0 n=2^16",
    4: "MATMUL 128x128",
    5: "PM text=2^18 pattern=8",
}


def data_seed(k: int) -> int:
    return 1000 + k


def challenge_seed(k: int) -> int:
    return 2000 + k


@dataclass
class Layer:
    log_size: int
    type: np.ndarray  # uint8  [2**log_size]
    in1: np.ndarray   # uint32 [2**log_size]
    in2: np.ndarray   # uint32 [2**log_size]


@dataclass
class Circuit:
    layers: List[Layer]          # [0] = output layer ... [d-1] = layer fed by the input
    log_input: int
    input: np.ndarray            # uint64 [2**log_input], canonical words (< 2**61 - 1)
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def d(self) -> int:
        return len(self.layers)

    def log_below(self, i: int) -> int:
        """log2 size of layer i+1 (the layer that feeds layer i)."""
        return self.layers[i + 1].log_size if i + 1 < self.d else self.log_input

    @property
    def gates(self) -> int:
        """Non-input gates (reading c-15)."""
        return sum(1 << L.log_size for L in self.layers)

    @property
    def rounds(self) -> int:
        return sum((1 if (i == 0 and self.sum_output) else 2) * self.log_below(i) for i in range(self.d))

    @property
    def gate_rounds(self) -> int:
        return sum((1 << self.layers[i].log_size) * (1 if (i == 0 and self.sum_output) else 2) * self.log_below(i)
                   for i in range(self.d))

    @property
    def sum_output(self) -> bool:
        """Layer 0 is the single sum gate of large fan-in (type code SUM)."""
        return self.layers[0].log_size == 0 and int(self.layers[0].type[0]) == SUM

    def transcript_words(self, i: int) -> int:
        """Words layer i writes: (G0,G1,G2) per round for 2s rounds, then q[0..s]; the sum gate: (G0,G1) for s rounds."""
        return 2 * self.log_below(i) if (i == 0 and self.sum_output) else 7 * self.log_below(i) + 1

    @property
    def total_transcript_words(self) -> int:
        return sum(self.transcript_words(i) for i in range(self.d))


def _layer(log_size, typ, in1, in2) -> Layer:
    n = 1 << log_size
    t = np.ascontiguousarray(np.broadcast_to(np.asarray(typ, dtype=np.uint8), (n,)))
    a = np.ascontiguousarray(np.asarray(in1, dtype=np.uint32).reshape(n))
    b = np.ascontiguousarray(np.asarray(in2, dtype=np.uint32).reshape(n))
    return Layer(log_size, t, a, b)


def _tree_layer(log_size: int, typ: int = ADD) -> Layer:
    """Binary tree wiring: in-neighbours of gate g are 2g and 2g+1 (reading c-9)."""
    g = np.arange(1 << log_size, dtype=np.uint32)
    return _layer(log_size, typ, 2 * g, 2 * g + 1)


def _square_layer(log_size: int) -> Layer:
    g = np.arange(1 << log_size, dtype=np.uint32)
    return _layer(log_size, MULT, g, g)


def _fermat_chain(log_n: int) -> List[Layer]:
    """Layers (INPUT SIDE FIRST) mapping n values a -> a^(p-1), p = 2^61-1 (reading c-8).

    MSB-first square-and-multiply on p-1 = 2^61-2 (bits 60..1 set, bit 0 clear): x = a;
    59 x {square layer, multiply layer}; one final square layer  => 119 layers.
    Every layer but the last is 2n wide: lane x (MULT) at [0,n), lane a (RELAY) at [n,2n).
    """
    n = 1 << log_n
    g = np.arange(n, dtype=np.uint32)
    typ2 = np.concatenate([np.full(n, MULT, np.uint8), np.full(n, RELAY, np.uint8)])
    out: List[Layer] = []
    # first square layer reads the n-wide layer below: x = a*a, and relays a
    out.append(_layer(log_n + 1, typ2, np.concatenate([g, g]), np.concatenate([g, g])))
    for step in range(59):
        # multiply layer: x = x*a ; relay a
        out.append(_layer(log_n + 1, typ2, np.concatenate([g, g + n]), np.concatenate([g + n, g + n])))
        if step < 58:
            # square layer on a 2n-wide layer below: x = x*x ; relay a
            out.append(_layer(log_n + 1, typ2, np.concatenate([g, g + n]), np.concatenate([g, g + n])))
    # final square (bit 0 of p-1 is clear): n wide, no relay lane
    out.append(_layer(log_n, MULT, g, g))
    assert len(out) == 119
    return out


def f2_circuit(log_n: int, seed: int) -> Circuit:
    """F2 = sum a_i^2 (Fig. 4 :220; BASELINE.json configs[0],[1]; reading c-7)."""
    rng = np.random.default_rng(seed)
    x = rng.integers(0, 1 << 20, size=1 << log_n, dtype=np.uint64)
    layers_in_first = [_square_layer(log_n)] + [_tree_layer(k) for k in range(log_n - 1, -1, -1)]
    return Circuit(layers_in_first[::-1], log_n, x, f"F2 n=2^{log_n}")


def _sum_gate() -> Layer:
    """Layer 0 of the paper's own F2 / F0 circuits: one gate that sums EVERY gate of layer 1 (reading c-19).
    in1 / in2 are placeholders (never read)."""
    return _layer(0, SUM, np.zeros(1, np.uint32), np.zeros(1, np.uint32))


def f2_sum_circuit(log_n: int, seed: int) -> Circuit:
    """F2 exactly as the paper draws it (Fig. 4): a layer of squaring gates, then one sum gate of fan-in n
    (instead of BASELINE.json's log n-layer binary add tree).  Same input recipe as f2_circuit."""
    base = f2_circuit(log_n, seed)
    return Circuit([_sum_gate(), base.layers[-1]], log_n, base.input, f"F2-sum n=2^{log_n}")


def f0_sum_circuit(log_n: int, seed: int) -> Circuit:
    """F0 with the paper's sum gate of high fan-in over the ^(p-1) chain.  Same input recipe as f0_circuit."""
    base = f0_circuit(log_n, seed)
    return Circuit([_sum_gate()] + base.layers[log_n:], log_n, base.input, f"F0-sum n=2^{log_n}")


def f0_circuit(log_n: int, seed: int) -> Circuit:
    """F0 = #{i : a_i != 0} via a^(p-1) (BASELINE.json configs[2])."""
    rng = np.random.default_rng(seed)
    n = 1 << log_n
    nz = rng.random(n) >= 0.5
    vals = rng.integers(1, 1 << 10, size=n, dtype=np.uint64)
    x = np.where(nz, vals, np.uint64(0)).astype(np.uint64)
    layers_in_first = _fermat_chain(log_n) + [_tree_layer(k) for k in range(log_n - 1, -1, -1)]
    return Circuit(layers_in_first[::-1], log_n, x, f"F0 n=2^{log_n}")


def matmul_circuit(log_m: int, seed: int) -> Circuit:
    """C = A B for m x m matrices, m = 2^log_m (BASELINE.json configs[3]; reading c-14).

    Input = A then B, row-major. Product gate g = (i*m + j)*m + k reads A[i,k] and B[k,j];
    log_m add-tree layers over k; output index i*m + j.
    """
    rng = np.random.default_rng(seed)
    m = 1 << log_m
    A = rng.integers(0, 1 << 10, size=(m, m), dtype=np.uint64)
    B = rng.integers(0, 1 << 10, size=(m, m), dtype=np.uint64)
    x = np.concatenate([A.reshape(-1), B.reshape(-1)])
    g = np.arange(m * m * m, dtype=np.uint64)
    i, j, k = g // (m * m), (g // m) % m, g % m
    prod = _layer(3 * log_m, MULT, i * m + k, m * m + k * m + j)
    layers_in_first = [prod] + [_tree_layer(t) for t in range(3 * log_m - 1, 2 * log_m - 1, -1)]
    return Circuit(layers_in_first[::-1], 2 * log_m + 1, x, f"MATMUL {m}x{m}", {"A": A, "B": B})


def matmul_eq_circuit(log_m: int, seed: int, wrong: int = 0) -> Circuit:
    """The paper's single-output MATMULT circuit: computes the m^2 entries of AB by
    naive multiplication, subtracts the claimed C from each, and counts the non-zero differences with the F0 circuit;
    the one output is 0 iff C = AB.

    Input = A, B, C row-major, then m^2 zeros (4 m^2 = 2^(2 log_m + 2) words); C = AB with `wrong` entries off by one.
    A layered circuit reads only the layer below, so -C[i,j] enters the sum over k as one more term: the inner dimension
    is 2m wide, gate g = (i*m + j)*2m + k' is A[i,k']*B[k',j] (MULT) for k' < m, 0 - C[i,j] (SUB) for k' = m and 0 - 0
    above; log_m + 1 add-tree layers give (AB - C)[i,j]; the ^(p-1) chain and a 2 log_m-layer add tree count the
    non-zero entries.
    """
    rng = np.random.default_rng(seed)
    m = 1 << log_m
    A = rng.integers(0, 1 << 10, size=(m, m), dtype=np.uint64)
    B = rng.integers(0, 1 << 10, size=(m, m), dtype=np.uint64)
    Cm = A @ B                                               # entries < 2^28: no wrap
    bad = rng.choice(m * m, size=wrong, replace=False) if wrong else np.zeros(0, dtype=np.int64)
    Cf = Cm.reshape(-1).copy()
    Cf[bad] += np.uint64(1)
    x = np.concatenate([A.reshape(-1), B.reshape(-1), Cf, np.zeros(m * m, dtype=np.uint64)])
    Z = 3 * m * m                                            # a zero word of the input
    g = np.arange(2 * m * m * m, dtype=np.uint64)
    ij, k = g // (2 * m), g % (2 * m)
    i, j = ij // m, ij % m
    kk = np.minimum(k, m - 1)
    in1 = np.where(k < m, i * m + kk, Z)
    in2 = np.where(k < m, m * m + kk * m + j, np.where(k == m, 2 * m * m + ij, Z))
    typ = np.where(k < m, MULT, SUB).astype(np.uint8)
    prod = _layer(3 * log_m + 1, typ, in1, in2)
    layers_in_first = [prod] + [_tree_layer(t) for t in range(3 * log_m, 2 * log_m - 1, -1)]
    layers_in_first += _fermat_chain(2 * log_m)
    layers_in_first += [_tree_layer(t) for t in range(2 * log_m - 1, -1, -1)]
    return Circuit(layers_in_first[::-1], 2 * log_m + 2, x, f"MATMUL-EQ {m}x{m}",
                   {"A": A, "B": B, "C": Cf.reshape(m, m), "wrong": np.sort(bad)})


def pm_circuit(log_t: int, log_q: int, seed: int, planted: int = 16) -> Circuit:
    """Pattern matching (BASELINE.json configs[4]; reading c-13).

    Text of 2^log_t symbols, pattern of 2^log_q symbols, both uniform in [0,2^8); the pattern is
    planted at `planted` random offsets. For each CYCLIC offset i: sum_j (t[(i+j) mod T] - q[j])^2,
    then ^(p-1) (1 on mismatch), then an add-tree: output = number of NON-matching offsets.
    Input = text || pattern || zeros, 2^(log_t+1) words.
    """
    rng = np.random.default_rng(seed)
    T, Q = 1 << log_t, 1 << log_q
    text = rng.integers(0, 1 << 8, size=T, dtype=np.uint64)
    pat = rng.integers(0, 1 << 8, size=Q, dtype=np.uint64)
    offs = rng.integers(0, T - Q + 1, size=planted)
    for o in offs:
        text[o:o + Q] = pat
    x = np.zeros(2 * T, dtype=np.uint64)
    x[:T] = text
    x[T:T + Q] = pat
    g = np.arange(T * Q, dtype=np.uint64)
    i, j = g // Q, g % Q
    sub = _layer(log_t + log_q, SUB, (i + j) % T, T + j)
    layers_in_first = [sub, _square_layer(log_t + log_q)]
    layers_in_first += [_tree_layer(t) for t in range(log_t + log_q - 1, log_t - 1, -1)]
    layers_in_first += _fermat_chain(log_t)
    layers_in_first += [_tree_layer(t) for t in range(log_t - 1, -1, -1)]
    return Circuit(layers_in_first[::-1], log_t + 1, x, f"PM text=2^{log_t} pattern={Q}",
                   {"text": text, "pattern": pat, "planted_offsets": np.sort(offs)})


def random_circuit(log_sizes, log_input: int, seed: int, types=(ADD, MULT, SUB, RELAY),
                   small_values: bool = False) -> Circuit:
    """Random wiring, random gate types: test fodder for the definitions (SURVEY.md §8c pins).

    log_sizes[i] = log2 size of layer i (0 = output). Input words are uniform in [0, 2^61-1)
    unless small_values.
    """
    rng = np.random.default_rng(seed)
    layers = []
    for i, ls in enumerate(log_sizes):
        below = log_sizes[i + 1] if i + 1 < len(log_sizes) else log_input
        n = 1 << ls
        typ = rng.choice(np.asarray(types, dtype=np.uint8), size=n)
        a = rng.integers(0, 1 << below, size=n, dtype=np.uint32)
        b = rng.integers(0, 1 << below, size=n, dtype=np.uint32)
        b = np.where(typ == RELAY, a, b).astype(np.uint32)
        layers.append(_layer(ls, typ, a, b))
    hi = (1 << 16) if small_values else (1 << 61) - 1
    x = rng.integers(0, hi, size=1 << log_input, dtype=np.uint64)
    return Circuit(layers, log_input, x, f"random {list(log_sizes)}<-{log_input} seed={seed}")


def config(k: int) -> Circuit:
    """BASELINE.json configs[k-1], k = 1..5, with data seed 1000+k (DESIGN.md input recipe)."""
    s = data_seed(k)
    if k == 1:
        c = f2_circuit(10, s)
    elif k == 2:
        c = f2_circuit(20, s)
    elif k == 3:
        c = f0_circuit(16, s)
    elif k == 4:
        c = matmul_circuit(7, s)
    elif k == 5:
        c = pm_circuit(18, 3, s)
    else:
        raise ValueError(f"config {k} not in 1..5")
    c.name = CONFIG_NAMES[k]
    c.meta["config"] = k
    c.meta["challenge_seed"] = challenge_seed(k)
    return c
