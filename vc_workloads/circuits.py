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
        return sum(2 * self.log_below(i) for i in range(self.d))

    @property
    def gate_rounds(self) -> int:
        return sum((1 << self.layers[i].log_size) * 2 * self.log_below(i) for i in range(self.d))

    def transcript_words(self, i: int) -> int:
        return 7 * self.log_below(i) + 1

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
