"""O-def: the GKR layer sum-check written out from its DEFINITION, in Python big-int arithmetic.

TEST INFRASTRUCTURE ONLY.  Imported by tests/ (and nothing in the product path).  Shares no
code with the CUDA path or with the C oracle (oracle/gkr_oracle.c): this file is what the C
oracle is pinned against on tiny circuits.

What it states (SURVEY.md §8(c) "Definition (O-def)"; §3.1 for the iteration
structure, §4.1.1 for "a large sum over roughly S^3 terms"):

    F_z(w1,w2) = sum_g eq(g,z) * eq(in1[g],w1) * eq(in2[g],w2) * f_type[g]( V~(w1), V~(w2) )

with V~ the multilinear extension of layer i+1's values, and round m's message

    g_m(t) = sum over Boolean suffixes of F_z(r_0..r_{m-1}, t, suffix),    t = 0,1,2

where the 2s variables are (w1 bits 0..s-1, then w2 bits 0..s-1), bit 0 least significant.
Everything here is exponential-time on purpose: no per-gate shortcut, no tables.
"""
from itertools import product

P = (1 << 61) - 1

ADD, MULT, SUB, RELAY = 0, 1, 2, 3
SUM = 4     # the single sum gate of large fan-in at the output


def chi(b: int, x: int) -> int:
    """chi(b,x) = x if b = 1 else 1 - x."""
    return x % P if b else (1 - x) % P


def bits(u: int, s: int):
    return [(u >> k) & 1 for k in range(s)]


def eq(u: int, x) -> int:
    """eq(u,x) = prod_k chi(u_k, x_k); bit k of the index u is variable k."""
    e = 1
    for k, xk in enumerate(x):
        e = e * chi((u >> k) & 1, xk) % P
    return e


def mle(V, x) -> int:
    """V~(x) = sum_u eq(u,x) V[u]   (multilinear extension, by definition)."""
    assert len(V) == 1 << len(x)
    return sum(eq(u, x) * int(V[u]) for u in range(len(V))) % P


def gate_f(t: int, L: int, R: int) -> int:
    if t == ADD:
        return (L + R) % P
    if t == MULT:
        return (L * R) % P
    if t == SUB:
        return (L - R) % P
    if t == RELAY:
        return L % P
    raise ValueError(t)


def evaluate(layers, x):
    """layers: list of (type[], in1[], in2[]) output first; returns [V_0, ..., V_d] (V_d = x)."""
    V = [None] * (len(layers) + 1)
    V[len(layers)] = [int(v) for v in x]
    for i in range(len(layers) - 1, -1, -1):
        typ, in1, in2 = layers[i]
        below = V[i + 1]
        if i == 0 and len(typ) == 1 and int(typ[0]) == SUM:       # the output is the sum of EVERY gate of layer 1
            V[0] = [sum(below) % P]
            continue
        V[i] = [gate_f(int(typ[g]), below[int(in1[g])], below[int(in2[g])]) for g in range(len(typ))]
    return V


def F_z(layer, Vbelow, z, w1, w2) -> int:
    """The layer polynomial at an arbitrary point (w1,w2) in F^s x F^s."""
    typ, in1, in2 = layer
    a, b = mle(Vbelow, w1), mle(Vbelow, w2)
    tot = 0
    for g in range(len(typ)):
        tot += eq(g, z) * eq(int(in1[g]), w1) % P * eq(int(in2[g]), w2) % P * gate_f(int(typ[g]), a, b)
    return tot % P


def round_message(layer, Vbelow, z, prefix, s):
    """g_m(t), t = 0,1,2, m = len(prefix): brute force over all Boolean suffixes."""
    m = len(prefix)
    out = []
    for t in (0, 1, 2):
        tot = 0
        for suffix in product((0, 1), repeat=2 * s - m - 1):
            x = list(prefix) + [t] + list(suffix)
            tot += F_z(layer, Vbelow, z, x[:s], x[s:])
        out.append(tot % P)
    return out


def interp2(G, r: int) -> int:
    """Value at r of the degree-<=2 polynomial through (0,G0),(1,G1),(2,G2), by Lagrange's formula."""
    inv2 = pow(2, P - 2, P)
    l0 = (r - 1) * (r - 2) % P * inv2 % P
    l1 = (-(r * (r - 2))) % P
    l2 = r * (r - 1) % P * inv2 % P
    return (G[0] * l0 + G[1] * l1 + G[2] * l2) % P


def lagrange_eval(q, tau: int) -> int:
    """Value at tau of the degree-<=len(q)-1 polynomial with q[k] at node k, k = 0..len(q)-1."""
    n = len(q)
    tot = 0
    for k in range(n):
        num, den = 1, 1
        for m in range(n):
            if m != k:
                num = num * (tau - m) % P
                den = den * (k - m) % P
        tot += q[k] * num % P * pow(den, P - 2, P)
    return tot % P


def line(r1, r2, t: int):
    """l(t) = r1 + t (r2 - r1), coordinate-wise."""
    return [(a + t * (b - a)) % P for a, b in zip(r1, r2)]


def wiring_sums(layer, z, r1, r2):
    """W_tau = sum_{g of type tau} eq(g,z) eq(in1[g],r1) eq(in2[g],r2), by definition."""
    typ, in1, in2 = layer
    W = [0, 0, 0, 0]
    for g in range(len(typ)):
        W[int(typ[g])] += eq(g, z) * eq(int(in1[g]), r1) % P * eq(int(in2[g]), r2)
    return [w % P for w in W]


def sum_gate_round_message(Vbelow, prefix, s):
    """The sum gate of large fan-in (reading c-19): the output is sum_{w Boolean} V~(w), so round m of its
    sum-check is  g_m(t) = sum over Boolean suffixes b of V~(prefix, t, b),  here for t = 0, 1, 2 (linear in t: the
    protocol sends t = 0, 1 only; the third value lets a test check the degree)."""
    m = len(prefix)
    out = []
    for t in (0, 1, 2):
        tot = 0
        for suffix in product((0, 1), repeat=s - m - 1):
            tot += mle(Vbelow, list(prefix) + [t] + list(suffix))
        out.append(tot % P)
    return out
