"""CPU oracle for the GKR prover hot path — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_1202_1350_b200 and shares no code with it.

  gkr_def.py     O-def: the definitions (exponential-time sums) in Python big ints
  gkr_oracle.c   O-cmt: the per-gate single-pass prover + verifier, plain C, unsigned __int128
  this file      gcc build step and ctypes marshalling for gkr_oracle.c (no arithmetic)
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "liboracle.so"
_SRC = _HERE / "gkr_oracle.c"

P = (1 << 61) - 1


class _Layer(C.Structure):
    _fields_ = [("log_size", C.c_uint32), ("type", C.c_void_p), ("in1", C.c_void_p), ("in2", C.c_void_p)]


class LayerDebug(C.Structure):
    _fields_ = [("r1", C.c_uint64 * 64), ("r2", C.c_uint64 * 64), ("v1", C.c_uint64), ("v2", C.c_uint64),
                ("Wsum", C.c_uint64 * 4), ("tau", C.c_uint64)]


def build(force: bool = False) -> Path:
    """Compile gkr_oracle.c -> liboracle.so with gcc -O2 (no OpenMP, single thread)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-o", str(tmp), str(_SRC)])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        u64, u32, vp = C.c_uint64, C.c_uint32, C.c_void_p
        for name in ("orc_add", "orc_sub", "orc_mul", "orc_pow", "orc_mix", "orc_draw"):
            getattr(L, name).restype = u64
            getattr(L, name).argtypes = [u64, u64]
        L.orc_p.restype = u64
        L.orc_inv.restype = u64
        L.orc_inv.argtypes = [u64]
        L.orc_eq_table.restype = None
        L.orc_eq_table.argtypes = [vp, u32, vp]
        L.orc_mle.restype = u64
        L.orc_mle.argtypes = [vp, u32, vp]
        L.orc_lagrange.restype = u64
        L.orc_lagrange.argtypes = [vp, u32, u64]
        L.orc_interp2.restype = u64
        L.orc_interp2.argtypes = [vp, u64]
        L.orc_evaluate.restype = C.c_int
        L.orc_evaluate.argtypes = [vp, u32, u32, vp, vp]
        L.orc_start.restype = C.c_int
        L.orc_start.argtypes = [vp, u32, u64, vp, vp, vp]
        L.orc_prove_layer.restype = C.c_int
        L.orc_prove_layer.argtypes = [vp, u32, vp, u64, vp, vp, vp, vp, vp]
        L.orc_transcript_words.restype = u64
        L.orc_transcript_words.argtypes = [vp, u32, u32]
        L.orc_prove.restype = C.c_int
        L.orc_prove.argtypes = [vp, u32, u32, vp, u64, vp, vp, u64, vp, vp]
        L.orc_layer_entry.restype = u64
        L.orc_layer_entry.argtypes = [vp, u32, u64, C.c_int, vp]
        L.orc_prove_sum_layer.restype = C.c_int
        L.orc_prove_sum_layer.argtypes = [u32, vp, u64, vp, vp, vp, vp]
        L.orc_verify.restype = C.c_int
        L.orc_verify.argtypes = [vp, u32, u32, vp, vp, u64, vp, u64, vp, vp, vp]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _u64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.uint64))


class OracleCircuit:
    """Marshals a vc_workloads.Circuit-like object (layers with log_size/type/in1/in2, log_input)."""

    def __init__(self, circuit):
        self.c = circuit
        self.d = len(circuit.layers)
        self.log_input = circuit.log_input
        self._keep = []
        arr = (_Layer * self.d)()
        for i, L in enumerate(circuit.layers):
            t = np.ascontiguousarray(L.type, dtype=np.uint8)
            a = np.ascontiguousarray(L.in1, dtype=np.uint32)
            b = np.ascontiguousarray(L.in2, dtype=np.uint32)
            self._keep += [t, a, b]
            arr[i] = _Layer(L.log_size, t.ctypes.data, a.ctypes.data, b.ctypes.data)
        self.arr = arr

    def log_below(self, i):
        return self.c.layers[i + 1].log_size if i + 1 < self.d else self.log_input

    def transcript_words(self) -> int:
        return int(lib().orc_transcript_words(self.arr, self.d, self.log_input))

    def evaluate(self, x):
        x = _u64(x)
        V = [np.empty(1 << L.log_size, dtype=np.uint64) for L in self.c.layers] + \
            [np.empty(1 << self.log_input, dtype=np.uint64)]
        ptrs = (C.c_void_p * (self.d + 1))(*[v.ctypes.data for v in V])
        rc = lib().orc_evaluate(self.arr, self.d, self.log_input, _ptr(x), ptrs)
        if rc:
            raise ValueError(f"orc_evaluate rc={rc}")
        return V

    def start(self, V0, seed):
        s0 = self.c.layers[0].log_size
        z = np.zeros(64, dtype=np.uint64)
        ctr, claim = C.c_uint64(0), C.c_uint64(0)
        lib().orc_start(_ptr(_u64(V0)), s0, seed, C.byref(ctr), _ptr(z), C.byref(claim))
        return z, int(claim.value), int(ctr.value)

    @property
    def sum_output(self) -> bool:
        """Layer 0 is the single large-fan-in sum gate (type code 4)."""
        L0 = self.c.layers[0]
        return L0.log_size == 0 and int(L0.type[0]) == 4

    def prove_layer(self, i, Vbelow, seed, ctr, z, claim, debug=True):
        """Returns (transcript words, z_out[64], claim_out, ctr_out, LayerDebug)."""
        s = self.log_below(i)
        z = _u64(z).copy()
        if z.size < 64:
            z = np.concatenate([z, np.zeros(64 - z.size, dtype=np.uint64)])
        if i == 0 and self.sum_output:
            tr = np.zeros(2 * s, dtype=np.uint64)
            c_ctr, c_claim = C.c_uint64(ctr), C.c_uint64(claim)
            rc = lib().orc_prove_sum_layer(s, _ptr(_u64(Vbelow)), seed, C.byref(c_ctr), _ptr(z), C.byref(c_claim), _ptr(tr))
            if rc:
                raise ValueError(f"orc_prove_sum_layer rc={rc}")
            return tr, z, int(c_claim.value), int(c_ctr.value), None
        tr = np.zeros(7 * s + 1, dtype=np.uint64)
        c_ctr, c_claim = C.c_uint64(ctr), C.c_uint64(claim)
        dbg = LayerDebug()
        Vb = _u64(Vbelow)
        rc = lib().orc_prove_layer(C.byref(self.arr[i]), s, _ptr(Vb), seed, C.byref(c_ctr), _ptr(z),
                                   C.byref(c_claim), _ptr(tr), C.byref(dbg) if debug else None)
        if rc:
            raise ValueError(f"orc_prove_layer rc={rc}")
        return tr, z, int(c_claim.value), int(c_ctr.value), dbg

    def prove(self, x, seed):
        """Whole proof. Returns (outputs, transcript, final_z, final_claim)."""
        x = _u64(x)
        n = self.transcript_words()
        out = np.zeros(1 << self.c.layers[0].log_size, dtype=np.uint64)
        tr = np.zeros(n, dtype=np.uint64)
        fz = np.zeros(max(self.log_input, 1), dtype=np.uint64)
        fc = C.c_uint64(0)
        rc = lib().orc_prove(self.arr, self.d, self.log_input, _ptr(x), seed, _ptr(out), _ptr(tr), n,
                             _ptr(fz), C.byref(fc))
        if rc:
            raise ValueError(f"orc_prove rc={rc}")
        return out, tr, fz, int(fc.value)

    def verify(self, x, outputs, seed, transcript):
        """Returns (accept, fail_layer, fail_round)."""
        x, outputs, transcript = _u64(x), _u64(outputs), _u64(transcript)
        acc, fl, fr = C.c_int(0), C.c_uint32(0), C.c_uint32(0)
        rc = lib().orc_verify(self.arr, self.d, self.log_input, _ptr(x), _ptr(outputs), seed, _ptr(transcript),
                              transcript.size, C.byref(acc), C.byref(fl), C.byref(fr))
        if rc:
            raise ValueError(f"orc_verify rc={rc}")
        return bool(acc.value), int(fl.value), int(fr.value)

    def layer_entry(self, i, seed, Vi):
        """Entry state (z, claim, counter) of layer i in isolation: orc_layer_entry for the point, orc_mle for the claim."""
        logs = np.array([l.log_size for l in self.c.layers] + [self.log_input], dtype=np.uint32)
        zz = np.zeros(64, dtype=np.uint64)
        ctr = int(lib().orc_layer_entry(logs.ctypes.data_as(C.c_void_p), i, seed, int(self.sum_output), _ptr(zz)))
        return zz, mle(Vi, zz), ctr


def mle(V, x) -> int:
    V, xx = _u64(V), _u64(x)
    s = int(V.size).bit_length() - 1
    assert V.size == 1 << s and xx.size >= s
    return int(lib().orc_mle(_ptr(V), s, _ptr(xx)))


def eq_table(x) -> np.ndarray:
    xx = _u64(x)
    T = np.zeros(1 << xx.size, dtype=np.uint64)
    lib().orc_eq_table(_ptr(xx), xx.size, _ptr(T))
    return T


def lagrange(q, tau) -> int:
    qq = _u64(q)
    return int(lib().orc_lagrange(_ptr(qq), qq.size, tau))


def interp2(G, r) -> int:
    return int(lib().orc_interp2(_ptr(_u64(G)), r))


def draw(seed, k) -> int:
    return int(lib().orc_draw(seed, k))


def mix(seed, k) -> int:
    return int(lib().orc_mix(seed, k))
