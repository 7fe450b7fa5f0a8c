"""Writes tests/golden/config<k>.txt and tests/golden/paper_<kind>_<n>.txt from the CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py 1 2 3 4 5                  # BASELINE.json configs
    python tests/golden/make_golden.py f2:22 f2:23 matmul:8 matmuleq:8 pm:19 f0:20 f0:21   # paper-scale constructions

For BASELINE.json config k (data seed 1000+k, challenge seed 2000+k; DESIGN.md input recipe) the
oracle (oracle/gkr_oracle.c, single thread) evaluates the circuit and produces the honest transcript;
the file stores, per layer, the SHA-256 of that layer's transcript words (little-endian uint64), plus
the first and last word in clear, the outputs' digest and the final claim.  The GPU parity tests
compare the CUDA transcript of the same config against these lines, which gives a bit-exact check at
the full sizes where re-running the oracle inside the test would take minutes (config 5: ~2.6e9
gate-rounds).  No value in the file is printed by the paper (it prints no worked example,
SURVEY.md §8(c) last row).
"""
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import vc_workloads as W  # noqa: E402


def sha(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a, dtype="<u8").tobytes()).hexdigest()


# paper-scale cases: (data seed, challenge seed) are the ones tests/test_gpu_verifier.py uses
PAPER_SEEDS = {"f2": (7, 31337), "matmul": (4, 4242), "pm": (5, 4242), "f0": (3, 4242), "matmuleq": (4, 4242)}


def paper_case(kind: str, n: int):
    from vc_workloads import circuits
    ds, cs = PAPER_SEEDS[kind]
    c = {"f2": lambda: circuits.f2_circuit(n, ds), "matmul": lambda: circuits.matmul_circuit(n, ds),
         "pm": lambda: circuits.pm_circuit(n, 3, ds), "f0": lambda: circuits.f0_circuit(n, ds),
         "matmuleq": lambda: circuits.matmul_eq_circuit(n, ds, wrong=3)}[kind]()
    return c, cs


def main(ks):
    for k in ks:
        if isinstance(k, str):
            kind, n = k.split(":")
            c, seed = paper_case(kind, int(n))
            fname, head = f"paper_{kind}_{n}.txt", f"# paper scale {kind}:{n}: {c.name}; data_seed={PAPER_SEEDS[kind][0]} challenge_seed={seed}"
        else:
            c = W.config(k)
            seed = W.challenge_seed(k)
            fname, head = f"config{k}.txt", f"# config {k}: {c.name}; data_seed={W.data_seed(k)} challenge_seed={seed}"
        oc = oracle.OracleCircuit(c)
        t0 = time.time()
        out, tr, fz, fc = oc.prove(c.input, seed)
        dt = time.time() - t0
        lines = [head,
                 f"# written by tests/golden/make_golden.py from oracle/gkr_oracle.c in {dt:.1f} s (1 thread)",
                 f"gates {c.gates}", f"transcript_words {tr.size}",
                 f"outputs_sha256 {sha(out)}", f"output0 {int(out[0])}",
                 f"transcript_sha256 {sha(tr)}", f"final_claim {fc}"]
        w = 0
        for i in range(c.d):
            n = c.transcript_words(i)
            seg = tr[w:w + n]
            lines.append(f"layer {i} {c.log_below(i)} {sha(seg)} {int(seg[0])} {int(seg[-1])}")
            w += n
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), fname)
        with open(path, "w") as f:
            f.write("\n".join(lines) + "\n")
        print(f"{k}: {dt:.1f} s -> {path}", flush=True)


if __name__ == "__main__":
    main([a if ":" in a else int(a) for a in sys.argv[1:]] or [1])
