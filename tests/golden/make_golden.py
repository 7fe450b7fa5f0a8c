"""Writes tests/golden/config<k>.txt from the CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py 1 2 3 4 5

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


def main(ks):
    for k in ks:
        c = W.config(k)
        seed = W.challenge_seed(k)
        oc = oracle.OracleCircuit(c)
        t0 = time.time()
        out, tr, fz, fc = oc.prove(c.input, seed)
        dt = time.time() - t0
        lines = [f"# config {k}: {c.name}; data_seed={W.data_seed(k)} challenge_seed={seed}",
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
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"config{k}.txt")
        with open(path, "w") as f:
            f.write("\n".join(lines) + "\n")
        print(f"config {k}: {dt:.1f} s -> {path}", flush=True)


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [1])
