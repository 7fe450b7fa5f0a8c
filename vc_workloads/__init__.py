"""Seeded synthetic circuits and inputs for the GKR prover hot path.

This package holds ONLY wiring/shape generators and seeded input generators (numpy).
It contains none of the method's arithmetic (no field operations, no sum-check, no
PRNG for challenges): both the CPU oracle's tests and the CUDA path's tests/bench take
their circuits and inputs from here, so that the two implementations see identical bytes
while sharing no code.  Recipes: DESIGN.md "Input recipe"; shapes: BASELINE.json configs.
"""
from .circuits import (  # noqa: F401
    ADD, MULT, SUB, RELAY, SUM, Circuit, Layer,
    f2_circuit, f0_circuit, matmul_circuit, matmul_eq_circuit, pm_circuit, f2_sum_circuit, f0_sum_circuit, random_circuit,
    config, CONFIG_NAMES, data_seed, challenge_seed,
)
