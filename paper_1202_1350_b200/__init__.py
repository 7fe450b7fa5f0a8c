"""paper_1202_1350_b200 — GKR/CMT prover hot path over F_p (p = 2^61-1) for one NVIDIA B200.

Thin Python binding over the C ABI of libvc.so (include/vc.h): argument marshalling only — every step of
the path (evaluation, beta weights, sum-check rounds, reductions, challenges, line restriction) runs in the
hand-written sm_100a kernels under csrc/.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: importing works anywhere, calling needs the built library and a CUDA device.
"""
from .binding import (  # noqa: F401
    VCError, Circuit, lib, library_path,
    vc_circuit_load, vc_evaluate, vc_prove_layer, vc_prove, vc_run_host, vc_verify_transcript,
    vc_verify_transcript_device, vc_debug_verifier_sums, vc_mle_device_noalloc,
    vc_circuit_free, vc_strerror, vc_transcript_words, vc_total_transcript_words,
    VC_OK, VC_ERR_ARG, VC_ERR_SHAPE, VC_ERR_STATE, VC_ERR_CUDA, VC_ERR_NOMEM, VC_ERR_LIMIT,
)
