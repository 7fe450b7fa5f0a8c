"""ctypes binding for libvc.so — same names as include/vc.h; marshalling only."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

VC_OK, VC_ERR_ARG, VC_ERR_SHAPE, VC_ERR_STATE, VC_ERR_CUDA, VC_ERR_NOMEM, VC_ERR_LIMIT = range(7)

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libvc.so"

EXPORTS = [
    "vc_circuit_load", "vc_evaluate", "vc_prove_layer", "vc_prove", "vc_run_host", "vc_verify_transcript",
    "vc_circuit_free", "vc_strerror", "vc_transcript_words", "vc_total_transcript_words", "vc_depth",
    "vc_log_size", "vc_debug_state", "vc_debug_values", "vc_status", "vc_launch_count", "vc_set_schedule",
    "vc_debug_fieldop", "vc_bench_modmul", "vc_profile_enable", "vc_profile_read", "vc_debug_layer_stamps", "vc_debug_trace",
    "vc_verify_transcript_device", "vc_debug_verifier_sums", "vc_debug_layer_kinds", "vc_debug_layer_wiring", "vc_circuit_load_hosted", "vc_debug_hosted_bytes", "vc_hosted_set_weights", "vc_mle_device_noalloc",
]


class VCError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {vc_strerror(code)} (code {code})")


class _Layer(C.Structure):
    _fields_ = [("log_size", C.c_uint32), ("type", C.c_void_p), ("in1", C.c_void_p), ("in2", C.c_void_p)]


def library_path() -> Path:
    return _SO


_lib = None


def lib():
    """Loads libvc.so; fails loudly if it has not been built (python __graft_entry__.py / build.py)."""
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise RuntimeError(f"{_SO} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                               "(there is no CPU fallback for the CUDA path)")
        L = C.CDLL(str(_SO))
        u64, u32, vp, i32 = C.c_uint64, C.c_uint32, C.c_void_p, C.c_int
        sig = {
            "vc_circuit_load": (i32, [vp, u32, u32, vp]),
            "vc_evaluate": (i32, [vp, vp, vp, vp]),
            "vc_prove_layer": (i32, [vp, u32, u64, vp, u64, vp]),
            "vc_prove": (i32, [vp, u64, vp, u64, vp]),
            "vc_run_host": (i32, [vp, vp, u64, vp, vp, u64, vp]),
            "vc_verify_transcript": (i32, [vp, vp, vp, u64, vp, u64, vp, vp, vp]),
            "vc_verify_transcript_device": (i32, [vp, vp, vp, u64, vp, u64, vp, vp, vp, vp]),
            "vc_debug_verifier_sums": (i32, [vp, vp, u64]),
            "vc_circuit_free": (None, [vp]),
            "vc_strerror": (C.c_char_p, [i32]),
            "vc_transcript_words": (u64, [vp, u32]),
            "vc_total_transcript_words": (u64, [vp]),
            "vc_depth": (u32, [vp]),
            "vc_log_size": (u32, [vp, u32]),
            "vc_debug_state": (i32, [vp, vp, vp, vp, vp]),
            "vc_debug_values": (i32, [vp, u32, vp, vp]),
            "vc_status": (i32, [vp, vp, vp]),
            "vc_launch_count": (u64, []),
            "vc_set_schedule": (i32, [vp, i32]),
            "vc_debug_fieldop": (i32, [i32, vp, vp, vp, u64, vp]),
            "vc_bench_modmul": (i32, [u32, u32, u32, u32, vp, vp]),
            "vc_debug_layer_stamps": (i32, [vp, vp, vp]),
            "vc_debug_trace": (i32, [vp, vp, u32, vp]),
            "vc_debug_layer_kinds": (i32, [vp, vp]),
            "vc_debug_layer_wiring": (i32, [vp, vp]),
            "vc_circuit_load_hosted": (i32, [vp, u32, u32, u32, vp]),
            "vc_debug_hosted_bytes": (i32, [vp, vp, vp]),
            "vc_hosted_set_weights": (i32, [vp, i32]),
            "vc_mle_device_noalloc": (i32, [vp, u32, vp, vp, vp]),
            "vc_profile_enable": (i32, [i32]),
            "vc_profile_read": (i32, [vp, vp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def vc_strerror(code: int) -> str:
    return lib().vc_strerror(code).decode()


def _check(rc: int, where: str):
    if rc != VC_OK:
        raise VCError(rc, where)


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


def _dev_ptr(t) -> int:
    """torch CUDA tensor (int64/uint64 storage of field words) -> device pointer."""
    if t is None:
        return 0
    assert t.is_cuda and t.is_contiguous() and t.element_size() == 8, "expected a contiguous CUDA tensor of 8-byte words"
    return t.data_ptr()


def _host_ptr(a) -> int:
    if hasattr(a, "data_ptr"):          # pinned / CPU torch tensor
        assert not a.is_cuda and a.is_contiguous() and a.element_size() == 8
        return a.data_ptr()
    assert isinstance(a, np.ndarray) and a.dtype == np.uint64 and a.flags.c_contiguous
    return a.ctypes.data


# ---------------------------------------------------------------------------- flat C-ABI mirrors
def vc_circuit_load(layers, log_input: int, hosted_chunk_log=None) -> int:
    """layers: sequence of objects with log_size/type/in1/in2 (numpy, host), output layer first. Returns the handle.
    hosted_chunk_log: vc_circuit_load_hosted with slots of 2^hosted_chunk_log gates (records and weights stay on the host)."""
    arr = (_Layer * len(layers))()
    keep = []
    for i, L in enumerate(layers):
        t = np.ascontiguousarray(L.type, dtype=np.uint8)
        a = np.ascontiguousarray(L.in1, dtype=np.uint32)
        b = np.ascontiguousarray(L.in2, dtype=np.uint32)
        keep += [t, a, b]
        arr[i] = _Layer(int(L.log_size), t.ctypes.data, a.ctypes.data, b.ctypes.data)
    h = C.c_void_p(0)
    if hosted_chunk_log is None:
        _check(lib().vc_circuit_load(arr, len(layers), int(log_input), C.byref(h)), "vc_circuit_load")
    else:
        _check(lib().vc_circuit_load_hosted(arr, len(layers), int(log_input), int(hosted_chunk_log), C.byref(h)), "vc_circuit_load_hosted")
    return h.value


def vc_mle_device_noalloc(d_values, log_n: int, d_point, d_out2, stream=None):
    """Enqueue out2 = (V~(point), status) for the 2^log_n-word device table d_values; allocates nothing (include/vc.h)."""
    _check(lib().vc_mle_device_noalloc(_dev_ptr(d_values), int(log_n), _dev_ptr(d_point), _dev_ptr(d_out2), _stream_ptr(stream)),
           "vc_mle_device_noalloc")


def vc_evaluate(handle: int, d_input, d_outputs=None, stream=None):
    _check(lib().vc_evaluate(handle, _dev_ptr(d_input), _dev_ptr(d_outputs), _stream_ptr(stream)), "vc_evaluate")


def vc_prove_layer(handle: int, layer: int, seed: int, d_transcript, stream=None, offset_words: int = 0):
    cap = d_transcript.numel() - offset_words
    _check(lib().vc_prove_layer(handle, layer, seed, _dev_ptr(d_transcript) + 8 * offset_words, cap,
                                _stream_ptr(stream)), "vc_prove_layer")


def vc_prove(handle: int, seed: int, d_transcript, stream=None):
    _check(lib().vc_prove(handle, seed, _dev_ptr(d_transcript), d_transcript.numel(), _stream_ptr(stream)), "vc_prove")


def vc_run_host(handle: int, h_input, seed: int, h_outputs, h_transcript, stream=None):
    n = h_transcript.numel() if hasattr(h_transcript, "numel") else h_transcript.size
    _check(lib().vc_run_host(handle, _host_ptr(h_input), seed, _host_ptr(h_outputs), _host_ptr(h_transcript), n,
                             _stream_ptr(stream)), "vc_run_host")


def vc_verify_transcript(handle: int, h_input, h_outputs, seed: int, h_transcript):
    """Returns (accept, fail_layer, fail_round)."""
    acc, fl, fr = C.c_int(0), C.c_uint32(0), C.c_uint32(0)
    h_input, h_outputs, h_transcript = (np.ascontiguousarray(x, dtype=np.uint64) for x in (h_input, h_outputs, h_transcript))
    _check(lib().vc_verify_transcript(handle, h_input.ctypes.data, h_outputs.ctypes.data, seed, h_transcript.ctypes.data,
                                      h_transcript.size, C.byref(acc), C.byref(fl), C.byref(fr)), "vc_verify_transcript")
    return bool(acc.value), int(fl.value), int(fr.value)


def vc_verify_transcript_device(handle: int, d_input, d_outputs, seed: int, d_transcript, stream=None):
    """The verifier with its O(S) sums on the GPU; device tensors in, (accept, fail_layer, fail_round) out."""
    acc, fl, fr = C.c_int(0), C.c_uint32(0), C.c_uint32(0)
    _check(lib().vc_verify_transcript_device(handle, _dev_ptr(d_input), _dev_ptr(d_outputs), seed, _dev_ptr(d_transcript),
                                             d_transcript.numel(), C.byref(acc), C.byref(fl), C.byref(fr),
                                             _stream_ptr(stream)), "vc_verify_transcript_device")
    return bool(acc.value), int(fl.value), int(fr.value)


def vc_debug_verifier_sums(handle: int, d: int) -> np.ndarray:
    out = np.zeros(4 * d + 2, dtype=np.uint64)
    _check(lib().vc_debug_verifier_sums(handle, out.ctypes.data, out.size), "vc_debug_verifier_sums")
    return out


def vc_circuit_free(handle: int):
    lib().vc_circuit_free(handle)


def vc_transcript_words(handle: int, layer: int) -> int:
    return int(lib().vc_transcript_words(handle, layer))


def vc_total_transcript_words(handle: int) -> int:
    return int(lib().vc_total_transcript_words(handle))


# ---------------------------------------------------------------------------- small convenience wrapper
class Circuit:
    """Owns a vc_circuit handle plus the torch device buffers a proof needs (input, outputs, transcript)."""

    def __init__(self, circuit, hosted_chunk_log=None):
        import torch
        self.torch = torch
        self.handle = vc_circuit_load(circuit.layers, circuit.log_input, hosted_chunk_log)
        self.d = len(circuit.layers)
        self.log_input = circuit.log_input
        self.n_out = 1 << circuit.layers[0].log_size
        self.words = vc_total_transcript_words(self.handle)
        self.d_input = torch.empty(1 << circuit.log_input, dtype=torch.int64, device="cuda")
        self.d_outputs = torch.empty(self.n_out, dtype=torch.int64, device="cuda")
        self.d_transcript = torch.zeros(self.words, dtype=torch.int64, device="cuda")

    def set_input(self, x: np.ndarray):
        t = self.torch.from_numpy(np.ascontiguousarray(x, dtype=np.uint64).view(np.int64))
        self.d_input.copy_(t)

    def set_schedule(self, schedule: int):
        _check(lib().vc_set_schedule(self.handle, schedule), "vc_set_schedule")

    def evaluate(self, stream=None):
        vc_evaluate(self.handle, self.d_input, self.d_outputs, stream)

    def prove(self, seed: int, stream=None):
        vc_prove(self.handle, seed, self.d_transcript, stream)

    def prove_layerwise(self, seed: int, stream=None):
        w = 0
        for i in range(self.d):
            vc_prove_layer(self.handle, i, seed, self.d_transcript, stream, offset_words=w)
            w += vc_transcript_words(self.handle, i)

    def outputs(self) -> np.ndarray:
        return self.d_outputs.cpu().numpy().view(np.uint64)

    def transcript(self) -> np.ndarray:
        return self.d_transcript.cpu().numpy().view(np.uint64)

    def values(self, layer: int) -> np.ndarray:
        n = 1 << int(lib().vc_log_size(self.handle, layer))
        out = np.empty(n, dtype=np.uint64)
        _check(lib().vc_debug_values(self.handle, layer, out.ctypes.data, _stream_ptr(None)), "vc_debug_values")
        return out

    def state(self):
        z = np.zeros(64, dtype=np.uint64)
        claim, ctr = C.c_uint64(0), C.c_uint64(0)
        _check(lib().vc_debug_state(self.handle, z.ctypes.data, C.byref(claim), C.byref(ctr), _stream_ptr(None)), "vc_debug_state")
        return z, int(claim.value), int(ctr.value)

    def layer_stamps(self) -> np.ndarray:
        """d+1 device timestamps (ns) of the last fused proof: start of each layer, [d] = end (vc_debug_layer_stamps)."""
        h = np.zeros(self.d + 1, dtype=np.uint64)
        _check(lib().vc_debug_layer_stamps(self.handle, _host_ptr(h), None), "vc_debug_layer_stamps")
        return h

    def layer_kinds(self) -> np.ndarray:
        """Per layer, the VC_K_* code of the kernel that proves it on the fused schedule (vc_debug_layer_kinds)."""
        h = np.zeros(self.d, dtype=np.uint32)
        _check(lib().vc_debug_layer_kinds(self.handle, h.ctypes.data), "vc_debug_layer_kinds")
        return h

    def layer_wiring(self) -> np.ndarray:
        """Per layer, how the prover gets its wiring: 0 records, 1 tree, 2 self, 3 bit-field rule (vc_debug_layer_wiring)."""
        h = np.zeros(self.d, dtype=np.uint32)
        _check(lib().vc_debug_layer_wiring(self.handle, h.ctypes.data), "vc_debug_layer_wiring")
        return h

    def set_hosted_weights(self, swap: bool):
        """Hosted circuits: recompute the weights per message (False, default) or swap them through host memory (True)."""
        _check(lib().vc_hosted_set_weights(self.handle, int(bool(swap))), "vc_hosted_set_weights")

    def hosted_bytes(self):
        """(h2d, d2h) bytes a hosted circuit moved in its last evaluation / proof (vc_debug_hosted_bytes)."""
        a, b = C.c_uint64(0), C.c_uint64(0)
        _check(lib().vc_debug_hosted_bytes(self.handle, C.byref(a), C.byref(b)), "vc_debug_hosted_bytes")
        return int(a.value), int(b.value)

    def flags(self) -> int:
        f = C.c_uint32(0)
        _check(lib().vc_status(self.handle, C.byref(f), _stream_ptr(None)), "vc_status")
        return int(f.value)

    def verify(self, x, outputs, seed, transcript):
        return vc_verify_transcript(self.handle, x, outputs, seed, transcript)

    def verify_device(self, seed: int, d_input=None, d_outputs=None, d_transcript=None, stream=None):
        """vc_verify_transcript_device on this object's device buffers (or the tensors given)."""
        return vc_verify_transcript_device(self.handle, self.d_input if d_input is None else d_input,
                                           self.d_outputs if d_outputs is None else d_outputs, seed,
                                           self.d_transcript if d_transcript is None else d_transcript, stream)

    def verifier_sums(self) -> np.ndarray:
        return vc_debug_verifier_sums(self.handle, self.d)

    def close(self):
        if self.handle:
            vc_circuit_free(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
