"""vc_mle_device_noalloc: the entry point that allocates nothing (scratch in a file-scope device array; include/vc.h).

Collected last on purpose (test_zz_*): the suite runs with pytest -x, so a failure here hides no other test.
The new entry point is compared, bit for bit (integer arithmetic: the tolerance of every test here is zero), with the
EXISTING path for the same sums — k_v_mle inside vc_verify_transcript_device, whose scratch is cudaMalloc'd per circuit
(start claim V~_0(z_0) of the outputs and closing extension V~_d(z_d) of the input, read with vc_debug_verifier_sums) —
and with the oracle's orc_mle, on two calls in a row without a synchronise between them.
"""
import random

import numpy as np
import pytest

import oracle
import vc_workloads as W

pytestmark = pytest.mark.gpu

P = (1 << 61) - 1


@pytest.fixture(scope="module")
def vc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1202_1350_b200 as v
    v.lib()
    return v


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint64).view(np.int64)).cuda()


def _host(t):
    return t.cpu().numpy().view(np.uint64)


def test_no_alloc_mle_matches_the_existing_path_on_two_calls_in_a_row(vc):
    import torch
    # 2^15 inputs = 64 blocks of partials, 2^9 outputs = one block: both sides of the reduction
    c = W.random_circuit([9, 12, 14], 15, 77)
    seed = 4321
    gc = vc.Circuit(c)
    gc.set_input(c.input)
    gc.evaluate(); gc.prove(seed)
    assert gc.verify_device(seed) == (True, 0, 0)                  # the existing path: k_v_mle on cudaMalloc'd scratch
    sums = gc.verifier_sums()
    want_start, want_close = int(sums[0]), int(sums[1 + 4 * c.d])
    s0, sd = c.layers[0].log_size, c.log_input
    z0 = np.array([oracle.draw(seed, k) for k in range(s0)], dtype=np.uint64)
    zd = gc.state()[0][:sd].copy()
    out = gc.outputs().copy()
    assert want_start == oracle.mle(out, z0) and want_close == oracle.mle(c.input, zd)     # the oracle agrees with the existing path

    d_in, d_outv, d_z0, d_zd = _dev(c.input), _dev(out), _dev(z0), _dev(zd)
    r1 = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    r2 = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):                                             # first pass includes the once-per-device set-up
        vc.vc_mle_device_noalloc(d_in, sd, d_zd, r1)               # two calls in a row, same stream, no synchronise between:
        vc.vc_mle_device_noalloc(d_outv, s0, d_z0, r2)             # the second finds the first one's partials in the array
        torch.cuda.synchronize()
        a, b = _host(r1), _host(r2)
        assert (int(a[0]), int(a[1])) == (want_close, 0)
        assert (int(b[0]), int(b[1])) == (want_start, 0)
        r1.fill_(-1); r2.fill_(-1)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == mem0
    assert torch.cuda.mem_get_info()[0] >= free0 - (2 << 20)       # no device allocation behind torch's back either (a module load would be once)
    gc.close()


def test_no_alloc_mle_clears_what_must_start_at_zero_and_rejects_sizes_beyond_the_limit(vc):
    import torch
    rng = random.Random(5)
    for s in (0, 1, 9, 13, 18):                                    # 1 word ... 2^18 words (512 blocks' worth capped at 296)
        x = np.array([rng.randrange(P) for _ in range(1 << s)], dtype=np.uint64)
        z = np.array([rng.randrange(P) for _ in range(max(s, 1))], dtype=np.uint64)
        res = torch.zeros(2, dtype=torch.int64, device="cuda")
        d_x, d_z = _dev(x), _dev(z)
        vc.vc_mle_device_noalloc(d_x, s, d_z, res)
        torch.cuda.synchronize()
        assert (int(_host(res)[0]), int(_host(res)[1])) == (oracle.mle(x, z[:s]) if s else int(x[0]), 0)
        # a non-canonical word is reported by THIS call and not by the next one (the status word is cleared per call)
        bad = x.copy(); bad[len(bad) // 2] = np.uint64((1 << 64) - 1)
        vc.vc_mle_device_noalloc(_dev(bad), s, d_z, res)
        torch.cuda.synchronize()
        assert int(_host(res)[1]) == 1
        vc.vc_mle_device_noalloc(d_x, s, d_z, res)
        torch.cuda.synchronize()
        assert (int(_host(res)[0]), int(_host(res)[1])) == (oracle.mle(x, z[:s]) if s else int(x[0]), 0)
    # the stated maximum: log_n <= 28; beyond it nothing is enqueued and the code says why
    res = torch.full((2,), 7, dtype=torch.int64, device="cuda")
    tiny = torch.zeros(64, dtype=torch.int64, device="cuda")
    with pytest.raises(vc.VCError) as e:
        vc.vc_mle_device_noalloc(tiny, 29, tiny, res)
    assert e.value.code == vc.VC_ERR_LIMIT and "maximum" in vc.vc_strerror(e.value.code)
    torch.cuda.synchronize()
    assert _host(res).tolist() == [7, 7]
    with pytest.raises(vc.VCError) as e:
        vc.lib().vc_mle_device_noalloc  # noqa: B018  (symbol exists)
        vc.vc_mle_device_noalloc(tiny, 3, tiny, None)
    assert e.value.code == vc.VC_ERR_ARG
