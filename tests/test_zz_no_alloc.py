"""The allocation-free entry point `bta_rows_times_block_noalloc` (include/bta.h): its scratch is a file-scope device
array inside the library, so callers that cannot call cudaMalloc (graph capture, serving loops) can use it.  Checked
against the existing path -- the sweeps' own launcher with caller-provided scratch, `bta_rows_times_block`
(include/bta_diag.h) -- and against numpy, on two calls in a row (the second smaller and triangular: stale contents of
the shared scratch must not matter).  Collected last on purpose (the suite runs with `pytest -x`)."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _case(P, K, J, tri, seed, alpha, beta):
    rng = np.random.default_rng(seed)
    R = rng.standard_normal((P, K))
    M = rng.standard_normal((K, J))
    if tri:
        M = np.tril(M)
    inp = rng.standard_normal((P, J))
    ref = alpha * (R @ M) + beta * inp
    return R, M, inp, ref


def test_noalloc_matches_existing_path_two_calls_in_a_row():
    import torch
    from paper_2605_06392_b200.binding import rows_times_block, rows_times_block_noalloc
    dev = torch.device("cuda", 0)
    t = lambda x: torch.tensor(x, dtype=torch.float64, device=dev)
    # first call fills most of the built-in scratch; the second is smaller, ragged and triangular
    for (P, K, J, tri, alpha, beta) in [(9, 1000, 1100, 0, -1.0, 1.0), (4, 300, 300, 1, 0.75, 0.0),
                                        (1, 4096, 4096, 0, 1.0, -2.0)]:
        R, M, inp, ref = _case(P, K, J, tri, 100 + P, alpha, beta)
        nks = -(-K // 128)
        part = torch.full((nks * P * J,), float("nan"), dtype=torch.float64, device=dev)
        out_old = torch.empty(P, J, dtype=torch.float64, device=dev)
        out_new = torch.empty(P, J, dtype=torch.float64, device=dev)
        Rd, Md, ind = t(R), t(M), t(inp)
        mem0 = torch.cuda.memory_allocated(dev)
        rows_times_block(Rd, Md, out_old, part, alpha, beta, ind if beta != 0.0 else None, tri)
        rows_times_block_noalloc(Rd, Md, out_new, alpha, beta, ind if beta != 0.0 else None, tri)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == mem0          # nothing allocated through torch's allocator either
        a, b = out_old.cpu().numpy(), out_new.cpu().numpy()
        scale = np.max(np.abs(ref))
        assert np.max(np.abs(b - a)) <= 1e-12 * scale              # same kernels, same summation order
        assert np.max(np.abs(b - ref)) <= 1e-12 * K * scale       # and the right product (tolerance of the GEMM tests)


def test_noalloc_in_place_and_repeatable():
    import torch
    from paper_2605_06392_b200.binding import rows_times_block_noalloc
    dev = torch.device("cuda", 0)
    R, M, inp, ref = _case(3, 517, 260, 0, 7, -0.5, 1.0)
    t = lambda x: torch.tensor(x, dtype=torch.float64, device=dev)
    Rd, Md = t(R), t(M)
    outs = []
    for _ in range(2):                                             # in == out (in-place update), twice: bit-identical
        buf = t(inp)
        rows_times_block_noalloc(Rd, Md, buf, -0.5, 1.0, buf, 0)
        outs.append(buf.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])
    assert np.max(np.abs(outs[0] - ref)) <= 1e-12 * 517 * np.max(np.abs(ref))


def test_noalloc_rejects_sizes_beyond_the_builtin_scratch():
    import torch
    from paper_2605_06392_b200 import BtaError
    from paper_2605_06392_b200.binding import NOALLOC_MAX_PART, lib, rows_times_block_noalloc
    dev = torch.device("cuda", 0)
    P, K, J = 9, 4224, 4096                                       # 33 chunks * 9 * 4096 > 32 * 9 * 4096
    assert -(-K // 128) * P * J > NOALLOC_MAX_PART
    R = torch.zeros(P, K, dtype=torch.float64, device=dev)
    M = torch.zeros(8, J, dtype=torch.float64, device=dev)        # never read: the call must fail before launching
    out = torch.zeros(P, J, dtype=torch.float64, device=dev)
    from paper_2605_06392_b200.binding import _check, _stream
    with pytest.raises(BtaError) as ei:
        _check(lib().bta_rows_times_block_noalloc(P, K, J, R.data_ptr(), K, M.data_ptr(), J, 0, 1.0, 0.0, None, 0,
                                                  out.data_ptr(), J, _stream()))
    assert ei.value.code == 1 and "BTA_NOALLOC_MAX_PART" in str(ei.value)
    with pytest.raises(BtaError):                                  # more than 9 rows
        _check(lib().bta_rows_times_block_noalloc(10, 128, 128, R.data_ptr(), K, M.data_ptr(), J, 0, 1.0, 0.0, None, 0,
                                                  out.data_ptr(), J, _stream()))
