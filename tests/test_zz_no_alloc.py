"""bfsc_compress_noalloc (include/bfsc.h): the single-buffer compress call with its workspace in the library's own
`static __device__` array, for callers that cannot allocate. Checked against the existing path (bfsc_compress with a
caller-owned workspace): same bytes, bit-exact (integer work), on two calls in a row that share the array — the second
on a different, shorter input, so anything the first call left behind in the scratch would show.
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

from paper_1704_00513_b200.workloads import streams

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1704_00513_b200 import build, binding
    build.build()
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def _existing_path(B, d_ids, n, W, thr):
    dev = d_ids.device
    cap = B.compress_bound(n, W)
    out = torch.full((cap + 64,), 0xAB, dtype=torch.uint8, device=dev)
    nbytes = torch.full((1,), -1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress(d_ids, n, W, thr, out, nbytes, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    return out[:int(nbytes.item())].cpu().numpy()


@pytest.mark.parametrize("W", [32, 64])
def test_noalloc_matches_existing_path_two_calls_in_a_row(B, W):
    dev = torch.device("cuda")
    # first call: the maximum size (512 tiles: tickets, look-back over every state of the scratch array), outliers;
    # second call: a shorter stream with other gaps and a ragged tail, then a RAW one (below the threshold)
    cases = [(B.NOALLOC_MAX_IDS, 256.0, 0.01, 0), (128 * 64 * 37 + 77, 2.0, 0.0, 0), (200, 3.0, 0.0, 4096)]
    inputs = [streams.gap_stream(n, mean, seed=31 + i, W=W, outlier_frac=outl, device=dev) for i, (n, mean, outl, _) in enumerate(cases)]
    expected = [_existing_path(B, ids, n, W, thr) for ids, (n, _, _, thr) in zip(inputs, cases)]
    outs = [torch.full((B.compress_bound(n, W) + 64,), 0xAB, dtype=torch.uint8, device=dev) for n, _, _, _ in cases]
    nbytes = [torch.full((1,), -1, dtype=torch.int64, device=dev) for _ in cases]
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    for ids, (n, _, _, thr), out, nb in zip(inputs, cases, outs, nbytes):     # back to back on one stream, no sync between
        B.compress_noalloc(ids, n, W, thr, out, nb, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    for (n, _, _, _), out, nb, exp in zip(cases, outs, nbytes, expected):
        total = int(nb.item())
        assert total == len(exp)
        got = out[:total].cpu().numpy()
        assert np.array_equal(got, exp), f"n={n}: first difference at byte {int(np.nonzero(got != exp)[0][0])}"
        assert bool((out[B.compress_bound(n, W):] == 0xAB).all()), "wrote beyond capacity"


def test_noalloc_rejects_sizes_beyond_the_scratch(B):
    dev = torch.device("cuda")
    n = B.NOALLOC_MAX_IDS + 1
    ids = torch.zeros(n, dtype=torch.int32, device=dev)
    out = torch.empty(B.compress_bound(n, 32), dtype=torch.uint8, device=dev)
    nbytes = torch.full((1,), -1, dtype=torch.int64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    with pytest.raises(B.BfscError) as e:
        B.compress_noalloc(ids, n, 32, 0, out, nbytes, status)
    assert e.value.code == B.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int(nbytes.item()) == -1 and int(status.item()) == 0          # nothing was enqueued


def test_checked_build_sees_a_violation(B):
    """Only under BFSC_CHECKED=1 (libbfsc_checked.so): a deliberately violated BFSC_CHECK is counted with its source line —
    the end-of-run assertion of tests/conftest.py would see a real one."""
    import ctypes
    if not B.CHECKED:
        pytest.skip("normal build: BFSC_CHECK compiles away")
    seen = (ctypes.c_uint * 2)()
    B.lib().bfsc_debug_check_selftest(seen)
    assert seen[0] == 1 and seen[1] > 0
    assert B.check_failures()[0][0] == 0                 # the selftest put the counters back
