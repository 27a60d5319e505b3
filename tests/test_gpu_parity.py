"""GPU parity: CUDA path (through the C ABI) vs the oracle, on the same seeded inputs.
Bar: compressed bytes memcmp-equal (headers, directory, pads), offsets equal, decoded IDs
equal to the input (integer work: bit-exact)."""
import numpy as np
import pytest
import torch

from paper_1704_00513_b200.workloads import rmat, streams

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1704_00513_b200 import build, binding
    build.build()
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def _np(t, W):
    a = t.cpu().numpy()
    return a.view(np.uint32) if W == 32 else a.view(np.uint64)


PFOR, BP128 = 1, 2           # bfsc_codec: encoder rule (FORMAT.md §7)
CODECS = [PFOR, BP128]


def run_batch(B, oracle_mod, ids_t, off_t, W, thr, check_oracle=True, codec=PFOR):
    """ids_t: CPU tensor (int32/int64 bit pattern), off_t: int64 offsets. Returns GPU bytes."""
    dev = torch.device("cuda")
    n, n_buf = ids_t.numel(), off_t.numel() - 1
    counts = (off_t[1:] - off_t[:-1]).tolist()
    cap = B.batch_compress_bound(counts, W)
    d_ids = torch.empty(n + 4, dtype=ids_t.dtype, device=dev)
    d_ids[:n] = ids_t.to(dev)
    d_off = off_t.to(dev)
    out = torch.full((cap + 64,), 0xAB, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    if codec == PFOR:
        B.compress_batch(d_ids, d_off, n_buf, W, thr, out, out_off, ws, status)
    else:
        B.compress_batch_codec(codec, d_ids, d_off, n_buf, W, thr, out, out_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    total = int(out_off[-1].item())
    assert total <= cap
    assert bool((out[cap:] == 0xAB).all()), "wrote beyond capacity"
    gpu_bytes = out[:total].cpu().numpy()
    gpu_off = out_off.cpu().numpy().astype(np.uint64)
    if check_oracle:
        ref, ref_off = oracle_mod.compress_batch(_np(ids_t, W), off_t.numpy().astype(np.uint64), thr, codec=codec)   # the plain serial oracle
        assert np.array_equal(gpu_off, ref_off)
        if not np.array_equal(gpu_bytes, ref):
            bad = int(np.nonzero(gpu_bytes != ref)[0][0])
            raise AssertionError(f"compressed bytes differ at {bad} of {len(ref)}")
    # decode on the GPU
    back = torch.full((n + 4,), -1, dtype=ids_t.dtype, device=dev)
    id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    status.zero_()
    B.decompress_batch(out, out_off, n_buf, W, back, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    assert torch.equal(id_off.cpu(), off_t)
    assert torch.equal(back[:n].cpu(), ids_t)
    assert bool((back[n:] == -1).all())
    run_scatter(B, d_ids, d_off, counts, W, thr, codec, out, out_off, ids_t, off_t)
    return gpu_bytes, gpu_off


def run_scatter(B, d_ids, d_off, counts, W, thr, codec, out, out_off, ids_t, off_t):
    """bfsc_compress_batch_scatter on the same batch: stream i lands in slot i of a slotted receive buffer (a guard
    zone behind every slot), byte-identical to stream i of the back-to-back output `out` (which the caller has compared
    with the oracle); then bfsc_decompress_batch straight from the slots."""
    dev = d_ids.device
    n, n_buf = ids_t.numel(), len(counts)
    slot = max([B.compress_bound(c, W) for c in set(counts)] + [32])
    pitch = slot + 48                                          # (a multiple of 16; 48 guard bytes)
    if n_buf == 0 or n_buf * pitch > (1 << 28):
        return
    recv = torch.full((n_buf * pitch,), 0xCD, dtype=torch.uint8, device=dev)
    dst = recv.data_ptr() + pitch * torch.arange(n_buf, dtype=torch.int64, device=dev)
    sizes = torch.full((n_buf,), -1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress_batch_scatter(codec, d_ids, d_off, n_buf, W, thr, dst, slot, sizes, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    assert torch.equal(sizes, out_off[1:] - out_off[:-1])
    # every slot: the stream, then untouched bytes up to the next slot
    col = torch.arange(pitch, device=dev).unsqueeze(0)
    live = col < sizes.unsqueeze(1)
    src_idx = (out_off[:-1].unsqueeze(1) + col).clamp_(max=out.numel() - 1)
    expect = torch.where(live, out[src_idx], torch.full_like(out[:1], 0xCD))
    got = recv.view(n_buf, pitch)
    if not torch.equal(got, expect):
        bad = torch.nonzero(got != expect)[0].tolist()
        raise AssertionError(f"scatter: slot {bad[0]} differs at byte {bad[1]} (stream of {int(sizes[bad[0]])} bytes)")
    # the receive side: decode the slots where they lie (a stream is shorter than its span)
    slot_off = pitch * torch.arange(n_buf + 1, dtype=torch.int64, device=dev)
    back = torch.full((n + 4,), -1, dtype=ids_t.dtype, device=dev)
    id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    B.decompress_batch(recv, slot_off, n_buf, W, back, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    assert torch.equal(id_off.cpu(), off_t)
    assert torch.equal(back[:n].cpu(), ids_t)


def run_single(B, oracle_mod, ids_t, W, thr, codec=PFOR):
    dev = torch.device("cuda")
    n = ids_t.numel()
    cap = B.compress_bound(n, W)
    d_ids = ids_t.to(dev) if n else torch.empty(4, dtype=ids_t.dtype, device=dev)
    out = torch.empty(cap, dtype=torch.uint8, device=dev)
    nbytes = torch.zeros(1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    if codec == PFOR:
        B.compress(d_ids, n, W, thr, out, nbytes, ws, status)
    else:
        B.compress_codec(codec, d_ids, n, W, thr, out, nbytes, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    total = int(nbytes.item())
    ref = oracle_mod.compress(_np(ids_t, W), thr, codec=codec)
    assert total == len(ref)
    assert np.array_equal(out[:total].cpu().numpy(), ref)
    back = torch.empty(max(n, 4), dtype=ids_t.dtype, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    B.decompress(out, total, W, back, n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and int(n_out.item()) == n
    assert torch.equal(back[:n].cpu(), ids_t)


@pytest.mark.parametrize("codec", CODECS)
@pytest.mark.parametrize("W", [32, 64])
def test_single_edge_sizes(B, oracle_mod, W, codec):
    for n in (0, 1, 2, 127, 128, 129, 255, 256, 257, 1000, 4097, 128 * 300 + 5):
        for mean in (1.0, 2.0, 256.0):
            t = streams.gap_stream(n, mean, seed=11, W=W)
            run_single(B, oracle_mod, t, W, 0, codec=codec)
    run_single(B, oracle_mod, streams.gap_stream(100, 2.0, seed=1, W=W), W, 1024, codec=codec)   # RAW
    run_single(B, oracle_mod, streams.gap_stream(300, 2.0, seed=1, W=W), W, 1024, codec=codec)


@pytest.mark.parametrize("codec", CODECS)
@pytest.mark.parametrize("W", [32, 64])
def test_adversarial_values(B, oracle_mod, W, codec):
    rng = np.random.default_rng(W)
    n = 128 * 40 + 77
    dt = np.uint32 if W == 32 else np.uint64
    tdt = torch.int32 if W == 32 else torch.int64
    cases = {
        "random_full_width": rng.integers(0, 1 << W, size=n, dtype=np.uint64, endpoint=False).astype(dt),
        "alt_extremes": np.where(np.arange(n) % 2 == 0, 0, (1 << W) - 1).astype(dt),
        "all_equal": np.full(n, 12345, dtype=dt),
        "max": np.full(n, (1 << W) - 1, dtype=dt),
        "wrap": ((np.uint64((1 << W) - 50) + np.arange(n, dtype=np.uint64)) & np.uint64((1 << W) - 1)).astype(dt),
    }
    for bits in (1, 3, 5, 7, 8, 9, 13, 16, 17, 24, 31, 32, 33, 40, 47, 63, 64):
        if bits > W:
            continue
        g = rng.integers(0, 1 << min(bits, 63), size=n, dtype=np.uint64)
        if bits == 64:
            g = g * np.uint64(2) + rng.integers(0, 2, size=n, dtype=np.uint64)
        cases[f"gaps_{bits}b"] = (np.cumsum(g) & np.uint64((1 << W) - 1)).astype(dt)
        # heavy tail: mostly small gaps plus a few of `bits` bits
        h = rng.integers(0, 4, size=n, dtype=np.uint64)
        idx = rng.integers(0, n, size=n // 50)
        h[idx] = g[idx]
        cases[f"tail_{bits}b"] = (np.cumsum(h) & np.uint64((1 << W) - 1)).astype(dt)
    for name, arr in cases.items():
        t = torch.from_numpy(arr.view(np.int32 if W == 32 else np.int64).copy()).to(tdt)
        off = torch.tensor([0, n], dtype=torch.int64)
        try:
            run_batch(B, oracle_mod, t, off, W, 0, codec=codec)
        except AssertionError as e:
            raise AssertionError(f"{name}: {e}")


@pytest.mark.parametrize("codec", CODECS)
@pytest.mark.parametrize("W", [32, 64])
def test_batch_ragged(B, oracle_mod, W, codec):
    counts = streams.log_uniform_counts(300, 6, 14, W, seed=5)
    counts[0] = 0
    counts[5] = 0
    counts[6] = 1
    counts[7] = 128
    counts[8] = 129
    counts[299] = 0
    ids, off = streams.batch_of_streams(counts, 16.0, seed=5, W=W)
    for thr in (0, 1024):
        run_batch(B, oracle_mod, ids, off, W, thr, codec=codec)
    # unaligned buffer starts (odd element offsets) exercise the scalar load/store path
    ids2, off2 = streams.batch_of_streams(torch.tensor([3, 130, 257, 1, 1000]), 2.0, seed=6, W=W)
    run_batch(B, oracle_mod, ids2, off2, W, 0, codec=codec)


@pytest.mark.parametrize("W", [32, 64])
def test_batch_alignments_and_many_buffers(B, oracle_mod, W):
    """Buffers that start at every element alignment (decode writes aligned windows shifted through the
    quad; encode stages unaligned chunks), blocks on the slow paths inside a batch, buffers that straddle
    tiles, and more buffers than one round of the plan kernels' scan (4096)."""
    g = torch.Generator().manual_seed(11)
    counts = torch.tensor([128 * 70 + e for e in (0, 1, 2, 3, 5, 6, 7, 9)] + [257, 3, 0, 129, 8191, 64 * 128, 1, 127])
    ids, off = streams.batch_of_streams(counts, 2.0, seed=9, W=W)
    ids = ids.clone()
    lo, hi = int(off[3]), int(off[4])                     # one buffer of incompressible values: blocks over the image cap
    ids[lo:hi] = torch.randint(-(2 ** 31), 2 ** 31 - 1, (hi - lo,), generator=g, dtype=torch.int64).to(ids.dtype) if W == 32 \
        else torch.randint(-(2 ** 62), 2 ** 62, (hi - lo,), generator=g, dtype=torch.int64)
    lo, hi = int(off[5]), int(off[6])                     # outliers: exceptions in most blocks
    sel = torch.rand(hi - lo, generator=g) < 0.02
    ids[lo:hi][sel] += 1 << 20
    for thr in (0, 1024):
        for codec in CODECS:
            run_batch(B, oracle_mod, ids, off, W, thr, codec=codec)
    # 9000 buffers: the one-CTA plan + block-table chain; 5000 and 8192: the fused plan of up to 8192 buffers
    # (two rounds of its decode-side scan, and the limit itself)
    for n_buf in (9000, 5000, 8192):
        many = torch.randint(0, 300, (n_buf,), generator=g)
        ids2, off2 = streams.batch_of_streams(many, 16.0, seed=10, W=W)
        for thr in (0, 1024):
            for codec in CODECS:
                run_batch(B, oracle_mod, ids2, off2, W, thr, codec=codec)


@pytest.mark.parametrize("codec", CODECS)
def test_tiny_rmat_config1(B, oracle_mod, codec):
    """BASELINE config 1: scale 12, 8 roots, 4 buffers by v mod 4, threshold 0, single + batch API."""
    G = rmat.Graph(12, 16, seed=1)
    for root in G.roots(8, seed=1):
        for f in G.bfs_frontiers(root):
            vals, off = streams.split_mod(f, 4)
            ids = streams.as_ids(vals, 32)
            run_batch(B, oracle_mod, ids, off, 32, 0, codec=codec)
            for q in range(4):
                run_single(B, oracle_mod, ids[int(off[q]):int(off[q + 1])].clone(), 32, 0, codec=codec)


@pytest.mark.parametrize("codec", CODECS)
def test_streams_config2_reduced(B, oracle_mod, codec):
    """config 2 recipes at 2^18 IDs (several thousand blocks, oracle in seconds)."""
    n = (1 << 18) + 37
    for mean, outl in ((2.0, 0.0), (256.0, 0.0), (256.0, 0.01)):
        for W in (32, 64):
            t = streams.gap_stream(n, mean, seed=2, W=W, outlier_frac=outl)
            run_batch(B, oracle_mod, t, torch.tensor([0, n], dtype=torch.int64), W, 0, codec=codec)
            run_single(B, oracle_mod, t, W, 0, codec=codec)


def test_errors_reported_on_device(B):
    dev = torch.device("cuda")
    t = streams.gap_stream(5000, 16.0, seed=3, W=32).to(dev)
    ws = torch.empty(B.workspace_bytes(5000, 1, 32), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    nbytes = torch.zeros(1, dtype=torch.int64, device=dev)
    small = torch.full((256 + 64,), 0xCD, dtype=torch.uint8, device=dev)
    B.lib().bfsc_compress(t.data_ptr(), 5000, 32, 0, small.data_ptr(), 256, nbytes.data_ptr(), ws.data_ptr(),
                          ws.numel(), status.data_ptr(), None)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_DST_TOO_SMALL
    assert bool((small[256:] == 0xCD).all())
    # corrupt stream -> BFSC_ERR_CORRUPT, no crash
    out = torch.empty(B.compress_bound(5000, 32), dtype=torch.uint8, device=dev)
    status.zero_()
    B.compress(t, 5000, 32, 0, out, nbytes, ws, status)
    torch.cuda.synchronize()
    total = int(nbytes.item())
    back = torch.empty(5000, dtype=torch.int32, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    for pos, val in ((0, 0x41), (5, 64), (36, 0)):
        bad = out.clone()
        bad[pos] = val
        status.zero_()
        B.decompress(bad, total, 32, back, n_out, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == B.ERR_CORRUPT, pos
    first_blk = 16 * int(out[32:36].cpu().numpy().view(np.uint32)[0])
    bad = out.clone()
    bad[first_blk + 8] = 33
    status.zero_()
    B.decompress(bad, total, 32, back, n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_CORRUPT
    # ids capacity too small
    status.zero_()
    B.decompress(out, total, 32, back[:100], n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_DST_TOO_SMALL


def test_batch_of_many_streams_rejects_corrupt_headers(B):
    """Batches of >= 512 streams read their headers through k_dec_headers (gathered by the whole GPU, then parsed
    by the one-CTA plan): the same rejections as the direct path (FORMAT.md §4), no crash, nothing decoded
    beyond capacity; and an intact batch of that size still round-trips."""
    dev = torch.device("cuda")
    W = 32
    counts = torch.randint(0, 600, (700,), generator=torch.Generator().manual_seed(5))
    ids, off = streams.batch_of_streams(counts, 16.0, seed=11, W=W)
    n, n_buf = ids.numel(), counts.numel()
    out = torch.empty(B.batch_compress_bound(counts.tolist(), W), dtype=torch.uint8, device=dev)
    out_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress_batch(ids.to(dev), off.to(dev), n_buf, W, 1024, out, out_off, ws, status)
    back = torch.full((n + 4,), -1, dtype=ids.dtype, device=dev)
    id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    B.decompress_batch(out, out_off, n_buf, W, back, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and torch.equal(back[:n].cpu(), ids) and torch.equal(id_off.cpu(), off)
    starts = out_off.cpu()
    for which, (rel, val) in ((3, (0, 0x41)), (350, (5, 64)), (699, (4, 9)), (512, (17, 0xFF))):   # magic, W, version, total_bytes
        bad = out.clone()
        bad[int(starts[which]) + rel] = val
        status.zero_()
        back.fill_(-1)
        B.decompress_batch(bad, out_off, n_buf, W, back, id_off, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == B.ERR_CORRUPT, which
        assert bool((back[n:] == -1).all())
    bad_off = out_off.clone()
    bad_off[100] += 8                                        # a stream that does not start on a 16-byte boundary
    status.zero_()
    B.decompress_batch(out, bad_off, n_buf, W, back, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_CORRUPT


@pytest.mark.parametrize("W", [32, 64])
def test_chained_decode_plan(B, oracle_mod, W):
    """Batches of >= 3072 streams are planned by k_dec_planchain (streams dealt out over the CTAs, prefixes from the
    lower tickets' published sums). Covered here: a batch with empty, RAW and one long stream (over 1024 blocks: written
    by the whole CTA); the same call replayed from a CUDA graph (same tag every replay: the tile kernel clears the states
    behind the plan) with a different, shorter batch decoded through the same workspace in between; rejected headers
    (status, nothing decoded, all ID offsets zero); the ID capacity exceeded; decode into frontier bitmaps."""
    dev = torch.device("cuda")
    g = torch.Generator().manual_seed(17 + W)
    counts = torch.randint(0, 400, (3500,), generator=g)
    counts[5] = 0
    counts[1777] = 150000                                   # 1172 blocks
    counts[3499] = 129
    ids, off = streams.batch_of_streams(counts, 16.0, seed=13, W=W)
    n, n_buf = ids.numel(), counts.numel()
    ref, ref_off = oracle_mod.compress_batch(_np(ids, W), off.numpy().astype(np.uint64), 256)
    d_in = torch.from_numpy(np.concatenate([ref, np.zeros(16, np.uint8)])).to(dev)
    d_off = torch.from_numpy(ref_off.astype(np.int64)).to(dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    back = torch.full((n + 4,), -1, dtype=ids.dtype, device=dev)
    id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    B.decompress_batch(d_in, d_off, n_buf, W, back, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and torch.equal(back[:n].cpu(), ids) and torch.equal(id_off.cpu(), off)
    assert bool((back[n:] == -1).all())
    # a second, shorter batch of many streams (its own tag, the same workspace), also the one captured below
    counts2 = torch.randint(1, 200, (3100,), generator=g)
    ids2, off2 = streams.batch_of_streams(counts2, 4.0, seed=14, W=W)
    ref2, ref2_off = oracle_mod.compress_batch(_np(ids2, W), off2.numpy().astype(np.uint64), 0)
    d_in2 = torch.from_numpy(np.concatenate([ref2, np.zeros(16, np.uint8)])).to(dev)
    d_off2 = torch.from_numpy(ref2_off.astype(np.int64)).to(dev)
    back2 = torch.full((ids2.numel() + 4,), -1, dtype=ids.dtype, device=dev)
    id_off2 = torch.zeros(counts2.numel() + 1, dtype=torch.int64, device=dev)
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        B.decompress_batch(d_in2, d_off2, counts2.numel(), W, back2, id_off2, ws, status)      # (warm-up outside the capture)
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            B.decompress_batch(d_in2, d_off2, counts2.numel(), W, back2, id_off2, ws, status)
    for rep in range(4):
        back2.fill_(-1); id_off2.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert int(status.item()) == 0 and torch.equal(back2[:ids2.numel()].cpu(), ids2) and torch.equal(id_off2.cpu(), off2), rep
        if rep == 1:                                        # another call through the same workspace between two replays
            back.fill_(-1)
            B.decompress_batch(d_in, d_off, n_buf, W, back, id_off, ws, status)
            torch.cuda.synchronize()
            assert int(status.item()) == 0 and torch.equal(back[:n].cpu(), ids)
    # rejected headers in the first, a middle and the last slice; a stream off its 16-byte boundary
    for which, (rel, val) in ((0, (0, 0x41)), (1777, (5, 64 if W == 32 else 32)), (3499, (4, 9)), (2000, (17, 0xFF))):
        bad = d_in.clone()
        bad[int(ref_off[which]) + rel] = val
        status.zero_(); back.fill_(-1); id_off.fill_(7)
        B.decompress_batch(bad, d_off, n_buf, W, back, id_off, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == B.ERR_CORRUPT, which
        assert bool((back == -1).all()) and not bool(id_off.any()), which
    status.zero_(); back.fill_(-1)
    small = torch.full((n - 1,), -1, dtype=ids.dtype, device=dev)              # one ID short
    B.decompress_batch(d_in, d_off, n_buf, W, small, id_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_DST_TOO_SMALL and bool((small == -1).all()) and not bool(id_off.any())
    # two such calls at the same time on two streams (own workspaces and outputs; the plans' CTAs interleave on the device)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    ws_b = torch.empty_like(ws)
    back_b = torch.full_like(back, -1)
    id_off_b = torch.zeros_like(id_off)
    status.zero_()
    torch.cuda.synchronize()
    for rep in range(20):
        with torch.cuda.stream(s1):
            B.decompress_batch(d_in, d_off, n_buf, W, back, id_off, ws, status)
        with torch.cuda.stream(s2):
            B.decompress_batch(d_in, d_off, n_buf, W, back_b, id_off_b, ws_b, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and torch.equal(back[:n].cpu(), ids) and torch.equal(back_b[:n].cpu(), ids)
    assert torch.equal(id_off.cpu(), off) and torch.equal(id_off_b.cpu(), off)
    # the same streams into frontier bitmaps (the bitmap sink behind the same plan)
    lo = int(_np(ids, W).min())
    n_bits = int(_np(ids, W).max()) - lo + 1
    if n_bits <= (1 << 27):
        words = (n_bits + 127) // 128 * 4
        d_fr = torch.zeros(words, dtype=torch.int32, device=dev)
        d_vis = torch.zeros(words, dtype=torch.int32, device=dev)
        n_dec = torch.zeros(1, dtype=torch.int64, device=dev)
        status.zero_()
        B.decompress_batch_to_frontier(d_in, d_off, n_buf, W, lo, d_fr, d_vis, n_bits, n_dec, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == 0 and int(n_dec.item()) == n
        exp = np.zeros(words * 32, dtype=bool)
        exp[(_np(ids, W).astype(np.uint64) - np.uint64(lo)).astype(np.int64)] = True
        exp_words = np.packbits(exp.reshape(-1, 32), axis=1, bitorder="little").view(np.uint32).reshape(-1)
        assert np.array_equal(d_fr.cpu().numpy().view(np.uint32), exp_words)
        assert np.array_equal(d_vis.cpu().numpy().view(np.uint32), exp_words)


def test_u64_wide_gap_blocks(B, oracle_mod):
    """u64 blocks whose deltas fit 32 bits but whose image does not fit the encoder's 288-byte slot (17 < b <= 32: gaps of
    2^17 .. 2^32 between sorted 64-bit IDs) are packed straight to the output once the tile's offsets are known, and the
    decoder stages them up to b = 32. Single stream over many tiles (k_enc_tiles<64, 0>, tickets), a batch on the general
    path (k_enc_tiles<64, 1>) with narrow and wide buffers side by side, exceptions on top (b + outliers), and the b = 32 /
    b = 33 boundary of the decoder's staging; bytes against the oracle."""
    rng = np.random.default_rng(64)
    n = 128 * 64 * 700 + 77                                  # 700 tiles: every CTA draws tickets
    for bits in (18, 21, 27, 32):
        g = rng.integers(1 << (bits - 1), 1 << bits, size=n, dtype=np.uint64)
        ids = np.cumsum(g).astype(np.uint64)
        t = torch.from_numpy(ids.view(np.int64).copy())
        run_single(B, oracle_mod, t, 64, 0)
    # outliers that still fit 32 bits on top of 20-bit gaps: exceptions inside directly emitted blocks
    g = rng.integers(1 << 19, 1 << 20, size=n, dtype=np.uint64)
    idx = rng.integers(0, n, size=n // 100)
    g[idx] = rng.integers(1 << 30, 1 << 32, size=idx.size, dtype=np.uint64)
    run_single(B, oracle_mod, torch.from_numpy(np.cumsum(g).astype(np.uint64).view(np.int64).copy()), 64, 0)
    # a batch on the general path: narrow, wide (b = 22), b = 32, b = 33 (wide deltas: the slow path) and ragged buffers
    parts, counts = [], []
    for k, (cnt, bits) in enumerate(((128 * 300 + 5, 4), (128 * 200 + 1, 22), (999, 22), (128 * 150, 32), (128 * 90 + 64, 33), (128 * 400, 19), (3, 25), (128 * 100 + 127, 8))):
        gg = rng.integers(1 << (bits - 1), 1 << bits, size=cnt, dtype=np.uint64)
        parts.append(np.cumsum(gg).astype(np.uint64) + np.uint64(k) * np.uint64(1 << 50))
        counts.append(cnt)
    ids = np.concatenate(parts)
    off = torch.zeros(len(counts) + 1, dtype=torch.int64)
    off[1:] = torch.cumsum(torch.tensor(counts), 0)
    t = torch.from_numpy(ids.view(np.int64).copy())
    for thr in (0, 1024):
        run_batch(B, oracle_mod, t, off, 64, thr)


def test_host_api_roundtrip(B, oracle_mod):
    dev = torch.device("cuda")
    for W in (32, 64):
        n = 50_000
        t = streams.gap_stream(n, 16.0, seed=4, W=W).pin_memory()
        scratch = torch.empty(B.host_scratch_bytes(n, W) + 256, dtype=torch.uint8, device=dev)
        h_out = torch.empty(B.compress_bound(n, W), dtype=torch.uint8).pin_memory()
        nbytes = B.compress_host(t, W, 0, h_out, scratch)
        ref = oracle_mod.compress(_np(t, W), 0)
        assert nbytes == len(ref) and np.array_equal(h_out[:nbytes].numpy(), ref)
        h_back = torch.empty(n, dtype=t.dtype).pin_memory()
        assert B.decompress_host(h_out, nbytes, W, h_back, scratch) == n
        assert torch.equal(h_back, t)


@pytest.mark.parametrize("codec", CODECS)
def test_rmat_config3_reduced(B, oracle_mod, codec):
    """config 3 recipe at scale 16: per-level frontiers, 16 buffers by contiguous vertex range, one
    batched call per level, 1 KB raw threshold (first/last levels go RAW or empty)."""
    G = rmat.Graph(16, 16, seed=3)
    for root in G.roots(2, seed=3):
        for f in G.bfs_frontiers(root):
            vals, off = streams.split_block(f, 16, 1 << 16)
            run_batch(B, oracle_mod, streams.as_ids(vals, 32), off, 32, 1024, codec=codec)


@pytest.mark.parametrize("codec", CODECS)
def test_rmat_config4_reduced(B, oracle_mod, codec):
    """config 4 recipe at scale 16: u64 IDs, 64 destination buffers (8x8 partition read as a 64-way
    block partition), 1 KB threshold."""
    G = rmat.Graph(16, 16, seed=4)
    for root in G.roots(2, seed=4):
        for f in G.bfs_frontiers(root):
            vals, off = streams.split_block(f, 64, 1 << 16)
            run_batch(B, oracle_mod, streams.as_ids(vals, 64), off, 64, 1024, codec=codec)


def test_rmat_config3_full_size_all_roots(B, oracle_mod):
    """config 3 at its BASELINE size (R-MAT scale 22, 16 buffers per level, u32, 1 KB threshold), ALL 16 roots:
    every level's batch byte-for-byte against the oracle (the graph and the BFS are built on the GPU by the
    workload module; the codec calls are the ones report.py times)."""
    G = rmat.Graph(22, 16, seed=3, device=torch.device("cuda"))
    roots = G.roots(16, seed=3)
    assert len(roots) == 16
    for root in roots:
        total = 0
        for f in G.bfs_frontiers(root):
            vals, off = streams.split_block(f, 16, 1 << 22)
            run_batch(B, oracle_mod, streams.as_ids(vals, 32).cpu(), off.cpu(), 32, 1024)
            total += vals.numel()
        assert total > 2_000_000                              # the giant component
    del G
    torch.cuda.empty_cache()


def test_rmat_config4_full_size_three_roots(B, oracle_mod):
    """config 4 at its BASELINE size (R-MAT scale 25, 64 buffers per level, u64, 1 KB threshold), three of the 8 roots
    (the graph is built once)."""
    G = rmat.Graph(25, 16, seed=4, device=torch.device("cuda"))
    for root in G.roots(8, seed=4)[:3]:
        total = 0
        for f in G.bfs_frontiers(root):
            vals, off = streams.split_block(f, 64, 1 << 25)
            run_batch(B, oracle_mod, streams.as_ids(vals, 64).cpu(), off.cpu(), 64, 1024)
            total += vals.numel()
        assert total > 16_000_000
    del G
    torch.cuda.empty_cache()


@pytest.mark.parametrize("W", [32, 64])
def test_sweep_config5_reduced(B, oracle_mod, W):
    """config 5 recipe: single buffers of 1 KB .. 4 MB (powers of 4), gap means 1, 16, 4096; plus a batch
    of 4096 buffers of 256 B .. 64 KB (log-uniform sizes), thresholds 0 and 1024."""
    for k in range(5, 12):
        n = (4 ** k) // (W // 8)
        for mean in (1.0, 16.0, 4096.0):
            if W == 32 and n * mean >= 2 ** 32:
                continue                                   # exceeds the u32 ID space
            t = streams.gap_stream(n, mean, seed=5, W=W)
            run_batch(B, oracle_mod, t, torch.tensor([0, n], dtype=torch.int64), W, 0)
    if W == 32:
        counts = streams.log_uniform_counts(4096, 8, 16, W, seed=5)
        ids, off = streams.batch_of_streams(counts, 16.0, seed=5, W=W)
        for thr in (0, 1024):
            run_batch(B, oracle_mod, ids, off, W, thr)


def test_random_batches_soak(B, oracle_mod):
    """Seeded random batches (buffer counts 1..6000, sizes 0..3 M IDs, u32/u64, gaps of mean 1..70000, optional
    outliers, both thresholds) byte-for-byte against the oracle: shakes the hand-overs between the warps of the
    encoder (tickets, look-back, deferred copy-out) and the plan / block-table kernels under varied timing."""
    g = torch.Generator().manual_seed(20261104)
    for _ in range(150):
        W = 32 if torch.rand(1, generator=g) < 0.6 else 64
        kind = int(torch.randint(0, 4, (1,), generator=g))
        if kind == 0:
            nbuf, hi = int(torch.randint(1, 40, (1,), generator=g)), 200000
        elif kind == 1:
            nbuf, hi = int(torch.randint(1000, 6000, (1,), generator=g)), 400
        elif kind == 2:
            nbuf, hi = int(torch.randint(1, 300, (1,), generator=g)), 20000
        else:
            nbuf, hi = 1, 3000000
        counts = torch.randint(0, hi, (nbuf,), generator=g)
        mean = [1.0, 2.0, 16.0, 256.0, 4096.0, 70000.0][int(torch.randint(0, 6, (1,), generator=g))]
        ids, off = streams.batch_of_streams(counts, mean, seed=int(torch.randint(0, 1 << 30, (1,), generator=g)), W=W)
        if torch.rand(1, generator=g) < 0.3 and ids.numel() > 10:
            sel = torch.rand(ids.numel(), generator=g) < 0.01
            ids = ids.clone()
            ids[sel] += 1 << 22
        thr = [0, 1024][int(torch.randint(0, 2, (1,), generator=g))]
        run_batch(B, oracle_mod, ids, off, W, thr)
        if nbuf == 1:
            run_single(B, oracle_mod, ids, W, thr)


@pytest.mark.parametrize("W", [32, 64])
def test_calls_replay_from_a_cuda_graph(B, oracle_mod, W):
    """include/bfsc.h: the device calls only enqueue kernels on the given stream (no allocation, no
    synchronisation), so a caller may capture them in a CUDA graph. One graph holding compress_batch +
    decompress_batch + compress + decompress is replayed on three different contents of the same buffers;
    every replay must give the oracle's bytes and the input back."""
    dev = torch.device("cuda")
    counts = torch.tensor([5000, 0, 129, 40000, 1, 300, 12800])
    n, n_buf = int(counts.sum()), counts.numel()
    off = torch.zeros(n_buf + 1, dtype=torch.int64)
    off[1:] = torch.cumsum(counts, 0)
    dt = torch.int32 if W == 32 else torch.int64
    d_ids = torch.zeros(n + 4, dtype=dt, device=dev)
    d_off = off.to(dev)
    cap = B.batch_compress_bound(counts.tolist(), W)
    out = torch.zeros(cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    back = torch.zeros(n + 4, dtype=dt, device=dev)
    id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
    cap1 = B.compress_bound(n, W)
    out1 = torch.zeros(cap1, dtype=torch.uint8, device=dev)
    nbytes1 = torch.zeros(1, dtype=torch.int64, device=dev)
    back1 = torch.zeros(n + 4, dtype=dt, device=dev)
    n_out1 = torch.zeros(1, dtype=torch.int64, device=dev)

    def calls():
        B.compress_batch(d_ids, d_off, n_buf, W, 1024, out, out_off, ws, status)
        B.decompress_batch(out, out_off, n_buf, W, back, id_off, ws, status)
        B.compress(d_ids, n, W, 0, out1, nbytes1, ws, status)
        B.decompress(out1, cap1, W, back1, n_out1, ws, status)

    calls()                                                  # first use outside the capture (one-time attribute set-up)
    torch.cuda.synchronize()
    side = torch.cuda.Stream(device=dev)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            calls()
    torch.cuda.synchronize()
    for rep, mean in enumerate((2.0, 300.0, 70000.0)):
        ids, off2 = streams.batch_of_streams(counts, mean, seed=100 + rep, W=W)
        assert torch.equal(off2, off)
        d_ids[:n] = ids.to(dev)
        out.zero_(); back.fill_(-1); out1.zero_(); back1.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        assert int(status.item()) == 0
        ref, ref_off = oracle_mod.compress_batch(_np(ids, W), off.numpy().astype(np.uint64), 1024)
        assert np.array_equal(out_off.cpu().numpy().astype(np.uint64), ref_off)
        assert np.array_equal(out[:len(ref)].cpu().numpy(), ref)
        assert torch.equal(back[:n].cpu(), ids) and torch.equal(id_off.cpu(), off)
        ref1 = oracle_mod.compress(_np(ids, W), 0)
        assert int(nbytes1.item()) == len(ref1) and np.array_equal(out1[:len(ref1)].cpu().numpy(), ref1)
        assert int(n_out1.item()) == n and torch.equal(back1[:n].cpu(), ids)


def _full_size(B, oracle_mod, ids, W, codec=PFOR):
    """One large single stream through bfsc_compress / bfsc_decompress (the launch configuration bench.py and
    report.py time): decoded IDs equal the input; the WHOLE compressed stream memcmp-equal to the serial oracle's;
    and, independently of the oracle, the directory walk (strictly increasing, sizes recomputed from the block
    headers, total = header + directory + blocks)."""
    dev = torch.device("cuda")
    n = ids.numel()
    E = W // 8
    cap = B.compress_bound(n, W)
    out = torch.empty(cap, dtype=torch.uint8, device=dev)
    nbytes = torch.zeros(1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    if codec == PFOR:
        B.compress(ids, n, W, 0, out, nbytes, ws, status)
    else:
        B.compress_codec(codec, ids, n, W, 0, out, nbytes, ws, status)
    back = torch.empty(n, dtype=ids.dtype, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    B.decompress(out, cap, W, back, n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and int(n_out.item()) == n
    assert torch.equal(back, ids)
    del back
    total = int(nbytes.item())
    s = out[:total].cpu().numpy()
    del out
    nb = (n + 127) // 128
    assert s[:4].tobytes() == b"BFSC" and s[4] == 1 and s[5] == W and s[6] == codec
    assert int(s[8:16].view(np.uint64)[0]) == n and int(s[16:24].view(np.uint64)[0]) == total
    assert int(s[24:28].view(np.uint32)[0]) == nb
    d = s[32:32 + 4 * (nb + 1)].view(np.uint32).astype(np.int64)
    assert d[0] * 16 == 32 + ((4 * (nb + 1) + 15) // 16) * 16 and d[nb] * 16 == total
    b = s[d[:-1] * 16 + 8].astype(np.int64)
    ne = s[d[:-1] * 16 + 9].astype(np.int64)
    exc = np.where(ne > 0, ((((ne + E - 1) // E) * E + E * ne + 15) // 16) * 16, 0)
    assert np.array_equal((d[1:] - d[:-1]) * 16, 16 + 16 * b + exc)
    host = ids.cpu().numpy().view(np.uint32 if W == 32 else np.uint64)
    ref = oracle_mod.compress(host, 0, codec=codec)              # serial oracle, whole stream
    assert len(ref) == total
    if not np.array_equal(s, ref):
        bad = int(np.nonzero(s != ref)[0][0])
        raise AssertionError(f"compressed bytes differ from the oracle at byte {bad} of {total}")


@pytest.mark.parametrize("codec", CODECS)
def test_config2_full_size(B, oracle_mod, codec):
    """BASELINE config 2 at its full size (3 streams of 2^24 IDs, the launch configuration bench.py times): every
    byte of every stream against the serial oracle, under both encoder rules."""
    for sub, (mean, outl) in enumerate(((2.0, 0.0), (256.0, 0.0), (256.0, 0.01))):
        ids = streams.gap_stream(1 << 24, mean, seed=2, W=32, outlier_frac=outl, sub=sub, device=torch.device("cuda"))
        _full_size(B, oracle_mod, ids, 32, codec=codec)


def test_config5_large_cells_full(B, oracle_mod):
    """The upper half of the config-5 sweep, every byte against the serial oracle: single buffers of 16 MB, 64 MB
    and 256 MB (u32 and u64; gap means 1, 16, 4096 where the IDs fit the type), plus ragged sizes around 2^23 IDs
    (the kernel is then several waves deep: every warp draws many tiles, look-backs span hundreds of super-tiles)."""
    dev = torch.device("cuda")
    for W in (32, 64):
        for k in (12, 13, 14):
            n = (4 ** k) // (W // 8)
            for mean in (1.0, 16.0, 4096.0):
                if W == 32 and n * mean >= 2 ** 32:
                    continue                               # exceeds the u32 ID space
                _full_size(B, oracle_mod, streams.gap_stream(n, mean, seed=5, W=W, device=dev), W)
                torch.cuda.empty_cache()
        _full_size(B, oracle_mod, streams.gap_stream((1 << 23) + 77, 256.0, seed=6, W=W, outlier_frac=0.01, device=dev), W)
        _full_size(B, oracle_mod, streams.gap_stream((1 << 23) - 129, 2.0, seed=7, W=W, device=dev), W, codec=BP128)


def test_config5_largest_buffers_full(B, oracle_mod):
    """The 1 GB ends of the config-5 sweep (2^28 u32 IDs with gaps of 1; 2^27 u64 IDs with gaps of mean 4096): tile
    counts, offsets and directory entries far beyond the 2^24-ID case (offsets over 2^32 / 16 are still exact)."""
    dev = torch.device("cuda")
    _full_size(B, oracle_mod, streams.gap_stream(1 << 28, 1.0, seed=5, W=32, device=dev), 32)
    torch.cuda.empty_cache()
    _full_size(B, oracle_mod, streams.gap_stream(1 << 27, 4096.0, seed=5, W=64, device=dev), 64)
    torch.cuda.empty_cache()


def test_decode_tma_staging_variant(B, oracle_mod, monkeypatch):
    """BFSC_DEC_STAGING=tma: single-stream decode stages every warp batch with one bulk copy (TMA) into a two-stage
    ring instead of per-lane cp.async (measured, slower, kept selectable). Same results: edge sizes,
    exceptions, blocks over the staged size, corrupt streams."""
    monkeypatch.setenv("BFSC_DEC_STAGING", "tma")
    for W in (32, 64):
        for n in (0, 1, 127, 128, 129, 1000, 128 * 300 + 5, (1 << 20) + 77):
            for mean, outl in ((2.0, 0.0), (256.0, 0.01), (70000.0, 0.0)):
                run_single(B, oracle_mod, streams.gap_stream(n, mean, seed=13, W=W, outlier_frac=outl), W, 0)
    rng = np.random.default_rng(5)
    x = np.cumsum(rng.integers(0, 1 << 26, size=128 * 20 + 3, dtype=np.uint64)).astype(np.uint32)   # b = 26: blocks over the staged size
    run_single(B, oracle_mod, torch.from_numpy(x.view(np.int32).copy()), 32, 0)
    test_errors_reported_on_device(B)


def test_exclusive_flag_same_bytes(B, oracle_mod):
    """BFSC_CODEC_FLAG_EXCLUSIVE (static first tiles, include/bfsc.h) changes the schedule, not the bytes: single and
    batch calls, both encoder rules, against the oracle."""
    dev = torch.device("cuda")
    for W in (32, 64):
        n = 128 * 64 * 700 + 99                                  # more tiles than one resident wave of CTAs
        x = streams.gap_stream(n, 16.0, seed=41, W=W, outlier_frac=0.01)
        for codec in CODECS:
            ref = oracle_mod.compress(_np(x, W), 0, codec=codec)
            cap = B.compress_bound(n, W)
            out = torch.empty(cap, dtype=torch.uint8, device=dev)
            nbytes = torch.zeros(1, dtype=torch.int64, device=dev)
            ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
            status = torch.zeros(1, dtype=torch.int32, device=dev)
            B.compress_codec(codec | B.CODEC_FLAG_EXCLUSIVE, x.to(dev), n, W, 0, out, nbytes, ws, status)
            torch.cuda.synchronize()
            assert int(status.item()) == 0 and int(nbytes.item()) == len(ref)
            assert np.array_equal(out[:len(ref)].cpu().numpy(), ref)
        counts = streams.log_uniform_counts(500, 6, 15, W, seed=42)
        ids, off = streams.batch_of_streams(counts, 16.0, seed=42, W=W)
        ref, ref_off = oracle_mod.compress_batch(_np(ids, W), off.numpy().astype(np.uint64), 1024)
        out = torch.empty(B.batch_compress_bound(counts.tolist(), W), dtype=torch.uint8, device=dev)
        out_off = torch.zeros(counts.numel() + 1, dtype=torch.int64, device=dev)
        ws = torch.empty(B.workspace_bytes(ids.numel(), counts.numel(), W), dtype=torch.uint8, device=dev)
        status = torch.zeros(1, dtype=torch.int32, device=dev)
        B.compress_batch_codec(PFOR | B.CODEC_FLAG_EXCLUSIVE, ids.to(dev), off.to(dev), counts.numel(), W, 1024, out, out_off, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == 0 and np.array_equal(out_off.cpu().numpy().astype(np.uint64), ref_off)
        assert np.array_equal(out[:len(ref)].cpu().numpy(), ref)


def test_two_compress_calls_run_concurrently(B, oracle_mod):
    """Two bfsc_compress calls on two CUDA streams of one device at the same time, 200 times (every tile is
    drawn by ticket: no co-residency assumption), each with its own workspace; bytes vs the
    oracle every time (the inputs alternate, so a stale result cannot pass)."""
    dev = torch.device("cuda")
    W = 32
    n = (1 << 21) + 333
    xs = [streams.gap_stream(n, m, seed=31 + i, W=W, outlier_frac=o, device=dev) for i, (m, o) in enumerate(((2.0, 0.0), (256.0, 0.01)))]
    refs = [oracle_mod.compress(_np(x, W), 0) for x in xs]
    cap = B.compress_bound(n, W)
    outs = [torch.empty(cap, dtype=torch.uint8, device=dev) for _ in range(2)]
    nbs = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(2)]
    wss = [torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev) for _ in range(2)]
    sts = [torch.zeros(1, dtype=torch.int32, device=dev) for _ in range(2)]
    cs = [torch.cuda.Stream(device=dev) for _ in range(2)]
    torch.cuda.synchronize()
    for rep in range(200):
        for k in range(2):
            with torch.cuda.stream(cs[k]):
                B.compress(xs[(k + rep) % 2], n, W, 0, outs[k], nbs[k], wss[k], sts[k])
        if rep % 20 == 19 or rep < 2:
            torch.cuda.synchronize()
            for k in range(2):
                ref = refs[(k + rep) % 2]
                assert int(sts[k].item()) == 0 and int(nbs[k].item()) == len(ref)
                assert np.array_equal(outs[k][:len(ref)].cpu().numpy(), ref), (rep, k)
    torch.cuda.synchronize()


def _mutations(rng, good, W, n_mut):
    """Seeded single-byte (and a few two-byte) mutations of a stream, biased to the bytes a decoder reads as
    structure: stream header, directory, block headers, exception areas."""
    nb = int(good[24:28].view(np.uint32)[0])
    d = good[32:32 + 4 * (nb + 1)].view(np.uint32).astype(np.int64)
    spots = list(range(4, 28)) + list(range(32, 32 + 4 * (nb + 1)))
    for k in range(nb):
        o = 16 * int(d[k])
        b, ne = int(good[o + 8]), int(good[o + 9])
        spots += [o + 8, o + 9]
        if ne:
            spots += list(range(o + 16 + 16 * b, o + 16 + 16 * b + ne + 2))
    spots = [x for x in spots if x < len(good)]
    for _ in range(n_mut):
        s = good.copy()
        for _ in range(1 if rng.random() < 0.8 else 2):
            p = spots[int(rng.integers(0, len(spots)))]
            s[p] = int(rng.integers(0, 256)) if rng.random() < 0.5 else (int(s[p]) + int(rng.choice([1, -1, 2, 16, 128]))) % 256
        yield s


@pytest.mark.parametrize("W", [32, 64])
def test_decoder_fuzz_matches_oracle_verdict(B, oracle_mod, W):
    """FORMAT.md §4 on the GPU, single and batch calls, staged fast path and wide (> 336 B) blocks: for seeded
    mutations of header, directory, block-header and exception bytes the device status equals the oracle's verdict
    (OK / CORRUPT / DST_TOO_SMALL); when both accept, the IDs are equal; guard elements behind the output are never
    written; truncated input is rejected."""
    dev = torch.device("cuda")
    rng = np.random.default_rng(1000 + W)
    dt = np.uint32 if W == 32 else np.uint64
    tdt = torch.int32 if W == 32 else torch.int64
    n = 128 * 9 + 50
    g = rng.integers(1, 40, size=n).astype(np.uint64)
    g[rng.integers(0, n, size=40)] = np.uint64(1) << np.uint64(21)                       # exceptions in most blocks
    g[128 * 4:128 * 6] = rng.integers(1 << 24, 1 << 26, size=256).astype(np.uint64)      # two blocks over the staged size (b = 26)
    x = (np.cumsum(g) & np.uint64((1 << W) - 1)).astype(dt)
    good = oracle_mod.compress(x, 0)
    cap_ids = n + 64
    ws = torch.empty(B.workspace_bytes(cap_ids + 200, 2, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    cap_b = cap_ids + 200                                            # the batch call decodes a 200-ID stream in front of the mutated one
    back = torch.empty(cap_b + 16, dtype=tdt, device=dev)
    id_off = torch.zeros(3, dtype=torch.int64, device=dev)
    small = oracle_mod.compress(x[:200], 0)
    verdicts = {0: 0, 2: 0, 3: 0}

    def oracle_verdict(s):
        try:
            return 0, oracle_mod.decompress(s, W, capacity=cap_ids)
        except oracle_mod.OracleError as ex:
            return ex.code, None

    def check(s, in_bytes=None):
        code, ids = oracle_verdict(s if in_bytes is None else s[:in_bytes])
        d_in = torch.from_numpy(s).to(dev)
        # single call
        back.fill_(-7); status.zero_()
        B.decompress(d_in, len(s) if in_bytes is None else in_bytes, W, back[:cap_ids], n_out, ws, status)
        torch.cuda.synchronize()
        st = int(status.item())
        assert st == code, f"single: device status {st}, oracle {code}"
        assert bool((back[cap_ids:] == -7).all())
        if code == 0:
            assert int(n_out.item()) == len(ids) and np.array_equal(_np(back[:len(ids)], W), ids)
        verdicts[code] = verdicts.get(code, 0) + 1
        # batch call: [intact small stream | s]
        if in_bytes is None:
            both = torch.from_numpy(np.concatenate([small, s])).to(dev)
            offs = torch.tensor([0, len(small), len(small) + len(s)], dtype=torch.int64, device=dev)
            back.fill_(-7); status.zero_()
            B.decompress_batch(both, offs, 2, W, back[:cap_b], id_off, ws, status)
            torch.cuda.synchronize()
            st = int(status.item())
            assert st == code, f"batch: device status {st}, oracle {code}"
            assert bool((back[cap_b:] == -7).all())
            if code == 0:
                assert np.array_equal(_np(back[200:200 + len(ids)], W), ids)

    check(good)
    for s in _mutations(rng, good, W, 400):
        check(s)
    for cut in (16, 31, 32, 48, len(good) - 16, len(good) - 1):
        check(good, in_bytes=cut)
    assert verdicts[0] > 20 and verdicts[3] > 100            # the mutations reach both outcomes


# ---- FORMAT.md §9: frontier bitmaps; §8: RAW fallback ------------------------------------------------------------
FALLBACK = 0x200


def _bitmap_ids(bm_np, n_bits, id_base, W):
    """numpy, independent of both sides: the ascending IDs of the set bits."""
    bits = np.unpackbits(bm_np.view(np.uint8), bitorder="little")[:n_bits]
    v = np.nonzero(bits)[0].astype(np.uint64)
    ids = v + np.uint64(id_base & 0xFFFFFFFFFFFFFFFF)
    return (ids & np.uint64(0xFFFFFFFF)).astype(np.uint32) if W == 32 else ids


def run_bitmap(B, oracle_mod, bm_t, n_bits, W, id_base=0, thr=0, codec=PFOR, check_list=True):
    dev = torch.device("cuda")
    bm_np = bm_t.numpy().view(np.uint32)
    d_bm = bm_t.to(dev)
    cap = B.compress_bound(n_bits, W)
    out = torch.full((cap + 64,), 0xAB, dtype=torch.uint8, device=dev)
    nbytes = torch.full((1,), -1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.bitmap_workspace_bytes(n_bits, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress_bitmap(codec, d_bm, n_bits, id_base, W, thr, out, nbytes, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    total = int(nbytes.item())
    ref = oracle_mod.compress_bitmap(bm_np, n_bits, W, id_base, thr, codec)
    got = out[:total].cpu().numpy()
    assert total == len(ref), (total, len(ref))
    if not np.array_equal(got, ref):
        raise AssertionError(f"bitmap stream differs at byte {int(np.nonzero(got != ref)[0][0])} of {len(ref)}")
    assert bool((out[cap:] == 0xAB).all()), "wrote beyond capacity"
    assert torch.equal(d_bm.cpu(), bm_t), "the bitmap is an input"
    if check_list:                                   # FORMAT.md §9: it IS the stream of the ID list
        ids = _bitmap_ids(bm_np, n_bits, id_base, W)
        assert np.array_equal(ref, oracle_mod.compress(ids, thr, codec=codec))
    # decode into a bitmap that already holds other bits: OR semantics, nothing beyond n_bits touched
    words = bm_t.numel()
    old = streams.frontier_bitmap(words * 32, 0.1, seed=77)[:words].clone()
    d_back = old.to(dev)
    n_out = torch.full((1,), -1, dtype=torch.int64, device=dev)
    ws2 = torch.empty(B.workspace_bytes(max(n_bits, 1), 1, W), dtype=torch.uint8, device=dev)
    B.decompress_to_bitmap(out, total, W, id_base, d_back, n_bits, n_out, ws2, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    exp = old.numpy().view(np.uint32).copy()
    n_ref = oracle_mod.decompress_to_bitmap(ref, W, exp, n_bits, id_base)
    assert int(n_out.item()) == n_ref
    assert np.array_equal(d_back.cpu().numpy().view(np.uint32), exp)
    return total


@pytest.mark.parametrize("codec", CODECS)
@pytest.mark.parametrize("W", [32, 64])
def test_bitmap_edge_sizes(B, oracle_mod, W, codec):
    bases = (0, 12345, (1 << 32) - 100) if W == 32 else (0, (1 << 40) + 7, (1 << 64) - 50)
    for n_bits in (0, 1, 31, 32, 33, 127, 128, 129, 1000, 1023, 1024, 1025, 4096 + 7, 128 * 64 * 3 + 5):
        for dens in (0.0, 1.0, 0.5, 0.03):
            bm = streams.frontier_bitmap(n_bits, dens, seed=n_bits + 1)
            run_bitmap(B, oracle_mod, bm, n_bits, W, id_base=bases[n_bits % 3], codec=codec)
    run_bitmap(B, oracle_mod, streams.frontier_bitmap(3000, 0.05, seed=2), 3000, W, thr=4096, codec=codec)   # RAW by the threshold
    run_bitmap(B, oracle_mod, streams.frontier_bitmap(3000, 0.9, seed=2), 3000, W, thr=4096, codec=codec)


@pytest.mark.parametrize("W", [32, 64])
def test_bitmap_densities_many_tiles(B, oracle_mod, W):
    """Several tiles per CTA and a ragged tail; dense (landing area), sparse (blocks that span many words: read from
    global memory), clustered, and one block spread over the whole bitmap."""
    n_bits = (1 << 22) + 4321
    for dens, run in ((0.5, 1), (0.25, 1), (0.03, 1), (0.002, 1), (0.3, 64), (0.01, 1024)):
        run_bitmap(B, oracle_mod, streams.frontier_bitmap(n_bits, dens, seed=5, run=run), n_bits, W, id_base=3,
                   check_list=dens >= 0.25)
    run_bitmap(B, oracle_mod, streams.frontier_bitmap(n_bits, 0.00002, seed=6), n_bits, W)     # ~84 IDs: one ragged block
    run_bitmap(B, oracle_mod, streams.frontier_bitmap(n_bits, 1.0, seed=6), n_bits, W)          # full


def test_bitmap_frontier_scale24(B, oracle_mod):
    """A frontier bitmap of a scale-24 graph (2^24 vertices), a quarter of the vertices in it."""
    n_bits = 1 << 24
    total = run_bitmap(B, oracle_mod, streams.frontier_bitmap(n_bits, 0.25, seed=24), n_bits, 32, check_list=False)
    assert total < n_bits // 8 * 3                   # (gap ~4: about 3.6 bits per ID)


@pytest.mark.parametrize("W", [32, 64])
def test_bitmap_decode_rejects_ids_outside(B, oracle_mod, W):
    dev = torch.device("cuda")
    ids = _np(streams.gap_stream(5000, 3.0, seed=4, W=W), W)
    stream = oracle_mod.compress(ids, 0)
    lo, hi = int(ids.min()), int(ids.max())
    for id_base, n_bits, ok in ((lo, hi - lo + 1, True), (lo + 1, hi - lo, False), (lo, hi - lo, False), (0, hi + 1, True)):
        words = max(4, ((n_bits + 31) // 32 + 3) // 4 * 4)
        d_bm = torch.zeros(words, dtype=torch.int32, device=dev)
        d_in = torch.from_numpy(np.concatenate([stream, np.zeros(16, np.uint8)])).to(dev)
        n_out = torch.zeros(1, dtype=torch.int64, device=dev)
        status = torch.zeros(1, dtype=torch.int32, device=dev)
        ws = torch.empty(B.workspace_bytes(len(ids), 1, W), dtype=torch.uint8, device=dev)
        B.decompress_to_bitmap(d_in, len(stream), W, id_base, d_bm, n_bits, n_out, ws, status)
        torch.cuda.synchronize()
        exp = np.zeros(words, np.uint32)
        try:
            oracle_mod.decompress_to_bitmap(stream, W, exp, n_bits, id_base)
            ref_ok = True
        except oracle_mod.OracleError as e:
            ref_ok = False
            assert e.code == 2                       # DST_TOO_SMALL
        assert ref_ok == ok
        assert (int(status.item()) == 0) == ok
        if ok:
            assert np.array_equal(d_bm.cpu().numpy().view(np.uint32), exp)
        else:
            assert int(status.item()) == 2


def _fallback_single(B, oracle_mod, ids_t, W, thr=0, codec=PFOR):
    dev = torch.device("cuda")
    n = ids_t.numel()
    cap = B.compress_bound(n, W)
    d_ids = ids_t.to(dev) if n else torch.empty(4, dtype=ids_t.dtype, device=dev)
    out = torch.full((cap + 64,), 0xAB, dtype=torch.uint8, device=dev)
    nbytes = torch.full((1,), -1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress_codec(codec | FALLBACK, d_ids, n, W, thr, out, nbytes, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    total = int(nbytes.item())
    ref = oracle_mod.compress(_np(ids_t, W), thr, codec=codec | oracle_mod.FLAG_RAW_FALLBACK)
    assert total == len(ref) and total <= 32 + (n * W // 8 + 15) // 16 * 16
    assert np.array_equal(out[:total].cpu().numpy(), ref)
    assert bool((out[cap:] == 0xAB).all())
    back = torch.empty(max(n, 4), dtype=ids_t.dtype, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    B.decompress(out, total, W, back, n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and int(n_out.item()) == n
    assert torch.equal(back[:n].cpu(), ids_t)
    return int(ref[6])                                # mode byte


@pytest.mark.parametrize("codec", CODECS)
@pytest.mark.parametrize("W", [32, 64])
def test_raw_fallback_single(B, oracle_mod, W, codec):
    rng = np.random.default_rng(W + codec)
    tdt = torch.int32 if W == 32 else torch.int64
    dt = np.uint32 if W == 32 else np.uint64
    modes = set()
    for n in (0, 1, 2, 3, 127, 128, 129, 1000, 128 * 64 + 3, 128 * 64 * 40 + 77):
        rnd = torch.from_numpy(rng.integers(0, 1 << W, size=n, dtype=np.uint64, endpoint=False).astype(dt).view(
            np.int32 if W == 32 else np.int64))
        modes.add(_fallback_single(B, oracle_mod, rnd, W, codec=codec))              # incompressible: RAW
        modes.add(_fallback_single(B, oracle_mod, streams.gap_stream(n, 3.0, seed=n, W=W), W, codec=codec))
        modes.add(_fallback_single(B, oracle_mod, streams.gap_stream(n, 3.0, seed=n, W=W), W, thr=2048, codec=codec))
    assert modes == {0, codec}
    # around the tie (FORMAT.md §8: a tie goes to RAW): one block of 128 IDs with a constant gap of 2^g packs into
    # 48 + 16 + 16 (g + 1) bytes against 32 + 16 W RAW — equal at g = W - 3, smaller below, larger above
    for gap_bits in (W - 4, W - 3, W - 2, W - 1):
        v = (np.arange(128, dtype=np.uint64) * np.uint64(1 << gap_bits)) & np.uint64((1 << W) - 1 if W < 64 else 0xFFFFFFFFFFFFFFFF)
        t = torch.from_numpy(v.astype(dt).view(np.int32 if W == 32 else np.int64))
        _fallback_single(B, oracle_mod, t, W, codec=codec)


def test_raw_fallback_batch_is_unsupported_and_bitmap_follows_the_rule(B, oracle_mod):
    dev = torch.device("cuda")
    ids = streams.gap_stream(1000, 2.0, seed=1, W=32).to(dev)
    off = torch.tensor([0, 400, 1000], dtype=torch.int64, device=dev)
    out = torch.empty(B.batch_compress_bound([400, 600], 32), dtype=torch.uint8, device=dev)
    out_off = torch.zeros(3, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(1000, 2, 32), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    with pytest.raises(B.BfscError) as e:
        B.compress_batch_codec(PFOR | FALLBACK, ids, off, 2, 32, 0, out, out_off, ws, status)
    assert e.value.code == B.ERR_UNSUPPORTED
    # bitmaps: a handful of set bits far apart do not shrink (n = 1: 64 bytes against 48 RAW); dense ones do
    for W in (32, 64):
        for n_bits, dens in ((0, 0.0), (5000, 0.0002), (5000, 0.001), (1 << 20, 0.000003), (1 << 20, 0.3)):
            bm = streams.frontier_bitmap(n_bits, dens, seed=9)
            run_bitmap(B, oracle_mod, bm, n_bits, W, codec=PFOR | FALLBACK)


# ---- FORMAT.md §9, last item: decode into the next frontier against the visited bitmap (Algorithm 4 lines 10-13) ----
def _frontier_case(B, oracle_mod, ids_np, W, n_bits, id_base, thr=0, seed=0, expect_ok=True):
    dev = torch.device("cuda")
    stream = oracle_mod.compress(ids_np, thr)
    words = max(4, ((n_bits + 31) // 32 + 3) // 4 * 4)
    vis0 = streams.frontier_bitmap(words * 32, 0.4, seed=seed + 1)[:words].numpy().view(np.uint32).copy()
    fr0 = streams.frontier_bitmap(words * 32, 0.1, seed=seed + 2)[:words].numpy().view(np.uint32).copy()
    d_in = torch.from_numpy(np.concatenate([stream, np.zeros(16, np.uint8)])).to(dev)
    d_vis = torch.from_numpy(vis0.view(np.int32).copy()).to(dev)
    d_fr = torch.from_numpy(fr0.view(np.int32).copy()).to(dev)
    n_out = torch.full((1,), -1, dtype=torch.int64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    ws = torch.empty(B.workspace_bytes(max(len(ids_np), 1), 1, W), dtype=torch.uint8, device=dev)
    B.decompress_to_frontier(d_in, len(stream), W, id_base, d_fr, d_vis, n_bits, n_out, ws, status)
    torch.cuda.synchronize()
    vis, fr = vis0.copy(), fr0.copy()
    try:
        n_ref = oracle_mod.decompress_to_frontier(stream, W, fr, vis, n_bits, id_base)
        ref_ok = True
    except oracle_mod.OracleError as e:
        assert e.code == 2
        ref_ok = False
    assert ref_ok == expect_ok
    if not ref_ok:
        assert int(status.item()) == 2                 # DST_TOO_SMALL; the bitmaps may hold the bits of other IDs
        return
    assert int(status.item()) == 0 and int(n_out.item()) == n_ref
    assert np.array_equal(d_vis.cpu().numpy().view(np.uint32), vis), "visited bitmap differs from the oracle"
    assert np.array_equal(d_fr.cpu().numpy().view(np.uint32), fr), "frontier bitmap differs from the oracle"


@pytest.mark.parametrize("W", [32, 64])
def test_decompress_to_frontier(B, oracle_mod, W):
    dt = np.uint32 if W == 32 else np.uint64
    rng = np.random.default_rng(W)
    bases = (0, 777, (1 << W) - 50)
    for k, (n, mean) in enumerate(((0, 1.0), (1, 1.0), (127, 2.0), (128, 2.0), (1000, 3.0), (128 * 64 * 3 + 5, 2.0), (50000, 40.0), (3000, 5000.0))):
        rel = _np(streams.gap_stream(n, mean, seed=40 + k, W=W), W).astype(np.uint64) if n else np.zeros(0, np.uint64)
        rel = rel - (rel[0] if n else 0)                                   # bit indices from 0
        n_bits = int(rel[-1]) + 1 + k if n else 100
        id_base = bases[k % 3]
        ids = ((rel + np.uint64(id_base)) & np.uint64((1 << W) - 1 if W < 64 else 0xFFFFFFFFFFFFFFFF)).astype(dt)
        _frontier_case(B, oracle_mod, ids, W, n_bits, id_base, seed=k)
        if n > 200:
            _frontier_case(B, oracle_mod, ids, W, n_bits, id_base, thr=1 << 30, seed=k)          # a RAW stream
            _frontier_case(B, oracle_mod, ids, W, n_bits - k - 1, id_base, seed=k, expect_ok=False)   # the last ID does not fit
    # IDs in any order and more than once (the codec takes any sequence): a vertex received twice counts once
    pool = rng.integers(0, 5000, size=20000, dtype=np.uint64)
    _frontier_case(B, oracle_mod, (pool + np.uint64(9)).astype(dt), W, 5000, 9, seed=99)
    # a 2^22-bit level: many tiles, all warps
    bits = rng.random(1 << 22) < 0.3
    _frontier_case(B, oracle_mod, np.nonzero(bits)[0].astype(dt), W, 1 << 22, 0, seed=5)


def _batch_frontier_case(B, oracle_mod, lists, W, n_bits, id_base, thr, pitch_pad, seed, with_visited=True, expect=0):
    """lists: the ID arrays of the received streams. The streams (oracle bytes) lie in slots of a receive buffer, each
    shorter than its span; expected bitmaps: the oracle's single-stream update applied stream after stream."""
    dev = torch.device("cuda")
    blobs = [oracle_mod.compress(x, thr) for x in lists]
    pitch = (max(len(b) for b in blobs) + 15) // 16 * 16 + pitch_pad
    recv = np.full(len(blobs) * pitch + 16, 0xCD, np.uint8)
    for i, b in enumerate(blobs):
        recv[i * pitch:i * pitch + len(b)] = b
    words = max(4, ((n_bits + 31) // 32 + 3) // 4 * 4)
    vis0 = streams.frontier_bitmap(words * 32, 0.4, seed=seed + 1)[:words].numpy().view(np.uint32).copy()
    fr0 = streams.frontier_bitmap(words * 32, 0.1, seed=seed + 2)[:words].numpy().view(np.uint32).copy()
    d_in = torch.from_numpy(recv).to(dev)
    d_off = pitch * torch.arange(len(blobs) + 1, dtype=torch.int64, device=dev)
    d_vis = torch.from_numpy(vis0.view(np.int32).copy()).to(dev)
    d_fr = torch.from_numpy(fr0.view(np.int32).copy()).to(dev)
    n_out = torch.full((1,), -1, dtype=torch.int64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    total = sum(len(x) for x in lists)
    ws = torch.empty(B.workspace_bytes(max(total, 1), len(blobs), W), dtype=torch.uint8, device=dev)
    B.decompress_batch_to_frontier(d_in, d_off, len(blobs), W, id_base, d_fr, d_vis if with_visited else None, n_bits, n_out,
                                   ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == expect
    if expect:
        return
    vis, fr = vis0.copy(), fr0.copy()
    for b in blobs:
        if with_visited:
            oracle_mod.decompress_to_frontier(b, W, fr, vis, n_bits, id_base)
        else:
            oracle_mod.decompress_to_bitmap(b, W, fr, n_bits, id_base)
    assert int(n_out.item()) == total
    assert np.array_equal(d_fr.cpu().numpy().view(np.uint32), fr), "frontier bitmap differs from the oracle"
    assert np.array_equal(d_vis.cpu().numpy().view(np.uint32), vis), "visited bitmap differs from the oracle"


@pytest.mark.parametrize("W", [32, 64])
def test_decompress_batch_to_frontier(B, oracle_mod, W):
    """Algorithm 4 lines 10-13 over all received streams in one call: the union of the streams' IDs, filtered by the
    visited set, whatever their order; streams that overlap (a vertex found by several ranks), empty and RAW streams,
    the one-launch path (small levels) and the planned one, ID base offsets, IDs outside the bitmap."""
    dt = np.uint32 if W == 32 else np.uint64
    rng = np.random.default_rng(100 + W)

    def draw(n_bits, n, id_base):
        v = np.sort(rng.choice(n_bits, size=min(n, n_bits), replace=False)).astype(np.uint64)
        return ((v + np.uint64(id_base)) & np.uint64(0xFFFFFFFFFFFFFFFF if W == 64 else 0xFFFFFFFF)).astype(dt)

    # a small level: 8 streams over 2^16 vertices (one launch), overlapping, one empty, one below the RAW threshold
    nb, base = 1 << 16, 1000
    small = [draw(nb, n, base) for n in (3000, 0, 17, 5000, 128, 129, 1, 2500)]
    _batch_frontier_case(B, oracle_mod, small, W, nb, base, 128, 64, seed=1)
    _batch_frontier_case(B, oracle_mod, small, W, nb, base, 128, 0, seed=2, with_visited=False)
    # a large level: 16 streams over 2^22 vertices (plan + tiles), heavy overlap
    nb = 1 << 22
    big = [draw(nb, n, 0) for n in (200000, 150000, 0, 1, 300000, 70000, 128 * 64, 90000, 5, 250000, 100000, 60000, 31, 0, 120000, 80000)]
    _batch_frontier_case(B, oracle_mod, big, W, nb, 0, 1024, 256, seed=3)
    # one stream carries an ID beyond the bitmap
    bad = [x.copy() for x in small]
    bad[3][-1] = base + (1 << 16) + 5
    _batch_frontier_case(B, oracle_mod, bad, W, 1 << 16, base, 0, 64, seed=4, expect=B.ERR_DST_TOO_SMALL)
    # a corrupt slot (no stream header) is rejected
    dev = torch.device("cuda")
    junk = torch.full((4096,), 0xCD, dtype=torch.uint8, device=dev)
    off = torch.tensor([0, 2048, 4096], dtype=torch.int64, device=dev)
    fr = torch.zeros(64, dtype=torch.int32, device=dev)
    vis = torch.zeros(64, dtype=torch.int32, device=dev)
    n_out = torch.full((1,), -1, dtype=torch.int64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    ws = torch.empty(B.workspace_bytes(1000, 2, W), dtype=torch.uint8, device=dev)
    B.decompress_batch_to_frontier(junk, off, 2, W, 0, fr, vis, 2048, n_out, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_CORRUPT and int(n_out.item()) == 0
    assert not bool(fr.any()) and not bool(vis.any())


# ---- the one-launch cluster kernel of small batches (k_enc_small: <= 1024 buffers, <= 2048 blocks by the workspace size) ----
@pytest.mark.parametrize("W", [32, 64])
def test_small_batch_cluster_kernel_boundaries(B, oracle_mod, W):
    """Batches around the limits of the small-batch path and inside it: 1 .. 4 tiles per CTA, exactly 2048 blocks and one
    more (the general path), 1024 buffers and 1025, empty / RAW / one-ID buffers between full ones, buffers at every
    element alignment, outliers (exceptions), incompressible blocks (largest images), u64 deltas over 2^32 (the wide
    path), both encoder rules, thresholds 0 and 1 KB."""
    g = torch.Generator().manual_seed(W)
    cases = []
    for nblk in (1, 63, 64, 65, 511, 512, 513, 1024, 1536, 2047, 2048, 2049):           # one buffer of nblk blocks (ragged tail)
        cases.append(torch.tensor([128 * nblk - 5]))
    cases.append(torch.randint(0, 300, (1024,), generator=g))                               # 1024 small buffers
    cases.append(torch.randint(0, 300, (1025,), generator=g))                               # one too many: the general path
    cases.append(torch.tensor([0, 0, 1, 0, 129, 0, 0, 127, 128, 0, 5000, 1, 1, 0, 255, 256, 257, 0]))
    cases.append(torch.tensor([128 * 3 + e for e in range(1, 40)]))                        # every alignment
    cases.append(torch.randint(100, 3000, (100,), generator=g))                             # ~ 1200 blocks in 100 buffers
    for ci, counts in enumerate(cases):
        ids, off = streams.batch_of_streams(counts, 2.0 if ci % 2 else 300.0, seed=60 + ci, W=W)
        ids = ids.clone()
        n = ids.numel()
        if n > 4000:                                                                         # outliers and an incompressible stretch
            sel = torch.rand(n, generator=g) < 0.01
            ids[sel] += 1 << 20
            lo = n // 3
            ids[lo:lo + 700] = torch.randint(-(2 ** 31), 2 ** 31 - 1, (700,), generator=g, dtype=torch.int64).to(ids.dtype) if W == 32 \
                else torch.randint(-(2 ** 62), 2 ** 62, (700,), generator=g, dtype=torch.int64)
        for thr in (0, 1024):
            for codec in CODECS:
                run_batch(B, oracle_mod, ids, off, W, thr, codec=codec)


def test_small_batch_cluster_kernel_errors(B):
    dev = torch.device("cuda")
    counts = torch.tensor([1000, 0, 77, 4096, 129])
    ids, off = streams.batch_of_streams(counts, 16.0, seed=7, W=32)
    n, n_buf = ids.numel(), counts.numel()
    d_ids, d_off = ids.to(dev), off.to(dev)
    ws = torch.empty(B.workspace_bytes(n, n_buf, 32), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    out_off = torch.full((n_buf + 1,), -1, dtype=torch.int64, device=dev)
    small = torch.full((1024,), 0xAB, dtype=torch.uint8, device=dev)                        # far too small an output buffer
    B.compress_batch(d_ids, d_off, n_buf, 32, 0, small[:512], out_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_DST_TOO_SMALL and bool((out_off == 0).all()) and bool((small[512:] == 0xAB).all())
    status.zero_()
    bad = off.clone(); bad[2] = bad[1] - 1                                                   # decreasing offsets
    out = torch.empty(B.batch_compress_bound(counts.tolist(), 32), dtype=torch.uint8, device=dev)
    B.compress_batch(d_ids, bad.to(dev), n_buf, 32, 0, out, out_off, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_INVALID_ARG and bool((out_off == 0).all())
    status.zero_()
    counts2 = torch.tensor([1000, 0, 77, 4096, 129, 20000])                                 # 199 blocks
    ids2, off2 = streams.batch_of_streams(counts2, 16.0, seed=7, W=32)
    tiny_ws = torch.empty(B.workspace_bytes(200, 6, 32), dtype=torch.uint8, device=dev)      # a workspace for far fewer IDs: 64 blocks
    out2 = torch.empty(B.batch_compress_bound(counts2.tolist(), 32), dtype=torch.uint8, device=dev)
    out_off2 = torch.full((7,), -1, dtype=torch.int64, device=dev)
    B.compress_batch(ids2.to(dev), off2.to(dev), 6, 32, 0, out2, out_off2, tiny_ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == B.ERR_INVALID_ARG and bool((out_off2 == 0).all())


def test_mixed_calls_overlap_on_four_streams(B, oracle_mod):
    """Large single-buffer calls, small batches (the one-cluster kernel) and mid-size batches enqueued on four streams
    without any synchronisation between them, three passes over the same buffers: every tile of every compress grid comes
    from a ticket and a cluster is scheduled as a whole, so whatever shares the device, nothing can wait for a CTA that
    is not running. Bytes against the oracle, decode against the input."""
    dev = torch.device("cuda")
    rng = np.random.default_rng(17)
    cu = [torch.cuda.Stream() for _ in range(4)]
    for rnd in range(12):
        jobs = []
        for s in range(4):
            W = int(rng.choice([32, 64])); thr = int(rng.choice([0, 1024])); kind = (rnd + s) % 3
            if kind == 0:
                n = int(rng.choice([1 << 20, (1 << 22) + 5])); n_buf = 1; off = None
                ids = streams.gap_stream(n, float(rng.choice([2.0, 256.0])), seed=100 * rnd + s, W=W, outlier_frac=0.01, device=dev)
            else:
                n_buf = int(rng.choice([16, 64])) if kind == 1 else 500
                counts = torch.randint(0, 3000 if kind == 1 else 400, (n_buf,), generator=torch.Generator().manual_seed(100 * rnd + s))
                ids, off = streams.batch_of_streams(counts, 16.0, seed=100 * rnd + s, W=W, device=dev)
                ids, off = ids.to(dev), off.to(dev); n = ids.numel()
            cap = B.compress_bound(n, W) if off is None else B.batch_compress_bound((off[1:] - off[:-1]).tolist(), W)
            jobs.append(dict(W=W, thr=thr, ids=ids, off=off, n=n, n_buf=n_buf, cap=cap,
                             out=torch.empty(cap, dtype=torch.uint8, device=dev),
                             ws=torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev),
                             st=torch.zeros(1, dtype=torch.int32, device=dev), oo=torch.zeros(n_buf + 1, dtype=torch.int64, device=dev),
                             back=torch.empty(max(n, 4), dtype=ids.dtype, device=dev), io=torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)))
        torch.cuda.synchronize()
        for _ in range(3):
            for s, j in enumerate(jobs):
                with torch.cuda.stream(cu[s]):
                    if j["off"] is None:
                        B.compress(j["ids"], j["n"], j["W"], j["thr"], j["out"], j["oo"][1:2], j["ws"], j["st"])
                        B.decompress(j["out"], j["cap"], j["W"], j["back"], j["io"][1:2], j["ws"], j["st"])
                    else:
                        B.compress_batch(j["ids"], j["off"], j["n_buf"], j["W"], j["thr"], j["out"], j["oo"], j["ws"], j["st"])
                        B.decompress_batch(j["out"], j["oo"], j["n_buf"], j["W"], j["back"], j["io"], j["ws"], j["st"])
        torch.cuda.synchronize()
        for j in jobs:
            assert int(j["st"].item()) == 0
            host = _np(j["ids"], j["W"])
            if j["off"] is None:
                ref = oracle_mod.compress(host, j["thr"])
                assert int(j["oo"][1].item()) == len(ref)
            else:
                ref, ro = oracle_mod.compress_batch(host, j["off"].cpu().numpy().astype(np.uint64), j["thr"])
                assert np.array_equal(j["oo"].cpu().numpy().astype(np.uint64), ro)
            assert np.array_equal(j["out"][:len(ref)].cpu().numpy(), ref)
            assert torch.equal(j["back"][:j["n"]], j["ids"])


def test_batch_scatter_errors(B, oracle_mod):
    """bfsc_compress_batch_scatter: a stream that does not fit its destination is reported (size 0, DST_TOO_SMALL) and
    nothing is written beyond any destination's capacity while the other streams arrive intact; a null or misaligned
    destination is INVALID_ARG on the device; host-side argument errors; the RAW-fallback flag is UNSUPPORTED."""
    dev = torch.device("cuda")
    W = 32
    # the one-cluster kernel (<= 2048 blocks), then the general path (plan -> tiles -> streams)
    for counts in (torch.tensor([1000, 128 * 64 * 3 + 5, 40, 0, 128 * 70]), torch.tensor([1000, 128 * 64 * 40 + 5, 40, 0, 128 * 700])):
        ids, off = streams.batch_of_streams(counts, 16.0, seed=77, W=W)
        n, n_buf = ids.numel(), counts.numel()
        d_ids, d_off = ids.to(dev), off.to(dev)
        ref, ref_off = oracle_mod.compress_batch(_np(ids, W), off.numpy().astype(np.uint64), 0)
        sizes_ref = np.diff(ref_off.astype(np.int64))
        ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
        status = torch.zeros(1, dtype=torch.int32, device=dev)
        cap = int(sizes_ref[4])                                    # stream 4 fits exactly, stream 1 (several tiles) does not
        assert sizes_ref[1] > cap > sizes_ref[0]
        pitch = (cap + 15) // 16 * 16 + 64
        recv = torch.full((n_buf * pitch,), 0xCD, dtype=torch.uint8, device=dev)
        dst = recv.data_ptr() + pitch * torch.arange(n_buf, dtype=torch.int64, device=dev)
        sizes = torch.full((n_buf,), -1, dtype=torch.int64, device=dev)
        B.compress_batch_scatter(PFOR, d_ids, d_off, n_buf, W, 0, dst, cap, sizes, ws, status)
        torch.cuda.synchronize()
        assert int(status.item()) == B.ERR_DST_TOO_SMALL
        got = recv.view(n_buf, pitch).cpu().numpy()
        for i in range(n_buf):
            if i == 1:
                assert int(sizes[i]) == 0
            else:
                assert int(sizes[i]) == sizes_ref[i]
                assert np.array_equal(got[i, :sizes_ref[i]], ref[int(ref_off[i]):int(ref_off[i + 1])]), f"stream {i}"
                assert (got[i, sizes_ref[i]:] == 0xCD).all()
            assert (got[i, cap:] == 0xCD).all(), f"slot {i}: wrote beyond its capacity"
        # a null and a misaligned destination
        cap2 = int(sizes_ref.max())
        pitch2 = cap2 + 64
        recv2 = torch.empty(n_buf * pitch2, dtype=torch.uint8, device=dev)
        for bad_addr in (0, recv2.data_ptr() + 2 * pitch2 + 4):
            recv2.fill_(0xCD); status.zero_(); sizes.fill_(-1)
            dst2 = recv2.data_ptr() + pitch2 * torch.arange(n_buf, dtype=torch.int64, device=dev)
            dst2[2] = bad_addr
            B.compress_batch_scatter(PFOR, d_ids, d_off, n_buf, W, 0, dst2, cap2, sizes, ws, status)
            torch.cuda.synchronize()
            assert int(status.item()) == B.ERR_INVALID_ARG
            assert int(sizes[2]) == 0 and [int(sizes[i]) for i in (0, 1, 3, 4)] == [int(sizes_ref[i]) for i in (0, 1, 3, 4)]
            assert bool((recv2.view(n_buf, pitch2)[2] == 0xCD).all())
    # host-side rejections: nothing is enqueued
    status.zero_()
    for kwargs in (dict(dst=None), dict(sizes=None), dict(codec=PFOR | B.CODEC_FLAG_RAW_FALLBACK, code=B.ERR_UNSUPPORTED)):
        with pytest.raises(B.BfscError) as e:
            B.compress_batch_scatter(kwargs.get("codec", PFOR), d_ids, d_off, n_buf, W, 0, kwargs.get("dst", dst), cap,
                                     kwargs.get("sizes", sizes), ws, status)
        assert e.value.code == kwargs.get("code", B.ERR_INVALID_ARG)


# ---- FORMAT.md §10: visited-bitmap containers (bfsc_compress_vbitmap / bfsc_decompress_vbitmap) ----
def _vb_case(B, oracle_mod, bm_words, n_bits, codec=PFOR, dirty_tail=False):
    dev = torch.device("cuda")
    words = (n_bits + 31) // 32
    src = bm_words.copy()
    if dirty_tail and n_bits % 32:
        src[-1] |= np.uint32(0xFFFFFFFF) << np.uint32(n_bits % 32)     # garbage beyond n_bits in the caller's last word
    d_bm = torch.from_numpy(src.view(np.int32).copy()).to(dev) if words else torch.zeros(1, dtype=torch.int32, device=dev)
    cap = B.vbitmap_bound(n_bits)
    out = torch.full((cap + 64,), 0xAB, dtype=torch.uint8, device=dev)
    nb = torch.full((1,), -1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.vbitmap_workspace_bytes(n_bits), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    B.compress_vbitmap(codec, d_bm, n_bits, out[:cap], nb, ws, status)
    torch.cuda.synchronize()
    ref = oracle_mod.compress_vbitmap(bm_words, n_bits, codec)
    assert int(status.item()) == 0 and int(nb.item()) == len(ref), (n_bits, int(nb.item()), len(ref))
    got = out[:len(ref)].cpu().numpy()
    assert np.array_equal(got, ref), f"n_bits {n_bits}: container differs at byte {int(np.nonzero(got != ref)[0][0])} (kind {ref[6]})"
    assert bool((out[cap:] == 0xAB).all()), "wrote beyond capacity"
    back = torch.full((max(words, 1) + 2,), 0x55555555, dtype=torch.int32, device=dev)
    B.decompress_vbitmap(out, len(ref), back, n_bits, ws, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    assert np.array_equal(back[:words].cpu().numpy().view(np.uint32), bm_words[:words]), f"n_bits {n_bits}: decoded bitmap differs (kind {ref[6]})"
    assert bool((back[words:] == 0x55555555).all()), "wrote beyond the bitmap"
    return ref


@pytest.mark.parametrize("codec", CODECS)
def test_vbitmap_container(B, oracle_mod, codec):
    """Bytes against the oracle and identity round trip: sizes 0 … 2^22 + 17 bits, densities from empty to full (set bits
    listed, clear bits listed, the bitmap itself), clustered bits, garbage beyond n_bits in the caller's last word."""
    rng = np.random.default_rng(7 + codec)
    kinds = set()
    for n_bits in (0, 1, 31, 32, 33, 384, 385, 1000, 4097, 128 * 64 * 3 + 5, 1 << 20, (1 << 22) + 17):
        for dens in (0.0, 1.0, 0.5, 0.001, 0.999, 0.05, 0.95, 0.12, 0.88):
            bits = rng.random(n_bits) < dens
            words = (n_bits + 31) // 32
            pad = np.zeros(words * 32, dtype=bool)
            pad[:n_bits] = bits
            bm = np.packbits(pad.reshape(-1, 32), axis=1, bitorder="little").view(np.uint32).reshape(-1) if words else np.zeros(0, np.uint32)
            kinds.add(int(_vb_case(B, oracle_mod, bm, n_bits, codec, dirty_tail=True)[6]))
    assert kinds == {0, 1, 2}
    # a late-BFS visited bitmap: 2^24 vertices, runs of unvisited ones
    n_bits = 1 << 24
    bm = streams.frontier_bitmap(n_bits, 0.02, seed=3, run=16).numpy().view(np.uint32)[:n_bits // 32]
    ref = _vb_case(B, oracle_mod, ~bm, n_bits, codec)
    assert ref[6] == 2 and len(ref) < n_bits // 8 // 3            # (2 % of the bits clear, in runs: under a third of the bitmap)


def test_vbitmap_rejects(B, oracle_mod):
    """The decoder's verdicts are the oracle's (FORMAT.md §10), and a rejected container leaves the caller's bitmap alone."""
    dev = torch.device("cuda")
    rng = np.random.default_rng(11)
    n_bits = 5000
    words = (n_bits + 31) // 32
    ws = torch.empty(B.vbitmap_workspace_bytes(n_bits), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)

    def pack(b):
        pad = np.zeros(words * 32, dtype=bool)
        pad[:n_bits] = b
        return np.packbits(pad.reshape(-1, 32), axis=1, bitorder="little").view(np.uint32).reshape(-1)

    def verdict(buf, nb=n_bits):
        d = torch.from_numpy(np.concatenate([buf, np.zeros(16, np.uint8)])).to(dev)
        back = torch.full((words,), 0x77777777, dtype=torch.int32, device=dev)
        status.zero_()
        w2 = ws if nb == n_bits else torch.empty(B.vbitmap_workspace_bytes(nb), dtype=torch.uint8, device=dev)
        B.decompress_vbitmap(d, len(buf), back, nb, w2, status)
        torch.cuda.synchronize()
        rc = int(status.item())
        if rc:
            assert bool((back == 0x77777777).all()), "a rejected container changed the bitmap"
        try:
            oracle_mod.decompress_vbitmap(buf, nb)
            ref = 0
        except oracle_mod.OracleError as e:
            ref = e.code
        assert rc == ref, (rc, ref)
        return rc

    sparse = oracle_mod.compress_vbitmap(pack(rng.random(n_bits) < 0.01), n_bits)        # kind 1
    dense = oracle_mod.compress_vbitmap(pack(rng.random(n_bits) < 0.99), n_bits)         # kind 2
    half = oracle_mod.compress_vbitmap(pack(rng.random(n_bits) < 0.5), n_bits)           # kind 0
    assert (sparse[6], dense[6], half[6]) == (1, 2, 0)
    for good in (sparse, dense, half):
        assert verdict(good) == 0
        for pos, val in ((0, 0x58), (4, 2), (5, 64), (6, 3), (7, 1), (16, (int(good[16]) + 16) & 0xff), (16, (int(good[16]) - 16) & 0xff), (24, (int(good[24]) + 1) & 0xff)):
            bad = good.copy()
            bad[pos] = val
            assert verdict(bad) != 0, (int(good[6]), pos)
        assert verdict(good[:-16]) == B.ERR_CORRUPT
        assert verdict(good, n_bits + 1) == B.ERR_DST_TOO_SMALL
    bad = half.copy()
    bad[32 + n_bits // 8] |= 1 << 7                                        # a pad bit of the kind-0 payload
    assert verdict(bad) == B.ERR_CORRUPT
    bad = sparse.copy()
    bad[32 + 40] ^= 0xFF                                                   # inside the stream: its first block header / directory
    verdict(bad)                                                           # (whatever the oracle says)
    far = sparse.copy()                                                    # the container claims fewer bits than its IDs need
    far[8:16] = np.frombuffer((600).to_bytes(8, "little"), dtype=np.uint8)
    assert verdict(far, 600) == B.ERR_CORRUPT
