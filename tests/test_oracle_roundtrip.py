"""Round-trip identity (PAPER.md L930-935 lossless criterion), walk-the-headers invariants,
second-witness decoding, threshold / batch semantics, corrupt-stream rejection and the
multi-threaded drivers of the oracle. CPU only."""
import struct

import numpy as np
import pytest
import torch

from oracle import witness
from paper_1704_00513_b200.workloads import rmat, streams


def _dt(W):
    return np.uint32 if W == 32 else np.uint64


def _np(t, W):
    a = t.cpu().numpy()
    return a.view(np.uint32) if W == 32 else a.view(np.uint64)


def walk_and_check(oracle_mod, s: bytes, x: np.ndarray, W: int):
    """FORMAT.md invariants recomputed from the block headers alone."""
    n = len(x)
    assert s[:4] == b"BFSC" and s[4] == 1 and s[5] == W and s[7] == 0 and s[28:32] == bytes(4)
    hn, total, nb = struct.unpack("<QQI", s[8:28])
    assert hn == n and total == len(s) and total % 16 == 0
    if s[6] == 0:
        assert nb == 0 and total == 32 + (n * W // 8 + 15) // 16 * 16
        assert s[32:32 + n * W // 8] == x.tobytes()
        assert not any(s[32 + n * W // 8:])
        return
    assert nb == (n + 127) // 128
    dirb = (4 * (nb + 1) + 15) // 16 * 16
    d = struct.unpack(f"<{nb + 1}I", s[32:32 + 4 * (nb + 1)])
    assert not any(s[32 + 4 * (nb + 1):32 + dirb])
    assert d[0] == (32 + dirb) // 16 and d[nb] == total // 16
    mask = (1 << W) - 1
    for k in range(nb):
        blk = s[16 * d[k]:16 * d[k + 1]]
        base, b, n_exc = struct.unpack("<QBB", blk[:10])
        assert blk[10:16] == bytes(6)
        assert len(blk) == witness.block_bytes(b, n_exc, W)          # dir span == size from header
        xs = [int(v) for v in x[128 * k:128 * k + 128]]
        assert base == xs[0]
        _, dl = witness.deltas_of_block(xs, W)
        assert n_exc == sum(1 for v in dl if v >> b)
        sizes = [witness.block_bytes(bb, sum(1 for v in dl if v >> bb), W) for bb in range(W + 1)]
        assert len(blk) == min(sizes)                                # chosen b is a minimiser
        assert b == max(bb for bb in range(W + 1) if sizes[bb] == min(sizes) and bb <= max(v.bit_length() for v in dl))
        if n_exc:
            e = blk[16 + 16 * b:]
            pos = list(e[:n_exc])
            assert pos == sorted(set(pos)) and pos == [j for j in range(128) if dl[j] >> b]
            hoff = -(-n_exc // (W // 8)) * (W // 8)
            assert not any(e[n_exc:hoff])
            highs = [int.from_bytes(e[hoff + i * (W // 8):hoff + (i + 1) * (W // 8)], "little") for i in range(n_exc)]
            assert all(h != 0 for h in highs)
            assert not any(e[hoff + n_exc * (W // 8):])
        assert blk == witness.build_block(dl, base & mask, b, W)     # every byte incl. pads


CASES_N = [0, 1, 2, 3, 127, 128, 129, 255, 256, 257, 1000, 4097]


@pytest.mark.parametrize("W", [32, 64])
def test_roundtrip_shapes(oracle_mod, W):
    rng = np.random.default_rng(W)
    for n in CASES_N:
        variants = {
            "sorted": np.sort(rng.integers(0, 1 << 24, size=n, dtype=np.uint64)),
            "unsorted": rng.integers(0, 1 << (W - 1), size=n, dtype=np.uint64),
            "equal": np.full(n, 77, dtype=np.uint64),
            "wrap": (np.uint64((1 << W) - 5) + np.arange(n, dtype=np.uint64) * np.uint64(3)) & np.uint64((1 << W) - 1),
            "max": np.full(n, (1 << W) - 1, dtype=np.uint64),
            "alt_extremes": np.where(np.arange(n) % 2 == 0, 0, (1 << W) - 1).astype(np.uint64),
        }
        for name, v in variants.items():
            x = v.astype(_dt(W))
            s = oracle_mod.compress(x)
            assert len(s) <= oracle_mod.compress_bound(n, W), (name, n)
            y = oracle_mod.decompress(s, W)
            assert np.array_equal(x, y), (name, n)
            if n <= 300:
                walk_and_check(oracle_mod, s.tobytes(), x, W)
                assert witness.decode_stream(s.tobytes(), W) == [int(t) for t in x]
            # canonical: re-encoding the decoded IDs gives the same bytes
            assert np.array_equal(oracle_mod.compress(y), s)


def test_monotone_output_and_streams(oracle_mod):
    for mean, out in ((1.0, 0.0), (2.0, 0.0), (16.0, 0.0), (256.0, 0.01)):
        t = streams.gap_stream(5000, mean, seed=2, W=64, outlier_frac=out)
        x = _np(t, 64)
        s = oracle_mod.compress(x)
        y = oracle_mod.decompress(s, 64)
        assert np.array_equal(x, y) and np.all(np.diff(y.astype(np.int64)) >= 0)
        walk_and_check(oracle_mod, s.tobytes(), x[:], 64) if mean == 256.0 else None
    # bits/ID sanity (SURVEY.md §8(c) ratio sanity row; not a pin, loose bounds)
    x = _np(streams.gap_stream(1 << 16, 2.0, seed=2, W=32), 32)
    bits = 8 * len(oracle_mod.compress(x)) / len(x)
    assert 4.0 < bits < 6.0


def test_threshold(oracle_mod):
    x = np.arange(255, dtype=np.uint32)            # 1020 B
    assert oracle_mod.compress(x, 1024)[6] == 0    # RAW
    assert oracle_mod.compress(x, 1020)[6] == 1    # strict <
    assert oracle_mod.compress(x, 0)[6] == 1
    x = np.arange(256, dtype=np.uint32)
    assert oracle_mod.compress(x, 1024)[6] == 1
    x64 = np.arange(127, dtype=np.uint64)
    s = oracle_mod.compress(x64, 1024)
    assert s[6] == 0 and len(s) == 32 + 1024 - 8 + 8
    assert np.array_equal(oracle_mod.decompress(s, 64), x64)
    walk_and_check(oracle_mod, s.tobytes(), x64, 64)
    e = oracle_mod.compress(np.zeros(0, np.uint32), 1024)
    assert len(e) == 32 and e[6] == 0


def test_tiny_rmat_batches(oracle_mod):
    """BASELINE config 1 through the oracle: scale-12 R-MAT, 8 roots, 4 buffers by v mod 4."""
    G = rmat.Graph(12, 16, seed=1)
    roots = G.roots(8, seed=1)
    assert len(set(roots)) == 8
    n_levels = 0
    for root in roots:
        for f in G.bfs_frontiers(root):
            n_levels += 1
            assert torch.all(f[1:] > f[:-1])
            vals, off = streams.split_mod(f, 4)
            ids = _np(streams.as_ids(vals, 32), 32)
            off = off.numpy().astype(np.uint64)
            out, out_off = oracle_mod.compress_batch(ids, off, 0)
            assert int(out_off[-1]) == len(out)
            for i in range(4):
                one = oracle_mod.compress(ids[int(off[i]):int(off[i + 1])], 0)
                assert np.array_equal(out[int(out_off[i]):int(out_off[i + 1])], one)
            back, id_off = oracle_mod.decompress_batch(out, out_off, 32, len(ids))
            assert np.array_equal(back, ids) and np.array_equal(id_off, off)
    assert n_levels > 20


def test_mt_matches_serial(oracle_mod):
    counts = streams.log_uniform_counts(64, 8, 14, 32, seed=5)
    counts[3] = 0
    counts[7] = 1
    t, off = streams.batch_of_streams(counts, 16.0, seed=5, W=32)
    ids, off = _np(t, 32), off.numpy().astype(np.uint64)
    for thr in (0, 1024):
        a, ao = oracle_mod.compress_batch(ids, off, thr)
        b, bo = oracle_mod.compress_batch(ids, off, thr, threads=3)
        assert np.array_equal(a, b) and np.array_equal(ao, bo)
        y, yo = oracle_mod.decompress_batch(a, ao, 32, len(ids), threads=3)
        assert np.array_equal(y, ids) and np.array_equal(yo, off)
    big = _np(streams.gap_stream(100_000, 256.0, seed=2, W=64, outlier_frac=0.01), 64)
    o1 = np.array([0, len(big)], dtype=np.uint64)
    a, ao = oracle_mod.compress_batch(big, o1, 0)
    b, bo = oracle_mod.compress_batch(big, o1, 0, threads=4)
    assert np.array_equal(a, b)
    y, _ = oracle_mod.decompress_batch(a, ao, 64, len(big), threads=4)
    assert np.array_equal(y, big)


def test_corrupt_streams_rejected(oracle_mod):
    x = _np(streams.gap_stream(700, 16.0, seed=9, W=32), 32)
    good = oracle_mod.compress(x)

    def bad(mut):
        s = good.copy()
        mut(s)
        with pytest.raises(oracle_mod.OracleError):
            oracle_mod.decompress(s, 32)
        with pytest.raises(ValueError):
            witness.decode_stream(s.tobytes(), 32)

    bad(lambda s: s.__setitem__(0, 0x41))                          # magic
    bad(lambda s: s.__setitem__(4, 2))                             # version
    bad(lambda s: s.__setitem__(5, 64))                            # W
    bad(lambda s: s.__setitem__(6, 9))                             # mode
    bad(lambda s: s.__setitem__(7, 1))                             # reserved header byte (FORMAT.md §4)
    bad(lambda s: s.__setitem__(slice(16, 24), np.frombuffer(struct.pack("<Q", len(good) + 16), np.uint8)))
    bad(lambda s: s.__setitem__(slice(24, 28), np.frombuffer(struct.pack("<I", 99), np.uint8)))
    bad(lambda s: s.__setitem__(slice(36, 40), np.frombuffer(struct.pack("<I", 1), np.uint8)))      # dir[1] backwards
    first_blk = 16 * struct.unpack("<I", good[32:36].tobytes())[0]
    bad(lambda s: s.__setitem__(first_blk + 8, 33))                # b > W
    bad(lambda s: s.__setitem__(first_blk + 9, 127))               # block larger than its span
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.decompress(good[:-16], 32)                      # truncated


def test_exception_positions_must_ascend(oracle_mod):
    """FORMAT.md §4: an exception list whose positions are not strictly ascending (a duplicate, or two swapped
    entries) is rejected by both decoders; the untouched stream and a stream whose positions were replaced by
    OTHER ascending ones still decode (to different IDs: positions are data)."""
    for W in (32, 64):
        d = np.ones(128, dtype=np.uint64)
        d[0] = 0
        d[[9, 40, 41, 100]] = np.uint64(1 << 20)
        x = (np.uint64(7) + np.cumsum(d)).astype(np.uint32 if W == 32 else np.uint64)
        good = oracle_mod.compress(x)
        blk = 16 * struct.unpack("<I", good[32:36].tobytes())[0]
        assert good[blk + 8] == 1 and good[blk + 9] == 4           # b = 1, four exceptions
        e = blk + 16 + 16
        assert list(good[e:e + 4]) == [9, 40, 41, 100]
        assert np.array_equal(oracle_mod.decompress(good, W), x)
        assert witness.decode_stream(good.tobytes(), W) == [int(v) for v in x]
        for pos in ([9, 40, 40, 100], [9, 41, 40, 100], [100, 41, 40, 9], [9, 9, 9, 9]):
            s = good.copy()
            s[e:e + 4] = pos
            with pytest.raises(oracle_mod.OracleError):
                oracle_mod.decompress(s, W)
            with pytest.raises(ValueError):
                witness.decode_stream(s.tobytes(), W)
        s = good.copy()
        s[e:e + 4] = [1, 2, 3, 127]                                # other ascending positions: well-formed
        y = oracle_mod.decompress(s, W)
        assert witness.decode_stream(s.tobytes(), W) == [int(v) for v in y] and not np.array_equal(y, x)
