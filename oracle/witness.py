"""Second witness — a pure-Python, big-integer reading of FORMAT.md v1, written from the
document alone (it does not call, import or mirror oracle/bfsc_ref.c). Test infrastructure.

It pins the byte layout of the oracle from the other side: `decode_stream` treats every
column as ONE big little-endian integer and slices rows out of it, and `build_block`
constructs a block for a FORCED b the same way, so that a test can brute-force the
canonical b ("smallest block over all b, ties to the largest b", FORMAT.md §2) without
using the oracle's width histogram.

Paper passages: delta coding L979-986; width eq. (6); blocks of 128 / b in 0..32
L987-998, L1052-1056; exceptions = values >= 2^b kept apart, L1000-1011.
Only for small inputs (pure Python loops).
"""
from __future__ import annotations


def _align(x: int, k: int) -> int:
    return -(-x // k) * k


def block_bytes(b: int, n_exc: int, W: int) -> int:
    e = _align(_align(n_exc, W // 8) + n_exc * (W // 8), 16) if n_exc else 0
    return 16 + 16 * b + e


def deltas_of_block(xs, W: int):
    """xs: the block's valid IDs (1..128 python ints) -> (base, [128 deltas])."""
    M = 1 << W
    d = [0] * 128
    for j in range(1, len(xs)):
        d[j] = (xs[j] - xs[j - 1]) % M
    return xs[0], d


def build_block(d, base: int, b: int, W: int) -> bytes:
    """FORMAT.md §2 with a forced b (0..W)."""
    assert len(d) == 128 and 0 <= b <= W
    exc = [j for j in range(128) if d[j] >> b]           # d_j >= 2^b
    cols = [0, 0, 0, 0]                                  # one big integer per column
    for j in range(128):
        c, r = j % 4, j // 4
        cols[c] |= (d[j] & ((1 << b) - 1)) << (r * b)
    payload = bytearray(16 * b)
    for c in range(4):
        raw = cols[c].to_bytes(4 * b, "little") if b else b""
        for k in range(b):
            payload[16 * k + 4 * c:16 * k + 4 * c + 4] = raw[4 * k:4 * k + 4]
    out = bytearray()
    out += base.to_bytes(8, "little") + bytes([b, len(exc)]) + bytes(6)
    out += payload
    if exc:
        e = bytearray(bytes(exc))
        e += bytes(_align(len(e), W // 8) - len(e))
        for j in exc:
            e += (d[j] >> b).to_bytes(W // 8, "little")
        e += bytes(_align(len(e), 16) - len(e))
        out += e
    assert len(out) == block_bytes(b, len(exc), W)
    return bytes(out)


def brute_force_b(d, W: int):
    """Build the block for EVERY b in 0..W; smallest wins, ties -> largest b."""
    best = None
    for b in range(W + 1):
        size = len(build_block(d, 0, b, W))
        if best is None or size <= best[1]:
            best = (b, size)
    return best


def stream_mode(s: bytes) -> int:
    return s[6]


def stream_blocks(s: bytes):
    """(b, n_exc) of every block of a mode 1 / mode 2 stream, by walking the directory."""
    nb = int.from_bytes(s[24:28], "little")
    dir_ = [int.from_bytes(s[32 + 4 * k:36 + 4 * k], "little") for k in range(nb + 1)]
    return [(s[16 * dir_[k] + 8], s[16 * dir_[k] + 9]) for k in range(nb)]


def decode_stream(s: bytes, W: int):
    """-> list of python ints. Raises ValueError on anything FORMAT.md §4 rejects."""
    if len(s) < 32 or s[0:4] != b"BFSC" or s[4] != 1 or s[5] != W or s[6] not in (0, 1, 2) or s[7] != 0:   # 2 = BP128-D1: decoded like 1 (FORMAT.md §7)
        raise ValueError("bad header")
    n = int.from_bytes(s[8:16], "little")
    total = int.from_bytes(s[16:24], "little")
    nb = int.from_bytes(s[24:28], "little")
    if total > len(s) or total % 16:
        raise ValueError("bad total_bytes")
    if s[6] == 0:
        if nb != 0 or 32 + n * (W // 8) > total:
            raise ValueError("bad raw stream")
        return [int.from_bytes(s[32 + i * (W // 8):32 + (i + 1) * (W // 8)], "little") for i in range(n)]
    if nb != -(-n // 128):
        raise ValueError("bad nb")
    dir_ = [int.from_bytes(s[32 + 4 * k:36 + 4 * k], "little") for k in range(nb + 1)]
    if dir_[nb] != total // 16 or dir_[0] != (32 + _align(4 * (nb + 1), 16)) // 16:
        raise ValueError("bad directory ends")
    M = 1 << W
    out = []
    for k in range(nb):
        if dir_[k + 1] <= dir_[k]:
            raise ValueError("directory not increasing")
        blk = s[16 * dir_[k]:16 * dir_[k + 1]]
        base = int.from_bytes(blk[0:8], "little")
        b, n_exc = blk[8], blk[9]
        if b > W or n_exc > 127 or block_bytes(b, n_exc, W) > len(blk):
            raise ValueError("bad block header")
        payload = blk[16:16 + 16 * b]
        cols = []
        for c in range(4):
            raw = b"".join(payload[16 * kk + 4 * c:16 * kk + 4 * c + 4] for kk in range(b))
            cols.append(int.from_bytes(raw, "little"))
        d = [(cols[j % 4] >> ((j // 4) * b)) & ((1 << b) - 1) for j in range(128)]
        if n_exc:
            e = blk[16 + 16 * b:]
            pos = list(e[:n_exc])
            hoff = _align(n_exc, W // 8)
            if any(pos[i] <= pos[i - 1] for i in range(1, n_exc)):
                raise ValueError("exception positions not strictly ascending")
            for i, p in enumerate(pos):
                if p >= 128:
                    raise ValueError("bad exception position")
                d[p] |= int.from_bytes(e[hoff + i * (W // 8):hoff + (i + 1) * (W // 8)], "little") << b
        m = min(128, n - 128 * k)
        v = base % M
        for j in range(m):
            v = (v + d[j]) % M
            out.append(v)
    return out
