"""Throughput / ratio report for BASELINE.json configs 3, 4 and 5 (configs[1] is bench.py's line).

    python -m paper_1704_00513_b200.report --config 3            # R-MAT 22, u32, 16 buffers/level, 1 KB threshold
    python -m paper_1704_00513_b200.report --config 4            # R-MAT 25, u64, 64 buffers/level
    python -m paper_1704_00513_b200.report --config 5            # message-size sweep + 4096-buffer batch
    (`python bench.py --config N ...` runs the same report with two more columns: the oracle (oracle/, multi-threaded
     driver) timed on the box's host cores on the very same buffers, beside every row. This module belongs to the
     product package and never imports the oracle: bench.py passes the timer in.)
    (--json adds one JSON line per report: totals, oracle included when timed)
    (--scale / --roots shrink configs 3 and 4 for a quick look; --codec bp128 runs the same cases under the
     no-exception rule, FORMAT.md §7 — the codec class the thesis ran; --graph replays
     each timed run from a CUDA graph captured around the same C-ABI calls: the host's 9-15 us per call from
     Python leave the figures, what remains is the device-side time of the kernel chain)

Every call goes through the C ABI (binding.py); each timed call is preceded by an L2 flush (a 256 MB
memset outside the timed region) and timed with CUDA events; every decoded batch is compared with its
input. Prints markdown rows: raw MB, ratio, bits/ID, encode GB/s (raw input bytes / time), decode GB/s
(raw output bytes / time) and both as fractions of the measured HBM copy peak counted on algorithmic
bytes (raw + compressed).
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1704_00513_b200 import binding as B  # noqa: E402
from paper_1704_00513_b200.workloads import rmat, streams  # noqa: E402


def peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"])
    except Exception:
        return 6650.0


class Runner:
    def __init__(self, dev, reps=5, codec=B.CODEC_PFOR, graph=False, cpu_timer=None, scatter=False):
        """cpu_timer(ids: device tensor, off: device int64 offsets, W, thr, codec) -> (encode seconds, decode seconds)
        of a CPU implementation on the same buffers, or None (bench.py --config passes the oracle's)."""
        self.dev, self.reps, self.codec, self.graph, self.cpu_timer = dev, reps, codec, graph, cpu_timer
        self.scatter = scatter                               # batch rows: the data path of exchange.SlotExchange (streams into / out of slots)
        self.totals = []                                     # one dict per report row marked as a total (--json)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        self.peak = peak_gbs()

    def _time(self, fns):
        """fns: the same call on `len(fns)` rotating copies of its buffers. Returns (per-call ms in a run of
        back-to-back calls, ms of one isolated call with a cold L2, host-bound flag: enqueueing the run took the
        host at least 90 % of the time the GPU needed, i.e. the figure is the host's, not the kernels')."""
        import time
        for f in fns:                                        # warm-up
            f()
        torch.cuda.synchronize()
        rounds = max(self.reps, -(-40 // len(fns)))
        if self.graph:
            return self._time_graph(fns, rounds)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(rounds):
            for f in fns:
                f()
        e1.record()
        host_ms = 1e3 * (time.perf_counter() - t0)
        torch.cuda.synchronize()
        gpu_ms = e0.elapsed_time(e1)
        stream_ms = gpu_ms / (rounds * len(fns))
        self.host_bound = self.host_bound or host_ms >= 0.9 * gpu_ms
        iso = None
        for _ in range(3):
            self.flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fns[0](); e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            iso = ms if iso is None else min(iso, ms)
        return stream_ms, iso

    def _time_graph(self, fns, rounds):
        """As _time, but the calls are captured once (stream capture around the same C-ABI calls: the library only
        enqueues kernels) and replayed: one graph holding a pass over all copies, one holding a single call."""
        side = torch.cuda.Stream(device=self.dev)
        g_all, g_one = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(g_all, stream=side):
                for f in fns:
                    f()
            with torch.cuda.graph(g_one, stream=side):
                fns[0]()
        torch.cuda.synchronize()
        g_all.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(rounds):
            g_all.replay()
        e1.record()
        torch.cuda.synchronize()
        stream_ms = e0.elapsed_time(e1) / (rounds * len(fns))
        iso = None
        for _ in range(3):
            self.flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); g_one.replay(); e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            iso = ms if iso is None else min(iso, ms)
        return stream_ms, iso

    def batch(self, ids, off, W, thr, single=False):
        """ids: device tensor (bit pattern), off: device int64 offsets. Returns dict of results. Timed on
        `copies` rotating copies of every buffer (working set >= 256 MB, 2..8 copies)."""
        dev = self.dev
        self.host_bound = False
        n, n_buf = ids.numel(), off.numel() - 1
        counts = (off[1:] - off[:-1]).tolist()
        cap = B.batch_compress_bound(counts, W)
        per_copy = 2 * n * (W // 8) + 1
        copies = int(max(2, min(8, -(-(256 << 20) // per_copy))))
        outs = [torch.empty(cap, dtype=torch.uint8, device=dev) for _ in range(copies)]
        out_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
        ws = torch.empty(B.workspace_bytes(n, n_buf, W), dtype=torch.uint8, device=dev)
        status = torch.zeros(1, dtype=torch.int32, device=dev)
        backs = [torch.empty(max(n, 4), dtype=ids.dtype, device=dev) for _ in range(copies)]
        id_off = torch.zeros(n_buf + 1, dtype=torch.int64, device=dev)
        pads = []
        for _ in range(copies):
            pad = torch.empty(n + 4, dtype=ids.dtype, device=dev)
            pad[:n] = ids
            pads.append(pad)
        cpu = {}
        if self.cpu_timer is not None:
            ce, cd = self.cpu_timer(ids, off, W, thr, self.codec)
            cpu = {"cpu_enc_ms": 1e3 * ce, "cpu_dec_ms": 1e3 * cd}
        if single:                                           # one buffer: the single-buffer entry points
            nbytes = torch.zeros(1, dtype=torch.int64, device=dev)
            n_out = torch.zeros(1, dtype=torch.int64, device=dev)
            enc, enc_iso = self._time([(lambda c=c: B.compress_codec(self.codec, pads[c], n, W, thr, outs[c], nbytes, ws, status)) for c in range(copies)])
            dec, dec_iso = self._time([(lambda c=c: B.decompress(outs[c], cap, W, backs[c], n_out, ws, status)) for c in range(copies)])
            assert int(status.item()) == 0 and int(n_out.item()) == n
            assert torch.equal(backs[copies - 1][:n], ids), "decode != input"
            comp = int(nbytes.item())
            return {"n": n, "n_buf": 1, "raw": n * (W // 8), "comp": comp, "enc_ms": enc, "dec_ms": dec,
                    "enc_iso_ms": enc_iso, "dec_iso_ms": dec_iso, "host_bound": self.host_bound} | cpu
        if self.scatter:
            # every stream into its own slot of a receive buffer (bfsc_compress_batch_scatter), decoded where it lies
            slot = max([B.compress_bound(c, W) for c in set(counts)] + [32])
            pitch = (slot + 255) // 256 * 256
            recvs = [torch.empty(n_buf * pitch, dtype=torch.uint8, device=dev) for _ in range(copies)]
            dsts = [r.data_ptr() + pitch * torch.arange(n_buf, dtype=torch.int64, device=dev) for r in recvs]
            slot_off = pitch * torch.arange(n_buf + 1, dtype=torch.int64, device=dev)
            sizes = torch.zeros(n_buf, dtype=torch.int64, device=dev)
            enc, enc_iso = self._time([(lambda c=c: B.compress_batch_scatter(self.codec, pads[c], off, n_buf, W, thr, dsts[c], slot, sizes, ws, status)) for c in range(copies)])
            dec, dec_iso = self._time([(lambda c=c: B.decompress_batch(recvs[c], slot_off, n_buf, W, backs[c], id_off, ws, status)) for c in range(copies)])
            assert int(status.item()) == 0
            assert torch.equal(backs[copies - 1][:n], ids) and torch.equal(id_off, off), "decode != input"
            return {"n": n, "n_buf": n_buf, "raw": n * (W // 8), "comp": int(sizes.sum().item()), "enc_ms": enc, "dec_ms": dec,
                    "enc_iso_ms": enc_iso, "dec_iso_ms": dec_iso, "host_bound": self.host_bound} | cpu
        enc, enc_iso = self._time([(lambda c=c: B.compress_batch_codec(self.codec, pads[c], off, n_buf, W, thr, outs[c], out_off, ws, status)) for c in range(copies)])
        dec, dec_iso = self._time([(lambda c=c: B.decompress_batch(outs[c], out_off, n_buf, W, backs[c], id_off, ws, status)) for c in range(copies)])
        assert int(status.item()) == 0
        assert torch.equal(backs[copies - 1][:n], ids) and torch.equal(id_off, off), "decode != input"
        comp = int(out_off[-1].item())
        return {"n": n, "n_buf": n_buf, "raw": n * (W // 8), "comp": comp, "enc_ms": enc, "dec_ms": dec,
                "enc_iso_ms": enc_iso, "dec_iso_ms": dec_iso, "host_bound": self.host_bound} | cpu

    def row(self, label, r):
        raw, comp = r["raw"], r["comp"]
        alg = raw + comp
        e, d = r["enc_ms"] * 1e-3, r["dec_ms"] * 1e-3
        ratio = raw / comp if comp else 0.0
        bits = 8.0 * comp / r["n"] if r["n"] else 0.0
        if r.get("host_bound"):
            label += " (*)"
        ora = "n/a | n/a"
        if r.get("cpu_enc_ms") and r.get("cpu_dec_ms"):
            ora = f"{raw / r['cpu_enc_ms'] / 1e6:.2f} | {raw / r['cpu_dec_ms'] / 1e6:.2f}"
        return (f"| {label} | {r['n_buf']} | {raw / 1e6:.3f} | {ratio:.2f} | {bits:.2f} | {r['enc_ms'] * 1e3:.1f} | "
                f"{raw / e / 1e9:.1f} | {100 * alg / e / 1e9 / self.peak:.1f} | {r['dec_ms'] * 1e3:.1f} | "
                f"{raw / d / 1e9:.1f} | {100 * alg / d / 1e9 / self.peak:.1f} | {r['enc_iso_ms'] * 1e3:.1f} | {r['dec_iso_ms'] * 1e3:.1f} | {ora} |")

    def total(self, label, r):
        """A totals row: printed like any row, and kept for --json."""
        self.totals.append({"case": label} | {k: r[k] for k in r if k != "host_bound"} |
                           {"enc_frac_of_peak": (r["raw"] + r["comp"]) / (r["enc_ms"] * 1e-3) / 1e9 / self.peak,
                            "dec_frac_of_peak": (r["raw"] + r["comp"]) / (r["dec_ms"] * 1e-3) / 1e9 / self.peak})
        return self.row(label, r)


HDR = ("enc us / dec us: per call, in a run of back-to-back calls on rotating copies of the buffers (working set >= 256 MB or 8 copies); "
       "isolated: ONE call between two events after an L2 flush (launch latency and cold caches included); "
       "(*) = the host needed as long to enqueue the run as the GPU to execute it (9-15 us per call from Python): "
       "the back-to-back figure is then the host's; oracle enc / dec GB/s: the CPU oracle (oracle/, all host cores) timed on the "
       "same buffers in the same run (only through `python bench.py --config N`; n/a otherwise)\n\n"
       "| case | buffers | raw MB | ratio | bits/ID | enc us | enc GB/s in | enc % peak | dec us | dec GB/s out | dec % peak | isolated enc us | isolated dec us | oracle enc GB/s | oracle dec GB/s |\n"
       "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")


def rmat_config(R, scale, seed, W, parts, n_roots, thr, per_level_roots=1):
    dev = R.dev
    G = rmat.Graph(scale, 16, seed=seed, device=dev)
    print(f"R-MAT scale {scale}, edgefactor 16, seed {seed}: {G.col.numel()} directed edges after dedupe; "
          f"{parts} buffers per level by contiguous vertex range, {'u32' if W == 32 else 'u64'} IDs, threshold {thr} B\n")
    print(HDR)
    for ri, root in enumerate(G.roots(n_roots, seed=seed)):
        tot = {"n": 0, "n_buf": parts, "raw": 0, "comp": 0, "enc_ms": 0.0, "dec_ms": 0.0, "enc_iso_ms": 0.0, "dec_iso_ms": 0.0}
        for level, f in enumerate(G.bfs_frontiers(root)):
            vals, off = streams.split_block(f, parts, 1 << scale)
            ids = streams.as_ids(vals, W).to(dev)
            r = R.batch(ids, off.to(dev), W, thr)
            for k in ("n", "raw", "comp", "enc_ms", "dec_ms", "enc_iso_ms", "dec_iso_ms", "cpu_enc_ms", "cpu_dec_ms"):
                if k in r:
                    tot[k] = tot.get(k, 0.0) + r[k]
            tot["host_bound"] = tot.get("host_bound", False) or r["host_bound"]
            if ri < per_level_roots:
                print(R.row(f"root {root} level {level} ({r['n']} IDs)", r))
        print(R.total(f"**root {root}, all levels** ({tot['n']} IDs)", tot))


def sweep(R):
    dev = R.dev
    print("Single sorted buffers (threshold 0); n/a = the stream would exceed the u32 ID space\n")
    print(HDR)
    for W in (32, 64):
        for k in range(5, 16):
            nbytes = 4 ** k
            n = nbytes // (W // 8)
            for mean in (1.0, 16.0, 4096.0):
                label = f"u{W} {nbytes >> 10} KB mean {int(mean)}"
                if W == 32 and n * mean >= 2 ** 32:
                    print(f"| {label} | 1 | {nbytes / 1e6:.3f} | n/a | | | | | | | | | |")
                    continue
                ids = streams.gap_stream(n, mean, seed=5, W=W, device=dev)
                off = torch.tensor([0, n], dtype=torch.int64, device=dev)
                print(R.row(label, R.batch(ids, off, W, 0, single=True)))
                del ids
    # BFS levels of up to ~1 MB (the one-launch paths of both directions) and just above (the general path)
    for n_buf, per in ((16, 2000), (16, 8000), (16, 16000), (16, 20000), (16, 100000)):
        counts = torch.full((n_buf,), per, dtype=torch.int64)
        ids, off = streams.batch_of_streams(counts, 16.0, seed=5, W=32, device=dev)
        print(R.total(f"level of {n_buf} buffers x {per} IDs, mean 16, threshold 1024", R.batch(ids.to(dev), off.to(dev), 32, 1024)))
    counts = streams.log_uniform_counts(64, 8, 12, 32, seed=5)
    ids, off = streams.batch_of_streams(counts, 16.0, seed=5, W=32, device=dev)
    print(R.total("level of 64 buffers 1 KB-16 KB (log-uniform), mean 16, threshold 1024", R.batch(ids.to(dev), off.to(dev), 32, 1024)))
    counts = streams.log_uniform_counts(4096, 8, 16, 32, seed=5)
    ids, off = streams.batch_of_streams(counts, 16.0, seed=5, W=32, device=dev)
    for thr in (0, 1024):
        print(R.total(f"batch of 4096 buffers 256 B-64 KB, mean 16, threshold {thr}", R.batch(ids.to(dev), off.to(dev), 32, thr)))


def run(a, cpu_timer=None):
    """The report of parsed arguments `a` (see main); cpu_timer: Runner's."""
    assert torch.cuda.is_available(), "needs a CUDA device (there is no CPU fallback)"
    dev = torch.device("cuda:0")
    B.lib()
    R = Runner(dev, a.reps, B.CODEC_BP128 if a.codec == "bp128" else B.CODEC_PFOR, a.graph, cpu_timer, a.scatter)
    if a.scatter:
        print("batch rows: bfsc_compress_batch_scatter into a slotted receive buffer (one slot per stream, the layout of "
              "exchange.SlotExchange) and bfsc_decompress_batch straight from the slots\n")
    if a.graph:
        print("timed runs replayed from CUDA graphs captured around the C-ABI calls (device-side time of the kernel chain)\n")
    print(f"encoder rule: {'BP128-D1 (mode 2, no exceptions)' if a.codec == 'bp128' else 'PFOR-D1 (mode 1)'}\n")
    if a.config == 3:
        rmat_config(R, a.scale or 22, 3, 32, 16, a.roots or 16, 1024)
    elif a.config == 4:
        rmat_config(R, a.scale or 25, 4, 64, 64, a.roots or 8, 1024)
    else:
        sweep(R)
    if a.json:
        print()
        print(json.dumps({"report": f"configs[{a.config - 1}]", "codec": a.codec, "graph_replay": bool(a.graph),
                          "peak_GBps": R.peak, "oracle_timed": cpu_timer is not None, "totals": R.totals}))


def add_arguments(ap):
    ap.add_argument("--scale", type=int, default=0)
    ap.add_argument("--roots", type=int, default=0)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--codec", default="pfor", choices=["pfor", "bp128"], help="encoder rule (bfsc_codec)")
    ap.add_argument("--graph", action="store_true", help="replay the timed calls from captured CUDA graphs")
    ap.add_argument("--json", action="store_true", help="one JSON line with the totals after the table")
    ap.add_argument("--scatter", action="store_true", help="batch rows through bfsc_compress_batch_scatter (streams into slots)")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[3, 4, 5])
    add_arguments(ap)
    run(ap.parse_args())


if __name__ == "__main__":
    main()
