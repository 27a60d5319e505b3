#!/usr/bin/env python
"""bench.py — headline benchmark of the bfsc hot path (BASELINE.json metric:
"encode/decode GB/s and % of HBM peak on 1 B200; compression ratio").

Workload (config.workload): BASELINE.json configs[1] — three synthetic sorted u32 streams of
2^24 IDs, seed 2: (a) geometric gaps mean 2, (b) mean 256, (c) mean 256 with 1 % of the gaps
replaced by U[2^16, 2^24). One STEP = one pass of the whole hot path over that batch:
bfsc_compress of a, b, c then bfsc_decompress of a, b, c (E0-E5, D0-D5 of SURVEY.md §8(a)).
value = (raw bytes encoded + raw bytes decoded) / time, inputs resident in HBM.
e2e   = the same through bfsc_compress_host / bfsc_decompress_host with pinned HOST buffers.
roofline = algorithmic bytes (raw + compressed) of the dominant call / its CUDA-event duration
           measured inside the timed region, against MEASURED_PEAKS.json hbm_gbs.
cpu_baseline = the oracle (oracle/, as it stands) on the host cores on the same workload.
`--impl reference` times the oracle alone (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

from paper_1704_00513_b200.workloads import streams  # noqa: E402

LOG2_N = 24
STREAMS = [("a_mean2", 2.0, 0.0), ("b_mean256", 256.0, 0.0), ("c_mean256_out1pct", 256.0, 0.01)]
SEED = 2
W = 32
METRIC = "codec_throughput_encode_plus_decode"
UNIT = "GB/s"
NCU_SUMMARIES = {"encode": "profiles/r2_enc_tiles_ncu_summary.txt", "decode": "profiles/r2_dec_tiles_ncu_summary.txt"}


def ncu_traffic(kind: str, stream: str):
    """dram__bytes_read.sum + dram__bytes_write.sum (bytes) of ONE launch of the encode / decode kernel on stream
    'a' | 'b' | 'c', read from the committed `ncu --set full` summary (profiles/README.md names the command that
    made it); None when the file or the section is missing."""
    path = os.path.join(ROOT, NCU_SUMMARIES[kind])
    try:
        sec, rd, wr = None, None, None
        for line in open(path):
            if line.startswith("== stream "):
                sec = line.split()[2]
            elif sec == stream and line.startswith("dram__bytes_read.sum "):
                rd = float(line.split()[1])
            elif sec == stream and line.startswith("dram__bytes_write.sum "):
                wr = float(line.split()[1])
        return None if rd is None or wr is None else int(round((rd + wr) * 1e6))     # ncu prints MB
    except OSError:
        return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 6 for i in range(4) if r[2 + i].startswith("Active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def make_streams(device, n):
    return [streams.gap_stream(n, mean, seed=SEED, W=W, outlier_frac=outl, sub=i, device=device)
            for i, (_, mean, outl) in enumerate(STREAMS)]


def np_view(t):
    return t.cpu().numpy().view(np.uint32 if W == 32 else np.uint64)


def max_over_ranks(x: float, world: int, device) -> float:
    """Replicas only: the job's time is the slowest rank's. MAX all-reduce over whatever backend
    the process group was initialised with (nccl on GPUs; gloo in the CPU test of this function)."""
    if world <= 1:
        return float(x)
    import torch.distributed as dist
    tt = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(per_rank_units: float, world: int, seconds: float) -> float:
    """value = units all ranks processed / max-over-ranks time (weak scaling: every rank does the same work)."""
    return world * per_rank_units / seconds


# --------------------------------------------------------------------------- oracle arm
def time_oracle(host_ids, threads, reps=1):
    """oracle encode+decode of every stream; returns (seconds, raw_bytes_processed, ratio)."""
    import oracle
    oracle.build()
    best = None
    raw = comp = 0
    for _ in range(reps):
        t0 = time.perf_counter()
        raw = comp = 0
        for a in host_ids:
            off = np.array([0, len(a)], dtype=np.uint64)
            s, so = oracle.compress_batch(a, off, 0, threads=threads)
            y, _ = oracle.decompress_batch(s, so, W, len(a), threads=threads)
            raw += 2 * a.nbytes
            comp += len(s)
            assert y[0] == a[0] and y[-1] == a[-1]
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best, raw, (raw / 2) / comp


def run_reference(args, rank, world):
    """This tier's reference arm: the oracle, as it stands, on the host cores — on the FULL workload (3 streams of
    2^log2n IDs, encode + decode per step: about 0.3 s at 16 threads), unless --steps of them would exceed
    --ref-budget-s; then, and only then, on the first 2^p IDs of every stream (said in config.sample)."""
    if rank != 0:
        return
    cores = len(os.sched_getaffinity(0))
    full = [np_view(t) for t in make_streams("cpu", 1 << args.log2n)]
    time_oracle([h[:1 << 16] for h in full], cores)                       # warm-up (builds the oracle's C library)
    cal, _, _ = time_oracle([h[:1 << 20] for h in full], cores)
    per_id = cal / (3 << 20)
    budget = args.ref_budget_s / max(args.steps + args.warmup, 1)
    p = args.log2n
    while p > 14 and per_id * (3 << p) > budget:
        p -= 1
    n = 1 << p
    host = [h[:n] for h in full]
    for _ in range(args.warmup):
        time_oracle(host, cores)
    times = []
    raw = ratio = 0
    for _ in range(args.steps):
        dt, raw, ratio = time_oracle(host, cores)
        times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    val = raw / (ms * 1e-3) / 1e9
    sample = (f"the full workload: all 2^{p} IDs of each of the 3 streams" if p == args.log2n else
              f"first 2^{p} of the 2^{args.log2n} IDs of each of the 3 streams (the full workload would exceed --ref-budget-s)")
    sample += f", encode+decode, {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic", "ratio": ratio,
        "config": workload_config(args.log2n, world) | {"sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_config_report(args):
    """`bench.py --config N`: the config-3/4/5 report of paper_1704_00513_b200/report.py with the oracle timed beside
    every row (same run, same inputs). The oracle runs its multi-threaded driver on all host cores
    under the PFOR rule, its serial functions under BP128 (the driver knows mode 1 only)."""
    import oracle
    from paper_1704_00513_b200 import report
    from paper_1704_00513_b200 import build as cuda_build
    cuda_build.build()
    oracle.build()
    cores = len(os.sched_getaffinity(0))

    def oracle_timer(ids, off, Wb, thr, codec):
        a = ids.cpu().numpy().view(np.uint32 if Wb == 32 else np.uint64)
        o = off.cpu().numpy().astype(np.uint64)
        threads = cores if codec == oracle.CODEC_PFOR else 0
        t0 = time.perf_counter()
        s, so = oracle.compress_batch(a, o, thr, threads=threads, codec=codec)
        t1 = time.perf_counter()
        y, _ = oracle.decompress_batch(s, so, Wb, len(a), threads=threads)
        t2 = time.perf_counter()
        assert len(a) == 0 or (y[0] == a[0] and y[len(a) - 1] == a[-1])
        return t1 - t0, t2 - t1

    print(f"oracle columns: oracle/ on {cores} host threads (PFOR rule; 1 thread under BP128), same buffers, same run\n")
    report.run(args, cpu_timer=oracle_timer)


def workload_config(log2n, world):
    """config of the JSON line: the same for both arms (the driver compares them)."""
    return {"workload": f"configs[1]: 3 sorted u32 streams of 2^{log2n} IDs (a: geometric gaps mean 2, b: mean 256, "
                        "c: mean 256 + 1% outliers in [2^16,2^24)), seed 2; step = compress a,b,c then decompress a,b,c",
            "raw_threshold_bytes": 0, "parallelism": "replicas only" if world > 1 else "single GPU"}


# --------------------------------------------------------------------------- CUDA arm
def run_ours(args, rank, local_rank, world):
    from paper_1704_00513_b200 import binding as B
    from paper_1704_00513_b200 import build as cuda_build
    if rank == 0:
        cuda_build.build()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    B.lib()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    n = 1 << args.log2n
    ids = make_streams(dev, n)
    S = len(ids)
    cap = B.compress_bound(n, W)
    outs = [torch.empty(cap, dtype=torch.uint8, device=dev) for _ in range(S)]
    nbytes = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(S)]
    backs = [torch.empty(n, dtype=ids[0].dtype, device=dev) for _ in range(S)]
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)
    ws = torch.empty(B.workspace_bytes(n, 1, W), dtype=torch.uint8, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    raw_bytes = n * (W // 8)

    def step():
        for s in range(S):
            B.compress(ids[s], n, W, 0, outs[s], nbytes[s], ws, status)
        for s in range(S):
            B.decompress(outs[s], cap, W, backs[s], n_out, ws, status)

    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    assert int(status.item()) == 0, f"device status {int(status.item())}"
    comp = [int(x.item()) for x in nbytes]
    for s in range(S):                                       # untimed sanity: decode == input
        assert torch.equal(backs[s], ids[s]), "decode != input"

    if args.ncu:
        # Capture mode (profiles/README.md): between cudaProfilerStart / Stop, ONE compress and ONE decompress call per
        # stream, in the order a, b, c — run under `ncu --profile-from-start off`; no number is reported from here.
        sampler.stop()
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        torch.cuda.synchronize()
        torch.cuda.profiler.start()
        for s in range(S):
            flush.zero_()
            B.compress(ids[s], n, W, 0, outs[s], nbytes[s], ws, status)
            flush.zero_()
            B.decompress(outs[s], cap, W, backs[s], n_out, ws, status)
        torch.cuda.synchronize()
        torch.cuda.profiler.stop()
        if rank == 0:
            print(json.dumps({"ncu_capture": "compress + decompress of streams a, b, c, one call each", "status": int(status.item())}))
        return

    mk = lambda: torch.cuda.Event(enable_timing=True)       # noqa: E731
    t0, t1 = mk(), mk()
    launches0 = B.kernel_launches()
    t_wait = time.time()
    while not sampler.rows and time.time() - t_wait < 3.0:   # nvidia-smi needs a moment to start streaming
        time.sleep(0.05)
    sampler.rows.clear()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()
    t0.record()
    for k in range(args.steps):
        step()
    t1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches_timed = B.kernel_launches() - launches0
    ms_total = t0.elapsed_time(t1)
    ms_total = max_over_ranks(ms_total, world, dev)
    ms_step = ms_total / args.steps
    # ---- per-call durations (roofline): CUDA events around a run of back-to-back launches of ONE call on
    # kCopies distinct copies of the stream (inputs and outputs rotate: > 250 MB of other traffic between a
    # buffer's write and its re-read, twice the L2), average per launch. No event sits between two launches:
    # an event record between two kernels costs 2-3 us of idle GPU and would be charged to the kernel.
    kCopies = 4
    reps = max(5, min(args.steps, 50))
    c_out = outs + [torch.empty(cap, dtype=torch.uint8, device=dev) for _ in range(kCopies - S)]
    c_back = backs + [torch.empty(n, dtype=ids[0].dtype, device=dev) for _ in range(kCopies - S)]
    kTrials = 5                                              # runs per call: median reported, min alongside
    enc_ms, dec_ms, enc_min, dec_min = [], [], [], []
    bp_enc_ms, bp_dec_ms = [], []                            # the same calls under the BP128 rule (FORMAT.md §7)
    ex_enc_ms = []                                           # bfsc_compress with BFSC_CODEC_FLAG_EXCLUSIVE (static first tiles, include/bfsc.h)
    nbytes_bp = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(S)]
    for s in range(S):
        c_ids = [ids[s]] + [ids[s].clone() for _ in range(kCopies - 1)]
        for c in range(kCopies):
            B.compress(c_ids[c], n, W, 0, c_out[c], nbytes[s], ws, status)
        torch.cuda.synchronize()

        def run_of(call):
            a0, a1 = mk(), mk()
            a0.record()
            for _ in range(reps):
                for c in range(kCopies):
                    call(c)
            a1.record()
            torch.cuda.synchronize()
            return a0.elapsed_time(a1) / (reps * kCopies)

        enc_call = lambda c: B.compress(c_ids[c], n, W, 0, c_out[c], nbytes[s], ws, status)          # noqa: E731
        dec_call = lambda c: B.decompress(c_out[c], cap, W, c_back[c], n_out, ws, status)           # noqa: E731
        enc_runs = [run_of(enc_call) for _ in range(kTrials)]
        for c in range(kCopies):
            dec_call(c)
        torch.cuda.synchronize()
        dec_runs = [run_of(dec_call) for _ in range(kTrials)]
        assert torch.equal(c_back[kCopies - 1], ids[s]), "decode != input"
        enc_ms.append(float(np.median(enc_runs)))
        dec_ms.append(float(np.median(dec_runs)))
        enc_min.append(min(enc_runs))
        dec_min.append(min(dec_runs))
        ex_call = lambda c: B.compress_codec(B.CODEC_PFOR | B.CODEC_FLAG_EXCLUSIVE, c_ids[c], n, W, 0, c_out[c], nbytes[s], ws, status)   # noqa: E731
        for c in range(kCopies):
            ex_call(c)
        torch.cuda.synchronize()
        ex_enc_ms.append(float(np.median([run_of(ex_call) for _ in range(kTrials)])))
        bp_call = lambda c: B.compress_codec(B.CODEC_BP128, c_ids[c], n, W, 0, c_out[c], nbytes_bp[s], ws, status)   # noqa: E731
        for c in range(kCopies):
            bp_call(c)
        torch.cuda.synchronize()
        bp_enc_ms.append(float(np.median([run_of(bp_call) for _ in range(kTrials)])))
        c_back[kCopies - 1].zero_()
        bp_dec_ms.append(float(np.median([run_of(dec_call) for _ in range(kTrials)])))
        assert torch.equal(c_back[kCopies - 1], ids[s]), "BP128: decode != input"
        del c_ids
    assert int(status.item()) == 0, f"device status {int(status.item())}"
    value = whole_job_value(2 * S * raw_bytes, world, ms_step * 1e-3) / 1e9
    # nvidia-smi is sampled every 20 ms from before the timed region (a few milliseconds long) to the end of the per-call
    # runs above (the same calls, a few seconds of them): the clocks under this load, not of one idle instant
    clocks = sampler.stop()
    clocks["window"] = "timed region + the per-call runs of the same calls that follow it"

    # ---- the batched path, reported beside the headline, not in it: (1) BASELINE configs[4]'s batch of 4096 buffers of
    # 256 B - 64 KB (log-uniform), gaps of mean 16, u32, threshold 0; (2) the largest BFS level of configs[3] (R-MAT 25,
    # u64 IDs, 64 destination buffers by contiguous vertex range, 1 KB threshold). One bfsc_compress_batch /
    # bfsc_decompress_batch per call, on rotating copies (> 2 x L2 between a buffer's write and its re-read); timed
    # twice: enqueued from Python (host time included when it is the longer one) and replayed from a CUDA graph
    # captured around the same C-ABI calls (device-side time of the kernel chain).
    batch = None
    if rank == 0 and args.log2n == LOG2_N and not args.no_batch:
        def measure_batch(b_ids, b_off, Wb, thr, label):
            bn, nbuf = b_ids.numel(), b_off.numel() - 1
            counts_l = (b_off[1:] - b_off[:-1]).tolist()
            bcap = B.batch_compress_bound(counts_l, Wb)
            kB = int(max(3, min(8, -(-(300 << 20) // (2 * bn * (Wb // 8) + 1)))))
            bi = [b_ids] + [b_ids.clone() for _ in range(kB - 1)]
            bo = [torch.empty(bcap, dtype=torch.uint8, device=dev) for _ in range(kB)]
            bb = [torch.empty(bn, dtype=b_ids.dtype, device=dev) for _ in range(kB)]
            b_out_off = torch.zeros(nbuf + 1, dtype=torch.int64, device=dev)
            b_id_off = torch.zeros(nbuf + 1, dtype=torch.int64, device=dev)
            bws = torch.empty(B.workspace_bytes(bn, nbuf, Wb), dtype=torch.uint8, device=dev)
            enc = lambda c: B.compress_batch(bi[c], b_off, nbuf, Wb, thr, bo[c], b_out_off, bws, status)         # noqa: E731
            dec = lambda c: B.decompress_batch(bo[c], b_out_off, nbuf, Wb, bb[c], b_id_off, bws, status)      # noqa: E731

            def run_b(call, reps_b=10):
                for c in range(kB):
                    call(c)
                torch.cuda.synchronize()
                a0, a1 = mk(), mk()
                a0.record()
                for _ in range(reps_b):
                    for c in range(kB):
                        call(c)
                a1.record()
                torch.cuda.synchronize()
                return a0.elapsed_time(a1) / (reps_b * kB)

            def run_graph(call, reps_b=10):
                side = torch.cuda.Stream(device=dev)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.stream(side):
                    with torch.cuda.graph(g, stream=side):
                        for c in range(kB):
                            call(c)
                torch.cuda.synchronize()
                g.replay()
                torch.cuda.synchronize()
                a0, a1 = mk(), mk()
                a0.record()
                for _ in range(reps_b):
                    g.replay()
                a1.record()
                torch.cuda.synchronize()
                return a0.elapsed_time(a1) / (reps_b * kB)

            b_enc = float(np.median([run_b(enc) for _ in range(3)]))
            b_dec = float(np.median([run_b(dec) for _ in range(3)]))
            g_enc = float(np.median([run_graph(enc) for _ in range(3)]))
            g_dec = float(np.median([run_graph(dec) for _ in range(3)]))
            assert int(status.item()) == 0 and torch.equal(bb[kB - 1], b_ids) and torch.equal(b_id_off, b_off), "batch: decode != input"
            b_raw, b_comp = bn * (Wb // 8), int(b_out_off[-1].item())
            pk = peaks()[0]
            # the same batch through the data path of the exchange: every stream into its own slot of a
            # receive buffer (bfsc_compress_batch_scatter: the encoder's stores are the transfer), decoded where it lies
            slot = max(B.compress_bound(c, Wb) for c in set(counts_l))
            pitch = (slot + 255) // 256 * 256
            recv = [torch.empty(nbuf * pitch, dtype=torch.uint8, device=dev) for _ in range(kB)]
            dsts = [r.data_ptr() + pitch * torch.arange(nbuf, dtype=torch.int64, device=dev) for r in recv]
            slot_off = pitch * torch.arange(nbuf + 1, dtype=torch.int64, device=dev)
            sizes = torch.zeros(nbuf, dtype=torch.int64, device=dev)
            sca = lambda c: B.compress_batch_scatter(B.CODEC_PFOR, bi[c], b_off, nbuf, Wb, thr, dsts[c], slot, sizes, bws, status)   # noqa: E731
            dsl = lambda c: B.decompress_batch(recv[c], slot_off, nbuf, Wb, bb[c], b_id_off, bws, status)                            # noqa: E731
            for x in bb:
                x.zero_()
            g_sca = float(np.median([run_graph(sca) for _ in range(3)]))
            g_dsl = float(np.median([run_graph(dsl) for _ in range(3)]))
            assert int(status.item()) == 0 and torch.equal(bb[kB - 1], b_ids) and int(sizes.sum().item()) == b_comp, "scatter: decode != input"
            del recv, dsts
            return {"workload": label, "n_buf": nbuf, "raw_bytes": b_raw, "ratio": b_raw / b_comp,
                    "scatter_encode_graph_ms": g_sca, "decode_from_slots_graph_ms": g_dsl,
                    "encode_ms": b_enc, "decode_ms": b_dec, "encode_graph_ms": g_enc, "decode_graph_ms": g_dec,
                    "encode_GBps_in": b_raw / g_enc / 1e6, "decode_GBps_out": b_raw / g_dec / 1e6,
                    "encode_frac_of_peak": (b_raw + b_comp) / g_enc / 1e6 / pk, "decode_frac_of_peak": (b_raw + b_comp) / g_dec / 1e6 / pk,
                    "encode_frac_of_peak_enqueued": (b_raw + b_comp) / b_enc / 1e6 / pk,
                    "decode_frac_of_peak_enqueued": (b_raw + b_comp) / b_dec / 1e6 / pk,
                    "note": "*_graph_ms and the fractions: replayed from a CUDA graph (device-side time of the call's kernel chain); "
                            "encode_ms / decode_ms: enqueued from Python, per call incl. the host's time when that is the longer one"}

        counts = streams.log_uniform_counts(4096, 8, 16, 32, seed=5)
        b_ids, b_off = streams.batch_of_streams(counts, 16.0, seed=5, W=W, device=dev)
        batch = {"b4096": measure_batch(b_ids.to(dev), b_off.to(dev), W, 0,
                                        "configs[4] batch: 4096 buffers of 256 B-64 KB (log-uniform), gaps mean 16, u32, threshold 0, seed 5")}
        del b_ids, b_off
        try:
            from paper_1704_00513_b200.workloads import rmat
            G = rmat.Graph(25, 16, seed=4, device=dev)
            root = G.roots(1, seed=4)[0]
            big = max(G.bfs_frontiers(root), key=lambda f: f.numel())
            del G
            torch.cuda.empty_cache()
            vals, off64 = streams.split_block(big, 64, 1 << 25)
            batch["rmat25_level"] = measure_batch(streams.as_ids(vals, 64).to(dev), off64.to(dev), 64, 1024,
                                                  f"configs[3]: largest BFS level of R-MAT 25 (seed 4, first root), {vals.numel()} u64 IDs "
                                                  "in 64 buffers by contiguous vertex range, threshold 1 KB")
            del vals, off64, big
            torch.cuda.empty_cache()
        except torch.cuda.OutOfMemoryError:
            batch["rmat25_level"] = None

    # ---- frontier bitmaps (FORMAT.md §9), beside the headline: stream a given as the bitmap of its IDs
    # (one bit per vertex: the form the BFS holds its frontier in) through bfsc_compress_bitmap /
    # bfsc_decompress_to_bitmap, on rotating copies; the stream is byte-identical to the ID-list call's (checked).
    bitmap = None
    if rank == 0 and args.log2n == LOG2_N and not args.no_batch:
        a_ids = ids[0].to(torch.int64) & 0xFFFFFFFF
        n_bits = int(a_ids.max().item()) + 1
        words = ((n_bits + 31) // 32 + 3) // 4 * 4
        bits = torch.zeros(words * 32, dtype=torch.bool, device=dev)
        bits[a_ids] = True
        bm = (bits.view(words, 32).to(torch.int64) << torch.arange(32, dtype=torch.int64, device=dev)).sum(1)
        bm = (bm & 0xFFFFFFFF).to(torch.uint32).view(torch.int32)
        del bits, a_ids
        kC = 4
        bms = [bm] + [bm.clone() for _ in range(kC - 1)]
        bm_back = [torch.zeros(words, dtype=torch.int32, device=dev) for _ in range(kC)]
        ws_bm = torch.empty(B.bitmap_workspace_bytes(n_bits, W), dtype=torch.uint8, device=dev)
        ws_d = torch.empty(B.workspace_bytes(n_bits, 1, W), dtype=torch.uint8, device=dev)
        nb_bm = torch.zeros(1, dtype=torch.int64, device=dev)
        enc_bm = lambda c: B.compress_bitmap(B.CODEC_PFOR, bms[c], n_bits, 0, W, 0, c_out[c], nb_bm, ws_bm, status)          # noqa: E731
        dec_bm = lambda c: B.decompress_to_bitmap(c_out[c], cap, W, 0, bm_back[c], n_bits, n_out, ws_d, status)             # noqa: E731

        def run_bm(call):
            for c in range(kC):
                call(c)
            torch.cuda.synchronize()
            a0, a1 = mk(), mk()
            a0.record()
            for _ in range(reps):
                for c in range(kC):
                    call(c)
            a1.record()
            torch.cuda.synchronize()
            return a0.elapsed_time(a1) / (reps * kC)

        bm_enc = float(np.median([run_bm(enc_bm) for _ in range(kTrials)]))
        comp_bm = int(nb_bm.item())
        bm_dec = float(np.median([run_bm(dec_bm) for _ in range(kTrials)]))
        assert int(status.item()) == 0 and comp_bm == comp[0], "bitmap stream != ID-list stream"
        mask_tail = torch.equal(bm_back[kC - 1][:n_bits // 32], bm[:n_bits // 32])
        assert mask_tail and int(n_out.item()) == n, "bitmap decode != input"
        # Algorithm 4 lines 10-13 fused into the decode (bfsc_decompress_to_frontier): every ID is new (visited bitmaps zeroed
        # outside the timed region), one call per fresh (frontier, visited) pair, 8 pairs back to back, best of 3 runs
        kF = 8
        fr_b = [torch.zeros(words, dtype=torch.int32, device=dev) for _ in range(kF)]
        vis_b = [torch.zeros(words, dtype=torch.int32, device=dev) for _ in range(kF)]
        fr_runs = []
        for _ in range(3):
            for c in range(kF):
                fr_b[c].zero_(); vis_b[c].zero_()
            torch.cuda.synchronize()
            a0, a1 = mk(), mk()
            a0.record()
            for c in range(kF):
                B.decompress_to_frontier(c_out[c % kC], cap, W, 0, fr_b[c], vis_b[c], n_bits, n_out, ws_d, status)
            a1.record()
            torch.cuda.synchronize()
            fr_runs.append(a0.elapsed_time(a1) / kF)
        assert int(status.item()) == 0 and torch.equal(fr_b[0][:n_bits // 32], bm[:n_bits // 32]) and torch.equal(vis_b[kF - 1], fr_b[kF - 1])
        bm_fr = float(min(fr_runs))
        del fr_b, vis_b
        alg_bm = n_bits // 8 + comp_bm
        pk = peaks()[0]
        bitmap = {"workload": f"stream a as a frontier bitmap: {n_bits} bits, {n} set (1 in {n_bits / n:.2f})", "n_bits": n_bits,
                  "bitmap_bytes": n_bits // 8, "stream_bytes": comp_bm, "encode_ms": bm_enc, "decode_ms": bm_dec, "decode_to_frontier_ms": bm_fr,
                  "id_list_encode_ms": enc_ms[0], "id_list_decode_ms": dec_ms[0],
                  "encode_frac_of_peak": alg_bm / bm_enc / 1e6 / pk, "decode_frac_of_peak": alg_bm / bm_dec / 1e6 / pk,
                  "note": "algorithmic bytes = bitmap + stream (the ID list is never materialised); the decode ORs into a bitmap that "
                          "already holds the bits after the first pass (same work: one atomic OR per touched word group)"}
        del bms, bm_back, bm, ws_bm, ws_d
        # a late-BFS VISITED bitmap through the container of FORMAT.md §10 (bfsc_compress_vbitmap / bfsc_decompress_vbitmap): 2^25
        # vertices, 98 % visited, the unvisited ones in runs of 16 — the clear bits are listed
        vb_bits = 1 << 25
        vb_bm = ~streams.frontier_bitmap(vb_bits, 0.02, seed=3, run=16).to(dev)
        vb_in = [vb_bm.clone() for _ in range(kC)]
        vb_cap = B.vbitmap_bound(vb_bits)
        vb_out = [torch.empty(vb_cap, dtype=torch.uint8, device=dev) for _ in range(kC)]
        vb_back = [torch.zeros_like(vb_bm) for _ in range(kC)]
        vb_ws = torch.empty(B.vbitmap_workspace_bytes(vb_bits), dtype=torch.uint8, device=dev)
        vb_nb = torch.zeros(1, dtype=torch.int64, device=dev)
        vb_enc = float(np.median([run_bm(lambda c: B.compress_vbitmap(B.CODEC_PFOR, vb_in[c], vb_bits, vb_out[c], vb_nb, vb_ws, status)) for _ in range(3)]))
        vb_dec = float(np.median([run_bm(lambda c: B.decompress_vbitmap(vb_out[c], vb_cap, vb_back[c], vb_bits, vb_ws, status)) for _ in range(3)]))
        assert int(status.item()) == 0 and torch.equal(vb_back[kC - 1], vb_bm), "visited bitmap: decode != input"
        bitmap["visited"] = {"workload": f"{vb_bits} vertices, 98 % visited, unvisited in runs of 16", "bitmap_bytes": vb_bits // 8,
                             "container_bytes": int(vb_nb.item()), "kind": int(vb_out[0][6].item()), "encode_ms": vb_enc, "decode_ms": vb_dec}
        del vb_in, vb_out, vb_back, vb_ws

    # ---- end to end through the host-buffer C-ABI calls (pinned host memory) ----
    e2e = None
    if not args.no_e2e:
        h_ids = [t.cpu().pin_memory() for t in ids]
        h_out = [torch.empty(cap, dtype=torch.uint8).pin_memory() for _ in range(S)]
        h_back = torch.empty(n, dtype=ids[0].dtype).pin_memory()
        scratch = torch.empty(B.host_scratch_bytes(n, W) + 256, dtype=torch.uint8, device=dev)
        e_steps = max(1, min(args.steps, 5))

        # Two host threads, two streams: compress calls (H2D-heavy) on one, decompress calls (D2H-heavy) on the
        # other, stream s decompressed as soon as its compress call has returned: PCIe runs in both directions.
        scratch2 = torch.empty(B.host_scratch_bytes(n, W) + 256, dtype=torch.uint8, device=dev)
        st_enc, st_dec = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        e_comp = [0] * S

        def e2e_step():
            done = [threading.Event() for _ in range(S)]
            err = []

            def enc_side():
                try:
                    with torch.cuda.stream(st_enc):
                        for s in range(S):
                            e_comp[s] = B.compress_host(h_ids[s], W, 0, h_out[s], scratch)
                            done[s].set()
                except Exception as ex:                       # noqa: BLE001
                    err.append(ex)
                    for d in done:
                        d.set()

            def dec_side():
                try:
                    with torch.cuda.stream(st_dec):
                        for s in range(S):
                            done[s].wait()
                            if err:
                                return
                            B.decompress_host(h_out[s], e_comp[s], W, h_back, scratch2)
                except Exception as ex:                       # noqa: BLE001
                    err.append(ex)

            ts = [threading.Thread(target=enc_side), threading.Thread(target=dec_side)]
            for t in ts:
                t.start()
            for t in ts:
                t.join()
            if err:
                raise err[0]

        e2e_step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        w0 = time.perf_counter()
        for _ in range(e_steps):
            e2e_step()
        torch.cuda.synchronize()
        e_ms = 1e3 * (time.perf_counter() - w0) / e_steps
        e_ms = max_over_ranks(e_ms, world, dev)
        assert torch.equal(h_back, h_ids[S - 1])
        e2e = {"value": whole_job_value(2 * S * raw_bytes, world, e_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": e_ms,
               "h2d_bytes_per_step": S * raw_bytes + sum(comp), "d2h_bytes_per_step": sum(comp) + S * raw_bytes + 32 * S,
               "api": "bfsc_compress_host + bfsc_decompress_host, pinned host buffers; compress calls and decompress calls "
                      "from two host threads on two streams (stream s is decompressed as soon as its compress call returned)"}

    if rank != 0:
        return
    peak, peak_src = peaks()
    per = {}
    for s, (name, _, _) in enumerate(STREAMS):
        alg = raw_bytes + comp[s] + 8
        per[name] = {"ratio": raw_bytes / comp[s], "bits_per_id": 8 * comp[s] / n,
                     "encode_ms": enc_ms[s], "decode_ms": dec_ms[s], "encode_ms_min": enc_min[s], "decode_ms_min": dec_min[s],
                     "encode_GBps_in": raw_bytes / enc_ms[s] / 1e6, "decode_GBps_out": raw_bytes / dec_ms[s] / 1e6,
                     "encode_alg_GBps": alg / enc_ms[s] / 1e6, "decode_alg_GBps": alg / dec_ms[s] / 1e6,
                     "encode_frac_of_peak": alg / enc_ms[s] / 1e6 / peak, "decode_frac_of_peak": alg / dec_ms[s] / 1e6 / peak,
                     "encode_frac_of_8TBps": alg / enc_ms[s] / 1e6 / 8000.0, "decode_frac_of_8TBps": alg / dec_ms[s] / 1e6 / 8000.0}
        cb = int(nbytes_bp[s].item())
        alg_bp = raw_bytes + cb + 8
        per[name]["bp128"] = {"ratio": raw_bytes / cb, "bits_per_id": 8 * cb / n, "encode_ms": bp_enc_ms[s], "decode_ms": bp_dec_ms[s],
                              "encode_alg_GBps": alg_bp / bp_enc_ms[s] / 1e6, "decode_alg_GBps": alg_bp / bp_dec_ms[s] / 1e6,
                              "encode_frac_of_peak": alg_bp / bp_enc_ms[s] / 1e6 / peak, "decode_frac_of_peak": alg_bp / bp_dec_ms[s] / 1e6 / peak,
                              "encode_frac_of_8TBps": alg_bp / bp_enc_ms[s] / 1e6 / 8000.0, "decode_frac_of_8TBps": alg_bp / bp_dec_ms[s] / 1e6 / 8000.0}
        per[name]["encode_exclusive_flag"] = {"encode_ms": ex_enc_ms[s], "encode_alg_GBps": alg / ex_enc_ms[s] / 1e6,
                                              "encode_frac_of_peak": alg / ex_enc_ms[s] / 1e6 / peak,
                                              "encode_frac_of_8TBps": alg / ex_enc_ms[s] / 1e6 / 8000.0,
                                              "note": "BFSC_CODEC_FLAG_EXCLUSIVE: the caller vouches that nothing else runs on the device (include/bfsc.h)"}
    # dominant kernel = k_enc_tiles<32> (96 of the 160 us of a step); the roofline object is that of its SLOWEST call,
    # the one furthest from the roofline (stream c: exceptions); a and b beside it
    names = [nm for nm, _, _ in STREAMS]
    dom_i = int(np.argmax(enc_ms))
    dom = names[dom_i]
    key = "abc"[dom_i]
    full = args.log2n == LOG2_N
    roof = {"bound": "hbm", "kernel": f"k_enc_tiles<32, 0> (+ its 1-CTA k_enc_plan): the bfsc_compress call on stream {key}, the slowest of a, b, c",
            "achieved": per[dom]["encode_alg_GBps"],
            "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": per[dom]["encode_alg_GBps"] / peak,
            "algorithmic_bytes_per_launch": raw_bytes + comp[dom_i] + 8,
            "traffic": ncu_traffic("encode", key) if full else None, "traffic_source": NCU_SUMMARIES["encode"],
            "per_stream": {"abc"[i]: {"encode_frac": per[names[i]]["encode_frac_of_peak"], "decode_frac": per[names[i]]["decode_frac_of_peak"],
                                      "encode_traffic": ncu_traffic("encode", "abc"[i]) if full else None,
                                      "decode_traffic": ncu_traffic("decode", "abc"[i]) if full else None} for i in range(S)},
            "decode": {"kernel": f"k_dec_tiles<32, 0, 0, 0, 0>: the bfsc_decompress call on stream {key}", "achieved": per[dom]["decode_alg_GBps"],
                       "frac": per[dom]["decode_alg_GBps"] / peak, "traffic": ncu_traffic("decode", key) if full else None,
                       "traffic_source": NCU_SUMMARIES["decode"]}}
    cpu = None
    if not args.no_cpu:
        cores = len(os.sched_getaffinity(0))
        host = [np_view(t) for t in ids]                     # the whole workload: same config as the GPU line
        dt, raw, _ = time_oracle(host, cores)
        m1 = 1 << min(args.log2n, 20)
        dt1, raw1, _ = time_oracle([h[:m1] for h in host], 1)
        cpu = {"value": raw / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
               "single_thread": {"value": raw1 / dt1 / 1e9, "unit": UNIT, "sample": f"first 2^{min(args.log2n, 20)} IDs of each stream, 1 thread"},
               "sample": f"the full workload: all 2^{args.log2n} IDs of each of the 3 streams, encode+decode, {cores} threads, 1 pass"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32",
        "data": "synthetic",
        "config": workload_config(args.log2n, world) | {
                   "l2_policy": "inputs larger than L2: >=170 MB of other streams' traffic between any write and its re-read",
                   "per_call_timing": "events around runs of back-to-back launches of one call on 4 rotating copies of the stream, "
                                      "average per launch; median of 5 runs (min alongside)"},
        "ratio": {k: v["ratio"] for k, v in per.items()},
        "encode_GBps_in": S * raw_bytes / sum(enc_ms) / 1e6, "decode_GBps_out": S * raw_bytes / sum(dec_ms) / 1e6,
        "per_stream": per, "batch": batch, "bitmap": bitmap, "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches_timed), "clocks": clocks,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1500)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--log2n", type=int, default=LOG2_N, help="IDs per stream = 2^log2n (default: the BASELINE size)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--ncu", action="store_true", help="capture mode for ncu --profile-from-start off: one compress + one "
                    "decompress per stream between cudaProfilerStart/Stop, nothing timed (profiles/README.md)")
    ap.add_argument("--no-batch", action="store_true", help="skip the batched-path section (4096-buffer batch, R-MAT 25 level)")
    ap.add_argument("--ref-budget-s", type=float, default=90.0, help="--impl reference: CPU seconds for the whole run")
    ap.add_argument("--config", type=int, default=0, choices=[0, 3, 4, 5],
                    help="instead of the bench line: the report of BASELINE configs 3, 4 or 5 (paper_1704_00513_b200/report.py) "
                         "with the oracle timed beside every row; takes report.py's flags (--graph --codec --json --scale --roots --reps)")
    from paper_1704_00513_b200 import report as _report
    _report.add_arguments(ap)
    args = ap.parse_args()
    if args.config:
        run_config_report(args)
        return
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_ours(args, rank, local_rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
