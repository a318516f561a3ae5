#!/usr/bin/env python
"""bench.py — BASELINE.json metric on configs[1]: whole-file device-resident decode of the 1 GiB synthetic FASTQ
(seed 2, 50 Mbp reference, 16 KB blocks).  A step = one aceapex_decode_all over the whole archive.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--size BYTES]

Prints one JSON line.  N > 1: replicas only: every rank decodes
its own copy of the same archive, no data-path collective; value = bytes of all ranks / max time over ranks."""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "decompressed GB/s (whole-file, range) vs HBM roofline; random-read latency ms"
WORKLOAD = "configs[1]: 1 GiB synthetic FASTQ (seed 2, 50 Mbp reference), 16 KB blocks, whole-file decode_all"


def make_input(size):
    from paper_2606_18900_b200 import datagen, encoder
    x = datagen.fastq(2, size, 50_000_000)
    a = encoder.encode(x, block_size=16384)
    return x, a


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                o = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                   stdout=subprocess.PIPE, text=True, timeout=5).stdout.strip()
                self.rows.append([c.strip() for c in o.split(",")])
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        reasons = []
        for name, col in (("hw_slowdown", 2), ("hw_thermal_slowdown", 3), ("sw_thermal_slowdown", 4), ("sw_power_cap", 5)):
            if any(len(r) > col and r[col] == "Active" for r in self.rows):
                reasons.append(name)
        mx = max([int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()] or [0])
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": reasons, "samples": len(sm)}


def oracle_sample(archive, n_bytes_total, target_s=12.0):
    """Times the oracle (as it stands, one thread) on a bounded prefix of the same archive."""
    from oracle import acx_oracle
    import numpy as np
    h = acx_oracle.header(archive)
    bs = 1 << h["log2_bs"]
    probe = min(h["n_blocks"], max(1, (32 << 20) // bs))
    out = np.zeros(min(h["N"], h["n_blocks"] * bs) + 1, dtype=np.uint8)   # pre-faulted output
    t = time.perf_counter()
    acx_oracle.decode_prefix(archive, probe, out=out)
    dt = time.perf_counter() - t
    rate = probe * bs / dt
    nblk = int(min(h["n_blocks"], max(probe, target_s * rate // bs)))
    t = time.perf_counter()
    got = acx_oracle.decode_prefix(archive, nblk, out=out)
    dt = time.perf_counter() - t
    return got, dt, "first %d of %d blocks (%.0f MiB of %.0f MiB) of the same archive, 1 thread" % (
        nblk, h["n_blocks"], got.size / 2**20, n_bytes_total / 2**20)


def range_and_reads(torch, ar, x, stream):
    """The other two access modes of the metric on the same archive: range decode of the whole file as 64 MiB windows
    through a bounded output buffer held by the library (aceapex_decode_stream; one slot of an eighth of the file, reused
    window after window like the chunks of PAPER.md:107-109: measured faster on FASTQ than two slots of half the size, 169 against
    126 GB/s, because the cost of a window is its number of distinct source segments, not its size), and read-level
    access by index (batch 1, batch 4096)."""
    from paper_2606_18900_b200 import datagen
    N = x.size
    W = min(128 << 20, max(1 << 20, N // 8))
    ring = ar.new_output(W)
    st = ar.decode_stream(0, N, ring, W)                     # the library's device FNV consumer checks every block
    ok = st["bad_blocks"] == 0 and st["bytes"] == N
    seen = []

    def consumer(w, lo, hi, ptr, cuda_stream):               # a second pass handing three windows to the host for a byte compare
        if w in (0, st["n_windows"] // 2, st["n_windows"] - 1):
            torch.cuda.synchronize()
            off = ptr - ring.data_ptr()
            seen.append(bool(torch.equal(ring[off:off + hi - lo].cpu(), torch.from_numpy(x[lo:hi]))))
        return 0
    ar.decode_stream(0, N, ring, W, consumer=consumer)
    ok = ok and len(seen) == 3 and all(seen)
    best = min(ar.decode_stream(0, N, ring, W, consumer=lambda *a_: 0)["device_ms"] for _ in range(3))   # timed: a consumer that does nothing
    ar.check()
    idx = datagen.fastq_index(N)
    off = (idx & np.uint64((1 << 40) - 1)).astype(np.int64)
    ln = (idx >> np.uint64(40)).astype(np.int64)
    rng = np.random.default_rng(5)
    out = ar.new_output(int(ln.max()) * 4096)
    ids = rng.integers(0, idx.size, 300).astype(np.uint64)
    lat = []
    for k, i in enumerate(ids):
        one = np.array([i], dtype=np.uint64)
        t0 = time.perf_counter()
        ar.decode_reads(idx, one, out=out)               # synchronous: returns with the read in device memory
        if k >= 20:
            lat.append((time.perf_counter() - t0) * 1e3)
        if k < 20:
            ok = ok and out[:ln[i]].cpu().numpy().tobytes() == x[off[i]:off[i] + ln[i]].tobytes()
    bms = []
    for k in range(8):
        bi = rng.integers(0, idx.size, 4096).astype(np.uint64)
        t0 = time.perf_counter()
        ar.decode_reads(idx, bi, out=out)
        if k >= 1:
            bms.append((time.perf_counter() - t0) * 1e3)
    # seeks (Table 3): one block and 100 blocks at random block-aligned positions, nothing resident
    BS = ar.info()["block_size"]
    seeks = {}
    sbuf = ar.new_output(100 * BS)
    for blocks in (1, 100):
        sl = []
        for k in range(120):
            b = int(rng.integers(0, N // BS - blocks))
            t0 = time.perf_counter()
            ar.decode_range(b * BS, (b + blocks) * BS, out=sbuf)
            torch.cuda.synchronize()
            if k >= 20:
                sl.append((time.perf_counter() - t0) * 1e3)
        seeks["%d_blocks_ms_median" % blocks] = float(np.median(sl))
    ar.check()
    return {"range_decode": {"value": N / best / 1e6, "unit": "GB/s", "window_bytes": W, "ring_bytes": W, "windows": st["n_windows"], "ms": best,
                             "min_window_gbs": st["min_window_gbs"], "max_window_gbs": st["max_window_gbs"], "peak_device_bytes": st["peak_device_bytes"],
                             "through": "aceapex_decode_stream (ring inside the library; every block checked by its device FNV consumer in an untimed pass: %.2f ms with it)" % st["device_ms"]},
            "random_read_latency": {"batch1_ms_median": float(np.median(lat)), "batch1_ms_p99": float(np.percentile(lat, 99)),
                                    "batch4096_ms": float(np.median(bms)), "batch4096_us_per_read": float(np.median(bms)) * 1e3 / 4096,
                                    "reads_in_index": int(idx.size), "timer": "host wall clock around the synchronous C-ABI call"},
            "seek_latency": dict(seeks, graph_launches=ar.graph_launch_count(), timer="host wall clock around aceapex_decode_range + synchronize"),
            "bit_exact": ok}


def entropy_microbench(torch):
    """SURVEY.md 8(f) rank 1 / PAPER.md:135: the rANS stage alone on 256 MiB of exponentially distributed bytes, 4096 rows of 64 KB
    (the paper's DietGPU shape), through aceapex_rans_encode / aceapex_rans_decode; decode(encode(x)) == x is checked."""
    from paper_2606_18900_b200.aceapex import RansBatch
    rng = np.random.default_rng(6)
    rows = np.minimum(rng.exponential(scale=12.0, size=(4096, 65536)), 255).astype(np.uint8)
    hist = np.bincount(rows.ravel(), minlength=256).astype(np.int64)
    freq = np.maximum((hist * 2048) // hist.sum(), (hist > 0).astype(np.int64))      # 2^11 slots, every present symbol >= 1
    while freq.sum() != 2048:
        freq[int(np.argmax(freq))] += 1 if freq.sum() < 2048 else -1
    rb = RansBatch(freq.astype(np.uint16), 65536)
    d = torch.from_numpy(rows).cuda()
    enc, sizes = rb.new_encoded(4096)
    out = torch.empty_like(d)
    st = torch.cuda.current_stream()
    res = {}
    for name, fn in (("encode", lambda: rb.encode(d, enc, sizes)), ("decode", lambda: rb.decode(enc, sizes, 4096, out))):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(10):
            fn()
        e1.record(st)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 10
        res[name] = {"ms": ms, "value": rows.size / ms / 1e6, "unit": "GB/s of symbols"}
    res["bit_exact"] = bool(torch.equal(out, d)) and rb.status() == 0
    res["ratio"] = rows.size / float(sizes.sum().item())
    res["shape"] = "4096 rows x 64 KB, exponential bytes (scale 12), one static table, 32 interleaved states per row"
    res["context"] = "DietGPU on one H100: encode 364.9, decode 592.5 GB/s (PAPER.md:135); not on this box"
    return res


def launch_overhead(torch, stream):
    """SURVEY.md 8(c) S19 ("launch-overhead floor near 270 us"): the schedule of decode_all on an archive of one
    8-byte block: nothing to decode, so the time of a step is what its launches cost."""
    from paper_2606_18900_b200 import encoder
    from paper_2606_18900_b200.aceapex import Archive
    ar = Archive(encoder.encode(np.frombuffer(b"ACGTACGT", dtype=np.uint8), block_size=16384))
    ar.set_stream(stream)
    out = ar.new_output()
    res = {}
    for sched in (None, "fused"):
        for _ in range(5):
            ar.decode_all(out, schedule=sched)
        torch.cuda.synchronize()
        l0 = ar.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(200):
            ar.decode_all(out, schedule=sched)
        e1.record(stream)
        torch.cuda.synchronize()
        n = (ar.launch_count() - l0) / 200
        t0 = time.perf_counter()
        for _ in range(200):
            ar.decode_all(out, schedule=sched)
            torch.cuda.synchronize()
        wall = (time.perf_counter() - t0) / 200 * 1e3
        res[sched or "default"] = {"launches_per_step": n, "empty_step_ms_device": e0.elapsed_time(e1) / 200, "empty_step_ms_wall_with_sync": wall,
                                   "per_launch_us": e0.elapsed_time(e1) / 200 / max(n, 1) * 1e3}
    ar.close()
    return res


def max_over_ranks(dist, value, device):
    """Replicas only: the job time is the slowest rank's time.  dist = None: single process."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, bytes_per_rank, ms_per_step):
    """Whole-job throughput in GB/s: every rank decodes its own copy, the step time is the maximum over ranks."""
    return world * bytes_per_rank / (ms_per_step * 1e-3) / 1e9


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    x, a = make_input(args.size)
    times, nbytes, sample = [], 0, ""
    for i in range(args.warmup + args.steps):
        got, dt, sample = oracle_sample(a, x.size, target_s=max(2.0, min(12.0, 150.0 / (args.warmup + args.steps))))
        assert np.array_equal(got, x[:got.size])
        if i >= args.warmup:
            times.append(dt)
            nbytes = got.size
    ms = 1e3 * sum(times) / len(times)
    v = nbytes / (ms * 1e-3) / 1e9
    line = {"metric": METRIC, "value": v, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8",
            "data": "synthetic", "impl": "reference", "config": {"workload": WORKLOAD, "size_bytes": int(x.size)},
            "cpu_baseline": {"value": v, "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import numpy as np
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_18900_b200.aceapex import Archive
    x, a = make_input(args.size)
    ar = Archive(a, device="cuda:%d" % local)
    info = ar.info()
    out = ar.new_output()
    stream = torch.cuda.current_stream()
    ar.set_stream(stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident metric: archive and output in HBM, K steps between two events
    for _ in range(args.warmup):
        ar.decode_all(out)
    ar.check()
    out.fill_(0xA5)           # poison: bit_exact below then proves that the TIMED launches wrote every byte
    barrier()
    l0 = ar.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    per_step = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0.record(stream)
    for a_ev, b_ev in per_step:
        a_ev.record(stream)
        ar.decode_all(out)
        b_ev.record(stream)
    e1.record(stream)
    barrier()
    launches = ar.launch_count() - l0
    total_ms = e0.elapsed_time(e1)
    if args.step_only:
        ar.check()
        print(json.dumps({"step_only": True, "ms_per_step": total_ms / args.steps, "bit_exact": bool(torch.equal(out[:x.size].cpu(), torch.from_numpy(x)))}))
        return
    kernel_ms = sum(p.elapsed_time(q) for p, q in per_step) / args.steps
    ar.check()
    ok = bool(torch.equal(out[:x.size].cpu(), torch.from_numpy(x)))
    fnv_bad = ar.verify_fnv(out) if info["has_fnv"] else 0
    total_ms = max_over_ranks(dist, total_ms, "cuda")
    ms = total_ms / args.steps
    value = aggregate_value(world, x.size, ms)
    # clocks under the same load: the timed region is a few ms, too short for nvidia-smi, so the identical step is
    # repeated for ~1.5 s while the sampler runs; the sustained rate of that loop is reported beside the clocks
    sampler = ClockSampler(local)
    sampler.start()
    torch.cuda.synchronize()
    n_sus = max(50, int(1500.0 / max(ms, 0.01)))
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record(stream)
    for _ in range(n_sus):
        ar.decode_all(out)
    s1.record(stream)
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    sustained_ms = s0.elapsed_time(s1) / n_sus
    ar.check()
    # per-kernel device times, live: the library records CUDA events on the launch stream around the step's three launches
    ar.set_phase_timing(True)
    phase = [0.0, 0.0, 0.0]
    for _ in range(args.steps):
        ar.decode_all(out)
        phase = [p_ + q_ / args.steps for p_, q_ in zip(phase, ar.phase_times())]
    ar.set_phase_timing(False)

    # ---- the same decode with the two-launch flag schedule (completion flags instead of one launch per level), for comparison
    ar.decode_all(out, schedule="flags")
    l0 = ar.launch_count()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    p0.record(stream)
    for _ in range(3):
        ar.decode_all(out, schedule="flags")
    p1.record(stream)
    torch.cuda.synchronize()
    lv_ms = p0.elapsed_time(p1) / 3
    ar.check()
    ok = ok and bool(torch.equal(out[:x.size].cpu(), torch.from_numpy(x)))
    levels_info = {"ms_per_step": lv_ms, "value": x.size / (lv_ms * 1e-3) / 1e9, "unit": "GB/s",
                   "launches_per_step": (ar.launch_count() - l0) // 3}
    ar.decode_all(out, schedule="fused")
    torch.cuda.synchronize()
    p0.record(stream)
    for _ in range(3):
        ar.decode_all(out, schedule="fused")
    p1.record(stream)
    torch.cuda.synchronize()
    ar.check()
    ok = ok and bool(torch.equal(out[:x.size].cpu(), torch.from_numpy(x)))
    fu_ms = p0.elapsed_time(p1) / 3
    fused_info = {"ms_per_step": fu_ms, "value": x.size / (fu_ms * 1e-3) / 1e9, "unit": "GB/s", "launches_per_step": 1}

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D archive + decode + D2H output per step
    h_arch = torch.from_numpy(a).pin_memory()
    h_out = torch.empty(x.size, dtype=torch.uint8).pin_memory()
    for _ in range(2):
        ar.decode_all_host(h_arch, out, h_out)
    barrier()
    n_e2e = max(2, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        ar.decode_all_host(h_arch, out, h_out)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / n_e2e
    e2e_s = max_over_ranks(dist, e2e_s, "cuda")
    ok = ok and bool(torch.equal(h_out, torch.from_numpy(x)))
    e2e = {"value": world * x.size / e2e_s / 1e9, "unit": "GB/s", "h2d_bytes_per_step": int(a.size), "d2h_bytes_per_step": int(x.size)}

    extra = range_and_reads(torch, ar, x, stream) if world == 1 else None
    if extra is not None:
        ok = ok and extra["bit_exact"]
    micro = entropy_microbench(torch) if world == 1 and rank == 0 else None
    if micro is not None:
        ok = ok and micro["bit_exact"]
    lo_info = launch_overhead(torch, stream) if world == 1 and rank == 0 else None
    if rank != 0:
        return
    # ---- roofline of the step's kernels: algorithmic bytes C + M + N per step / measured time of its launches
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    alg_bytes = info["archive_bytes"] + info["total_match_bytes"] + info["raw_bytes"]
    achieved = alg_bytes / (kernel_ms * 1e-3) / 1e9
    # dram__bytes_read.sum + dram__bytes_write.sum of one step and what bounds each kernel, from the committed summary of one
    # ncu --set full capture (profiles/step_capture.json, written by paper_2606_18900_b200/ncu_summary.py); it names the
    # hash of the CUDA sources it was taken on, and is ignored when those have changed since
    cap = {}
    try:
        from paper_2606_18900_b200 import ncu_summary
        cap = json.load(open(os.path.join(ROOT, "profiles", "step_capture.json")))
        if cap.get("source_hash") != ncu_summary.source_hash():
            cap = {"stale": "the CUDA sources changed after profiles/step_capture.json was taken"}
    except Exception:
        pass
    kern = cap.get("kernels", {})
    traffic = cap.get("dram_bytes_per_step")
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured)" if peaks else "fallback 6650 GB/s",
                "kernel": "k_literals + k_copy (the launches of one decode_all step)", "kernel_ms": kernel_ms,
                "algorithmic_bytes": {"C": info["archive_bytes"], "M": info["total_match_bytes"], "N": info["raw_bytes"]},
                "capture": cap.get("stale") or cap.get("command")}
    # the dominant kernel on its own: k_literals reads the archive and writes the literal bytes; k_copy reads and writes
    # the match bytes
    lit_bytes = info["archive_bytes"] + info["total_lit_bytes"]
    cp_bytes = 2 * info["total_match_bytes"]
    t_copy = phase[1] + phase[2]
    roofline["per_kernel"] = [
        {"kernel": "k_literals", "ms": phase[0], "share_of_step": phase[0] / max(sum(phase), 1e-9), "algorithmic_bytes": lit_bytes,
         "achieved": lit_bytes / (phase[0] * 1e-3) / 1e9, "frac": lit_bytes / (phase[0] * 1e-3) / 1e9 / peak, "bound_observed": kern.get("k_literals", {}).get("bound_observed")},
        {"kernel": "k_copy", "ms": t_copy, "share_of_step": t_copy / max(sum(phase), 1e-9),
         "algorithmic_bytes": cp_bytes, "achieved": cp_bytes / (t_copy * 1e-3) / 1e9,
         "frac": cp_bytes / (t_copy * 1e-3) / 1e9 / peak, "bound_observed": kern.get("k_copy", {}).get("bound_observed")}]
    cpu, cpu_mt = None, None
    if args.cpu_baseline:
        got, dt, sample = oracle_sample(a, x.size)
        assert np.array_equal(got, x[:got.size])
        cpu = {"value": got.size / dt / 1e9, "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": sample}
        from oracle import acx_mt                      # second reported baseline: multithreaded CPU decoder, all host cores
        cores = os.cpu_count() or 1
        buf = np.zeros(x.size + 1, dtype=np.uint8)
        best = None
        for _ in range(2):
            t0 = time.perf_counter()
            got = acx_mt.decode(a, threads=cores, out=buf)
            dt = time.perf_counter() - t0
            best = dt if best is None else min(best, dt)
        assert np.array_equal(got, x)
        cpu_mt = {"value": x.size / best / 1e9, "unit": "GB/s", "cores": cores, "kind": "multithreaded CPU decoder (oracle/acx_mt.c)",
                  "sample": "the whole archive, best of 2"}
    line = {"metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "size_bytes": int(x.size), "archive_bytes": int(a.size),
                       "ratio": x.size / a.size, "n_blocks": info["n_blocks"], "n_segments": info["n_segments"], "max_level": info["max_level"],
                       "format": "ACX-B200 v3: q_min %d, LITQ %s, %.0f %% of the literal bytes in LITQ" % (info["q_min"], "aligned pairs" if info["q_mode"] else "bytes", 100.0 * info["total_litq_bytes"] / max(info["total_lit_bytes"], 1)),
                       "l2": "output (1 GiB) and archive are larger than the 126 MB L2; no flush needed",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "resident_warps": info["resident_warps"]},
            "bit_exact": ok and fnv_bad == 0,
            "clocks": dict(sampler.summary(), sustained_ms_per_step=sustained_ms, sustained_steps=n_sus), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "cpu_multithreaded": cpu_mt, "range_and_reads": extra, "flag_schedule": levels_info, "fused_schedule": fused_info,
            "entropy_microbench": micro, "launch_overhead": lo_info}
    print(json.dumps(line))
    if not (ok and fnv_bad == 0):
        sys.exit(1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=1 << 30, help="bytes of FASTQ (default: configs[1], 1 GiB)")
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--step-only", action="store_true", help="only the timed decode_all steps (for ncu captures); prints a short line")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
