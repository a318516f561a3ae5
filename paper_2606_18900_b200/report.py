#!/usr/bin/env python
"""Measurements for BASELINE.json configs[0..4] (one JSON line per measurement).

  python -m paper_2606_18900_b200.report --config 1            # 1 GiB FASTQ: whole-file, range windows, reads
  python -m paper_2606_18900_b200.report --config 2            # 3.1 GB FASTA + 10^6 region reads (batch 1 / 4096)
  python -m paper_2606_18900_b200.report --config 3 --size N   # N bytes of FASTA (default 50 GiB) through an 8 GiB ring
  python -m paper_2606_18900_b200.report --config 4            # block-size sweep on the configs[1] FASTQ, launch overhead
  python -m paper_2606_18900_b200.report --config 5            # the rANS stage alone (PAPER.md:135 shape)
  python -m paper_2606_18900_b200.report --config 6            # encoder options (level cap, source window, LITQ mode) vs speed
  python -m paper_2606_18900_b200.report --config 7            # one isolated 64 MiB window of configs[1] (the ncu target of range decode)

Everything is verified against the ORIGINAL bytes (direct compare where the data fits, per-block FNV-1a otherwise).
Timing: CUDA events on the handle's stream around the C-ABI calls, after warm-up; GB = 10^9 bytes.
CPU baselines (oracle, multithreaded decoder) are timed by bench.py, not here: the product never imports oracle/."""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

PEAK_FALLBACK = 6650.0


def peak_gbs():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured"
    except Exception:
        return PEAK_FALLBACK, "fallback"


def emit(**kw):
    print(json.dumps(kw), flush=True)


def timed(torch, stream, fn, reps, warmup=1):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def roofline(info, ms, out_bytes=None):
    peak, how = peak_gbs()
    n = info["raw_bytes"] if out_bytes is None else out_bytes
    scale = n / max(info["raw_bytes"], 1)
    alg = (info["archive_bytes"] + info["total_match_bytes"] + info["raw_bytes"]) * scale
    ach = alg / (ms * 1e-3) / 1e9
    return {"bound": "hbm", "achieved": ach, "peak": peak, "peak_source": how, "unit": "GB/s", "frac": ach / peak,
            "frac_of_8TBs": ach / 8000.0}


def whole_file(torch, ar, x, label, reps=5):
    stream = torch.cuda.current_stream()
    ar.set_stream(stream)
    out = ar.new_output()
    info = ar.info()
    res = {}
    xt = torch.from_numpy(x).to(out.device) if x is not None else None
    for sched in (None, "flags", "fused"):
        out.zero_()
        ar.decode_all(out, schedule=sched)
        ar.check()
        ok = bool(torch.equal(out[:info["raw_bytes"]], xt)) if xt is not None else None
        fnv_bad = ar.verify_fnv(out) if info["has_fnv"] else None
        l0 = ar.launch_count()
        ms = timed(torch, stream, lambda: ar.decode_all(out, schedule=sched), reps)
        res[sched or "default"] = {"ms": ms, "GBps": info["raw_bytes"] / ms / 1e6, "bit_exact": ok, "fnv_bad_blocks": fnv_bad,
                                   "launches": (ar.launch_count() - l0) // (reps + 1)}
    d = res["default"]
    emit(config=label, what="decode_all", raw_bytes=info["raw_bytes"], archive_bytes=info["archive_bytes"],
         ratio=info["raw_bytes"] / info["archive_bytes"], n_blocks=info["n_blocks"], block_size=info["block_size"],
         max_level=info["max_level"], schedules=res, roofline=roofline(info, d["ms"]))
    del out, xt
    return res


def windows(torch, ar, x, label, window, ring_slots, reps=1, sample_check=None):
    """Whole file as consecutive windows through a ring of `ring_slots` slots: aceapex_decode_stream owns the window order, the
    slot rotation and the resident registration.  Pass 1: the library's device FNV consumer checks every block; pass 2:
    a consumer that compares sampled windows with the original bytes; then `reps` timed passes with a consumer that does
    nothing."""
    stream = torch.cuda.current_stream()
    ar.set_stream(stream)
    info = ar.info()
    N = info["raw_bytes"]
    ring = ar.new_output(window * ring_slots)
    st = ar.decode_stream(0, N, ring, window)
    bad = st["bad_blocks"] if info["has_fnv"] else 0
    mism = []

    def consumer(w, lo, hi, ptr, cuda_stream):
        if x is not None and (sample_check is None or w in sample_check):
            torch.cuda.synchronize()
            off = ptr - ring.data_ptr()
            if not torch.equal(ring[off:off + hi - lo].cpu(), torch.from_numpy(x[lo:hi])):
                mism.append(w)
        return 0
    ar.decode_stream(0, N, ring, window, consumer=consumer)
    best = None
    for _ in range(max(reps, 1)):
        t = ar.decode_stream(0, N, ring, window, consumer=lambda *a_: 0)
        best = t if best is None or t["device_ms"] < best["device_ms"] else best
    ar.check()
    emit(config=label, what="range_windows_through_ring", window_bytes=window, ring_bytes=window * ring_slots, windows=best["n_windows"],
         total_ms=best["device_ms"], GBps=N / best["device_ms"] / 1e6, GBps_min=best["min_window_gbs"], GBps_max=best["max_window_gbs"],
         total_ms_with_fnv_consumer=st["device_ms"], bad=int(bad) + len(mism), roofline=roofline(info, best["device_ms"]),
         peak_device_bytes=best["peak_device_bytes"], torch_peak_bytes=int(torch.cuda.max_memory_allocated()))
    return int(bad) + len(mism)


def isolated_windows(torch, ar, x, label, window):
    """1 GiB-style windows decoded in isolation (nothing resident): start / middle / end of the file."""
    stream = torch.cuda.current_stream()
    info = ar.info()
    N = info["raw_bytes"]
    buf = ar.new_output(window)
    res = {}
    for name, lo in (("start", 0), ("middle", (N // 2) & ~(window - 1) if N >= 2 * window else 0), ("end", max(0, N - window))):
        hi = min(N, lo + window)
        ar.decode_range(lo, hi, out=buf)
        ar.check()
        ok = None
        if x is not None:
            ok = bool(torch.equal(buf[:hi - lo].cpu(), torch.from_numpy(x[lo:hi])))
        ms = timed(torch, stream, lambda: ar.decode_range(lo, hi, out=buf), 2, warmup=0)
        res[name] = {"lo": lo, "hi": hi, "ms": ms, "GBps": (hi - lo) / ms / 1e6, "bit_exact": ok}
    emit(config=label, what="isolated_windows", window_bytes=window, windows=res)


def seeks(torch, ar, x, label, n=300, seed=11):
    """PAPER.md:81-91 Table 3: latency of decoding 1 block and 100 consecutive blocks at random positions (host wall clock
    around decode_range + synchronize, nothing resident)."""
    info = ar.info()
    BS, nb = info["block_size"], info["n_blocks"]
    rng = np.random.default_rng(seed)
    res = {}
    for blocks in (1, 100):
        if nb <= blocks:
            continue
        buf = ar.new_output(blocks * BS)
        lat, ok = [], True
        for k in range(n + 10):
            b = int(rng.integers(0, nb - blocks))
            lo, hi = b * BS, min(info["raw_bytes"], (b + blocks) * BS)
            t = time.perf_counter()
            ar.decode_range(lo, hi, out=buf)
            torch.cuda.synchronize()
            if k >= 10:
                lat.append((time.perf_counter() - t) * 1e3)
            if k < 10:
                ok = ok and buf[:hi - lo].cpu().numpy().tobytes() == x[lo:hi].tobytes()
        ar.check()
        lat = np.array(lat)
        res["%d_blocks" % blocks] = {"ms_median": float(np.median(lat)), "ms_p99": float(np.percentile(lat, 99)), "ms_min": float(lat.min()),
                                     "bytes": blocks * BS, "bit_exact": ok}
    emit(config=label, what="seek_latency", n=n, seeks=res, graph_launches=ar.graph_launch_count())


def reads(torch, ar, x, idx, label, n_single=1000, n_batches=20, batch=4096, seed=5):
    stream = torch.cuda.current_stream()
    rng = np.random.default_rng(seed)
    off = (idx & np.uint64((1 << 40) - 1)).astype(np.int64)
    ln = (idx >> np.uint64(40)).astype(np.int64)
    out = ar.new_output(int(ln.max()) * batch)
    # batch 1: sequential single calls (the call synchronises and returns the read); wall clock per call
    ids = rng.integers(0, idx.size, n_single).astype(np.uint64)
    for i in ids[:20]:
        ar.decode_reads(idx, np.array([i], dtype=np.uint64), out=out)
    lat = []
    ok = True
    for i in ids:
        one = np.array([i], dtype=np.uint64)
        t = time.perf_counter()
        ar.decode_reads(idx, one, out=out)
        lat.append((time.perf_counter() - t) * 1e3)
    for i in ids[:50]:
        ar.decode_reads(idx, np.array([i], dtype=np.uint64), out=out)
        got = out[:ln[i]].cpu().numpy()
        ok = ok and got.tobytes() == x[off[i]:off[i] + ln[i]].tobytes()
    ar.check()
    lat = np.array(lat)
    b_ms, ok_b = [], True
    for k in range(n_batches):
        bi = rng.integers(0, idx.size, batch).astype(np.uint64)
        if k == 0:
            ar.decode_reads(idx, bi, out=out)           # warm-up
        t = time.perf_counter()
        ar.decode_reads(idx, bi, out=out)
        b_ms.append((time.perf_counter() - t) * 1e3)
        if k < 2:
            total, offs = ar.reads_bytes(idx, bi)
            got = out[:total].cpu().numpy()
            for j in range(0, batch, 37):
                r = int(bi[j])
                ok_b = ok_b and got[int(offs[j]):int(offs[j]) + ln[r]].tobytes() == x[off[r]:off[r] + ln[r]].tobytes()
    ar.check()
    b_ms = np.array(b_ms)
    emit(config=label, what="random_reads", index_entries=int(idx.size), index_bytes=int(idx.nbytes),
         batch1={"n": n_single, "ms_median": float(np.median(lat)), "ms_p99": float(np.percentile(lat, 99)), "ms_min": float(lat.min()),
                 "bit_exact": ok},
         batched={"batch": batch, "n_batches": n_batches, "ms_per_batch_median": float(np.median(b_ms)),
                  "us_per_read": float(np.median(b_ms)) * 1e3 / batch, "bit_exact": ok_b})


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--size", type=int, default=0)
    ap.add_argument("--src-window", type=int, default=0, help="encoder option: sources at most this far back (0 = unlimited)")
    ap.add_argument("--max-levels", default="", help="config 3: comma-separated encoder level caps to measure (default: the encoder's)")
    args = ap.parse_args()
    import torch
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    emit(what="box", cores=os.cpu_count(), gpu=torch.cuda.get_device_name(0), peak=peak_gbs())
    if args.config in (0, 1):
        size, seed, ref = ((4 << 20), 1, 1_000_000) if args.config == 0 else ((1 << 30), 2, 50_000_000)
        size = args.size or size
        x = datagen.fastq(seed, size, ref)
        t = time.time()
        a = encoder.encode(x, block_size=16384)
        emit(config=args.config, what="encode", seconds=time.time() - t, MBps=x.size / (time.time() - t) / 1e6)
        ar = Archive(a)
        whole_file(torch, ar, x, args.config)
        win = min(64 << 20, max(1 << 20, size // 16))
        windows(torch, ar, x, args.config, win, 2)
        windows(torch, ar, x, args.config, 2 * win, 1)         # the same ring bytes as ONE reused buffer (chunks)
        isolated_windows(torch, ar, x, args.config, win)
        reads(torch, ar, x, datagen.fastq_index(size), args.config)
        seeks(torch, ar, x, args.config)
        ar.close()
        os.environ["ACEAPEX_NO_GRAPHS"] = "1"                  # read at open: the same seeks with plain launches
        ar = Archive(a)
        del os.environ["ACEAPEX_NO_GRAPHS"]
        seeks(torch, ar, x, "%d/plain launches (ACEAPEX_NO_GRAPHS=1)" % args.config)
        ar.close()
    elif args.config == 2:
        size = args.size or 3_100_000_000
        t = time.time()
        x = datagen.fasta(3, size)
        emit(config=2, what="generate", seconds=time.time() - t)
        t = time.time()
        a = encoder.encode(x, block_size=16384)
        emit(config=2, what="encode", seconds=time.time() - t, MBps=x.size / (time.time() - t) / 1e6)
        ar = Archive(a)
        whole_file(torch, ar, x, 2, reps=3)
        idx = datagen.region_index(3, size, 1_000_000, 150)
        reads(torch, ar, x, idx, 2, n_single=2000, n_batches=1_000_000 // 4096)
        isolated_windows(torch, ar, x, 2, 1 << 28)
        seeks(torch, ar, x, 2)
        ar.close()
    elif args.config == 3:
        size = args.size or (50 << 30)
        t = time.time()
        x = datagen.fasta(4, size)
        emit(config=3, what="generate", seconds=time.time() - t, bytes=size)
        for max_level in ([int(v) for v in args.max_levels.split(",")] if args.max_levels else [None]):
            kw = {} if max_level is None else {"max_level": max_level}
            t = time.time()
            a = encoder.encode(x, block_size=16384, src_window=args.src_window, **kw)
            emit(config=3, what="encode", src_window=args.src_window, encoder_max_level=max_level, seconds=time.time() - t,
                 MBps=x.size / (time.time() - t) / 1e6, archive_bytes=int(a.size))
            ar = Archive(a)
            info = ar.info()
            emit(config=3, what="archive", raw_bytes=info["raw_bytes"], archive_bytes=info["archive_bytes"], n_blocks=info["n_blocks"],
                 offset_width=info["offset_width"], max_level=info["max_level"], workspace_bytes=info["workspace_bytes"])
            window = min(1 << 30, max(1 << 24, size // 8))
            nwin = (size + window - 1) // window
            windows(torch, ar, x, 3, window, 8, reps=1, sample_check={0, nwin // 2, nwin - 1})
            isolated_windows(torch, ar, x, 3, window)
            ar.close()
            del ar, a
            torch.cuda.empty_cache()
    elif args.config == 5:
        # the entropy stage alone on the workload shape of PAPER.md:135 (DietGPU: 256 MB of
        # exponentially distributed bytes, 4096 x 64 KB): aceapex_rans_encode / aceapex_rans_decode, one warp per row
        sys.path.insert(0, ROOT)
        import bench
        emit(config=5, what="rans_microbench", **bench.entropy_microbench(torch))
    elif args.config == 4:
        size = args.size or (1 << 30)
        x = datagen.fastq(2, size, 50_000_000)
        sys.path.insert(0, ROOT)
        import bench
        emit(config=4, what="launch_overhead", note="SURVEY.md 8(c) S19 (c): the schedule of decode_all on an archive of one 8-byte block",
             **bench.launch_overhead(torch, torch.cuda.current_stream()))
        for bs in (4096, 8192, 16384, 65536, 262144, 1 << 20):
            for max_level in ((2, 0, 3) if bs == 16384 else (2,)):          # 2 = the encoder's default
                t = time.time()
                a = encoder.encode(x, block_size=bs, max_level=max_level)
                enc_s = time.time() - t
                ar = Archive(a)
                info = ar.info()
                res = whole_file(torch, ar, x, "4/bs=%d/max_level=%d" % (bs, max_level), reps=3)
                n_blocks, bt_off = int(a[24:32].view(np.uint64)[0]), int(a[104:112].view(np.uint64)[0])   # FORMAT.md §1.1
                lv = np.frombuffer(a[bt_off:bt_off + 8 * n_blocks].tobytes(), dtype=np.uint16).reshape(-1, 4)[:, 2]   # §1.4 level
                # S19 (a), (b): launches per decode; time of a call not covered by its kernels, per launch (phase timers = CUDA events
                # around each launch; the rest of the call is launch gaps)
                ar.set_phase_timing(True)
                ms_call = timed(torch, torch.cuda.current_stream(), lambda: ar.decode_all(res_out(ar)), 3)
                ph = ar.phase_times()
                ar.set_phase_timing(False)
                emit(config=4, what="block_size_point", block_size=bs, encoder_max_level=max_level, ratio=x.size / a.size, encode_seconds=enc_s,
                     n_segments=info["n_segments"], GBps=res["default"]["GBps"], ms=res["default"]["ms"], mean_level=float(lv.mean()), max_level=int(lv.max()),
                     wavefront_depth=int(lv.max()) + 1, launches_default=res["default"]["launches"], ms_flags=res["flags"]["ms"], ms_fused=res["fused"]["ms"],
                     call_ms=ms_call, kernels_ms=float(sum(ph)), gap_per_launch_us=(ms_call - float(sum(ph))) * 1e3 / max(res["default"]["launches"], 1))
                if bs == 16384 and max_level == 2:
                    seeks(torch, ar, x, "4/bs=16384")
                ar.close()
                del ar
                torch.cuda.empty_cache()
    elif args.config == 6:
        # encoder options against range-decode speed (measure, do not dismiss): level cap, source window, LITQ mode
        size = args.size or (1 << 30)
        x = datagen.fastq(2, size, 50_000_000)
        for kw in (dict(), dict(max_level=0), dict(max_level=3), dict(q_mode=0), dict(q_min=0), dict(src_window=256 << 20), dict(src_window=64 << 20), dict(log2_seg=12)):
            t = time.time()
            a = encoder.encode(x, block_size=16384, **kw)
            ar = Archive(a)
            res = whole_file(torch, ar, x, "6/%s" % kw, reps=3)
            win = min(128 << 20, max(1 << 20, size // 8))       # one reused buffer of an eighth of the file
            ring = ar.new_output(win)
            st = min((ar.decode_stream(0, size, ring, win, consumer=lambda *a_: 0) for _ in range(2)), key=lambda q: q["device_ms"])
            bad = ar.decode_stream(0, size, ring, win)["bad_blocks"]
            emit(config=6, what="encoder_option", options=kw, ratio=x.size / a.size, encode_seconds=time.time() - t, decode_all_GBps=res["default"]["GBps"],
                 ring_GBps=size / st["device_ms"] / 1e6, ring_min_window_GBps=st["min_window_gbs"], bad_blocks=int(bad))
            seeks(torch, ar, x, "6/%s" % kw, n=100)
            ar.close()
            del ar, ring
            torch.cuda.empty_cache()
    elif args.config == 7:
        # one isolated 64 MiB window in the middle of configs[1] (nothing resident: every source before it is foreign), three
        # times: the command profiles/r2_range_window.md captures with ncu
        size = args.size or (1 << 30)
        x = datagen.fastq(2, size, 50_000_000)
        ar = Archive(encoder.encode(x, block_size=16384))
        W = min(64 << 20, size // 4)
        lo = (size // 2) & ~(W - 1)
        buf = ar.new_output(W)
        for _ in range(3):
            ar.decode_range(lo, lo + W, out=buf)
        torch.cuda.synchronize()
        ar.check()
        ms = timed(torch, torch.cuda.current_stream(), lambda: ar.decode_range(lo, lo + W, out=buf), 3, warmup=0)
        emit(config=7, what="isolated_window", lo=lo, hi=lo + W, ms=ms, GBps=W / ms / 1e6, launches=ar.launch_count() // 6,
             bit_exact=bool(torch.equal(buf[:W].cpu(), torch.from_numpy(x[lo:lo + W]))))
        ar.close()


_OUT = {}


def res_out(ar):
    """one output buffer per archive handle (timing helper)"""
    k = id(ar)
    if k not in _OUT:
        _OUT.clear()
        _OUT[k] = ar.new_output()
    return _OUT[k]


if __name__ == "__main__":
    main()
