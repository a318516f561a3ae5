"""Turns one `ncu --page raw --csv` export of a decode_all step into profiles/step_capture.json, the file bench.py reads its
`roofline.traffic` and `bound_observed` entries from.

  python bench.py --steps 2 --warmup 3 --no-cpu-baseline --step-only                      # plain run first (exit 0)
  ncu --set full --clock-control none --import-source on -k regex:'k_literals|k_copy' -s <launches of warm-up> -c <launches of one step> \\
      -f -o gpurun_out/step python bench.py --steps 2 --warmup 3 --no-cpu-baseline --step-only
  ncu -i gpurun_out/step.ncu-rep --page raw --csv > gpurun_out/step_raw.csv
  python -m paper_2606_18900_b200.ncu_summary gpurun_out/step_raw.csv "<the ncu command>"   # -> profiles/step_capture.json + .md

The summary names the SHA-256 of the CUDA sources it was taken on; bench.py ignores it when they have changed since."""
import csv
import hashlib
import json
import os
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)

WANT = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "smsp__inst_executed.sum",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
        "dram__cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "launch__registers_per_thread", "launch__grid_size", "launch__block_size", "lts__t_sector_hit_rate.pct"]
STALLS = ["long_scoreboard", "short_scoreboard", "wait", "not_selected", "no_instruction", "math_pipe_throttle", "mio_throttle",
          "branch_resolving", "barrier", "lg_throttle"]
UNIT = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0}


def source_hash():
    h = hashlib.sha256()
    cs = os.path.join(PKG, "csrc")
    for f in sorted(os.listdir(cs)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(cs, f), "rb").read())
    return h.hexdigest()[:16]


def summarise(raw_csv, command):
    rows = list(csv.reader(open(raw_csv)))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    launches = []
    for r in rows[2:]:
        if len(r) < len(hdr):
            continue
        name = r[col["Kernel Name"]]
        d = {"kernel": name}
        for k in WANT:
            if k in col:
                v = float(r[col[k]].replace(",", "")) * UNIT.get(units[col[k]], 1.0)
                d[k] = v
        for sname in STALLS:
            k = "smsp__average_warps_issue_stalled_%s_per_issue_active.ratio" % sname
            if k in col:
                d["stall_" + sname] = float(r[col[k]].replace(",", ""))
        launches.append(d)
    out = {"command": command, "source_hash": source_hash(), "launches": launches, "kernels": {}}
    out["dram_bytes_per_step"] = int(sum(d["dram__bytes_read.sum"] + d["dram__bytes_write.sum"] for d in launches))
    out["dram_bytes_read_per_step"] = int(sum(d["dram__bytes_read.sum"] for d in launches))
    out["dram_bytes_write_per_step"] = int(sum(d["dram__bytes_write.sum"] for d in launches))
    for key in ("k_literals", "k_copy"):
        ds = [d for d in launches if key in d["kernel"]]
        if not ds:
            continue
        d = max(ds, key=lambda q: q["gpu__time_duration.sum"])
        stalls = sorted(((k[6:], v) for k, v in d.items() if k.startswith("stall_")), key=lambda t: -t[1])[:3]
        out["kernels"][key] = {
            "time_ms": sum(q["gpu__time_duration.sum"] for q in ds) * 1e3,
            "dram_bytes": int(sum(q["dram__bytes_read.sum"] + q["dram__bytes_write.sum"] for q in ds)),
            "bound_observed": "issue slots %.0f %% busy, LSU data pipe %.0f %%, DRAM %.0f %% active; top stalls per issue: %s (ncu --set full, %s)" % (
                d["smsp__issue_active.avg.pct_of_peak_sustained_active"], d["l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"],
                d["dram__cycles_active.avg.pct_of_peak_sustained_elapsed"], ", ".join("%s %.2f" % s for s in stalls), "profiles/step_capture.md")}
    return out


def main():
    raw, command = sys.argv[1], sys.argv[2]
    out = summarise(raw, command)
    json.dump(out, open(os.path.join(ROOT, "profiles", "step_capture.json"), "w"), indent=1)
    with open(os.path.join(ROOT, "profiles", "step_capture.md"), "w") as f:
        f.write("# ncu --set full capture of one decode_all step on configs[1]\n\nCommand (after the same command had exited 0 without ncu):\n\n```\n%s\n```\n\n" % command)
        f.write("CUDA source hash %s.  Per launch:\n\n| kernel | grid x block | us | instructions | issue %% | LSU pipe %% | DRAM %% | DRAM read MB | DRAM write MB | L2 hit %% | top stalls per issue |\n|---|---|---|---|---|---|---|---|---|---|---|\n" % out["source_hash"])
        for d in out["launches"]:
            stalls = sorted(((k[6:], v) for k, v in d.items() if k.startswith("stall_")), key=lambda t: -t[1])[:4]
            f.write("| %s | %d x %d | %.1f | %.3e | %.1f | %.1f | %.1f | %.1f | %.1f | %.1f | %s |\n" % (
                d["kernel"][:48], d.get("launch__grid_size", 0), d.get("launch__block_size", 0), d["gpu__time_duration.sum"] * 1e6, d["smsp__inst_executed.sum"],
                d["smsp__issue_active.avg.pct_of_peak_sustained_active"], d["l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"],
                d["dram__cycles_active.avg.pct_of_peak_sustained_elapsed"], d["dram__bytes_read.sum"] / 1e6, d["dram__bytes_write.sum"] / 1e6,
                d.get("lts__t_sector_hit_rate.pct", 0.0), ", ".join("%s %.2f" % s for s in stalls)))
        f.write("\nDRAM bytes per step: %d (read %d, write %d).\n" % (out["dram_bytes_per_step"], out["dram_bytes_read_per_step"], out["dram_bytes_write_per_step"]))
    print(json.dumps(out["kernels"], indent=1))


if __name__ == "__main__":
    main()
