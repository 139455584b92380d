"""Per-kernel work counts from an ncu capture, in the form bench.py reads.

    ncu -i <capture>.ncu-rep --page raw --csv > raw.csv
    python -m paper_2410_09146_b200.profile_counts raw.csv profiles/<round>_kernel_counts.csv --capture <id> --zones 16777216 \
        --workload cfg4_256

One row per kernel class (launches of the same class averaged): executed fp64 thread-instructions per interior zone
(dadd + dmul + dfma, predicated on), flop per zone (dfma counted twice), DRAM bytes read / written per launch, duration,
registers, fp64-pipe and warp-slot utilisation, and the hash of the kernel sources the capture was taken from.
bench.py refuses to derive achieved fp64 figures from these counts when the sources it runs have a different hash.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import os
import re

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = [os.path.join(HERE, "csrc", "phx_kernels.cu"), os.path.join(HERE, "csrc", "phx_device.cuh")]
FIELDS = ["capture", "workload", "class", "kernel", "launches", "time_ms", "registers", "fp64_instr_per_zone", "flop_per_zone",
          "dram_read_bytes", "dram_write_bytes", "fp64_pipe_pct", "warps_active_pct", "src_sha16"]


def source_hash() -> str:
    h = hashlib.sha256()
    for f in SOURCES:
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def kernel_class(name: str) -> str | None:
    m = re.search(r"k_sweep_march<\(int\)\d+, \(int\)\d+, \(int\)(\d)", name) or re.search(r"k_sweep_march<\d+, \d+, (\d)", name)
    if m:
        return "sweep_y" if m.group(1) == "1" else "sweep_z"
    if "k_sweep_x" in name:
        return "sweep_x"
    m = re.search(r"k_update<\(int\)\d+, \(bool\)\d, \(bool\)(\d)", name) or re.search(r"k_update<\d+, \d+, (\d)", name)
    if m:
        return "update_cfl" if m.group(1) == "1" else "update"
    for k in ("k_fill_ghosts", "k_cfl_partial", "k_cfl_final", "k_prim_to_cons", "k_c2p"):
        if k in name:
            return k[2:]
    return None


def to_unit(value: str, unit: str) -> float:
    v = float(value.replace(",", ""))
    scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1.0, "us": 1e-3, "ns": 1e-6, "s": 1e3}
    return v * scale.get(unit, 1.0)


def read_raw(path):
    with open(path, newline="") as fh:
        rows = list(csv.reader(fh))
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}

    def get(r, name):
        return to_unit(r[col[name]], units[col[name]])
    out = []
    for r in data:
        if len(r) != len(hdr):
            continue
        cyc = get(r, "smsp__cycles_elapsed.avg")
        ops = {k: get(r, f"smsp__sass_thread_inst_executed_op_{k}_pred_on.sum.per_cycle_elapsed") * cyc for k in ("dadd", "dmul", "dfma")}
        out.append(dict(name=r[col["Kernel Name"]], time_ms=get(r, "gpu__time_duration.sum"),
                        registers=int(float(r[col["launch__registers_per_thread"]])),
                        instr=ops["dadd"] + ops["dmul"] + ops["dfma"], flop=ops["dadd"] + ops["dmul"] + 2.0 * ops["dfma"],
                        rd=get(r, "dram__bytes_read.sum"), wr=get(r, "dram__bytes_write.sum"),
                        pipe=float(r[col["sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"]]),
                        warps=float(r[col["sm__warps_active.avg.pct_of_peak_sustained_active"]])))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("out_csv")
    ap.add_argument("--capture", required=True)
    ap.add_argument("--workload", required=True)
    ap.add_argument("--zones", type=int, required=True)
    ap.add_argument("--append", action="store_true")
    a = ap.parse_args()
    groups = {}
    for k in read_raw(a.raw_csv):
        c = kernel_class(k["name"])
        if c:
            groups.setdefault(c, []).append(k)
    sha = source_hash()
    mode = "a" if a.append and os.path.exists(a.out_csv) else "w"
    with open(a.out_csv, mode, newline="") as fh:
        w = csv.DictWriter(fh, fieldnames=FIELDS)
        if mode == "w":
            w.writeheader()
        for c, ks in groups.items():
            n = len(ks)
            avg = lambda key: sum(k[key] for k in ks) / n
            w.writerow(dict(capture=a.capture, workload=a.workload, **{"class": c}, kernel=re.sub(r"\(.*", "", ks[0]["name"].replace("void ", "")),
                            launches=n, time_ms=round(avg("time_ms"), 6), registers=ks[0]["registers"],
                            fp64_instr_per_zone=round(avg("instr") / a.zones, 2), flop_per_zone=round(avg("flop") / a.zones, 2),
                            dram_read_bytes=int(avg("rd")), dram_write_bytes=int(avg("wr")), fp64_pipe_pct=round(avg("pipe"), 2),
                            warps_active_pct=round(avg("warps"), 2), src_sha16=sha))
    print(f"{a.out_csv}: {len(groups)} kernel classes, sources {sha}")


def load(path, workload):
    """{class: row dict with numbers} of one workload from a counts file, plus the source hash the rows carry."""
    out, sha = {}, None
    with open(path, newline="") as fh:
        for r in csv.DictReader(fh):
            if r["workload"] != workload:
                continue
            sha = r["src_sha16"]
            out[r["class"]] = {k: (float(v) if k not in ("capture", "workload", "class", "kernel", "src_sha16") else v) for k, v in r.items()}
    return out, sha


if __name__ == "__main__":
    main()
