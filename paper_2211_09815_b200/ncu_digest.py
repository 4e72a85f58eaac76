"""Digest of `ncu --page raw --csv` exports into the text files kept under profiles/.

    python -m paper_2211_09815_b200.ncu_digest full  <workload> <raw.csv> [<raw.csv> ...]  > profiles/<name>.md
    python -m paper_2211_09815_b200.ncu_digest traffic <workload> <raw.csv> [...]          >> profiles/r02_traffic.csv
    python -m paper_2211_09815_b200.ncu_digest launches <launches.csv>                     > profiles/<name>.md

`full`: one row per captured launch with the counters north_star asks for (DRAM bytes, achieved DRAM throughput,
shared-memory atomic instructions and their rate, shared-memory wavefronts and bank conflicts, sectors per request of the
global loads, occupancy).  `traffic`: dram__bytes_read.sum + dram__bytes_write.sum per launch, averaged per kernel class,
stamped with the hash of the kernel sources and the commit (bench.py only trusts rows whose hash matches the running
sources).  `launches`: per-kernel totals and shares of a `--metrics gpu__time_duration.sum` launch list.
No arithmetic of the method lives here; nothing in the package imports this module.
"""
import csv
import hashlib
import os
import subprocess
import sys
from collections import OrderedDict

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# kernel name fragment -> timing class of bench.py's kernel table
CLASSES = [("scatter_kernel<1", "scatter1"), ("scatter_kernel<3", "scatter3"), ("gather_kernel<4", "gather_fused"),
           ("gather_kernel<3, 0, 0, 1>", "gather_kick"), ("gather_kernel<3", "gather"), ("gather_kernel<1", "gather_grad"),
           ("fft_x_force", "kspace_force"), ("fft_x_adjoint", "kspace_adjoint"), ("kspace_force", "kspace_force"),
           ("kspace_adjoint", "kspace_adjoint"), ("fft_z_r2c", "fft_z_r2c"), ("fft_z_c2r", "fft_z_c2r"), ("fft_y", "fft_y"),
           ("bin_reorder", "bin_reorder"), ("bin_count", "bin_count"), ("scan_kernel", "bin_scan"), ("kick_drift", "kick_drift"),
           ("objective", "objective")]


def klass(name):
    for frag, c in CLASSES:
        if frag in name:
            return c
    return None


def source_hash():
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2211_09815_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".inc")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def commit():
    try:
        return subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip() or "?"
    except OSError:
        return "?"


def read_raw(path):
    rows = list(csv.reader(open(path)))
    hi = [i for i, r in enumerate(rows) if r and r[0] == "ID"][0]
    hdr, units = rows[hi], rows[hi + 1]
    out = []
    for r in rows[hi + 2:]:
        if len(r) >= len(hdr):
            out.append({h: r[i] for i, h in enumerate(hdr)})
    return out, {h: units[i] for i, h in enumerate(hdr)}


def num(rec, key, unit=None):
    v = rec.get(key, "")
    try:
        x = float(v.replace(",", ""))
    except ValueError:
        return None
    if unit:
        u = unit.get(key, "")
        scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0,
                 "msecond": 1e-3, "usecond": 1e-6, "nsecond": 1e-9, "second": 1.0}
        for k, s in scale.items():
            if u == k:
                return x * s
    return x


def fmt(x, f="%.3g"):
    return "-" if x is None else f % x


T = "gpu__time_duration.sum"
RD, WR = "dram__bytes_read.sum", "dram__bytes_write.sum"


def cmd_full(workload, paths):
    print(f"# ncu --set full digest: {workload}\n")
    print(f"Kernel sources `{source_hash()}`, commit `{commit()}`.  One row per captured launch (cold cache, serialised: compare")
    print("shares and ratios, not absolute times).  `atom/s` = shared-memory atomic instructions per second of kernel time;")
    print("`conf` = bank-conflict share of the shared-memory wavefronts; `sect/req` = sectors per request of the global loads.\n")
    print("| kernel | class | us | DRAM rd MB | DRAM wr MB | DRAM % | L1/smem % | issue % | warps act % | regs | smem atom inst | atom/s | smem wavefronts | conf | sect/req ld |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for p in paths:
        recs, unit = read_raw(p)
        for r in recs:
            name = r.get("Kernel Name", "?")
            t = num(r, T, unit)
            rd, wr = num(r, RD, unit), num(r, WR, unit)
            atom = num(r, "smsp__inst_executed_op_shared_atom.sum")
            wf = num(r, "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")
            cf = num(r, "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum")
            sec = num(r, "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum")
            req = num(r, "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum")
            print("| `%s` | %s | %s | %s | %s | %s | %s | %s | %s | %s | %s | %s | %s | %s | %s |" % (
                name[:44], klass(name) or "-", fmt(t * 1e6 if t else None, "%.1f"), fmt(rd / 1e6 if rd is not None else None, "%.0f"),
                fmt(wr / 1e6 if wr is not None else None, "%.0f"), fmt(num(r, "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"), "%.0f"),
                fmt(num(r, "l1tex__throughput.avg.pct_of_peak_sustained_active"), "%.0f"),
                fmt(num(r, "smsp__issue_active.avg.pct_of_peak_sustained_active"), "%.0f"),
                fmt(num(r, "sm__warps_active.avg.pct_of_peak_sustained_active"), "%.0f"), fmt(num(r, "launch__registers_per_thread"), "%.0f"),
                fmt(atom, "%.3g"), fmt(atom / t if atom and t else None, "%.3g"), fmt(wf, "%.3g"),
                fmt(cf / wf if cf is not None and wf else None, "%.2f"), fmt(sec / req if sec and req else None, "%.1f")))


def cmd_traffic(workload, paths):
    agg = OrderedDict()
    for p in paths:
        recs, unit = read_raw(p)
        for r in recs:
            c = klass(r.get("Kernel Name", ""))
            rd, wr = num(r, RD, unit), num(r, WR, unit)
            if c and rd is not None and wr is not None:
                agg.setdefault(c, []).append(rd + wr)
    h, cm = source_hash(), commit()
    for c, v in agg.items():
        print(f"{workload},{c},{sum(v) / len(v):.0f},{h},{cm}")


def cmd_launches(path):
    rows = list(csv.reader(open(path)))
    hi = [i for i, r in enumerate(rows) if r and r[0] == "ID"][0]
    hdr = rows[hi]
    kn, mn, mv, mu = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value"), hdr.index("Metric Unit")
    scale = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "nsecond": 1e-3, "usecond": 1.0, "msecond": 1e3, "s": 1e6, "second": 1e6}
    agg = OrderedDict()
    for r in rows[hi + 1:]:
        if len(r) > mv and r[mn] == T:
            us = float(r[mv].replace(",", "")) * scale.get(r[mu], 1.0)
            a = agg.setdefault(r[kn][:60], [0, 0.0])
            a[0] += 1
            a[1] += us
    tot = sum(a[1] for a in agg.values()) or 1.0
    print(f"# ncu launch list digest ({os.path.basename(path)})\n")
    print(f"Kernel sources `{source_hash()}`, commit `{commit()}`.  Per-launch times are cold-cache and serialised: the SHARE column is")
    print("what is comparable with bench.py's kernel table.\n")
    print("| kernel | launches | total ms | avg us | share |")
    print("|---|---|---|---|---|")
    for k, (n, us) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        print(f"| `{k}` | {n} | {us / 1e3:.2f} | {us / n:.1f} | {us / tot:.3f} |")
    print(f"\ntotal {tot / 1e3:.1f} ms over {sum(a[0] for a in agg.values())} launches")


if __name__ == "__main__":
    if len(sys.argv) >= 4 and sys.argv[1] == "full":
        cmd_full(sys.argv[2], sys.argv[3:])
    elif len(sys.argv) >= 4 and sys.argv[1] == "traffic":
        cmd_traffic(sys.argv[2], sys.argv[3:])
    elif len(sys.argv) == 3 and sys.argv[1] == "launches":
        cmd_launches(sys.argv[2])
    else:
        sys.exit(__doc__)
