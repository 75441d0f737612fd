"""Reading the tracked ncu captures and the SASS of the built library (measurement support; no arithmetic of the method).

* `kernel_source_hash()`  -- first 10 hex digits of the SHA-1 over csrc/* and the nvcc flags: names a build of the
  kernels.  The raw ncu exports under profiles/ carry it in their file name, so a figure read from one of them can be
  told apart from a figure measured on other kernels.
* `ncu_table(workload)`   -- per launcher, from profiles/ncu_raw_<workload>_<hash>.csv (the `ncu -i X.ncu-rep --page
  raw --csv` export of one `ncu --set full --clock-control none` capture of `bench.py --workload <workload>`): DRAM
  bytes read + written, duration, fp64 pipe utilisation, registers ...; `stale` when the only file present was captured
  on other kernel sources.
* `sass_digest()`         -- per kernel of libfargo_b200.so: registers, spills, and counts of the SASS mnemonics that
  matter here (DFMA/DMUL/DADD, MUFU, SHFL, LDG/STG, LDGSTS = cp.async, UBLKCP/UTMALDG = TMA, BAR, SYNCS = mbarrier).
      python -m paper_1602_02359_b200.profiling sass   > profiles/sass_digest_<hash>.md
      python -m paper_1602_02359_b200.profiling hash
"""
from __future__ import annotations

import csv
import glob
import hashlib
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
PROFILES = os.path.join(ROOT, "profiles")

# kernel function -> launcher name of fargo_profile_report (a launcher may own several kernels: times and bytes add up)
LAUNCHER_OF = [
    (r"k_bc_b", "bc_b"), (r"k_mhd_pressure|k_mhd_curv", "mhd_pressure"), (r"k_mhd_emf", "mhd_emf"), (r"k_mhd_tension", "mhd_tension"),
    (r"k_mhd_ct", "mhd_ct"), (r"k_mhd_resid", "mhd_resid"), (r"k_mhd_arc|k_mhd_orbital", "mhd_orbital"),
    (r"k_source_fused|k_source_tile", "source"), (r"k_visc3d_fused", "source_d"), (r"k_visc3d_(tensor|force)", "source_d"),
    (r"k_momenta", "momenta"), (r"k_visc_(tensor|force)", "source_d"), (r"k_source_c\b", "source_c"),
    (r"k_source_a\b", "source_a"), (r"k_source_bc\b", "source_bc"), (r"k_source_b\b", "source_b"),
    (r"k_sweep_x", "sweep_x"), (r"k_sweep_ring<\w+, *\(?int\)?1|k_sweep_ring<\w+, *1", "sweep_y"),
    (r"k_sweep_ring<\w+, *\(?int\)?2|k_sweep_ring<\w+, *2", "sweep_z"), (r"k_sweep_last", "sweep_last"),
    (r"k_orbital", "orbital"), (r"k_newvel_dt", "newvel_dt"), (r"k_newvel", "newvel"), (r"k_dt_", "dt"),
    (r"k_vmean", "vmean"), (r"k_potential", "potential"), (r"k_planet", "planets"), (r"k_bc", "bc"), (r"k_advance", "advance"),
]


def launcher_of(kernel_name: str):
    for pat, name in LAUNCHER_OF:
        if re.search(pat, kernel_name):
            return name
    return None


def kernel_source_hash() -> str:
    from . import build as B
    h = hashlib.sha1()
    for f in sorted(os.listdir(B.CSRC)):
        with open(os.path.join(B.CSRC, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    h.update(" ".join(B.NVCC_FLAGS).encode())
    return h.hexdigest()[:10]


def _num(s):
    try:
        return float(s.replace(",", ""))
    except (ValueError, AttributeError):
        return None


def read_ncu_raw(path: str):
    """Rows of an `ncu --page raw --csv` export: one dict per kernel launch, metric name -> (value, unit)."""
    with open(path, newline="") as f:
        lines = [ln for ln in f if not ln.startswith("==")]
    rows = list(csv.reader(lines))
    if len(rows) < 3:
        return []
    names, units = rows[0], rows[1]
    return [{n: (v, u) for n, u, v in zip(names, units, r)} for r in rows[2:]]


_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
          "ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "ms": 1.0, "msecond": 1.0, "nsecond": 1e-6, "second": 1e3, "s": 1e3}


def _val(row, name):
    v = row.get(name)
    if not v:
        return None
    x = _num(v[0])
    return None if x is None else x * _SCALE.get(v[1], 1.0)


def ncu_table(workload: str):
    """({launcher: {...}}, source file, stale flag) from the tracked raw export of this workload; ({}, None, None)
    when there is none."""
    h = kernel_source_hash()
    exact = os.path.join(PROFILES, "ncu_raw_%s_%s.csv" % (workload, h))
    stale = False
    path = exact
    if not os.path.exists(exact):
        others = sorted(glob.glob(os.path.join(PROFILES, "ncu_raw_%s_*.csv" % workload)), key=os.path.getmtime)
        if not others:
            return {}, None, None
        path, stale = others[-1], True
    acc = {}
    for row in read_ncu_raw(path):
        kname = row.get("Kernel Name", ("", ""))[0]
        name = launcher_of(kname)
        if name is None:
            continue
        e = acc.setdefault(name, {"launches": 0, "dram_bytes": 0.0, "ms": 0.0, "fp64": [], "regs": [], "kernels": set(),
                                  "inst": 0.0, "ipc": []})
        e["launches"] += 1
        e["kernels"].add(kname)
        rd, wr = _val(row, "dram__bytes_read.sum"), _val(row, "dram__bytes_write.sum")
        if rd is not None and wr is not None:
            e["dram_bytes"] += rd + wr
        t = _val(row, "gpu__time_duration.sum")
        if t is not None:
            e["ms"] += t
        ni = _val(row, "smsp__inst_executed.sum")   # warp-level instructions
        if ni is not None:
            e["inst"] += ni
        for key, dst in (("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "fp64"),
                         ("launch__registers_per_thread", "regs"), ("sm__inst_executed.avg.per_cycle_active", "ipc")):
            x = _val(row, key)
            if x is not None:
                e[dst].append(x)
    return acc, os.path.relpath(path, ROOT), stale


def per_update(table, name, updates_captured):
    """DRAM bytes and fp64-pipe % of launcher `name` per UPDATE (a launcher runs once per update, `bc` twice)."""
    e = table.get(name)
    if not e or not updates_captured:
        return None, None
    fp = sum(e["fp64"]) / len(e["fp64"]) if e["fp64"] else None
    return e["dram_bytes"] / updates_captured, fp


# ---------------------------------------------------------------------------------- SASS ------------
MNEMONICS = ["DFMA", "DMUL", "DADD", "DSETP", "MUFU", "FFMA", "SHFL", "LDG", "STG", "LDS", "STS", "LDGSTS", "UBLKCP", "UTMALDG",
             "SYNCS", "BAR", "ATOM", "RED", "BRA", "WARPSYNC"]


def sass_digest() -> str:
    from . import build as B
    lib = B.build()
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True).stdout
    usage, cur = {}, None
    for ln in res.splitlines():
        m = re.match(r"\s*Function (\S+):", ln)
        if m:
            cur = m.group(1)
        m = re.search(r"REG:(\d+).*?SHARED:(\d+).*?LOCAL:(\d+)", ln)
        if m and cur:
            usage[cur] = tuple(int(x) for x in m.groups())
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    counts, cur = {}, None
    for ln in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", ln)
        if m:
            cur = m.group(1)
            counts[cur] = dict.fromkeys(MNEMONICS, 0)
            counts[cur]["total"] = 0
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", ln)
        if m and cur:
            op = m.group(1)
            counts[cur]["total"] += 1
            if op in counts[cur]:
                counts[cur][op] += 1
    dem = subprocess.run(["cu++filt"] + list(counts), capture_output=True, text=True).stdout.splitlines()
    pretty = dict(zip(counts, dem)) if len(dem) == len(counts) else {k: k for k in counts}
    out = ["# SASS digest of libfargo_b200.so, kernel sources %s" % kernel_source_hash(), "",
           "`python -m paper_1602_02359_b200.profiling sass` (cuobjdump -res-usage / -sass of the in-tree build; static",
           "instruction counts of the whole kernel body, loops counted once).  LDGSTS = cp.async, UBLKCP / UTMALDG = bulk /",
           "tensor TMA copies, SYNCS = mbarrier operations; LOCAL > 0 means spills.", "",
           "| kernel | REG | SHARED B | LOCAL B | total | " + " | ".join(MNEMONICS) + " |",
           "|---|---|---|---|---|" + "---|" * len(MNEMONICS)]
    for k in sorted(counts, key=lambda k: pretty[k]):
        name = re.sub(r"^void fg::", "", pretty[k])
        cut = name.find(">(")
        name = name[:cut + 1] if cut >= 0 else name.split("(")[0]
        name = name.replace("(int)", "").replace("(bool)", "").replace("double", "f64").replace("float", "f32")
        if not name.startswith("k_"):
            continue
        u = usage.get(k, ("?", "?", "?"))
        c = counts[k]
        out.append("| %s | %s | %s | %s | %d | " % (name, u[0], u[1], u[2], c["total"]) + " | ".join(str(c[m]) for m in MNEMONICS) + " |")
    return "\n".join(out) + "\n"


if __name__ == "__main__":
    what = sys.argv[1] if len(sys.argv) > 1 else "hash"
    if what == "sass":
        sys.stdout.write(sass_digest())
    else:
        print(kernel_source_hash())
