"""Turns an `ncu --set full` capture of `bench.py` into the per-stage counter table bench.py reads.

    python -m paper_2607_04230_b200.ncu_summary --hash                  # sha256 of csrc/*.cu, *.cuh (run where the capture runs)
    python -m paper_2607_04230_b200.ncu_summary REP.ncu-rep SHA OUT.csv  # per-stage counters of the LAST captured frame

Measurement tooling only: nothing on the render path imports it. bench.py uses read_stage_csv / source_hash to label
the committed capture fresh or stale.
"""
from __future__ import annotations

import csv
import hashlib
import io
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
STAGE_OF = (("k_generate", "generate"), ("k_raster", "raster"), ("k_hiz", "raster"), ("k_shade", "shade"), ("k_filter", "filter"))
METRICS = {
    "dram_bytes": ("dram__bytes_read.sum", "dram__bytes_write.sum"),
    "warp_inst": ("smsp__inst_executed.sum",),
    "duration_ns": ("gpu__time_duration.sum",),
}
PCT = {"lts_throughput_pct": "lts__throughput.avg.pct_of_peak_sustained_elapsed",
       "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active"}
UNIT_SCALE = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1, "us": 1e3, "ms": 1e6, "s": 1e9, "nsecond": 1,
              "usecond": 1e3, "msecond": 1e6, "second": 1e9, "inst": 1, "": 1, "%": 1}


def source_hash() -> str:
    """sha256[:16] of csrc/*.cu, *.cuh with comments and white space removed (a comment edit does not make a capture
    stale; any token change does)."""
    import re
    h = hashlib.sha256()
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh")):
            txt = open(os.path.join(CSRC, f), encoding="utf-8").read()
            txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
            txt = re.sub(r"//[^\n]*", "", txt)
            h.update(f.encode())
            h.update("".join(txt.split()).encode())
    return h.hexdigest()[:16]


def read_stage_csv(path: str):
    """-> ({stage: {column: number | str}}, sha)"""
    stages, sha = {}, None
    rows = list(csv.reader(open(path)))
    head = rows[0]
    for r in rows[1:]:
        if not r:
            continue
        if r[0] == "_src_sha256":
            sha = r[1]
            continue
        d = {}
        for k, v in zip(head[1:], r[1:]):
            try:
                d[k] = float(v) if "." in v else int(v)
            except ValueError:
                d[k] = v
        stages[r[0]] = d
    return stages, sha


def _num(v: str, unit: str) -> float:
    return float(v.replace(",", "")) * UNIT_SCALE.get(unit, 1)


def summarise(rep: str, sha: str, out: str) -> None:
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw[raw.index('"ID"'):])))
    head, units, body = rows[0], rows[1], rows[2:]
    col = {n: i for i, n in enumerate(head)}
    kn = col["Kernel Name"]
    for r in body:  # "void k_raster<...>(...)" -> "k_raster<...>(...)"
        r[kn] = r[kn][5:] if r[kn].startswith("void ") else r[kn]
    # the last frame of the capture: walk back from the end to the last k_generate launch
    # (a complete one: a k_generate launch that has a k_filter launch behind it; the frame ends at that k_filter)
    ends = [i for i, r in enumerate(body) if r[kn].startswith("k_filter")]
    start = max(i for i, r in enumerate(body) if r[kn].startswith("k_generate") and any(e > i for e in ends))
    frame = body[start:min(e for e in ends if e > start) + 1]
    acc = {}
    for r in frame:
        stage = next((s for k, s in STAGE_OF if r[kn].startswith(k)), None)
        if stage is None:
            continue
        a = acc.setdefault(stage, {"kernels": [], **{m: 0.0 for m in METRICS}, **{p: [] for p in PCT}})
        a["kernels"].append(r[kn].split("(")[0])
        for m, names in METRICS.items():
            a[m] += sum(_num(r[col[n]], units[col[n]]) for n in names)
        for p, n in PCT.items():
            a[p].append(r[col[n]])
    with open(out, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["stage"] + list(METRICS) + list(PCT) + ["kernels"])
        for stage in ("generate", "raster", "shade", "filter"):
            a = acc[stage]
            w.writerow([stage] + [int(a[m]) for m in METRICS] + ["/".join(a[p]) for p in PCT] + [" + ".join(a["kernels"])])
        w.writerow(["_src_sha256", sha, "sha256[:16] of csrc/*.cu, *.cuh when the capture ran"])


if __name__ == "__main__":
    if sys.argv[1:] == ["--hash"]:
        print(source_hash())
    else:
        summarise(sys.argv[1], sys.argv[2], sys.argv[3])
