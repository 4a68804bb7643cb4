"""FP64 work per accepted integrator step of the shipped kernels: the numerator of bench.py's roofline.

The counts are MEASURED, not typed in: one ncu pass per workload W over the same bench command,

    python bench.py --workload W --steps 1 --warmup 3 --no-cpu-baseline > gpurun_out/bench_W.json   (must exit 0) &&
    ncu --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__sass_thread_inst_executed_op_ffma_pred_on.sum,\
smsp__sass_thread_inst_executed_op_fmul_pred_on.sum,smsp__sass_thread_inst_executed_op_fadd_pred_on.sum,\
smsp__inst_executed_pipe_fp64.sum,smsp__inst_executed.sum,\
smsp__thread_inst_executed.sum,gpu__time_duration.sum,sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active,\
dram__bytes_read.sum,dram__bytes_write.sum \
        --clock-control none -k regex:k_render -s 3 -c 1 --csv --log-file gpurun_out/flops_W.csv \
        python bench.py --workload W --steps 1 --warmup 3 --no-cpu-baseline

and then, here,

    python -m paper_1801_10452_b200.roofline_counts gpurun_out profiles/fp64_inst_per_step.json

divides the thread-level counters of that k_render launch by the accepted steps of the image (the library's own
counter, printed by the plain run as steps_per_image) and stamps the result with the SHA-256 of the kernel sources
(csrc/*).  bench.py recomputes that hash from the sources it runs and reports roofline = null with the reason when
they differ: a kernel edit cannot silently falsify the roofline fraction.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
DEFAULT_JSON = os.path.join(os.path.dirname(HERE), "profiles", "fp64_inst_per_step.json")
WORKLOADS = ("C0", "C1", "C2", "C3", "C4", "PB1", "PB1F32", "LC", "C3B")

METRICS = {
    "dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "ffma": "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum",
    "fmul": "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum",
    "fadd": "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum",
    "fp64_pipe_warp_inst": "smsp__inst_executed_pipe_fp64.sum",
    "warp_inst": "smsp__inst_executed.sum",
    "thread_inst": "smsp__thread_inst_executed.sum",
    "kernel_ns": "gpu__time_duration.sum",
    "fp64_pipe_pct": "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
    "dram_read_bytes": "dram__bytes_read.sum",
    "dram_write_bytes": "dram__bytes_write.sum",
}


def csrc_sha256() -> str:
    """SHA-256 over the kernel sources (names and contents, sorted): identifies the kernel the counts belong to."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode())
            with open(os.path.join(CSRC, name), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()


_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "nsecond": 1.0, "usecond": 1e3, "msecond": 1e6, "second": 1e9,
         "ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9}


def parse_ncu_csv(path: str) -> dict:
    """Metric name -> value (bytes, ns, counts) of the FIRST profiled launch in an ncu --csv log."""
    with open(path, newline="") as fh:
        lines = [ln for ln in fh if ln.startswith('"')]
    rows = list(csv.reader(lines))
    head = rows[0]
    i_name, i_unit, i_val, i_id = head.index("Metric Name"), head.index("Metric Unit"), head.index("Metric Value"), head.index("ID")
    first = rows[1][i_id]
    out = {}
    for r in rows[1:]:
        if r[i_id] != first:
            continue
        out[r[i_name]] = float(r[i_val].replace(",", "")) * _UNIT.get(r[i_unit], 1.0)
    return out


def collect(run_dir: str) -> dict:
    table = {}
    for w in WORKLOADS:
        f_csv, f_json = os.path.join(run_dir, f"flops_{w}.csv"), os.path.join(run_dir, f"bench_{w}.json")
        if not (os.path.exists(f_csv) and os.path.exists(f_json)):
            continue
        with open(f_json) as fh:
            bench = json.loads(fh.read().strip().splitlines()[-1])
        steps = float(bench["steps_per_image"]) * float(bench.get("frames_per_step", 1))     # accepted steps of ONE launch
        m = parse_ncu_csv(f_csv)
        row = {"steps_per_launch": steps}
        for key, name in METRICS.items():
            if name in m:
                row[key] = m[name] if key in ("kernel_ns", "fp64_pipe_pct", "dram_read_bytes", "dram_write_bytes") else m[name] / steps
        table[w] = row
    return table


def operand_forms(source_csv: str, lib_path: str, mangled: str, steps_per_launch: float) -> dict:
    """FP64 instructions per accepted step by operand form, for the operand-aware bound of DESIGN.md 5.1.

    ``source_csv`` = ``ncu -i prof.ncu-rep --page source --csv --print-source sass`` of one k_render launch (executed
    count per SASS instruction); ``lib_path`` + ``mangled`` (a substring of the mangled kernel name) give the same
    kernel's SASS from ``cuobjdump -sass``, which -- unlike ncu's listing -- carries the ``.reuse`` flags.  The two
    listings are joined by instruction order.  A DFMA whose three sources are three different registers, none of them
    served by the operand-reuse cache (flagged ``.reuse`` on the PREVIOUS instruction's same slot is not tracked here:
    the count below is an upper bound of the slow form), issues every 3.17 cycles on B200; every other FP64
    instruction every 2.06 (raptor_fp64_probe)."""
    import re
    import subprocess
    sass, take = [], False
    out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True).stdout
    for line in out.splitlines():
        if "Function :" in line:
            take = mangled in line
            continue
        if take:
            m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
            if m:
                sass.append(m.group(2).strip())
    with open(source_csv, newline="") as fh:
        rows = list(csv.reader(fh))
    head = next(r for r in rows if "Source" in r and "Instructions Executed" in r)
    i_s, i_e = head.index("Source"), head.index("Instructions Executed")
    prof = [(r[i_s].strip(), int(r[i_e])) for r in rows[rows.index(head) + 1:] if len(r) > i_e and r[i_e].isdigit()]
    n = min(len(sass), len(prof))
    mismatch = sum(1 for a, (b, _) in zip(sass[:n], prof[:n]) if a.replace(".reuse", "").split()[:1] != b.split()[:1])
    warp_steps = steps_per_launch / 32.0
    out_counts = {"dfma_3reg": 0.0, "dfma_3reg_reuse_flagged": 0.0, "dfma_other": 0.0, "dmul": 0.0, "dadd": 0.0, "dsetp": 0.0}
    for text, (_, cnt) in zip(sass[:n], prof[:n]):
        t = re.sub(r"^@!?U?P\d+\s+", "", text)
        op = t.split()[0].split(".")[0]
        if op not in ("DFMA", "DMUL", "DADD", "DSETP"):
            continue
        srcs = [o.strip() for o in t.split(None, 1)[1].split(",")[1:]]
        regs, reuse = set(), 0
        for o in srcs:
            m = re.match(r"^[-|~]*\|?(R\d+)(\.reuse)?", o)
            if m:
                regs.add(m.group(1))
                reuse += 1 if m.group(2) else 0
        key = {"DMUL": "dmul", "DADD": "dadd", "DSETP": "dsetp"}.get(op)
        if op == "DFMA":
            key = "dfma_other" if len(regs) < 3 else ("dfma_3reg_reuse_flagged" if reuse else "dfma_3reg")
        out_counts[key] += cnt / warp_steps
    out_counts["listing_mismatch"] = mismatch
    return out_counts


def by_function(disasm: str, source_csv: str, mangled: str, steps_per_launch: float) -> dict:
    """FP64-pipe and all warp instructions per warp-step by device function: where a step's instructions go.

    ``disasm`` = ``nvdisasm -g -c`` of a cubin of the kernel built with the library's flags, e.g.

        nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -std=c++17 --fmad=true -DRAPTOR_MODEL=3 -DRAPTOR_INTEG=0 \
             -cubin paper_1801_10452_b200/csrc/raptor_render.cu -o m3.cubin && nvdisasm -g -c m3.cubin > m3.dis

    (its ``//## File ..., line N`` marks name the innermost inlined source line of every instruction);
    ``source_csv`` = ``ncu -i prof.ncu-rep --page source --csv --print-source sass`` of one launch of that kernel (executed
    count per SASS instruction).  The two listings are joined by instruction order (the opcodes must agree), lines of
    raptor_device.cuh are mapped to the ``__device__`` function they lie in, everything in raptor_render.cu is the RK4
    combination and the loop.  Run:  python -m paper_1801_10452_b200.roofline_counts --by-function m3.dis source_C2.csv
    k_renderILi3ELb0ELb0ELb0ELi0ELb0ELb0E <accepted steps of the launch>."""
    import re
    starts = []
    with open(os.path.join(CSRC, "raptor_device.cuh")) as fh:
        for i, line in enumerate(fh, 1):
            m = re.match(r"^(?:static )?__device__ .*?(\w+)\(", line)
            if m:
                starts.append((i, m.group(1)))

    def func_of(path, line):
        if path.endswith("raptor_device.cuh"):
            name = "?"
            for s0, n0 in starts:
                if s0 <= line:
                    name = n0
            return name
        return "raptor_render.cu" if path.endswith("raptor_render.cu") else "library:" + os.path.basename(path)

    ins, take, path, line = [], False, "?", 0
    with open(disasm) as fh:
        for text in fh:
            if text.startswith("//---") and ".text." in text:
                take = mangled in text
                continue
            if not take:
                continue
            m = re.match(r'\s*//## File "(.*)", line (\d+)', text)
            if m:
                path, line = m.group(1), int(m.group(2))
                continue
            m = re.match(r"\s*/\*([0-9a-f]{4,})\*/\s+(.*?);", text)
            if m:
                op = re.sub(r"^@!?U?P\d+\s+", "", m.group(2).strip()).split()[0].split(".")[0]
                ins.append((op, func_of(path, line)))
    with open(source_csv, newline="") as fh:
        rows = list(csv.reader(fh))
    head = next(r for r in rows if "Source" in r and "Instructions Executed" in r)
    i_s, i_e = head.index("Source"), head.index("Instructions Executed")
    prof = [(r[i_s].strip(), int(r[i_e])) for r in rows[rows.index(head) + 1:] if len(r) > i_e and r[i_e].isdigit()]
    n = min(len(ins), len(prof))
    mismatch = sum(1 for (op, _), (src, _) in zip(ins[:n], prof[:n])
                   if op != re.sub(r"^@!?U?P\d+\s+", "", src).split()[0].split(".")[0])
    warp_steps = steps_per_launch / 32.0
    out = {}
    for (op, fn), (_, cnt) in zip(ins[:n], prof[:n]):
        row = out.setdefault(fn, {"all": 0.0, "fp64_pipe": 0.0})
        row["all"] += cnt / warp_steps
        if op in ("DFMA", "DMUL", "DADD", "DSETP", "DMNMX"):
            row["fp64_pipe"] += cnt / warp_steps
    out["_listing"] = {"instructions": n, "mismatch": mismatch}
    return out


def load(path: str = DEFAULT_JSON):
    """(table, None) if the committed counts belong to the sources in this tree, else (None, reason)."""
    if not os.path.exists(path):
        return None, f"{os.path.relpath(path, os.path.dirname(HERE))} is missing"
    with open(path) as fh:
        doc = json.load(fh)
    have = csrc_sha256()
    if doc.get("csrc_sha256") != have:
        return None, (f"profiles/fp64_inst_per_step.json was measured on csrc {str(doc.get('csrc_sha256'))[:12]}, "
                      f"the sources here hash to {have[:12]}: re-run the ncu pass (paper_1801_10452_b200/roofline_counts.py)")
    return doc["per_step"], None


# mangled-name substrings of the kernels bench.py's workloads launch (for operand_forms)
KERNEL_OF = {"C0": "k_renderILi1ELb1ELb0ELb0ELi0ELb0ELb0E", "C1": "k_renderILi2ELb1ELb0ELb0ELi0ELb0ELb0E",
             "C2": "k_renderILi3ELb0ELb0ELb0ELi0ELb0ELb0E", "C3": "k_renderILi3ELb0ELb1ELb0ELi0ELb0ELb0E",
             "C4": "k_renderILi4ELb0ELb0ELb1ELi0ELb0ELb0E", "PB1": "k_renderILi3ELb0ELb0ELb1ELi3ELb0ELb0E"}


def main(argv):
    if len(argv) > 1 and argv[1] == "--by-function":
        table = by_function(argv[2], argv[3], argv[4], float(argv[5]))
        for fn, row in sorted(table.items(), key=lambda kv: -kv[1].get("all", 0.0)):
            print(f"{fn:28s} " + "  ".join(f"{k} {v:9.1f}" if isinstance(v, float) else f"{k} {v}" for k, v in row.items()))
        return
    run_dir = argv[1] if len(argv) > 1 else "gpurun_out"
    out = argv[2] if len(argv) > 2 else DEFAULT_JSON
    table = collect(run_dir)
    if not table:
        raise SystemExit(f"no flops_<W>.csv + bench_<W>.json pairs under {run_dir}")
    # optional: operand forms, where `ncu -i prof_<W>_r2.ncu-rep --page source --csv --print-source sass > source_<W>.csv` exists
    lib_path = os.path.join(HERE, "libraptor_b200.so")
    for w, mangled in KERNEL_OF.items():
        src = os.path.join(run_dir, f"source_{w}.csv")
        if w in table and os.path.exists(src) and os.path.exists(lib_path):
            table[w]["operand_forms"] = operand_forms(src, lib_path, mangled, table[w]["steps_per_launch"])
    doc = {"csrc_sha256": csrc_sha256(),
           "what": "thread-level executed FP64 instructions of one k_render launch / accepted steps of that launch; "
                   "flop = 2 dfma + dmul + dadd; fp64_pipe_warp_inst = warp-level instructions issued to the FP64 pipe "
                   "(arithmetic + DSETP etc.); kernel_ns, dram bytes: that launch under ncu (cold cache, serialised)",
           "command": "see the docstring of paper_1801_10452_b200/roofline_counts.py",
           "per_step": table}
    with open(out, "w") as fh:
        json.dump(doc, fh, indent=1, sort_keys=True)
        fh.write("\n")
    print(json.dumps(doc, indent=1, sort_keys=True))


if __name__ == "__main__":
    main(sys.argv)
