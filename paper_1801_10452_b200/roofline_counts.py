"""FP64 work per accepted integrator step of the shipped kernels: the numerator of bench.py's roofline.

``profiles/fp64_inst_per_step.json`` holds, per workload, the thread-level executed DFMA / DMUL / DADD (FP32 kernel:
FFMA / FMUL / FADD) instructions of one ``k_render`` launch divided by the accepted integrator steps of that launch,
measured with ncu over ``python bench.py --workload W --steps 1 --warmup 3 --no-cpu-baseline``; the ncu command line, the
metric names and the table made from them are in ``profiles/flop_per_step_r*.md``.  The file is stamped with the
SHA-256 of the kernel sources (``csrc/*``) it was measured on.  ``load()`` recomputes that hash from the sources
bench.py is about to run and returns no table, with the reason, when they differ: a kernel edit cannot silently
falsify the roofline fraction.

This module only READS the committed counts.  The scripts that turn ncu logs into that file (and into the operand-form
and per-function breakdowns quoted in ``profiles/``) are measurement tooling and are not part of the package.
"""
from __future__ import annotations

import hashlib
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
DEFAULT_JSON = os.path.join(os.path.dirname(HERE), "profiles", "fp64_inst_per_step.json")


def csrc_sha256() -> str:
    """SHA-256 over the kernel sources (names and contents, sorted): identifies the kernel the counts belong to."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode())
            with open(os.path.join(CSRC, name), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()


def load(path: str = DEFAULT_JSON):
    """(table, None) if the committed counts belong to the sources in this tree, else (None, reason)."""
    if not os.path.exists(path):
        return None, f"{os.path.relpath(path, os.path.dirname(HERE))} is missing"
    with open(path) as fh:
        doc = json.load(fh)
    have = csrc_sha256()
    if doc.get("csrc_sha256") != have:
        return None, (f"profiles/fp64_inst_per_step.json was measured on csrc {str(doc.get('csrc_sha256'))[:12]}, "
                      f"the sources here hash to {have[:12]}: repeat the ncu pass of profiles/flop_per_step_r*.md")
    return doc["per_step"], None
