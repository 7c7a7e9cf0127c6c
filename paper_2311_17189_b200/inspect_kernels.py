"""Inspection of the specialised kernels of a workload without a GPU: compiles them with NVRTC through
ami_table_kernel_cubin_variant, runs ``cuobjdump -sass`` on the result and prints, per kernel, the
registers / spills ptxas reports, the histogram of SASS opcodes (FP64-pipe opcodes first) and the register operands
of the FP64 instructions with the register-file ceiling they imply.

    python -m paper_2311_17189_b200.inspect_kernels cfg3 [--unit 0] [--complex] [--dim 2] [--band 0] [--top 25]

Workloads are the names of ami_inputs.get_config plus ``order7``.  This is how the opcode tables under
profiles/ are made.
"""
from __future__ import annotations

import argparse
import collections
import os
import re
import subprocess
import tempfile

FP64 = ("DFMA", "DMUL", "DADD", "DSETP", "MUFU")


def histogram(cubin: bytes) -> dict:
    """{kernel or function name: Counter(opcode -> static count)} from cuobjdump -sass."""
    with tempfile.NamedTemporaryFile(suffix=".cubin", delete=False) as f:
        f.write(cubin)
        path = f.name
    try:
        text = subprocess.run([os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump"), "-sass", path],
                              capture_output=True, text=True, check=True).stdout
    finally:
        os.unlink(path)
    out, cur = collections.OrderedDict(), None
    for line in text.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = out.setdefault(m.group(1), collections.Counter())
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", line)
        if m and cur is not None:
            cur[m.group(1)] += 1
    return out


def operand_classes(cubin: bytes) -> dict:
    """{kernel: {"fp64": Counter((opcode, distinct register operands, of which flagged .reuse) -> count),
    "other_reads": register reads of all other instructions, "other": their number}} from cuobjdump -sass.
    The register file hands out one 64-bit operand per lane and cycle, so a DFMA with three distinct
    register operands costs three cycles where the pipe needs two."""
    with tempfile.NamedTemporaryFile(suffix=".cubin", delete=False) as f:
        f.write(cubin)
        path = f.name
    try:
        text = subprocess.run([os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump"), "-sass", path],
                              capture_output=True, text=True, check=True).stdout
    finally:
        os.unlink(path)
    out, cur = collections.OrderedDict(), None
    for line in text.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = out.setdefault(m.group(1), {"fp64": collections.Counter(), "other_reads": 0, "other": 0})
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)\s*(.*?);", line)
        if not m or cur is None:
            continue
        op, args = m.group(1).split(".")[0], [x.strip() for x in m.group(2).split(",")]
        regs, reuse = set(), 0
        for x in args[1:]:                       # source operands (the first is the destination)
            r = re.match(r"[-|~!]*(R\d+)((?:\.\w+)*)", x)
            if r and r.group(1) != "RZ" and r.group(1) not in regs:
                regs.add(r.group(1))
                reuse += ".reuse" in r.group(2)
        if op in ("DFMA", "DMUL", "DADD", "DSETP"):
            cur["fp64"][(op, len(regs), reuse)] += 1
        else:
            cur["other"] += 1
            cur["other_reads"] += len(regs)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload")
    ap.add_argument("--unit", type=int, default=0)
    ap.add_argument("--complex", action="store_true")
    ap.add_argument("--dim", type=int, default=2)
    ap.add_argument("--band", type=int, default=0)
    ap.add_argument("--top", type=int, default=25)
    args = ap.parse_args()
    import ami_inputs as A
    from . import AmiTable
    cfg = A.get_config("stress8" if args.workload == "order7" else args.workload)
    diagram = A.random_self_energy(7, 0) if args.workload == "order7" else cfg.diagram
    tab = AmiTable.from_diagram(diagram, device=None)
    info = tab.info
    print(f"workload {args.workload}: T_flat {info['n_terms']}, U_F {info['n_fermi_leaves']}, U_D {info['n_den_leaves']}, "
          f"plan kind {info['plan_kind']} (1 register, 2 split), translation units {tab.kernel_units()}, unit {args.unit}")
    cubin, log = tab.kernel_cubin(unit=args.unit, dim=args.dim, band=args.band, complex_energies=args.complex)
    fn = None
    for line in log.splitlines():
        m = re.search(r"(?:Compiling entry function|Function properties for) '?([\w]+)'?", line)
        if m:
            fn = m.group(1)
        if "registers" in line or "spill" in line:
            print(f"ptxas {fn}: {line.split(':', 1)[-1].strip() if 'Used' in line else line.strip()}")
    for name, cnt in histogram(cubin).items():
        total = sum(cnt.values())
        fp = sum(cnt[o] for o in FP64)
        print(f"\n{name}: {total} SASS instructions, FP64 pipe (DFMA DMUL DADD DSETP) {fp - cnt['MUFU']} + MUFU {cnt['MUFU']}")
        order = [o for o in FP64 if cnt[o]] + [o for o, _ in cnt.most_common() if o not in FP64]
        print("  " + "  ".join(f"{o} {cnt[o]}" for o in order[: args.top]))
    print("\nregister operands of the FP64 instructions (static; (opcode, distinct register operands, flagged .reuse): count)")
    for name, c in operand_classes(cubin).items():
        n_fp = sum(c["fp64"].values())
        pairs = sum(k[1] * v for k, v in c["fp64"].items())
        three = sum(v for k, v in c["fp64"].items() if k[1] == 3)
        rf = pairs + c["other_reads"] / 2.0          # cycles of register-file bandwidth: one 64-bit operand per cycle
        print(f"{name}: {n_fp} FP64 instructions reading {pairs / max(n_fp, 1):.2f} register pairs on average, {three} with three; "
              f"{c['other']} other instructions with {c['other_reads']} 32-bit register reads; register-file cycles "
              f"{rf:.0f} against {2 * n_fp} FP64-pipe cycles -> ceiling {min(1.0, 2 * n_fp / max(rf, 1)):.2f} of the issue rate")
        print("  " + "  ".join(f"{k[0]}/{k[1]}/{k[2]}: {v}" for k, v in sorted(c["fp64"].items())))


if __name__ == "__main__":
    main()
