"""Static instruction counts of the main kernels from `cuobjdump -sass` (test infrastructure).

bench.py's roofline multiplies FP64-pipe instruction counts per template-bin / per node interval by the
units one launch processes; test_cabi.py re-derives those counts from the SASS of the built library with
the functions here, so the constants in bench.py cannot drift from the code."""
import re
import subprocess

FP64_OPS = ("DFMA", "DMUL", "DADD", "DSETP")


def kernel_instructions(lib_path: str, kernel: str):
    """[(address, opcode-without-modifiers, full text)] of one kernel."""
    out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, check=True).stdout
    starts = [m.start() for m in re.finditer(r"Function : \S*" + re.escape(kernel), out)]
    if not starts:
        raise KeyError(kernel)
    i = starts[0]
    j = out.find("Function :", i + 10)
    ins = []
    for line in out[i:j if j > 0 else None].splitlines():
        m = re.search(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);", line)
        if not m:
            continue
        words = m.group(2).split()
        op = words[1] if words[0].startswith("@") else words[0]
        ins.append((int(m.group(1), 16), op.split(".")[0], m.group(2).strip()))
    return ins


def loops(ins):
    """[(start, end)] address ranges closed by a backward branch, innermost first (sorted by length)."""
    found = []
    for addr, op, text in ins:
        if op != "BRA":
            continue
        m = re.search(r"(0x[0-9a-f]+)\s*$", text)
        if m and int(m.group(1), 16) < addr:
            found.append((int(m.group(1), 16), addr))
    return sorted(found, key=lambda r: r[1] - r[0])


def count(ins, lo, hi, ops=FP64_OPS):
    return sum(1 for a, op, _ in ins if lo <= a <= hi and op in ops), sum(1 for a, _, _ in ins if lo <= a <= hi)


def fast_kernel_counts(lib_path: str):
    """FP64 instructions per template-bin of fstat_fast_kernel: its per-bin loops are the innermost loops
    that read the folded data from shared memory (one LDS.128 per bin); every variant the compiler emits
    must have the same FP64 count per bin.  (Per node interval and per work item the executed counts are
    measured with ncu, profiles/r1_v6.md: rare paths and loop peeling make the static count ambiguous.)"""
    ins = kernel_instructions(lib_path, "fstat_fast_kernel")
    per_bin, per_bin_all = set(), []
    all_loops = loops(ins)
    for lo, hi in all_loops:
        if any(lo <= l2 and h2 <= hi and (l2, h2) != (lo, hi) for l2, h2 in all_loops):
            continue                                      # not innermost
        n_lds = sum(1 for a, op, _ in ins if lo <= a <= hi and op == "LDS")
        n64, ntot = count(ins, lo, hi)
        if n_lds >= 1 and n64 >= 10:
            per_bin.add(n64 / n_lds)
            per_bin_all.append(ntot / n_lds)
    assert per_bin, "no per-bin loop found"
    return {"per_bin": sorted(per_bin), "per_bin_all_pipes": min(per_bin_all)}


def direct_kernel_counts(lib_path: str):
    ins = kernel_instructions(lib_path, "fstat_main_kernel")
    best = max(loops(ins), key=lambda r: count(ins, *r)[0] if r[1] - r[0] < 0x4000 else 0)
    # the per-bin loop is the innermost loop that holds (nearly) all of the kernel's FP64 work
    cands = [r for r in loops(ins) if count(ins, *r)[0] >= 200]
    lo, hi = cands[0] if cands else best
    n, t = count(ins, lo, hi)
    return {"per_bin": float(n), "per_bin_all_pipes": float(t)}
