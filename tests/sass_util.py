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
    """FP64 instructions of fstat_fast_kernel: per template-bin (inner loop, unrolled by 2), per node
    interval (outer loop body without the inner loop) and before the outer loop (work-item prologue:
    three node evaluations, linear phase term)."""
    ins = kernel_instructions(lib_path, "fstat_fast_kernel")
    ls = [r for r in loops(ins) if count(ins, *r)[0] >= 20]
    inner, outer = ls[0], ls[-1]
    assert outer[0] < inner[0] and inner[1] < outer[1]
    n_inner, t_inner = count(ins, *inner)
    n_outer, t_outer = count(ins, *outer)
    n_pre, _ = count(ins, 0, outer[0] - 1)
    unroll = 2
    return {"per_bin": n_inner / unroll, "per_bin_all_pipes": t_inner / unroll,
            "per_interval": n_outer - n_inner, "per_item": n_pre}


def direct_kernel_counts(lib_path: str):
    ins = kernel_instructions(lib_path, "fstat_main_kernel")
    best = max(loops(ins), key=lambda r: count(ins, *r)[0] if r[1] - r[0] < 0x4000 else 0)
    # the per-bin loop is the innermost loop that holds (nearly) all of the kernel's FP64 work
    cands = [r for r in loops(ins) if count(ins, *r)[0] >= 200]
    lo, hi = cands[0] if cands else best
    n, t = count(ins, lo, hi)
    return {"per_bin": float(n), "per_bin_all_pipes": float(t)}
