"""SASS cost model of the interaction kernels' hot loops (developer tool; reads the built library with cuobjdump).

    python -m paper_2101_08226_b200.sass_cost_model [function-substring] [-v]

Finds the straight-line blocks that hold a pair body (>= 40 DFMAs) in the SASS of the named kernel (default: the
headline instantiation m2l_staged_kernel<correction on, no fused L2L, plain>) and prints per block the FP64 instruction
tally (DFMA / DMUL / DADD: the operation count of DESIGN.md section 7), the DFMAs by number of FRESH register
operands, and the modelled cycles per pair; -v lists every instruction with its modelled cost.
Model (register file: two banks, a 64-bit operand takes one read slot of each): an FP64
instruction holds the sub-partition's dispatch port for max(2, number of distinct 64-bit register operands that do not
come from the operand-reuse cache) cycles; every other instruction for 1.  An operand comes from the reuse cache if the
instruction before carried `.reuse` on the same register in the same operand slot.  "FP64 pipe" is the sum over the FP64
instructions alone: measured kernel times follow THAT number (the other instructions issue in the shadow of the FP64
pipe: removing six of them per pair in round 2 changed nothing, removing FP64 pipe cycles always did).
profiles/r02_sass_cost_model.md is the output of this tool for the shipped kernels."""
import re
import subprocess
import sys

FP64 = ("DFMA", "DMUL", "DADD")


def dump(lib, fn):
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    lines = out.splitlines()
    start = None
    res = []
    for i, l in enumerate(lines):
        if "Function :" in l:
            if start is not None:
                break
            if fn in l:
                start = i
        elif start is not None:
            res.append(l)
    return res


INS = re.compile(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);")


def parse(lines):
    ins = []
    for l in lines:
        m = INS.search(l)
        if not m:
            continue
        addr = int(m.group(1), 16)
        text = m.group(2).strip()
        pred = None
        if text.startswith("@"):
            pred, text = text.split(None, 1)
        parts = text.split(None, 1)
        op = parts[0]
        ops = [o.strip() for o in parts[1].split(",")] if len(parts) > 1 else []
        ins.append((addr, op, ops, pred))
    return ins


REG = re.compile(r"^[-|~!]*\|?(R\d+)(\.reuse)?\|?$")


def srcregs(op, ops):
    """list of (slot, reg, reuse) of the source operands of an FP64 instruction"""
    res = []
    for slot, o in enumerate(ops[1:]):
        m = REG.match(o.replace(".64", ""))
        if m:
            res.append((slot, m.group(1), bool(m.group(2))))
    return res


def model(ins, lo, hi, verbose=False):
    prev_reuse = {}
    cyc = 0
    n = {"DFMA": 0, "DMUL": 0, "DADD": 0, "other": 0}
    fresh3 = 0
    hist = {}
    for addr, op, ops, pred in ins:
        if addr < lo or addr >= hi:
            continue
        base = op.split(".")[0]
        cur_reuse = {}
        if base in FP64:
            regs = srcregs(op, ops)
            fresh = set()
            for slot, r, ru in regs:
                if prev_reuse.get(slot) != r:
                    fresh.add(r)
                if ru:
                    cur_reuse[slot] = r
            c = max(2, len(fresh))
            n[base] += 1
            if base == "DFMA":
                hist[len(fresh)] = hist.get(len(fresh), 0) + 1
                if len(fresh) >= 3:
                    fresh3 += 1
            if verbose:
                print("%05x %d %-6s %s" % (addr, c, op, ", ".join(ops)))
        else:
            c = 1
            n["other"] += 1
            # a non-FP64 instruction keeps the cache only for the slots it flags itself
            for slot, o in enumerate(ops[1:]):
                m = REG.match(o)
                if m and m.group(2):
                    cur_reuse[slot] = m.group(1)
            if verbose:
                print("%05x %d %-6s %s" % (addr, c, op, ", ".join(ops)))
        cyc += c
        prev_reuse = cur_reuse
    return cyc, n, fresh3, hist


def blocks(ins):
    """maximal straight-line runs with >= 60 DFMAs (the pair bodies)"""
    res = []
    start = None
    cnt = 0
    for i, (addr, op, ops, pred) in enumerate(ins):
        if start is None:
            start = addr
            cnt = 0
        if op.startswith("DFMA"):
            cnt += 1
        if op.startswith(("BRA", "EXIT", "BSYNC", "BSSY", "RET", "CALL", "WARPSYNC")):
            if cnt >= 40:
                res.append((start, addr + 16, cnt))
            start = None
    return res


def main(argv):
    import os
    args = [a for a in argv if not a.startswith("-")]
    lib = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libocto_fmm.so")
    if args and os.path.exists(args[0]):
        lib = args.pop(0)
    fn = args[0] if args else "m2l_staged_kernelILb1ELb0ELi0E"
    ins = parse(dump(lib, fn))
    if not ins:
        raise SystemExit("no function matching %r in %s" % (fn, lib))
    rng = blocks(ins)
    verbose = "-v" in argv
    print("# %s in %s" % (fn, os.path.basename(lib)))
    for lo, hi, cnt in rng:
        cyc, n, f3, hist = model(ins, lo, hi, verbose)
        fp = n["DFMA"] + n["DMUL"] + n["DADD"]
        print("block %05x-%05x: cycles %d (FP64 pipe %d)  DFMA %d DMUL %d DADD %d other %d | fp64 %d flop %d | DFMA fresh-operand histogram %s" % (
            lo, hi, cyc, cyc - n["other"], n["DFMA"], n["DMUL"], n["DADD"], n["other"], fp, 2 * n["DFMA"] + n["DMUL"] + n["DADD"],
            dict(sorted(hist.items()))))


if __name__ == "__main__":
    main(sys.argv[1:])
