"""Search for the statement order of m2l_pair_folded (developer tool; needs nvcc and cuobjdump, no GPU).

    python -m paper_2101_08226_b200.order_search [--function folded|components] [--minutes M] [--seed S] [--random N]
                                                 [--weights A B] [--apply]

Why: the interaction kernel is bound by the FP64 pipe, and a DFMA whose three source registers all have to be read
fresh holds the pipe for 3 cycles instead of 2.  Whether consecutive instructions share an
operand slot is decided by ptxas's schedule of the loop body; ptxas is deterministic and starts from the order of the
source, so the order of the (mutually independent) statements of the body is a free parameter.  This tool
  1. reads the statements of m2l_pair_folded (correction on; or, with --function components, of m2l_pair_components, the
     body with the correction off) from csrc/m2l_math.cuh (one statement per line) and builds their
     dependency graph (a statement depends on the last writer of every name it reads; updates of one accumulator stay
     in their order),
  2. generates variants -- `--random N` random topological orders first, then hill climbing by single-statement moves
     from the best order so far for `--minutes M` --,
  3. compiles each variant of the ONE kernel m2l_staged_kernel<correction on (off), no fused L2L, plain> (1.5 s) in a
     temporary directory and scores its SASS with sass_cost_model: FP64-pipe cycles of the two copies of the
     software-pipelined loop body on the general path, plus a quarter of those of the path without dipole terms,
  4. prints the best order; `--apply` writes it into csrc/m2l_math.cuh.
The order in the repository is the result of about 2000 variants (round 2).  The search is reproducible for a given seed
and compiler version; a different nvcc will want a new search."""
import json
import os
import random
import re
import shutil
import subprocess
import sys
import tempfile
import time
from concurrent.futures import ProcessPoolExecutor

from . import sass_cost_model as scm

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
MATH = os.path.join(CSRC, "m2l_math.cuh")
# the two pair bodies: (function, comment line that follows it in m2l_math.cuh, kernel whose SASS is scored, its instantiation)
TARGETS = {
    "folded": ("void m2l_pair_folded(", "// Body of one ordered pair with the correction OFF, component form",
               "m2l_staged_kernelILb1ELb0ELi0E", "true"),
    "components": ("void m2l_pair_components(", "// Body of one ordered pair A <- B.",
                   "m2l_staged_kernelILb0ELb0ELi0E", "false"),
}
TARGET = "folded"


def one_cu():
    return ('#include "kernels.cuh"\ntemplate __global__ void octo::m2l_staged_kernel<%s, false, octo::MODE_PLAIN>'
            "(const __grid_constant__ octo::SlabMaps, const __grid_constant__ octo::Params);\n" % TARGETS[TARGET][3])
IDENT = re.compile(r"a\.\w+(?:\[\d\])?|[A-Za-z_]\w*")
NOT_NAMES = {"const", "double", "fma", "if", "DIPOLE", "s", "tA", "x", "y", "z", "w", "a", "c_fold"}


def body_span(src):
    start, after = TARGETS[TARGET][0], TARGETS[TARGET][1]
    a = src.index("{", src.index(start)) + 1
    b = src.rindex("}", a, src.index(after, a))
    return a, b


def read_statements():
    src = open(MATH).read()
    a, b = body_span(src)
    return [l.strip() for l in src[a:b].splitlines() if l.strip() and not l.strip().startswith("//")]


def analyse(stmts):
    """per statement: (name it defines, names it reads); an accumulator update reads and defines the accumulator"""
    info = []
    for st in stmts:
        body = st[len("if (DIPOLE) "):] if st.startswith("if (DIPOLE) ") else st
        if body.startswith("const double "):
            lhs, rhs = body[len("const double "):].split("=", 1)
            info.append((lhs.strip(), set(IDENT.findall(rhs)) - NOT_NAMES))
        else:
            m = re.match(r"(a\.\w+(?:\[\d\])?)\s*\+?=\s*(.*)", body)
            if not m:
                raise SystemExit("order_search: cannot parse statement %r" % st)
            info.append((m.group(1), (set(IDENT.findall(m.group(2))) - NOT_NAMES) | {m.group(1)}))
    last, dep = {}, []
    for i, (d, uses) in enumerate(info):
        dep.append({last[u] for u in uses if u in last})
        last[d] = i
    succ = [[] for _ in info]
    for i, ds in enumerate(dep):
        for j in ds:
            succ[j].append(i)
    return dep, succ


def random_order(n, dep, succ, rng, locality):
    indeg = [len(d) for d in dep]
    ready = [i for i in range(n) if indeg[i] == 0]
    stamp = {i: 0 for i in ready}
    order, t = [], 0
    while ready:
        t += 1
        if rng.random() < locality:                    # depth first: prefer what became ready last
            m = max(stamp[i] for i in ready)
            pick = rng.choice([i for i in ready if stamp[i] == m])
        else:
            pick = rng.choice(ready)
        ready.remove(pick)
        order.append(pick)
        for k in succ[pick]:
            indeg[k] -= 1
            if indeg[k] == 0:
                ready.append(k)
                stamp[k] = t
    return order


def mutate(order, dep, succ, rng, moves):
    order = list(order)
    n = len(order)
    for _ in range(moves):
        i = rng.randrange(n)
        st = order.pop(i)
        pos = {s: k for k, s in enumerate(order)}
        lo = max([pos[d] for d in dep[st]], default=-1) + 1
        hi = min([pos[s] for s in succ[st]], default=n - 1)
        order.insert(rng.randint(lo, hi) if lo <= hi else i, st)
    return order


def score(args):
    """FP64-pipe cycles of the pair-body blocks of one variant, or None if it does not compile or spills"""
    global TARGET
    workdir, stmts, order, TARGET = args
    os.makedirs(workdir, exist_ok=True)
    for f in os.listdir(CSRC):
        if f.endswith(".cuh"):
            shutil.copy(os.path.join(CSRC, f), os.path.join(workdir, f))
    src = open(MATH).read()
    a, b = body_span(src)
    open(os.path.join(workdir, "m2l_math.cuh"), "w").write(src[:a] + "\n" + "".join("    %s\n" % stmts[i] for i in order) + src[b:])
    open(os.path.join(workdir, "one.cu"), "w").write(one_cu())
    r = subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-cubin", "-o", "one.cubin",
                        "one.cu", "-Xptxas", "-v"], cwd=workdir, capture_output=True, text=True)
    spill = re.search(r"(\d+) bytes spill stores", r.stderr)
    if r.returncode != 0 or not spill or int(spill.group(1)) != 0:
        return None
    ins = scm.parse(scm.dump(os.path.join(workdir, "one.cubin"), TARGETS[TARGET][2]))
    cyc = []
    for lo, hi, _ in scm.blocks(ins):
        c, n, _, _ = scm.model(ins, lo, hi)
        cyc.append(c - n["other"])
    return cyc if len(cyc) >= 6 else None


WEIGHTS = (1.0, 0.25)       # of the general path and of the path without dipole terms (--weights A B)


def objective(cyc):
    return 1e9 if cyc is None else WEIGHTS[0] * (cyc[0] + cyc[1]) + WEIGHTS[1] * (cyc[3] + cyc[4])


def main(argv):
    def opt(name, default):
        return type(default)(argv[argv.index(name) + 1]) if name in argv else default
    global TARGET, WEIGHTS
    minutes, seed, nrandom = opt("--minutes", 10.0), opt("--seed", 1), opt("--random", 64)
    if "--weights" in argv:
        WEIGHTS = (float(argv[argv.index("--weights") + 1]), float(argv[argv.index("--weights") + 2]))
    TARGET = opt("--function", "folded")
    if TARGET not in TARGETS:
        raise SystemExit("order_search: --function folded | components")
    rng = random.Random(seed)
    stmts = read_statements()
    dep, succ = analyse(stmts)
    n = len(stmts)
    tmp = tempfile.mkdtemp(prefix="order_search_")
    workers = max(1, min(8, os.cpu_count() or 1))
    try:
        with ProcessPoolExecutor(workers) as ex:
            def evaluate(orders):
                return list(ex.map(score, [(os.path.join(tmp, "w%d" % (k % workers)), stmts, o, TARGET) for k, o in enumerate(orders)],
                                   chunksize=max(1, len(orders) // workers)))
            cur = list(range(n))
            best_cyc = evaluate([cur])[0]
            best = objective(best_cyc)
            print("source order: objective %.2f, FP64-pipe cycles per block %s" % (best, best_cyc), flush=True)
            cands = [random_order(n, dep, succ, rng, rng.choice([0.0, 0.3, 0.6, 0.8, 0.9, 0.97])) for _ in range(nrandom)]
            for o, c in zip(cands, evaluate(cands) if cands else []):
                if objective(c) < best:
                    best, best_cyc, cur = objective(c), c, o
            print("after %d random orders: objective %.2f %s" % (nrandom, best, best_cyc), flush=True)
            t0 = time.time()
            while time.time() - t0 < 60 * minutes:
                cands = [mutate(cur, dep, succ, rng, rng.choice([1, 1, 2, 3, 5])) for _ in range(workers)]
                for o, c in zip(cands, evaluate(cands)):
                    if objective(c) <= best:
                        if objective(c) < best:
                            print("  objective %.2f %s" % (objective(c), c), flush=True)
                        best, best_cyc, cur = objective(c), c, o
    finally:
        shutil.rmtree(tmp, ignore_errors=True)
    print("best: objective %.2f, FP64-pipe cycles per block %s" % (best, best_cyc))
    print(json.dumps(cur))
    if "--apply" in argv:
        src = open(MATH).read()
        a, b = body_span(src)
        open(MATH, "w").write(src[:a] + "\n" + "".join("    %s\n" % stmts[i] for i in cur) + src[b:])
        print("written to", MATH)


if __name__ == "__main__":
    main(sys.argv[1:])
