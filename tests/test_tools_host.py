"""The two developer tools that DESIGN.md section 7 leans on, checked against the built library (no GPU needed:
cuobjdump reads the sm_100a cubin here).

1. sass_cost_model: the FP64 tally of the hot loops in the SHIPPED SASS equals what octo_fmm_flops_per_interaction(_path)
   reports -- the roofline's flop count is pinned to the code, not to a comment.
2. order_search: the statements of m2l_pair_folded parse, the order in the source respects their dependencies, and the
   orders the search generates are permutations that respect them too."""
import random
import shutil

import pytest

cuobjdump = pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")


def _loop_blocks(fn):
    from paper_2101_08226_b200 import build
    from paper_2101_08226_b200 import sass_cost_model as scm
    lib = build.build()
    ins = scm.parse(scm.dump(lib, fn))
    assert ins, fn
    res = []
    for lo, hi, _ in scm.blocks(ins):
        cyc, n, fresh3, hist = scm.model(ins, lo, hi)
        res.append((cyc, n, fresh3))
    return res


@cuobjdump
@pytest.mark.parametrize("corr,fn", [(True, "m2l_staged_kernelILb1ELb0ELi0E"), (False, "m2l_staged_kernelILb0ELb0ELi0E")])
def test_flop_counts_are_those_of_the_shipped_sass(corr, fn):
    import paper_2101_08226_b200 as p
    blocks = _loop_blocks(fn)
    # blocks 1-2: the two copies of the pipelined loop body, general path; 3: its drain; 4-6: the path without dipole terms
    assert len(blocks) == 6
    for first, dipole in ((0, True), (3, False)):
        flops, instr = p.octo_fmm_flops_per_interaction_path(p.MULTIPOLE, corr, dipole)
        for cyc, n, _ in blocks[first:first + 2]:
            fp64 = n["DFMA"] + n["DMUL"] + n["DADD"]
            # the per-(class, dz) segment carries one more DADD (Rz0) that the per-pair count includes
            assert fp64 in (instr, instr - 1), (fn, dipole, n, instr)
            assert 2 * n["DFMA"] + n["DMUL"] + n["DADD"] in (flops, flops - 1), (fn, dipole, n, flops)
            # an FP64 instruction costs 2 or 3 pipe cycles in the model
            assert 2 * fp64 <= cyc - n["other"] <= 3 * fp64
    if corr:
        # at most half of the DFMAs of the headline loop read three fresh registers (round 1: 60 of 86)
        for cyc, n, fresh3 in blocks[:2]:
            assert fresh3 <= 45 and n["DFMA"] == 82


@pytest.mark.parametrize("target,count,accumulators", [("folded", 100, 1 + 1 + 3 + 5 + 7 + 3), ("components", 118, 1 + 1 + 3 + 5 + 7)])
def test_order_search_respects_the_dependencies_of_the_pair_body(target, count, accumulators, monkeypatch):
    from paper_2101_08226_b200 import order_search as osr
    monkeypatch.setattr(osr, "TARGET", target)
    stmts = osr.read_statements()
    assert len(stmts) == count and len(set(stmts)) == count
    dep, succ = osr.analyse(stmts)
    n = len(stmts)
    # the order in the source is a valid one (every statement after what it reads)
    assert all(d < i for i in range(n) for d in dep[i])
    # every accumulator update depends on the previous update of the same accumulator
    acc = {}
    for i, st in enumerate(stmts):
        body = st[len("if (DIPOLE) "):] if st.startswith("if (DIPOLE) ") else st
        if body.startswith("a."):
            name = body.split("=")[0].replace("+", "").strip()
            if name in acc:
                assert acc[name] in dep[i], st
            acc[name] = i
    assert len(acc) == accumulators                     # l0, l0b, l1, l2, l3 (, c): the accumulators of DESIGN.md section 6
    rng = random.Random(5)

    def valid(order):
        pos = {s: k for k, s in enumerate(order)}
        return sorted(order) == list(range(n)) and all(pos[d] < pos[i] for i in range(n) for d in dep[i])

    for loc in (0.0, 0.6, 0.97):
        o = osr.random_order(n, dep, succ, rng, loc)
        assert valid(o)
        for moves in (1, 3, 5):
            o = osr.mutate(o, dep, succ, rng, moves)
            assert valid(o)
    assert osr.objective(None) > osr.objective([300, 300, 0, 270, 270, 0])
