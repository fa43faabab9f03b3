"""The boundary really is a C ABI: a plain C client (tests/c_abi_client.c: include/octo_fmm.h + the CUDA runtime, no
Python, no torch) runs cfg 1 through the shared library and its output is compared with the oracle."""
import os
import shutil
import subprocess

import numpy as np
import pytest

import fmm_inputs as fi
import oracle
from helpers import parity_error

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plain_c_client(tmp_path):
    import torch
    assert torch.cuda.is_available()
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not on PATH")
    from paper_2101_08226_b200 import build
    build.build()
    libdir = os.path.join(ROOT, "paper_2101_08226_b200")
    exe = str(tmp_path / "c_abi_client")
    subprocess.run(["nvcc", "-O1", "-x", "cu", "-I", os.path.join(ROOT, "include"), os.path.join(ROOT, "tests", "c_abi_client.c"),
                    "-o", exe, "-L", libdir, "-locto_fmm", "-Xlinker", "-rpath", "-Xlinker", libdir], check=True)
    w = fi.config1()
    inp, outp = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(inp, "wb") as f:
        np.array(list(w.n) + list(w.out_lo) + list(w.out_hi) + [1], dtype=np.int32).tofile(f)
        np.array([w.h, w.theta], dtype=np.float64).tofile(f)
        w.moments.astype(np.float64).tofile(f)
        w.com_off.astype(np.float64).tofile(f)
    r = subprocess.run([exe, inp, outp], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    raw = np.fromfile(outp, dtype=np.uint8)
    ocell = 8 * 8 * 8
    vals = raw[:ocell * 23 * 8].view(np.float64)
    count = int(raw[ocell * 23 * 8:ocell * 23 * 8 + 8].view(np.uint64)[0])
    nst = int(raw[ocell * 23 * 8 + 8:ocell * 23 * 8 + 12].view(np.int32)[0])
    L, Lc = vals[:ocell * 20].reshape(20, 8, 8, 8), vals[ocell * 20:].reshape(3, 8, 8, 8)
    Lr, Lcr, cnt = oracle.interact_multipole(w.n, w.h, w.theta, w.moments, w.com_off, w.out_lo, w.out_hi, True)
    assert count == cnt == 118272 and nst == 231
    assert parity_error(L, Lr) < 1e-12 and parity_error(Lc, Lcr) < 1e-11


def test_plain_c_client_of_the_tree_solve(tmp_path):
    """The adaptive-tree calls from plain C (tests/c_abi_tree_client.c): a 4-level tree stored in boxes, pair counts and
    (phi, g) against the oracle."""
    import torch
    assert torch.cuda.is_available()
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not on PATH")
    from paper_2101_08226_b200 import build
    build.build()
    libdir = os.path.join(ROOT, "paper_2101_08226_b200")
    exe = str(tmp_path / "c_abi_tree_client")
    subprocess.run(["nvcc", "-O1", "-x", "cu", "-I", os.path.join(ROOT, "include"), os.path.join(ROOT, "tests", "c_abi_tree_client.c"),
                    "-o", exe, "-L", libdir, "-locto_fmm", "-Xlinker", "-rpath", "-Xlinker", libdir], check=True)
    tree = fi.star_tree(32, 4)
    boxes = fi.tree_boxes(tree)
    kind, mass = fi.crop_tree(tree, boxes)
    inp, outp = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(inp, "wb") as f:
        np.array([tree.n0, tree.depth, 1], dtype=np.int32).tofile(f)
        np.array([tree.h0, 0.5], dtype=np.float64).tofile(f)
        np.array(boxes, dtype=np.int32).tofile(f)
        for k, m in zip(kind, mass):
            k.astype(np.uint8).tofile(f)
            m.astype(np.float64).tofile(f)
    r = subprocess.run([exe, inp, outp], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    raw = np.fromfile(outp, dtype=np.uint8)
    ref, cref = oracle.solve_tree(tree.n0, tree.h0, 0.5, kind, mass, True, box=boxes)
    pos = 0
    gmax = max(np.abs(x[1:]).max() for x in ref)
    for l, b in enumerate(boxes):
        nc = b[3] * b[4] * b[5]
        got = raw[pos:pos + 4 * nc * 8].view(np.float64).reshape(4, b[5], b[4], b[3])
        pos += 4 * nc * 8
        leaf = kind[l] == fi.TREE_LEAF
        if leaf.any():
            assert (np.abs(got[0] - ref[l][0])[leaf] / np.abs(ref[l][0])[leaf]).max() < 1e-12
            assert np.abs(got[1:] - ref[l][1:])[:, leaf].max() / gmax < 1e-12
        assert np.all(got[:, ~leaf] == 0.0)
    counts = raw[pos:pos + 24].view(np.uint64)
    assert [int(c) for c in counts] == [cref["m2l"], cref["p2p"], cref["cross"]]
