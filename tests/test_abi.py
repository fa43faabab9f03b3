"""C-ABI checks that need no GPU: the shared library loads, exports every symbol the header
declares, sizes workspaces, and rejects bad configurations.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    from paper_2101_08226_b200 import build
    build.build()
    import paper_2101_08226_b200 as p
    return p


def test_every_declared_symbol_is_exported(pkg):
    header = open(os.path.join(ROOT, "include", "octo_fmm.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    names = sorted(set(re.findall(r"\b(octo_fmm_[a-z0-9_]+)\s*\(", header)))
    assert {"octo_fmm_create", "octo_fmm_set_moments", "octo_fmm_interact", "octo_fmm_get_expansions",
            "octo_fmm_destroy"} <= set(names)
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2101_08226_b200", "libocto_fmm.so"))
    for n in names:
        assert hasattr(lib, n), n
        assert hasattr(pkg, n), "binding lacks " + n


def test_config_struct_matches_header(pkg):
    # field order/types of the ctypes mirror follow the header's struct
    header = open(os.path.join(ROOT, "include", "octo_fmm.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} octo_fmm_config;", header, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"\b([a-z_]+)(?:\[3\])?\s*[;,]", body)
    assert fields == [f[0] for f in pkg.octo_fmm_config._fields_]


def test_workspace_sizing_and_validation(pkg):
    ok = pkg.make_config((256, 256, 256), 1.0 / 256, 0.5)
    nbytes = pkg.octo_fmm_workspace_bytes(ok)
    ncell = 256 ** 3
    assert nbytes >= ncell * 8 * (20 + 20 + 3) and nbytes < ncell * 8 * 44   # staged sources: 10 component pairs
    assert pkg.octo_fmm_host_scratch_bytes(ok) >= ncell * 8 * 46
    mono = pkg.make_config((128, 128, 128), 1.0 / 128, 0.5, kind=pkg.MONOPOLE)
    assert pkg.octo_fmm_workspace_bytes(mono) >= (138 ** 3 + 4 * 128 ** 3) * 8
    for bad in (pkg.make_config((0, 256, 256), 1.0 / 256, 0.5),            # empty grid
                pkg.make_config((-8, 8, 8), 1.0 / 8, 0.5),
                pkg.make_config((250, 256, 256), 1.0 / 256, 0.5),          # not a multiple of 8
                pkg.make_config((256, 256, 256), 1.0 / 256, 1.0 / 3.0),    # theta <= theta_min reach (L137)
                pkg.make_config((256, 256, 256), 1.0 / 256, 1.0),
                pkg.make_config((256, 256, 256), 0.0, 0.5),
                pkg.make_config((24, 24, 24), 1.0 / 24, 0.5, out_lo=(8, 8, 8), out_hi=(16, 16, 12)),
                pkg.make_config((24, 24, 24), 1.0 / 24, 0.5, kind=7)):
        assert pkg.octo_fmm_workspace_bytes(bad) == 0
        with pytest.raises(pkg.OctoFmmError) as ei:
            pkg.octo_fmm_create(bad)
        assert ei.value.status == pkg.EINVAL


def test_create_without_workspace_or_device_fails_cleanly(pkg):
    cfg = pkg.make_config((24, 24, 24), 1.0 / 24, 0.5)
    with pytest.raises(pkg.OctoFmmError) as ei:      # NULL workspace
        pkg.octo_fmm_create(cfg)
    assert ei.value.status == pkg.EINVAL
    assert pkg.octo_fmm_flops_per_interaction(pkg.MULTIPOLE, True) == (212, 130)        # executed, counted in the SASS
    assert pkg.octo_fmm_flops_per_interaction_path(pkg.MULTIPOLE, True, False) == (180, 113)
    assert pkg.octo_fmm_flops_per_interaction(pkg.MULTIPOLE, False) == (202, 118)
    assert pkg.octo_fmm_flops_per_interaction(pkg.MONOPOLE, False) == (8, 4)


def test_product_path_does_not_touch_the_oracle():
    """The package must not import, load or reference anything under oracle/ (no CPU fallback)."""
    pkgdir = os.path.join(ROOT, "paper_2101_08226_b200")
    for base, _, files in os.walk(pkgdir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "fmm_oracle" not in text, f


def test_marshalling_refuses_strided_arrays_and_cpu_tensors():
    """_ptr() hands plain addresses to the C ABI: a strided array or tensor would be read as if it were dense."""
    import numpy as np
    import torch
    import paper_2101_08226_b200 as p
    a = np.zeros((4, 6))
    assert p._ptr(a) == a.ctypes.data and p._ptr(None) is None
    with pytest.raises(ValueError):
        p._ptr(a[:, ::2])
    with pytest.raises(ValueError):
        p._ptr(torch.zeros((4, 6))[:, ::2])
    with pytest.raises(ValueError):
        p._check_device_tensor(torch.zeros(8, dtype=torch.float64), "moments", torch.float64, 8, torch.device("cuda", 0))
