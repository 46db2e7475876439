"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/iris_so.h declares, validates arguments before touching the GPU and fails loudly without one."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from iris_inputs import make_workload

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_01338_b200 import build, binding
    build.build()
    return binding.load_library()


def test_header_symbols_are_exported(lib):
    from paper_2607_01338_b200 import DECLARED_SYMBOLS
    text = open(os.path.join(ROOT, "include", "iris_so.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(iris_so_[a-z_]+)\s*\(", text))
    assert declared == set(DECLARED_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), "library does not export %s" % name
    assert lib.iris_so_version() == 100
    assert lib.iris_so_status_string(1) == b"invalid argument"


def test_library_is_sm100a_only(lib):
    from paper_2607_01338_b200 import lib_path
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", lib_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out)


def test_config_struct_layout_matches_header():
    """The ctypes mirror must match the C struct field by field (names and order)."""
    from paper_2607_01338_b200.binding import _Config
    text = open(os.path.join(ROOT, "include", "iris_so.h")).read()
    body = text[text.index("typedef struct {"):text.index("} iris_so_config;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(int32_t|uint64_t|double)\s*", "", decl)
        names += [n.strip().lstrip("*") for n in decl.split(",")]
    assert names == [n for n, _ in _Config._fields_]


def test_create_validates_before_touching_the_device(lib):
    from paper_2607_01338_b200 import IrisSO, IrisSOError
    cfg, _ = make_workload("tiny")
    bad = [cfg.with_(nx=0), cfg.with_(cell_cm=-1.0), cfg.with_(nv=0), cfg.with_(dv_cms=0.0),
           cfg.with_(line_upper=1, line_lower=2), cfg.with_(line_upper=3, line_lower=1),
           cfg.with_(energy_K=cfg.energy_K[::-1].copy()), cfg.with_(weight=np.zeros(5)),
           cfg.with_(out_unit=1, subtract_space=1), cfg.with_(beam_fwhm_px=-1.0), cfg.with_(T_inf=float("nan")),
           cfg.with_(einstein_A=cfg.einstein_A.T.copy()), cfg.with_(noise_gamma_mode=3)]
    for c in bad:
        with pytest.raises(IrisSOError) as e:
            IrisSO(c)
        assert e.value.status == 1, str(e.value)
    with pytest.raises(IrisSOError) as e:
        IrisSO(cfg, transfer_algo=7)
    assert e.value.status == 1
    with pytest.raises(IrisSOError) as e:
        IrisSO(cfg.with_(beam_fwhm_px=40.0))
    assert e.value.status == 2            # unsupported, not invalid


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2607_01338_b200 import IrisSO, IrisSOError
    cfg, _ = make_workload("tiny")
    with pytest.raises(IrisSOError) as e:
        IrisSO(cfg)
    assert e.value.status == 3 and "no CPU fallback" in str(e.value)


def test_product_does_not_import_the_oracle():
    """Neither side may import the other; the product path must not route through oracle/."""
    for d, forbidden in (("paper_2607_01338_b200", ("oracle",)), ("oracle", ("paper_2607_01338_b200",)),
                         ("iris_inputs", ("oracle", "paper_2607_01338_b200"))):
        for dirpath, _, files in os.walk(os.path.join(ROOT, d)):
            for fn in files:
                if not fn.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                    continue
                src = open(os.path.join(dirpath, fn)).read()
                for name in forbidden:
                    assert not re.search(r"^\s*(from|import)\s+%s\b" % name, src, flags=re.M), (fn, name)
                    assert not re.search(r'#include\s+"[^"]*%s' % name, src), (fn, name)
