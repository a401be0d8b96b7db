"""The C-ABI library loads without a GPU and exports every symbol include/sdm.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "sdm.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(sdm_[a-z_0-9]+)\s*\(", txt)))


@pytest.fixture(scope="module")
def lib():
    from paper_1310_1905_b200 import build

    return ctypes.CDLL(build.build())


def test_header_declares_the_boundary_of_survey_8b():
    syms = declared_symbols()
    for s in ("sdm_create", "sdm_destroy", "sdm_step_sync", "sdm_step_async", "sdm_step_async_result", "sdm_diag_sd_conc",
              "sdm_diag_dry_rng", "sdm_diag_wet_rng", "sdm_diag_dry_mom", "sdm_diag_wet_mom", "sdm_outbuf", "sdm_export_state",
              "sdm_init", "sdm_init_from_arrays", "sdm_last_error", "sdm_stats"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_1310_1905_b200 import binding

    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(binding.EXPORTS) == syms   # the Python binding has the same names


def test_create_fails_loudly_without_a_gpu(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1310_1905_b200 import binding

    with pytest.raises(binding.SdmError, match="no CUDA device|not sm_100"):
        binding.Particles(nx=2, nz=2, max_sd=16)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1310_1905_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace("oracle/.", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            assert "paper_1310_1905_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "imports nothing from ``paper_1310_1905_b200``", "").replace("(paper_1310_1905_b200/csrc)", ""), f
