"""The C ABI library: loads, exports every symbol include/admm_b200.h declares, and fails loudly
(no CPU fallback) when there is no CUDA device.  No compute calls here.  CPU only."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2509_08602_b200 import build
    build.build()                      # nvcc cross-compiles sm_100a without a GPU
    from paper_2509_08602_b200 import binding as b
    return b


def test_library_exports_every_declared_symbol(binding):
    header = open(os.path.join(ROOT, "include", "admm_b200.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(admm_[a-z_0-9]+)\s*\(", header)))
    assert "admm_setup" in declared and "admm_solve_batch" in declared and len(declared) >= 10
    for name in declared:
        assert hasattr(binding._lib, name), f"{name} declared in the header but not exported"
    assert sorted(binding.EXPORTS) == declared
    assert "sm_100a" in binding.admm_version()


def test_option_struct_matches_header(binding):
    o = binding.admm_default_options()
    assert (o.storage, o.kernel_path, o.check_every, o.compaction) == (0, 0, 10, 1)
    assert abs(o.eps_abs - 1e-6) < 1e-12
    import ctypes
    assert ctypes.sizeof(binding.admm_options) == 4 * 3 + 4 + 8 + 4 * 10 + 4 + 4 + 8     # incl. pointer alignment padding (80 bytes)


def test_no_cpu_fallback_and_argument_errors(binding):
    import torch
    from workloads import make_tiny_workload
    w = make_tiny_workload(3, 6, 8, 3)
    if not torch.cuda.is_available():
        with pytest.raises(binding.AdmmError) as e:
            binding.admm_setup(w.phi, w.point_class, w.classes)
        assert e.value.status == binding.ADMM_ECUDA and "no CPU fallback" in str(e.value)
    # argument validation happens before any device work
    with pytest.raises(binding.AdmmError) as e:
        binding.admm_setup(w.phi, w.point_class, w.classes, storage=7)                      # unknown storage mode
    assert e.value.status == binding.ADMM_EINVAL
    with pytest.raises(binding.AdmmError) as e:
        binding.admm_setup(w.phi, w.point_class, w.classes, storage=binding.ADMM_STORAGE_BF16, kernel_path=binding.ADMM_PATH_SIMT)
    assert e.value.status == binding.ADMM_EINVAL
    for kw in (dict(warm_start_ratio=0.5), dict(warm_start_ratio=float("nan")), dict(bot_rows=np.full(w.n, 2, np.uint8))):
        with pytest.raises(binding.AdmmError) as e:                                            # new options: range checks
            binding.admm_setup(w.phi, w.point_class, w.classes, **kw)
        assert e.value.status == binding.ADMM_EINVAL, kw
    for cls in (dict(sense=1, threshold=1.0, hard=3), dict(sense=1, threshold=0.5, hard=2)):   # hard in {0,1,2}; hard = 2 needs threshold 1
        with pytest.raises(binding.AdmmError) as e:
            binding.admm_setup(w.phi, w.point_class, [type("C", (), cls)(), w.classes[1]])
        assert e.value.status == binding.ADMM_EINVAL, cls
    bad = [type("C", (), dict(sense=2, threshold=1.0, hard=0))(), w.classes[1]]
    with pytest.raises(binding.AdmmError) as e:
        binding.admm_setup(w.phi, w.point_class, bad)
    assert e.value.status == binding.ADMM_EINVAL


def test_product_package_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the product package or bench's GPU arm may import it."""
    pkg = os.path.join(ROOT, "paper_2509_08602_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith(".py"):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+paper_2509_08602_b200\b", src, flags=re.M), f
                assert "ctypes" not in src and "libadmm" not in src, f
