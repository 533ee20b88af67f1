"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/*.h declares,
validates arguments, and fails loudly (no fallback) when no CUDA device is present."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1701_07559_b200 import binding as b, build
    build.build()
    return b


def test_every_declared_symbol_is_exported(binding):
    inc = os.path.join(ROOT, "include")
    hdr = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    declared = set(re.findall(r"\b(mdwf_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    lib = binding.lib()
    for name in declared:
        assert hasattr(lib, name)


def test_create_validates_arguments(binding):
    for bad in [(3, 4, 4, 4, 8), (4, 4, 4, 4, 1), (4, 4, 4, 4, 33), (4, 0, 4, 4, 8)]:
        with pytest.raises(binding.MdwfError) as e:
            binding.mdwf_create(*bad, 1.3, 1.5, 0.5, 0.05)
        assert e.value.code == binding.MDWF_EARG
    h = binding.mdwf_create(4, 4, 4, 4, 12, 1.1, 1.5, 0.5, 0.005)
    assert binding.mdwf_flops_per_site(h) == 2880 + 48 * 12
    for k, v in (("ladder", "dsh"), ("reconstruct", "12"), ("apply_precision", "half"), ("reliable_delta", "0.2"),
                 ("matpc", "asym"), ("matpc", "sym"), ("kernels", "auto"), ("kernels", "v5"), ("tile_l2_mb", "64")):
        binding.mdwf_set_option(h, k, v)
    for k, v in (("ladder", "x"), ("reconstruct", "8"), ("matpc", "both"), ("kernels", "v4"), ("nope", "1"), ("reliable_delta", "2")):
        with pytest.raises(binding.MdwfError):
            binding.mdwf_set_option(h, k, v)
    binding.mdwf_destroy(h)


def test_no_silent_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = binding.mdwf_create(4, 4, 4, 4, 8, 1.3, 1.5, 0.5, 0.05)
    U = torch.zeros(4 ** 4 * 4 * 18, dtype=torch.float64)
    with pytest.raises(binding.MdwfError) as e:
        binding.mdwf_load_gauge_host(h, U.data_ptr(), 8)
    assert e.value.code in (binding.MDWF_ECUDA, binding.MDWF_ENOMEM)
    x = torch.zeros(10, dtype=torch.float64)
    with pytest.raises(binding.MdwfError) as e:
        binding.mdwf_apply(h, 0, x.data_ptr(), x.data_ptr() + 8, 8)
    assert e.value.code == binding.MDWF_ENOGAUGE
    binding.mdwf_destroy(h)


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1701_07559_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("oracle and the CUDA path", "").replace("imports oracle/", "") \
                    .replace("by the oracle", "") or f in ("inputs.py", "__init__.py"), f
    for f in ("mdwf_oracle.py", "mdwf_oracle.c", "build.py"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_1701_07559_b200" not in src and "from paper_1701_07559_b200" not in src
