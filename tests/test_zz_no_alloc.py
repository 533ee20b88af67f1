"""mdwf_blas_norm2_noalloc (include/mdwf.h): the ||x||^2 entry point that allocates nothing (per-block partials in a file-scope
__device__ array of the library) against the existing path mdwf_blas_norm2 (partials in a cudaMalloc'ed buffer of the context).
Collected last on purpose (test_zz_*): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _ctx():
    from paper_1701_07559_b200 import binding
    return binding, binding.Mdwf((4, 4, 4, 4), 8, 1.3, 1.5, 0.5, 0.05)


def test_noalloc_norm2_matches_existing_path_two_calls_in_a_row():
    binding, m = _ctx()
    binding.noalloc_setup()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    g = torch.Generator(device="cuda").manual_seed(11)
    # second call smaller than the first (fewer blocks: stale partials of the first call must not leak into it), third fp32,
    # fourth spans the full grid of 4096 blocks with a ragged tail
    cases = [(torch.float64, 1_000_003), (torch.float64, 4_099), (torch.float32, 777_777), (torch.float64, 4096 * 256 * 4 + 13)]
    for dtype, n in cases:
        x = torch.randn(n, dtype=dtype, device="cuda", generator=g)
        want = m.norm2(x)                                   # existing path (fp64 accumulation, fixed order)
        binding.blas_norm2_noalloc(x, out)
        binding.blas_norm2_noalloc(x, out)                  # twice in a row on the shared scratch
        got = float(out.item())
        ref = float((x.double() ** 2).sum().item())
        assert got == want, (dtype, n, got, want)           # same arithmetic, same order: bit-identical
        assert abs(got - ref) <= 1e-12 * ref, (dtype, n, got, ref)
    # empty input
    binding.blas_norm2_noalloc(torch.empty(0, dtype=torch.float64, device="cuda"), out)
    assert float(out.item()) == 0.0
    m.close()


def test_noalloc_rejects_sizes_beyond_the_maximum():
    from paper_1701_07559_b200 import binding
    L = binding.lib()
    nmax = binding.noalloc_max_n()
    assert nmax == 1 << 30
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    x = torch.ones(16, dtype=torch.float64, device="cuda")
    rc = L.mdwf_blas_norm2_noalloc(x.data_ptr(), nmax + 1, 8, out.data_ptr(), None)      # rejected before anything is touched
    assert rc == binding.MDWF_EARG
    assert b"maximum" in L.mdwf_noalloc_last_error()
    assert L.mdwf_blas_norm2_noalloc(x.data_ptr(), -1, 8, out.data_ptr(), None) == binding.MDWF_EARG
    assert L.mdwf_blas_norm2_noalloc(x.data_ptr(), 16, 2, out.data_ptr(), None) == binding.MDWF_EARG
    assert L.mdwf_blas_norm2_noalloc(x.data_ptr(), 16, 8, None, None) == binding.MDWF_EARG
    torch.cuda.synchronize()
    assert float(out.item()) == 7.0
    assert L.mdwf_blas_norm2_noalloc(x.data_ptr(), 16, 8, out.data_ptr(), None) == 0
    assert float(out.item()) == 16.0


def test_noalloc_on_a_side_stream():
    from paper_1701_07559_b200 import binding
    st = torch.cuda.Stream()
    x = torch.arange(1, 1001, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    binding.blas_norm2_noalloc(x, out, stream=st.cuda_stream)
    st.synchronize()
    assert float(out.item()) == 1000 * 1001 * 2001 / 6
