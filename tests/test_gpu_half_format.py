"""The 16-bit storage format is integer work: the stored words and scales must match a restatement of the formula BIT
FOR BIT (include/mdwf.h, mdwf_half_encode; reading A8 of SURVEY.md 8(c) -- the paper says only
"double-half").  The restatement below is numpy, written from the formula, and shares nothing with csrc/."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def np_encode(x):
    """x: complex array [L5][Vh][4][3] -> (uint16 words [L5][Vh][24], float32 scales [L5][Vh])"""
    v = np.ascontiguousarray(x).view(np.float64 if x.dtype == np.complex128 else np.float32).reshape(x.shape[0], x.shape[1], 24)
    v32 = v.astype(np.float32)                                     # the kernels quantise fp32 values
    m = np.abs(v32).max(axis=2)                                    # one scale per (s, site)
    with np.errstate(divide="ignore"):
        isc = np.where(m > 0, np.float32(32767.0) / m, np.float32(0.0)).astype(np.float32)   # fp32 division
    # one rounding, to nearest even, of the exact product (fp32 x fp32 is exact in fp64)
    q = np.rint(v32.astype(np.float64) * isc.astype(np.float64)[:, :, None]).astype(np.int64)
    return (q + 32768).astype(np.uint16), m


def np_decode(words, scales):
    sc = scales.astype(np.float32) * np.float32(np.float32(1.0) / np.float32(32767.0))        # fp32 product
    q = words.astype(np.int64) - 32768
    return (q.astype(np.float32) * sc[:, :, None]).astype(np.float32)                          # fp32 product


def _vector(L5, Vh, seed, decay):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((L5, Vh, 4, 3)) + 1j * rng.standard_normal((L5, Vh, 4, 3))
    # domain-wall-like profile: slices differ by orders of magnitude, which is what the per-(site, s) scale is for
    x *= np.exp(-decay * np.arange(L5))[:, None, None, None]
    x[1, 3] = 0.0                                                  # an all-zero site: scale 0, words 32768
    x[0, 0, 0, 0] = 1.0 + 0.5j                                     # exact ties and exact max
    x[0, 0, 1, 1] = -x[0, 0].real.max() * 3.0
    return x


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("via_fp64", [False, True])
def test_half_words_and_scales_bit_exact(dtype, via_fp64):
    from paper_1701_07559_b200 import binding
    L, L5 = (4, 4, 2, 6), 12                                       # Vh = 96: three 32-site groups
    Vh = L[0] * L[1] * L[2] * L[3] // 2
    m = binding.Mdwf(L, L5, 1.1, 1.5, 0.5, 0.005)
    x = _vector(L5, Vh, 5, 0.9).astype(dtype)
    words, scales = m.half_encode(torch.from_numpy(x).cuda(), via_fp64=via_fp64)
    w_ref, s_ref = np_encode(x)
    assert np.array_equal(scales.cpu().numpy().view(np.uint32), s_ref.view(np.uint32))
    assert np.array_equal(words.cpu().numpy().view(np.uint16), w_ref)
    m.close()


def test_half_decode_bit_exact_and_roundtrip_bound():
    from paper_1701_07559_b200 import binding
    L, L5 = (4, 4, 2, 6), 8
    Vh = L[0] * L[1] * L[2] * L[3] // 2
    m = binding.Mdwf(L, L5, 1.1, 1.5, 0.5, 0.005)
    x = _vector(L5, Vh, 6, 1.5).astype(np.complex64)
    words, scales = m.half_encode(torch.from_numpy(x).cuda())
    back = m.half_decode(words, scales).cpu().numpy()
    ref = np_decode(words.cpu().numpy().view(np.uint16), scales.cpu().numpy())
    assert np.array_equal(back.view(np.float32).reshape(L5, Vh, 24).view(np.uint32), ref.view(np.uint32))
    # |decode(encode(v)) - v| <= (1/2 + 2^-8) m / 32767 per component (half a step + the fp32 roundings), per (site, s)
    err = np.abs(back.view(np.float32).reshape(L5, Vh, 24) - x.view(np.float32).reshape(L5, Vh, 24))
    bound = (0.5 + 2.0 ** -8) * scales.cpu().numpy()[:, :, None] / 32767.0
    assert (err <= bound).all()
    m.close()
