"""CPU checks of the seeded input module's bf16 rounding (the values a bf16 record holds; the GPU twin of this test is
test_rec16_pack_keeps_nan_and_inf in test_rec_gpu.py, which holds the pack kernel to the same bits)."""
import numpy as np

from paper_2606_09794_b200 import workloads as W


def _f(bits):
    return np.array(bits, dtype=np.uint32).view(np.float32)


def test_to_bf16_rounds_to_nearest_even():
    x = _f([0x3F800000, 0x3F808000, 0x3F818000, 0x3F808001, 0x3F807FFF, 0xBF808000, 0x00000001, 0x80000000])
    want = [0x3F800000, 0x3F800000, 0x3F820000, 0x3F810000, 0x3F800000, 0xBF800000, 0x00000000, 0x80000000]
    assert W.to_bf16(x).view(np.uint32).tolist() == want          # ties go to the even bf16; -0 keeps its sign
    import torch
    r = np.random.default_rng(5).standard_normal(10_000).astype(np.float32) * np.float32(1e3)
    assert np.array_equal(W.to_bf16(r), torch.from_numpy(r).to(torch.bfloat16).float().numpy())


def test_to_bf16_keeps_nan_and_inf():
    """Plain add-and-shift rounding turns the NaN 0x7FFFFFFF into 0x8000 (-0.0) and 0xFFFFFFFF into +0.0: a NaN
    quaternion or amplitude would be stored as a finite number and every isfinite check downstream would pass."""
    nans = _f([0x7FFFFFFF, 0xFFFFFFFF, 0x7FC00000, 0x7F800001, 0xFF80FFFF, 0x7FBFFFFF])
    got = W.to_bf16(nans)
    assert np.isnan(got).all()
    assert (got.view(np.uint32) >> 31).tolist() == [0, 1, 0, 0, 1, 0]                     # the sign survives
    assert (got.view(np.uint32) & 0xFFFF).tolist() == [0] * 6                              # a bf16 value
    inf = _f([0x7F800000, 0xFF800000])
    assert W.to_bf16(inf).view(np.uint32).tolist() == [0x7F800000, 0xFF800000]
    big = _f([0x7F7FFFFF, 0xFF7FFFFF, 0x7F7F0000, 0x7F7F7FFF])                           # beyond the largest bf16: rounds to inf
    assert W.to_bf16(big).view(np.uint32).tolist() == [0x7F800000, 0xFF800000, 0x7F7F0000, 0x7F7F0000]
