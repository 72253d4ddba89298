"""The allocation-free slice encoder (fdtd_codec_encode_slices_noalloc: reduction scratch in a static device array of the
library, no cudaMalloc in the call) against the existing path (fdtd_codec_encode, slice by slice, caller-supplied scratch):
bit-exact codes and scales — the tolerance of the codec tests — on two calls in a row that share the static array.

Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2603_24027_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _slices(nslices, slice_len, seed, amp):
    rng = np.random.default_rng(seed)
    x = (amp * rng.standard_normal((nslices, slice_len)) * np.exp(rng.uniform(-8, 2, (nslices, slice_len)))).astype(np.float32)
    x[0, :4] = [0.0, -0.0, 1e-45, -3e-39]
    if nslices > 2:
        x[2] = 0.0                      # an all-zero slice: scale 0, codes 0
    return x


@pytest.mark.parametrize("dtype", [W.F8E4M3_SCALED, W.BF16, W.F16, W.F32, W.F8E4M3B11FNUZ])
def test_noalloc_encoder_matches_existing_path_on_two_calls_in_a_row(dtype):
    import torch
    from paper_2603_24027_b200 import fdtd
    # second call: fewer, shorter slices with much smaller values — a scratch word left over from the first call (a larger
    # absmax) would give it a wrong scale
    for call, (nslices, slice_len, amp) in enumerate([(36, 5003, 30.0), (7, 1300, 1e-3)]):
        x = torch.from_numpy(_slices(nslices, slice_len, 100 + call, amp)).cuda()
        codes = torch.full((nslices, slice_len * fdtd.ELEM_BYTES[dtype]), 0xAB, dtype=torch.uint8, device="cuda")
        scales = torch.full((nslices,), -1.0, dtype=torch.float32, device="cuda")
        fdtd.codec_encode_slices_noalloc(dtype, x, codes, scales)
        torch.cuda.synchronize()
        for sl in range(nslices):
            ref_codes, ref_scale = fdtd.codec_encode(dtype, x[sl])
            assert np.array_equal(codes[sl].cpu().numpy(), ref_codes.cpu().numpy()), (call, sl)
            assert np.float32(scales[sl].item()) == np.float32(ref_scale), (call, sl, scales[sl].item(), ref_scale)
        if dtype == W.F8E4M3_SCALED and nslices > 2:
            assert scales[2].item() == 0.0 and not codes[2].any().item()


def test_noalloc_encoder_rejects_sizes_beyond_its_static_scratch():
    import torch
    from paper_2603_24027_b200 import fdtd
    assert fdtd.NOALLOC_MAX_SLICES == 4096
    x = torch.zeros((fdtd.NOALLOC_MAX_SLICES + 1, 8), dtype=torch.float32, device="cuda")
    with pytest.raises(fdtd.FdtdError) as e:
        fdtd.codec_encode_slices_noalloc(W.F8E4M3_SCALED, x)
    assert e.value.status == 1 and "FDTD_NOALLOC_MAX_SLICES" in str(e.value)
    with pytest.raises(fdtd.FdtdError) as e:
        fdtd.codec_encode_slices_noalloc(W.F8E4M3_MX32, x[:4].contiguous())
    assert e.value.status == 5
    # the maximum itself is accepted
    codes, scales = fdtd.codec_encode_slices_noalloc(W.F8E4M3_SCALED, x[:fdtd.NOALLOC_MAX_SLICES].contiguous())
    torch.cuda.synchronize()
    assert not codes.any().item() and not scales.any().item()
