"""higs_sh32_encode_static (include/higs.h): the SH encoder for callers that cannot allocate.  Its work area is a static
device array inside the library, shared by every call.  Checked here against the existing path
(higs_scene_upload + higs_scene_compress_sh + higs_get_sh32) on two calls in a row with different inputs - the second call
finds the first one's counters, prefixes and scales in the array - bit for bit (byte work: the tolerance of
test_sh32_codec_bytes_and_render).  Collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

import higs_scenes as hs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hg():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device: the CUDA path has no fallback")
    import paper_2606_00352_b200 as m
    m.load()
    return m


def _existing_path(hg, scene):
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    ctx = hg.higs_create(0, scene.N, 64, 64)
    hg.higs_scene_upload(ctx, f(scene.means), f(scene.scales), f(scene.quats), f(scene.opacities), f(scene.sh), 3)
    hg.higs_scene_compress_sh(ctx)
    codes, scales = hg.higs_get_sh32(ctx, scene.N)
    hg.higs_destroy(ctx)
    return codes, scales


def test_static_encoder_matches_the_context_path_on_two_calls_in_a_row(hg):
    import torch
    a = hs.scene_cfg1()                                                   # 100,000 gaussians, SH degree 3
    b = hs.scene_cfg1(N=37_123, seed=77)                                  # other size (ragged tail), other values
    b.sh[:] = (b.sh * np.float32(3.7) + np.float32(0.01)).astype(np.float32)          # other percentiles than the first call's
    want = [_existing_path(hg, s) for s in (a, b)]
    d_sh = [torch.from_numpy(np.ascontiguousarray(s.sh, dtype=np.float32)).cuda() for s in (a, b)]
    d_codes = [torch.full((s.N, 32), 0xAB, dtype=torch.uint8, device="cuda") for s in (a, b)]
    d_scales = [torch.full((16, 3), -7.0, dtype=torch.float32, device="cuda") for _ in (a, b)]
    torch.cuda.synchronize()
    for k, s in enumerate((a, b)):                                        # back to back on one stream, nothing in between
        hg.higs_sh32_encode_static(d_sh[k], s.N, d_codes[k], d_scales[k])
    torch.cuda.synchronize()
    for k in range(2):
        codes, scales = want[k]
        got_scales = d_scales[k].cpu().numpy()
        assert np.array_equal(got_scales.view(np.uint32), scales.view(np.uint32)), f"call {k}: scale table"
        got = d_codes[k].cpu().numpy()
        assert np.array_equal(got, codes), f"call {k}: {int((got != codes).any(axis=1).sum())} codes differ"
    # a third call repeating the first input after the second one's state: same bytes again
    d_codes[0].fill_(0)
    hg.higs_sh32_encode_static(d_sh[0], a.N, d_codes[0], d_scales[0])
    torch.cuda.synchronize()
    assert np.array_equal(d_codes[0].cpu().numpy(), want[0][0])


def test_static_encoder_limits_and_empty_input(hg):
    import torch
    d_scales = torch.zeros((16, 3), dtype=torch.float32, device="cuda")
    hg.higs_sh32_encode_static(None, 0, None, d_scales)
    torch.cuda.synchronize()
    assert (d_scales.cpu().numpy() == 1.0).all()
    with pytest.raises(hg.HigsError) as e:
        hg.higs_sh32_encode_static(d_scales, hg.HIGS_SH32_STATIC_MAX_N + 1, d_scales, d_scales)
    assert e.value.status == hg.HIGS_E_CAPACITY and "HIGS_SH32_STATIC_MAX_N" in str(e.value)
    with pytest.raises(hg.HigsError) as e:
        hg.higs_sh32_encode_static(None, 5, None, d_scales)
    assert e.value.status == hg.HIGS_E_ARG
