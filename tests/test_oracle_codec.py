"""Pins for the oracle's 32-byte SH codec (bit layout and quantiser: DESIGN.md reading Q20).

The codec is an encoding the paper describes in one sentence, so it is pinned by what the description and the
mathematics fix, not by a second copy of itself: the bit layout read back field by field from hand-placed values,
fixed points of the quantiser, its error bound and monotonicity, the YCoCg-R lifting being exactly invertible and
leaving grey coefficients with zero chroma, the scales being the stated order statistics, and the 6x size."""
import numpy as np

import higs_scenes as hs
import oracle


def _fields(code_row):
    """Unpack one 32-byte code by the layout of DESIGN.md Q20 (written here independently of the oracle's packer)."""
    b = [int(x) for x in code_row]
    stream = sum(b[i] << (8 * i) for i in range(12))
    y6 = [(stream >> (6 * k)) & 63 for k in range(16)]
    co4 = [b[12 + k] & 15 for k in range(16)]
    cg4 = [b[12 + k] >> 4 for k in range(16)]
    ext = b[28] | (b[29] << 8) | (b[30] << 16) | (b[31] << 24)
    dc = ((y6[0] << 10) | (ext & 0x3ff), (co4[0] << 11) | ((ext >> 10) & 0x7ff), (cg4[0] << 11) | (ext >> 21))
    return y6, co4, cg4, dc


def test_size_and_layout_fields_read_back():
    """One gaussian whose every (basis, channel) value sits exactly on a known code: Y_k on code 32 + (k - 8) * 3 (k >= 1),
    Co_k on 8 + (k % 7) - 3, Cg_k on 8 - (k % 5) + 2, DC on (40000, 20000, 9000).  Scales 1."""
    scales = np.ones((16, 3), np.float32)
    want_y = [0] + [32 + (k - 8) * 3 for k in range(1, 16)]
    want_co = [0] + [8 + (k % 7) - 3 for k in range(1, 16)]
    want_cg = [0] + [8 - (k % 5) + 2 for k in range(1, 16)]
    dq = lambda c, L: np.sign(c - (L + 1)) * ((c - (L + 1)) / L) ** 2
    sh = np.zeros((1, 16, 3), np.float64)
    for k in range(16):
        if k == 0:
            y, co, cg = dq(40000, 32767), dq(20000, 16383), dq(9000, 16383)
        else:
            y, co, cg = dq(want_y[k], 31), dq(want_co[k], 7), dq(want_cg[k], 7)
        t = y - cg / 2; g = cg + t; b = t - co / 2; r = b + co            # inverse YCoCg-R
        sh[0, k] = (r, g, b)
    codes = oracle.sh32_encode(sh.astype(np.float32), scales)
    assert codes.shape == (1, 32) and codes.dtype == np.uint8             # 192 B -> 32 B
    y6, co4, cg4, dc = _fields(codes[0])
    assert dc == (40000, 20000, 9000)
    assert y6[1:] == want_y[1:] and co4[1:] == want_co[1:] and cg4[1:] == want_cg[1:]
    assert (y6[0], co4[0], cg4[0]) == (40000 >> 10, 20000 >> 11, 9000 >> 11)
    dec = oracle.sh32_decode(codes, scales)
    assert np.abs(dec - sh).max() < 2e-6                                   # code points are fixed points of the round trip


def test_quantiser_error_bound_monotone_and_clamp():
    """Square-root gamma: |decode(encode(v)) - v| <= s (2 sqrt|u| d + d^2), d = 1 / (2 L), for |u| = |v / s| <= 1; decode is
    monotone in v; values beyond the scale clamp to +-s; zero stays zero."""
    rng = np.random.default_rng(0)
    n = 4000
    for ch, L in ((0, 31), (1, 7), (2, 7)):
        s = 0.37
        scales = np.ones((16, 3), np.float32); scales[5, ch] = s
        v = rng.uniform(-1.3 * s, 1.3 * s, n).astype(np.float32)
        v[0] = 0.0
        v = np.sort(v)
        ycc = np.zeros((n, 3), np.float64); ycc[:, ch] = v
        t = ycc[:, 0] - ycc[:, 2] / 2; g = ycc[:, 2] + t; b = t - ycc[:, 1] / 2; r = b + ycc[:, 1]
        sh = np.zeros((n, 16, 3), np.float32); sh[:, 5] = np.stack([r, g, b], axis=1)
        dec = oracle.sh32_decode(oracle.sh32_encode(sh, scales), scales).astype(np.float64)[:, 5]
        co = dec[:, 0] - dec[:, 2]; tt = dec[:, 2] + co / 2; cg = dec[:, 1] - tt; yy = tt + cg / 2
        got = (yy, co, cg)[ch]
        others = [x for i, x in enumerate((yy, co, cg)) if i != ch]
        assert max(np.abs(o).max() for o in others) < 1e-6                 # the other two channels stay zero
        u = np.clip(np.abs(v.astype(np.float64)) / s, 0, 1)
        d = 0.5 / L
        bound = s * (2 * np.sqrt(u) * d + d * d) + 1e-6
        inside = np.abs(v) <= s
        assert (np.abs(got - v)[inside] <= bound[inside]).all()
        assert np.allclose(got[v > s], s, atol=1e-6) and np.allclose(got[v < -s], -s, atol=1e-6)
        assert (np.diff(got) >= -1e-6).all()                          # (fp32 storage of the decoded r, g, b)
        assert abs(got[np.nonzero(v == 0.0)[0][0]]) < 1e-9


def test_grey_coefficients_have_zero_chroma_and_lifting_inverts():
    s = hs.scene_cfg1(N=3000)
    sh = s.sh.copy()
    sh[:, :, 1] = sh[:, :, 0]; sh[:, :, 2] = sh[:, :, 0]                   # r = g = b
    scales = oracle.sh32_scales(sh)
    codes = oracle.sh32_encode(sh, scales)
    for row in codes[:50]:
        y6, co4, cg4, dc = _fields(row)
        assert all(c == 8 for c in co4[1:]) and all(c == 8 for c in cg4[1:]) and dc[1] == 16384 and dc[2] == 16384
    dec = oracle.sh32_decode(codes, scales)
    assert np.array_equal(dec[:, :, 0], dec[:, :, 1]) and np.array_equal(dec[:, :, 0], dec[:, :, 2])


def test_scales_are_the_stated_order_statistics():
    s = hs.scene_cfg1(N=5000)
    sh = s.sh.astype(np.float32)
    r, g, b = sh[..., 0], sh[..., 1], sh[..., 2]
    co = r - b; t = b + np.float32(0.5) * co; cg = g - t; y = t + np.float32(0.5) * cg
    ycc = np.stack([y, co, cg], axis=-1)                                    # [N][16][3], fp32 like the encoder
    scales = oracle.sh32_scales(sh)
    N = sh.shape[0]
    for k in (0, 1, 7, 15):
        for c in range(3):
            col = np.sort(np.abs(ycc[:, k, c]))
            idx = N - 1 if k == 0 else min(N - 1, int(N * 0.999))
            assert scales[k, c] == col[idx]


def test_round_trip_on_a_scene_and_dc_precision():
    s = hs.scene_cfg1(N=20000)
    scales = oracle.sh32_scales(s.sh)
    dec = oracle.sh32_decode(oracle.sh32_encode(s.sh, scales), scales)
    err = np.abs(dec.astype(np.float64) - s.sh)
    assert err[:, 0].max() < 1e-3 * scales[0].max()                        # DC: 15-16 bits
    assert np.median(err[:, 1:]) < 0.02                                    # higher bands: 6 / 4 bits of N(0, 0.1) values
