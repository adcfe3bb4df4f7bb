"""Pins for the oracle's integer lists (O-LIST) and for the three renderers agreeing.

* row scan (N-SCAN) against an independent exact test written here in fp64 numpy: a cell is hit
  iff the minimum of the quadratic form over the (clipped) cell rectangle is <= tau_s (the scan
  threshold: tau with the conditioning margin of DESIGN.md reading Q8);
* conservativeness by brute force: every pixel centre with q <= tau lies in a listed macro-tile; for
  ill-conditioned needles: every pixel the fp32 test accepts lies inside the ellipse of tau_s, which
  the scan covers exactly by the previous pin;
* counts / offsets / sorted segments against numpy (bincount, cumsum, lexsort);
* orc_render == orc_brute (bounding box logic) and == orc_render_batched (Eq. (1)),
  with B_r = 16 forcing many batches per macro-tile.
No GPU, no product code."""
import math

import numpy as np
import pytest

import higs_scenes as hs
import oracle


def _min_q_over_rect(mux, muy, A, B2, C, x0, x1, y0, y1):
    """Exact minimum of q(dx,dy) = A dx^2 + B2 dx dy + C dy^2 over the rectangle, in fp64."""
    if x0 <= mux <= x1 and y0 <= muy <= y1:
        return 0.0
    best = math.inf
    for y in (y0, y1):                       # horizontal edges: minimise over x in [x0, x1]
        dy = y - muy
        dx = min(max(-B2 * dy / (2 * A), x0 - mux), x1 - mux)
        best = min(best, A * dx * dx + B2 * dx * dy + C * dy * dy)
    for x in (x0, x1):                       # vertical edges
        dx = x - mux
        dy = min(max(-B2 * dx / (2 * C), y0 - muy), y1 - muy)
        best = min(best, A * dx * dx + B2 * dx * dy + C * dy * dy)
    return best


def _cells_by_rect_test(geo, W, H, cw, ch):
    mux, muy, a, b, c = (float(v) for v in geo[:5])
    tau = float(geo[8])                      # the scan runs on tau_s
    det = a * c - b * b
    A, B2, C = c / det, -2 * b / det, a / det
    ncx, ncy = (W + cw - 1) // cw, (H + ch - 1) // ch
    hit, near = [], []
    for r in range(ncy):
        for m in range(ncx):
            q = _min_q_over_rect(mux, muy, A, B2, C, m * cw, min((m + 1) * cw, W), r * ch, min((r + 1) * ch, H))
            if q <= tau:
                hit.append(r * ncx + m)
            if abs(q - tau) <= 2e-3 * tau:  # too close to call across fp32 / fp64
                near.append(r * ncx + m)
    return set(hit), set(near)


@pytest.mark.parametrize("W,H,cw,ch", [(640, 480, 64, 32), (100, 70, 64, 32), (129, 129, 8, 8), (640, 480, 8, 8)])
def test_row_scan_equals_min_q_over_rectangle(W, H, cw, ch):
    s = hs.scene_cfg1(N=6000)
    rng = np.random.default_rng(5)
    s.scales[:] = s.scales * np.exp(rng.normal(0.8, 0.8, s.scales.shape)).astype(np.float32)  # some big, skewed ones
    cam = hs.make_camera(W, H, eye=(0.4, 0.2, -1.0), centre=(0.0, 0.0, 5.0))
    pr = oracle.project(s, cam)
    idx = np.nonzero(pr.valid)[0]
    assert idx.size > 1500
    checked = 0
    for i in idx[:: max(1, idx.size // 700)]:
        got = set(oracle.scan(pr.geo[i], W, H, cw, ch).tolist())
        want, near = _cells_by_rect_test(pr.geo[i], W, H, cw, ch)
        assert got - near == want - near, (i, sorted(got ^ want))
        assert len(got) > 0
        checked += 1
    assert checked > 500


def test_row_scan_is_conservative_for_pixel_centres():
    s = hs.scene_cfg0()
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    nmx, _ = oracle.grid_dims(cam.W, cam.H)
    ys, xs = np.mgrid[0:cam.H, 0:cam.W]
    for i in range(0, s.N, 3):
        cells = set(oracle.scan(pr.geo[i], cam.W, cam.H).tolist())
        mux, muy, _, _, _, tau = (np.float32(v) for v in pr.geo[i, :6])
        A, B2, C = (np.float32(v) for v in pr.conic[i])
        dx = (xs.astype(np.float32) + np.float32(0.5)) - mux
        dy = (ys.astype(np.float32) + np.float32(0.5)) - muy
        q = A.astype(np.float64) * dx * dx + B2.astype(np.float64) * dx * dy + C.astype(np.float64) * dy * dy
        inside = q <= float(tau) * (1 + 1e-5)
        need = set(((ys[inside] // 32) * nmx + xs[inside] // 64).tolist())
        assert need <= cells, i


def _fp32_pixel_test(pr, i, xs, ys):
    """The pinned fp32 sequence N-Q on every pixel centre (numpy float32 ops, fma through float64)."""
    A, B2, C = (np.float32(v) for v in pr.conic[i])
    dx = (xs + 0.5).astype(np.float32) - pr.geo[i, 0]
    dy = (ys + 0.5).astype(np.float32) - pr.geo[i, 1]
    u = A * dx
    a0 = u * dx
    b0 = B2 * dx
    t = (np.float64(C) * dy.astype(np.float64) + b0.astype(np.float64)).astype(np.float32)
    q = (t.astype(np.float64) * dy.astype(np.float64) + a0.astype(np.float64)).astype(np.float32)
    return q <= pr.geo[i, 5]


def test_scan_threshold_covers_the_fp32_pixel_test_of_needles():
    """Elongated gaussians: the region the fp32 conic test accepts leaves the ellipse {q_cov <= tau} of the
    covariance by up to ~3 * 2^-24 * cond in tau (cancellation in the cross term).  tau_s
    must cover it with room to spare; without the margin 60-odd of these 500 needles fail."""
    W, H = 960, 540
    s = hs.needle_scene(500, W, H, seed=11, sigma_lo_px=20, sigma_hi_px=600)
    pr = oracle.project(s, s.cameras[0])
    ys, xs = np.mgrid[0:H, 0:W]
    outside_plain, worst = 0, 0.0
    for i in np.nonzero(pr.valid)[0]:
        ins = _fp32_pixel_test(pr, i, xs, ys)
        if not ins.any():
            continue
        a, b, c = (np.float64(pr.geo[i, k]) for k in (2, 3, 4))
        det = a * c - b * b
        dx = (xs[ins] + 0.5) - np.float64(pr.geo[i, 0])
        dy = (ys[ins] + 0.5) - np.float64(pr.geo[i, 1])
        q_cov = ((c * dx * dx - 2 * b * dx * dy + a * dy * dy) / det).max()
        tau, tau_s = float(pr.geo[i, 5]), float(pr.geo[i, 8])
        assert tau_s >= tau
        det32 = np.float32(a * c - np.float64(np.float32(b) * np.float32(b)))     # fma(a, c, -(b*b)) as N-PROJ rounds it
        assert tau_s / tau - 1 == pytest.approx(2.0 ** -20 * a * c / np.float64(det32), rel=1e-3, abs=1e-7)
        outside_plain += q_cov > tau
        if q_cov > tau:
            worst = max(worst, (q_cov / tau - 1) / (tau_s / tau - 1))
        assert q_cov <= tau + 0.5 * (tau_s - tau), i       # at most half of the margin is ever used
    assert outside_plain > 20                               # the hazard is real on this scene
    assert worst < 0.5


def test_render_equals_brute_equals_batched_on_needles():
    """Same three renderers on ill-conditioned needles at 1080p: before the margin one pixel of this frame
    differed between the bounding-box renderer and brute force."""
    s = hs.needle_scene(300, 1920, 1080, seed=6)
    pr = oracle.project(s, s.cameras[0])
    assert pr.n_vis == 300
    brute = oracle.brute(pr)
    assert np.array_equal(oracle.render(pr), brute)
    ls = oracle.bin_lists(pr)
    batched = oracle.render_batched(pr, ls)
    assert np.abs(batched - brute).max() < 1e-4 * float(pr.rgb.max())     # only the termination point is free (Q2)
    assert np.abs(oracle.render_batched(pr, ls, terminate=False) - oracle.brute(pr, terminate=False)).max() < 1e-12


@pytest.mark.parametrize("B_r", [1024, 16])
def test_lists_against_numpy(B_r):
    s = hs.scene_cfg1(N=30_000)
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    ls = oracle.bin_lists(pr, B_r=B_r)
    nmx, nmy = oracle.grid_dims(cam.W, cam.H)
    NM = nmx * nmy
    cell, gid = [], []
    for i in np.nonzero(pr.valid)[0]:
        c = oracle.scan(pr.geo[i], cam.W, cam.H)
        cell.append(c); gid.append(np.full(c.size, i, np.int64))
    cell = np.concatenate(cell); gid = np.concatenate(gid)
    cnt = np.bincount(cell, minlength=NM)
    assert (ls.mt_count == cnt).all()
    assert (ls.mt_offset == np.concatenate([[0], np.cumsum(cnt)])).all()
    assert ls.n_pairs == cell.size == int(ls.mt_count.sum())
    order = np.lexsort((gid, pr.key[gid], cell))           # by cell, then key, then id
    assert (ls.ids == gid[order]).all()
    assert (ls.keys == pr.key[gid[order]]).all()
    nb = -(-cnt // B_r)
    assert (ls.batch_offset == np.concatenate([[0], np.cumsum(nb)])).all()
    assert ls.n_units == int(nb.sum())
    assert (cnt > 1024).any() or B_r == 16                 # at least one multi-batch macro-tile at the paper's B_r


def test_render_equals_brute_equals_batched_cfg0():
    s = hs.scene_cfg0()
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    img = oracle.render(pr)
    brute = oracle.brute(pr)
    assert np.array_equal(img, brute)                      # same arithmetic, bbox only prunes
    ls = oracle.bin_lists(pr)
    full = oracle.render_batched(pr, ls, B_r=1 << 30, terminate=False)
    np.testing.assert_allclose(full, oracle.render(pr, terminate=False), atol=1e-12)
    for B_r in (1024, 16, 1):
        split = oracle.render_batched(pr, oracle.bin_lists(pr, B_r=B_r), B_r=B_r, terminate=False)
        np.testing.assert_allclose(split, full, atol=1e-12)            # Eq. (1) is associative
        split_t = oracle.render_batched(pr, oracle.bin_lists(pr, B_r=B_r), B_r=B_r, terminate=True)
        assert np.abs(split_t - img).max() < 1e-4 * float(pr.rgb.max())  # termination point is free (Q2)


def test_render_equals_brute_on_a_window_of_cfg1():
    s = hs.scene_cfg1(N=20_000)
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    win = (300, 200, 340, 232)
    assert np.array_equal(oracle.render(pr, window=win), oracle.brute(pr, window=win))
    full = oracle.render(pr)
    assert np.array_equal(full[200:232, 300:340], oracle.render(pr, window=win))
    assert np.array_equal(oracle.render(pr, threads=1), oracle.render(pr, threads=3))


def test_odd_sizes_empty_and_all_culled():
    s = hs.scene_cfg0(N=300, W=100, H=70)
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    ls = oracle.bin_lists(pr)
    assert ls.mt_count.size == 2 * 3
    np.testing.assert_allclose(oracle.render_batched(pr, ls, terminate=False), oracle.render(pr, terminate=False), atol=1e-12)
    s.means[:, 2] = -1.0                                    # everything behind the camera
    pr = oracle.project(s, cam)
    assert pr.n_vis == 0
    ls = oracle.bin_lists(pr)
    assert ls.n_pairs == 0 and ls.n_units == 0
    assert not oracle.render(pr).any()


def test_lists_and_batched_render_with_16x16_tiles():
    """The 16x16-tile variant (Table 2): macro-tiles of 8x4 tiles = 128x64 px.  Counts and sorted
    segments against numpy on the scan at 128x64 cells, and the batched renderer on those lists equals O-IMG."""
    s = hs.scene_cfg1(N=4000, W=320, H=240)
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    ls = oracle.bin_lists(pr, B_r=64, tile=16)
    nmx, nmy = (cam.W + 127) // 128, (cam.H + 63) // 64
    assert ls.mt_count.size == nmx * nmy
    cells = [oracle.scan(pr.geo[i], cam.W, cam.H, 128, 64) for i in np.nonzero(pr.valid)[0]]
    flat = np.concatenate(cells)
    assert np.array_equal(ls.mt_count, np.bincount(flat, minlength=nmx * nmy).astype(np.uint32))
    assert np.array_equal(ls.batch_offset[1:], np.cumsum((ls.mt_count + 63) // 64))
    owner = np.concatenate([np.full(len(c), i, np.uint32) for c, i in zip(cells, np.nonzero(pr.valid)[0])])
    for m in (0, nmx * nmy // 2, nmx * nmy - 1):
        ids = owner[flat == m]
        order = np.lexsort((ids, pr.key[ids]))
        a, b = int(ls.mt_offset[m]), int(ls.mt_offset[m + 1])
        assert np.array_equal(ls.ids[a:b], ids[order])
    img = oracle.render(pr)
    assert np.abs(oracle.render_batched(pr, ls, B_r=64, tile=16) - img).max() <= 1e-6


@pytest.mark.parametrize("mt", [(4, 8), (16, 2)])
def test_lists_and_batched_render_with_other_macro_tile_shapes(mt):
    """Macro-tile shape sweep: 32 render tiles grouped 4 x 8 or 16 x 2 instead of the paper's 8 x 4
    (PAPER.md:73).  Counts and sorted segments against numpy on the scan at cells of that extent; the image cannot depend on
    the grouping: the batched renderer on those lists equals O-IMG."""
    s = hs.scene_cfg1(N=4000, W=320, H=240)
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    ls = oracle.bin_lists(pr, B_r=64, mt=mt)
    mw, mh = 8 * mt[0], 8 * mt[1]
    nmx, nmy = (cam.W + mw - 1) // mw, (cam.H + mh - 1) // mh
    assert ls.mt_count.size == nmx * nmy
    vis = np.nonzero(pr.valid)[0]
    cells = [oracle.scan(pr.geo[i], cam.W, cam.H, mw, mh) for i in vis]
    flat = np.concatenate(cells)
    assert np.array_equal(ls.mt_count, np.bincount(flat, minlength=nmx * nmy).astype(np.uint32))
    owner = np.concatenate([np.full(len(c), i, np.uint32) for c, i in zip(cells, vis)])
    for m in (0, nmx * nmy // 2, nmx * nmy - 1):
        ids = owner[flat == m]
        order = np.lexsort((ids, pr.key[ids]))
        a, b = int(ls.mt_offset[m]), int(ls.mt_offset[m + 1])
        assert np.array_equal(ls.ids[a:b], ids[order])
    assert np.abs(oracle.render_batched(pr, ls, B_r=64, mt=mt) - oracle.render(pr)).max() <= 1e-6
