"""Pins for the CPU oracle (``oracle/``): closed forms, invariants, library special cases and
brute force, chosen so that a plausible mistake anywhere in the oracle (dropped term, wrong sign
or index, transposed operand) fails at least one of them.  No GPU, no product code.

Every expected value is either a closed form re-derived here in numpy from the definition the
fixture cites, or produced by a library routine (numpy sort, scipy spherical harmonics)."""
import math

import numpy as np
import pytest

import higs_scenes as hs
import oracle
from conftest import load_golden

W129 = 129
CX = 64  # pixel whose centre is the principal point of the 129x129 camera


def _one(mean=(0, 0, 3), scale=0.05, quat=(1, 0, 0, 0), o=0.8, rgb=(0.9, 0.5, 0.1)):
    s = hs.single_gaussian(mean, scale, quat, o, rgb, W129, W129)
    return s, s.cameras[0]


# ------------------------------------------------------------------ fixtures are self-consistent
def test_golden_single_isotropic_is_the_closed_form():
    g = load_golden("single_isotropic.txt")
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    assert g["fx"] == pytest.approx(fx, rel=1e-12)
    s2 = (fx * 0.05 / 3) ** 2 + 0.3
    tau = 2 * math.log(255 * 0.8)
    assert g["sigma2"] == pytest.approx(s2, rel=1e-12)
    assert g["tau"] == pytest.approx(tau, rel=1e-12)
    assert g["radius2"] == pytest.approx(tau * s2, rel=1e-12)
    d = np.arange(-12, 13)
    r2 = d[:, None] ** 2 + d[None, :] ** 2
    inside = r2 <= tau * s2
    assert int(inside.sum()) == g["covered_pixels"]
    assert float((0.8 * np.exp(-r2 / (2 * s2)))[inside].sum()) == pytest.approx(g["sum_alpha"], rel=1e-12)
    for (dx, dy) in [(1, 0), (2, 0), (3, 3), (6, 2)]:
        assert 0.8 * math.exp(-(dx * dx + dy * dy) / (2 * s2)) == pytest.approx(g[f"alpha_{dx}_{dy}"], rel=1e-12)
    assert (5 * 5 + 4 * 4 <= tau * s2) == bool(g["inside_5_4"])


def test_golden_ewa_is_the_closed_form():
    g = load_golden("ewa_offaxis.txt")
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    sx, sy, sz, x, z = 0.05, 0.03, 0.2, 1.0, 3.0
    assert g["a"] == pytest.approx(fx * fx * (sx * sx / z ** 2 + sz * sz * x * x / z ** 4) + 0.3, rel=1e-12)
    assert g["c"] == pytest.approx((fx * sy / z) ** 2 + 0.3, rel=1e-12)
    assert g["mux"] == pytest.approx(fx * x / z + 64.5, rel=1e-12)


def test_golden_ewa_clamp_active_is_the_closed_form():
    g = load_golden("ewa_clamp_active.txt")
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    sx, sy, sz, z = 0.05, 0.03, 0.6, 3.0
    lim = 0.65 * 129 / fx
    assert g["lim"] == pytest.approx(lim, rel=1e-12) and 0.9 > lim
    assert g["A_a"] == pytest.approx(fx * fx * (sx * sx + lim * lim * sz * sz) / z ** 2 + 0.3, rel=1e-12)
    assert g["A_c"] == pytest.approx((fx * sy / z) ** 2 + 0.3, rel=1e-12)
    assert g["A_mux"] == pytest.approx(fx * 0.9 + 64.5, rel=1e-12)
    assert g["A_a_if_unclamped"] == pytest.approx(fx * fx * (sx * sx + 0.81 * sz * sz) / z ** 2 + 0.3, rel=1e-12)
    assert g["B_a"] == pytest.approx((fx * sx / z) ** 2 + 0.3, rel=1e-12)
    assert g["B_c"] == pytest.approx(fx * fx * (sy * sy + lim * lim * sz * sz) / z ** 2 + 0.3, rel=1e-12)
    assert g["B_muy"] == pytest.approx(-fx * 0.9 + 64.5, rel=1e-12)
    assert g["C_b"] == pytest.approx(-(fx * lim / z) ** 2 * sz * sz, rel=1e-12)
    assert g["C_a"] == g["A_a"] and g["C_c"] == g["B_c"]


def test_golden_grid_counts():
    g = load_golden("grid.txt")
    assert oracle.MT_W == g["mt_w"] and oracle.MT_H == g["mt_h"] and oracle.B_R == g["batch_cap"]
    assert (oracle.MT_W // oracle.TILE) * (oracle.MT_H // oracle.TILE) == g["tiles_per_macro_tile"]
    nx, ny = oracle.grid_dims(1920, 1080)
    assert nx * ny == g["n_mt_1080p"]
    nx, ny = oracle.grid_dims(3840, 2160)
    assert nx * ny == g["n_mt_4k"]


# ------------------------------------------------------------------ one isotropic gaussian
def test_single_isotropic_gaussian_image():
    g = load_golden("single_isotropic.txt")
    s, cam = _one()
    pr = oracle.project(s, cam)
    assert pr.n_vis == 1
    assert pr.geo[0, 2] == pytest.approx(g["sigma2"], rel=2e-6)      # a
    assert pr.geo[0, 4] == pytest.approx(g["sigma2"], rel=2e-6)      # c
    assert abs(pr.geo[0, 3]) < 1e-6                                   # b
    assert pr.geo[0, 5] == pytest.approx(g["tau"], abs=2e-6)
    assert pr.geo[0, 0] == pytest.approx(64.5, abs=1e-5) and pr.geo[0, 1] == pytest.approx(64.5, abs=1e-5)
    img, T, ncomp = oracle.render(pr, want_T=True)
    assert ncomp == g["covered_pixels"]
    assert int((T < 1.0).sum()) == g["covered_pixels"]
    np.testing.assert_allclose(img[CX, CX], [g["centre_r"], g["centre_g"], g["centre_b"]], atol=1e-6)
    assert T[CX, CX] == pytest.approx(g["centre_T"], abs=1e-6)
    alpha = 1.0 - T                                       # one gaussian: alpha = 1 - T
    assert float(alpha.sum()) == pytest.approx(g["sum_alpha"], rel=1e-5)
    for (dx, dy) in [(1, 0), (2, 0), (3, 3), (6, 2)]:
        for sx, sy in [(1, 1), (-1, 1), (1, -1), (-1, -1)]:
            assert alpha[CX + sy * dy, CX + sx * dx] == pytest.approx(g[f"alpha_{dx}_{dy}"], rel=2e-5)
            assert alpha[CX + sy * dx, CX + sx * dy] == pytest.approx(g[f"alpha_{dx}_{dy}"], rel=2e-5)
    assert alpha[CX + 4, CX + 5] == 0.0 and alpha[CX + 5, CX + 4] == 0.0
    # colour is alpha * rgb everywhere
    np.testing.assert_allclose(img, alpha[..., None] * np.array([0.9, 0.5, 0.1]), atol=1e-6)
    ls = oracle.bin_lists(pr)
    assert ls.n_pairs == g["macro_tile_pairs"]
    nmx, _ = oracle.grid_dims(W129, W129)
    assert sorted(np.nonzero(ls.mt_count)[0].tolist()) == sorted([1 * nmx + 0, 1 * nmx + 1, 2 * nmx + 0, 2 * nmx + 1])


# ------------------------------------------------------------------ compositing by hand
def test_two_gaussian_compositing_and_order():
    g = load_golden("compositing.txt")
    s = hs.stack_gaussians([(0, 0, 3), (0, 0, 4)], [0.05, 0.05], [(1, 0, 0, 0)] * 2, [0.6, 0.5],
                           [(1, 0, 0), (0, 1, 0)], W129, W129)
    pr = oracle.project(s, s.cameras[0])
    img, T, _ = oracle.render(pr, want_T=True)
    np.testing.assert_allclose(img[CX, CX], [g["two_r"], g["two_g"], g["two_b"]], atol=1e-6)
    assert T[CX, CX] == pytest.approx(g["two_T"], abs=1e-6)
    # swap depths: id order must not matter, depth order must
    s2 = hs.stack_gaussians([(0, 0, 4), (0, 0, 3)], [0.05, 0.05], [(1, 0, 0, 0)] * 2, [0.6, 0.5],
                            [(1, 0, 0), (0, 1, 0)], W129, W129)
    img2 = oracle.render(oracle.project(s2, s2.cameras[0]))
    np.testing.assert_allclose(img2[CX, CX], [g["swap_r"], g["swap_g"], g["swap_b"]], atol=1e-6)


def test_equal_depth_ties_break_by_id():
    # same depth -> lower id is in front (reading Q7)
    s = hs.stack_gaussians([(0, 0, 3), (0, 0, 3)], [0.05, 0.05], [(1, 0, 0, 0)] * 2, [0.6, 0.5],
                           [(1, 0, 0), (0, 1, 0)], W129, W129)
    pr = oracle.project(s, s.cameras[0])
    assert pr.key[0] == pr.key[1]
    np.testing.assert_allclose(oracle.render(pr)[CX, CX], [0.6, 0.2, 0.0], atol=1e-6)
    ls = oracle.bin_lists(pr)
    m = np.nonzero(ls.mt_count)[0][0]
    seg = ls.ids[ls.mt_offset[m]:ls.mt_offset[m + 1]]
    assert seg.tolist() == [0, 1]


def test_alpha_clamp():
    g = load_golden("compositing.txt")
    s, cam = _one(o=0.999, rgb=(1, 1, 1))
    img, T, _ = oracle.render(oracle.project(s, cam), want_T=True)
    assert T[CX, CX] == pytest.approx(g["clamp_T"], abs=1e-9)
    # colour 1.0 goes through an fp32 SH DC coefficient, (1 - 0.5)/C0 rounded: 1.5e-8 off
    assert img[CX, CX, 0] == pytest.approx(g["clamp_alpha"], abs=1e-7)


@pytest.mark.parametrize("o,n_key,c_key,t_key", [(0.5, "half_composites", "half_C", "half_T"),
                                                  (0.999, "clamp_stack_composites", "clamp_stack_C", "clamp_stack_T")])
def test_termination_counts(o, n_key, c_key, t_key):
    g = load_golden("compositing.txt")
    n = 40
    s = hs.stack_gaussians([(0, 0, 3 + 0.01 * k) for k in range(n)], [0.05] * n, [(1, 0, 0, 0)] * n, [o] * n,
                           [(1, 1, 1)] * n, W129, W129)
    pr = oracle.project(s, s.cameras[0])
    win = (CX, CX, CX + 1, CX + 1)
    img, T, ncomp = oracle.render(pr, window=win, want_T=True)
    assert ncomp == g[n_key]
    assert img[0, 0, 0] == pytest.approx(g[c_key], abs=1e-7)     # rgb = 1 passes through an fp32 SH coefficient
    assert T[0, 0] == pytest.approx(g[t_key], rel=1e-9)
    # termination is only an optimisation: switching it off moves the pixel by < eps * max(rgb)
    img_nt, T_nt, ncomp_nt = oracle.render(pr, window=win, terminate=False, want_T=True)
    assert ncomp_nt == n
    assert 0 <= img_nt[0, 0, 0] - img[0, 0, 0] < 1e-4


def test_transmittance_monotone_and_bounded():
    s = hs.scene_cfg0()
    cam = s.cameras[0]
    pr = oracle.project(s, cam)
    img, T, _ = oracle.render(pr, terminate=False, want_T=True)
    assert (T >= 0).all() and (T <= 1).all()
    assert (img >= 0).all()
    assert (img <= pr.rgb.max() * (1 - T)[..., None] + 1e-12).all()
    # T is non-increasing as gaussians are appended in depth order
    order = np.lexsort((np.arange(pr.N), pr.key))
    prev = np.ones_like(T)
    for frac in (0.1, 0.3, 0.6, 1.0):
        keep = np.zeros(pr.N, np.uint8)
        keep[order[: int(frac * pr.N)]] = 1
        sub = oracle.Projected(pr.N, pr.W, pr.H, int(keep.sum()), (pr.valid & keep).astype(np.uint8), pr.reason,
                               pr.key, pr.geo, pr.conic, pr.rgb, pr.opac)
        _, Tk, _ = oracle.render(sub, terminate=False, want_T=True)
        assert (Tk <= prev + 1e-15).all()
        prev = Tk


# ------------------------------------------------------------------ EWA projection
def test_ewa_on_axis_axis_aligned():
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    s, cam = _one(mean=(0, 0, 2.5), scale=(0.04, 0.09, 0.5))
    pr = oracle.project(s, cam)
    assert pr.geo[0, 2] == pytest.approx((fx * 0.04 / 2.5) ** 2 + 0.3, rel=3e-6)
    assert pr.geo[0, 4] == pytest.approx((fx * 0.09 / 2.5) ** 2 + 0.3, rel=3e-6)
    assert abs(pr.geo[0, 3]) < 1e-6
    # conic is the inverse of the covariance
    a, b, c = (float(v) for v in pr.geo[0, 2:5])
    A, B2, Cc = (float(v) for v in pr.conic[0])
    det = a * c - b * b
    assert A == pytest.approx(c / det, rel=3e-6) and Cc == pytest.approx(a / det, rel=3e-6)
    assert B2 == pytest.approx(-2 * b / det, abs=1e-7)


def test_ewa_off_axis_golden():
    g = load_golden("ewa_offaxis.txt")
    s, cam = _one(mean=(1, 0, 3), scale=(0.05, 0.03, 0.2))
    pr = oracle.project(s, cam)
    assert pr.geo[0, 0] == pytest.approx(g["mux"], rel=1e-6)
    assert pr.geo[0, 1] == pytest.approx(g["muy"], rel=1e-6)
    assert pr.geo[0, 2] == pytest.approx(g["a"], rel=3e-6)
    assert pr.geo[0, 3] == pytest.approx(g["b"], abs=1e-6)
    assert pr.geo[0, 4] == pytest.approx(g["c"], rel=3e-6)
    d = oracle.project_f64((1, 0, 3), (0.05, 0.03, 0.2), (1, 0, 0, 0), 0.8, cam)
    # the fp64 definition still sees the fp32-rounded inputs (0.05f, 0.2f, ...): 3e-8 relative
    assert d["a"] == pytest.approx(g["a"], rel=2e-7) and d["c"] == pytest.approx(g["c"], rel=2e-7)


def test_ewa_frustum_clamp_active_golden():
    """The Jacobian clamp (reading Q11) with the clamp ACTIVE, against the hand-worked closed form - not against the
    oracle's own fp64 twin: a wrong limit, a clamp that also moves the centre, a clamp on the wrong axis or with
    the wrong sign each fail here."""
    g = load_golden("ewa_clamp_active.txt")
    sc = (0.05, 0.03, 0.6)
    for name, mean in (("A", (2.7, 0.0, 3.0)), ("B", (0.0, -2.7, 3.0)), ("C", (2.7, -2.7, 3.0))):
        s, cam = _one(mean=mean, scale=sc)
        pr = oracle.project(s, cam)
        assert pr.n_vis == 1, name                        # centre 36 px outside, ellipse (55 px) still reaches the image
        assert pr.geo[0, 2] == pytest.approx(g[name + "_a"], rel=3e-6), name
        assert pr.geo[0, 4] == pytest.approx(g[name + "_c"], rel=3e-6), name
        if g[name + "_b"] == 0.0:
            assert abs(pr.geo[0, 3]) < 1e-4, name
        else:
            assert pr.geo[0, 3] == pytest.approx(g[name + "_b"], rel=3e-6), name
        if name + "_mux" in g:                            # the centre itself is never clamped
            assert pr.geo[0, 0] == pytest.approx(g[name + "_mux"], rel=1e-6), name
            assert pr.geo[0, 1] == pytest.approx(g[name + "_muy"], rel=1e-6), name
    s, cam = _one(mean=(2.7, 0.0, 3.0), scale=sc)
    assert abs(float(oracle.project(s, cam).geo[0, 2]) - g["A_a_if_unclamped"]) > 100.0
    # just inside the limit the clamp is inactive and the plain closed form holds
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    x = 0.74 * 3.0
    s, cam = _one(mean=(x, 0.0, 3.0), scale=sc)
    assert oracle.project(s, cam).geo[0, 2] == pytest.approx(fx * fx * (0.05 ** 2 + (0.74 * 0.6) ** 2) / 9.0 + 0.3, rel=3e-6)


def test_ewa_monte_carlo_small_scale_limit():
    """Sample the 3D gaussian, project the samples exactly, compare the sample covariance of the
    pixel positions with the EWA covariance (minus the 0.3 dilation); exact as scale -> 0."""
    rng = np.random.default_rng(7)
    cam = hs.make_camera(640, 480, eye=(0.3, -0.2, -4.0), centre=(0.1, 0.0, 0.0))
    mean = np.array([0.4, -0.3, 0.5]); scale = np.array([2e-3, 5e-3, 1e-3]); quat = np.array([0.3, -0.5, 0.2, 0.7])
    d = oracle.project_f64(mean, scale, quat, 0.5, cam)
    q = quat / np.linalg.norm(quat); w, x, y, z = q
    R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                  [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                  [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
    pts = mean + (rng.normal(size=(400_000, 3)) * scale) @ R.T
    V = cam.view.reshape(3, 4).astype(np.float64)
    pc = pts @ V[:, :3].T + V[:, 3]
    u = cam.fx * pc[:, 0] / pc[:, 2] + cam.cx
    v = cam.fy * pc[:, 1] / pc[:, 2] + cam.cy
    cov = np.cov(np.stack([u, v]))
    assert d["a"] - 0.3 == pytest.approx(cov[0, 0], rel=0.01)
    assert d["c"] - 0.3 == pytest.approx(cov[1, 1], rel=0.01)
    assert d["b"] == pytest.approx(cov[0, 1], rel=0.02)
    assert d["mux"] == pytest.approx(u.mean(), abs=5e-3) and d["muy"] == pytest.approx(v.mean(), abs=5e-3)


def test_fp32_pinned_projection_agrees_with_fp64_definition():
    s = hs.scene_cfg1(N=20_000)
    cam = hs.make_camera(640, 480, eye=(1.0, 0.5, -2.0), centre=(0.0, 0.0, 5.0))
    pr = oracle.project(s, cam)
    idx = np.nonzero(pr.valid)[0][:: 37]
    assert idx.size > 200
    for i in idx:
        d = oracle.project_f64(s.means[i], s.scales[i], s.quats[i], s.opacities[i], cam)
        mux, muy, a, b, c, tau = (float(v) for v in pr.geo[i, :6])
        assert mux == pytest.approx(d["mux"], abs=2e-3) and muy == pytest.approx(d["muy"], abs=2e-3)
        assert a == pytest.approx(d["a"], rel=2e-4, abs=1e-5)
        assert c == pytest.approx(d["c"], rel=2e-4, abs=1e-5)
        assert b == pytest.approx(d["b"], rel=2e-4, abs=2e-4 * math.sqrt(d["a"] * d["c"]))
        assert tau == pytest.approx(d["tau"], abs=2e-6)
        A, B2, Cc = (float(v) for v in pr.conic[i])
        sc = max(abs(d["A"]), abs(d["C"]))
        assert A == pytest.approx(d["A"], rel=1e-3, abs=1e-3 * sc)
        assert Cc == pytest.approx(d["C"], rel=1e-3, abs=1e-3 * sc)
        assert B2 == pytest.approx(d["B2"], rel=1e-3, abs=1e-3 * sc)
        assert pr.key[i] == np.float32(d["zc"]).view(np.uint32) or abs(
            float(np.array(pr.key[i], np.uint32).view(np.float32)) - d["zc"]) < 1e-5


def test_quaternion_rotates_footprint_and_normalisation():
    fx = float(np.float32(64.5 / math.tan(math.radians(30.0))))
    th = math.radians(35.0)
    sx, sy, z = 0.08, 0.02, 3.0
    for mult in (1.0, 3.7):
        quat = tuple(mult * v for v in (math.cos(th / 2), 0.0, 0.0, math.sin(th / 2)))   # rotation about z
        s, cam = _one(mean=(0, 0, z), scale=(sx, sy, 0.01), quat=quat)
        pr = oracle.project(s, cam)
        l1, l2 = (fx * sx / z) ** 2, (fx * sy / z) ** 2
        c_, s_ = math.cos(th), math.sin(th)
        assert pr.geo[0, 2] == pytest.approx(c_ * c_ * l1 + s_ * s_ * l2 + 0.3, rel=5e-6)
        assert pr.geo[0, 4] == pytest.approx(s_ * s_ * l1 + c_ * c_ * l2 + 0.3, rel=5e-6)
        assert pr.geo[0, 3] == pytest.approx(c_ * s_ * (l1 - l2), rel=5e-6)


def test_depth_key_is_float_bits_and_orders_like_depth():
    s = hs.scene_cfg0()
    pr = oracle.project(s, s.cameras[0])                  # identity pose: z_cam = mean z exactly
    assert (pr.key == s.means[:, 2].view(np.uint32)).all()
    # positive floats sort correctly under unsigned integer comparison
    z = np.abs(np.random.default_rng(0).normal(size=10000)).astype(np.float32) + np.float32(0.2)
    assert (np.argsort(z, kind="stable") == np.argsort(z.view(np.uint32), kind="stable")).all()


def test_culls():
    cam = hs.make_camera(W129, W129)
    s = hs.stack_gaussians(
        [(0, 0, 0.1), (0, 0, -1), (0, 0, 3), (0, 0, 3), (50, 0, 3), (0, 0, 3)],
        [0.05] * 6, [(1, 0, 0, 0)] * 4 + [(1, 0, 0, 0), (0, 0, 0, 0)],
        [0.8, 0.8, 1.0 / 255.0, 0.8, 0.8, 0.8], [(1, 1, 1)] * 6, W129, W129)
    pr = oracle.project(s, cam)
    assert pr.valid.tolist() == [0, 0, 0, 1, 0, 0]
    assert pr.reason.tolist() == [1, 1, 4, 0, 5, 2]


# ------------------------------------------------------------------ ln_spec, q
def test_ln_spec_accuracy():
    xs = np.concatenate([np.linspace(1.0001, 255.0, 20001), 255.0 * np.logspace(-2.4, 0, 3000)])
    err = max(abs(oracle.ln_spec(float(np.float32(x))) - math.log(float(np.float32(x)))) for x in xs)
    assert err < 6e-7
    assert 2 * oracle.ln_spec(float(np.float32(255 * np.float32(0.8)))) == pytest.approx(2 * math.log(204.0), abs=2e-6)


def test_pixel_q_is_the_quadratic_form():
    rng = np.random.default_rng(3)
    for _ in range(2000):
        mux, muy = rng.uniform(0, 2000, 2)
        a, c = rng.uniform(0.3, 50, 2); b = rng.uniform(-0.95, 0.95) * math.sqrt(a * c)
        det = a * c - b * b
        A, B2, Cc = np.float32(c / det), np.float32(-2 * b / det), np.float32(a / det)
        px, py = np.float32(int(mux) + rng.integers(-8, 9) + 0.5), np.float32(int(muy) + rng.integers(-8, 9) + 0.5)
        q = oracle.pixel_q(px, py, np.float32(mux), np.float32(muy), A, B2, Cc)
        dx, dy = float(px) - float(np.float32(mux)), float(py) - float(np.float32(muy))
        ref = float(A) * dx * dx + float(B2) * dx * dy + float(Cc) * dy * dy
        mag = float(A) * dx * dx + abs(float(B2) * dx * dy) + float(Cc) * dy * dy
        assert q == pytest.approx(ref, abs=4e-7 * mag + 1e-12)


# ------------------------------------------------------------------ spherical harmonics
def _real_sh_scipy(l, m, d):
    from scipy.special import sph_harm_y
    theta = math.acos(max(-1.0, min(1.0, d[2])))
    phi = math.atan2(d[1], d[0])
    if m == 0:
        return float(sph_harm_y(l, 0, theta, phi).real)
    y = sph_harm_y(l, abs(m), theta, phi)       # includes the Condon-Shortley phase
    return math.sqrt(2.0) * float(y.real if m > 0 else y.imag)


def test_sh_basis_matches_library_real_harmonics():
    rng = np.random.default_rng(11)
    for _ in range(200):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        Y = oracle.sh_basis(d)
        k = 0
        for l in range(4):
            for m in range(-l, l + 1):
                assert Y[k] == pytest.approx(_real_sh_scipy(l, m, d), abs=1e-12), (l, m)
                k += 1


def test_sh_basis_orthonormal_by_quadrature():
    xs, ws = np.polynomial.legendre.leggauss(16)
    nphi = 32
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = math.sqrt(1 - ct * ct)
        for j in range(nphi):
            ph = 2 * math.pi * (j + 0.5) / nphi
            Y = oracle.sh_basis([st * math.cos(ph), st * math.sin(ph), ct])
            G += w * (2 * math.pi / nphi) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), atol=1e-12)


def test_sh_degree0_colour_is_direction_independent():
    for mean in [(0, 0, 3), (1, -0.5, 2.5), (-0.7, 0.6, 4)]:
        s = hs.single_gaussian(mean, 0.05, (1, 0, 0, 0), 0.8, (0.2, 0.6, 0.9), 640, 480)
        pr = oracle.project(s, s.cameras[0])
        np.testing.assert_allclose(pr.rgb[0], 0.5 + 0.28209479177387814 * s.sh[0, 0].astype(np.float64), atol=1e-12)
        np.testing.assert_allclose(pr.rgb[0], [0.2, 0.6, 0.9], atol=1e-6)


def test_sh_degree3_colour_uses_view_direction_and_clamps_at_zero():
    s = hs.scene_cfg1(N=2000)
    cam = hs.make_camera(640, 480, eye=(0.5, -0.3, -1.0), centre=(0.0, 0.0, 5.0))
    pr = oracle.project(s, cam)
    for i in np.nonzero(pr.valid)[0][:100]:
        d = s.means[i].astype(np.float64) - cam.cam_pos.astype(np.float64)
        d /= np.linalg.norm(d)
        Y = np.array([_real_sh_scipy(l, m, d) for l in range(4) for m in range(-l, l + 1)])
        ref = np.maximum(0.0, 0.5 + Y @ s.sh[i].astype(np.float64))
        np.testing.assert_allclose(pr.rgb[i], ref, atol=1e-10)
    assert (pr.rgb >= 0).all()


def test_cholesky_identity_and_factors():
    """Sigma^-1 = L L^T gives q = (l0 dx + l1 dy)^2 + (l2 dy)^2, equal to the conic form
    A dx^2 + B2 dx dy + C dy^2.  Checked against an independent fp64 evaluation written here from the covariance
    (numpy inverse and numpy Cholesky), on ordinary gaussians of cfg1 and on ill-conditioned needles, where the
    conic form cancels but the sum of squares does not; a swapped l1 / l2, a wrong sign of l1 or an upper-triangular
    factor each fail."""
    rng = np.random.default_rng(12)
    for scene in (hs.scene_cfg1(N=400), hs.needle_scene(200, 1920, 1080, seed=3, sigma_lo_px=50, sigma_hi_px=1500)):
        pr = oracle.project(scene, scene.cameras[0])
        for i in np.nonzero(pr.valid)[0][:150]:
            a, b, c = (float(v) for v in pr.geo[i, 2:5])
            l = oracle.cholesky(a, b, c)
            Sinv = np.linalg.inv(np.array([[a, b], [b, c]], np.float64))
            Lnp = np.linalg.cholesky(Sinv)                      # lower triangular, positive diagonal: unique
            assert np.allclose([l[0], l[1], l[2]], [Lnp[0, 0], Lnp[1, 0], Lnp[1, 1]], rtol=1e-9, atol=0)
            for _ in range(4):
                dx, dy = rng.normal(0, 3 * math.sqrt(a)), rng.normal(0, 3 * math.sqrt(c))
                d = np.array([dx, dy])
                q_ref = float(d @ Sinv @ d)
                assert abs(oracle.q_cholesky(dx, dy, l) - q_ref) <= 1e-6 * max(q_ref, 1e-12)
