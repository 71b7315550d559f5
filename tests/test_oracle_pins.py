"""Pins for the oracle (oracle/oracle.cpp) -- CPU only, no GPU, no CUDA library.

The paper prints no worked example for the rasterizer, so every pin is what the paper's equations
and the mathematics fix: closed forms (Eq. 1, Eq. 7), invariants, a dense "tent function" brute
force that restates Eq. 7 without floor() or buckets, the adjoint of torch's grid_sample (a library
routine), central finite differences, and an independent torch-autograd restatement.
A plausible mistake in the oracle (dropped term, wrong sign / index, transposed weight, wrong
pixel-centre convention, wrong tie-break, off-by-one cut-off) fails at least one of these.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2403_16862_b200.workloads import Camera, make_workload, second_pose

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
TINY = dict(fx=64.0, fy=64.0, cx=32.0, cy=32.0, width=64, height=64)


def _golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    return rows


def _one(pos, op, feat, cam=None):
    cam = cam or Camera(**TINY)
    r = oracle.Raster.from_points(np.array(pos, np.float32).reshape(-1, 3), np.array(op, np.float32).reshape(-1),
                                  np.array(feat, np.float32).reshape(len(op), -1), cam)
    return r


# ---------------------------------------------------------------- Eq. 7 closed forms (S1, S2)

def test_single_point_weights_golden():
    f = np.array([[0.25, 0.5, 0.75, 1.0]], np.float32)
    op = 0.8
    r = _one([[0.3, -0.2, 4.0]], [op], f)
    img, alpha, nb, _ = r.blend()
    cnt = r.counts()
    rows = _golden("single_point.txt")
    assert cnt.sum() == 4 and r.total == 4
    wsum = 0.0
    for px, py, w in rows:
        px, py = int(px), int(py)
        assert cnt[py, px] == 1
        # isolated point: composited value is f * a * w, alpha is a * w  (north_star closed form)
        np.testing.assert_allclose(alpha[py, px], np.float32(op) * w, rtol=0, atol=2e-6)
        np.testing.assert_allclose(img[py, px], f[0].astype(np.float64) * np.float32(op) * w, rtol=0, atol=2e-6)
        wsum += alpha[py, px] / np.float32(op)
    assert abs(wsum - 1.0) < 1e-6                       # four weights sum to 1
    np.testing.assert_allclose(img.sum(axis=(0, 1)), f[0] * np.float32(op), atol=2e-6)
    assert (cnt > 0).sum() == 4


def test_point_on_pixel_centre_weights_1000_and_four_fragments():
    # u = 64*x/z+32 = 40.5 exactly: x/z = 8.5/64 with z = 4 -> x = 0.53125 (exact in fp32)
    r = _one([[0.53125, -0.46875, 4.0]], [0.5], [[1, 2, 3, 4]])   # v = 64*(-0.46875)/4+32 = 24.5
    img, alpha, _, _ = r.blend()
    cnt = r.counts()
    assert cnt[24, 40] == 1 and cnt[24, 41] == 1 and cnt[25, 40] == 1 and cnt[25, 41] == 1   # A6: zero-weight kept
    assert cnt.sum() == 4
    assert alpha[24, 40] == 0.5 and alpha[24, 41] == 0 and alpha[25, 40] == 0 and alpha[25, 41] == 0
    np.testing.assert_array_equal(img[24, 40], 0.5 * np.array([1, 2, 3, 4.0]))


def test_border_fragments_dropped_per_fragment():
    # u = 0.2 -> fu = -0.3 -> x0 = -1: only the right column (pixel 0) survives, with weight tx = 0.7
    z = 4.0
    x = (0.2 - 32) * z / 64
    y = (10.5 - 32) * z / 64
    r = _one([[x, y, z]], [1.0], [[1, 1, 1, 1]])
    _, alpha, _, _ = r.blend()
    cnt = r.counts()
    assert cnt.sum() == 2 and cnt[10, 0] == 1 and cnt[11, 0] == 1
    assert r.kept == 1 and r.border_dropped == 2
    np.testing.assert_allclose(alpha[10, 0], 0.7, atol=1e-5)
    # completely outside: nothing
    r = _one([[(-1.2 - 32) * z / 64, y, z]], [1.0], [[1, 1, 1, 1]])
    assert r.total == 0 and r.kept == 0


def test_near_far_strict_and_nan_culled():
    cam = Camera(**TINY)
    pts = [[0, 0, cam.near_z], [0, 0, cam.far_z], [0, 0, -1.0], [0, 0, np.nan], [np.inf, 0, 1.0], [0, 0, 1.0]]
    r = _one(pts, [1.0] * 6, [[1, 1, 1, 1]] * 6)
    assert r.kept == 1 and r.total == 4


# ---------------------------------------------------------------- dense tent brute force (S1-S4)

def _project_np32(pos, cam):
    """Independent restatement of the canonical fp32 projection in numpy (every op rounds to fp32)."""
    R = np.asarray(cam.R, np.float32).reshape(9)
    t = np.asarray(cam.t, np.float32)
    x, y, z = (pos[:, k].astype(np.float32) for k in range(3))
    f32 = np.float32
    xc = ((R[0] * x + R[1] * y) + R[2] * z) + t[0]
    yc = ((R[3] * x + R[4] * y) + R[5] * z) + t[1]
    zc = ((R[6] * x + R[7] * y) + R[8] * z) + t[2]
    assert xc.dtype == np.float32
    with np.errstate(all="ignore"):
        u = (f32(cam.fx) * xc) / zc + f32(cam.cx)
        v = (f32(cam.fy) * yc) / zc + f32(cam.cy)
    keep = (zc > f32(cam.near_z)) & (zc < f32(cam.far_z)) & np.isfinite(u) & np.isfinite(v)
    return u, v, zc, keep


def _brute_force(pos, op, feat, cam, t_min=1e-4):
    """O(N*P): for every pixel scan all points; Eq. 7 as the tent max(0,1-|du|)max(0,1-|dv|)."""
    u, v, zc, keep = _project_np32(pos, cam)
    fu = (u - np.float32(0.5)).astype(np.float64)
    fv = (v - np.float32(0.5)).astype(np.float64)
    zb = zc.view(np.uint32).astype(np.int64)
    H, W, D = cam.height, cam.width, feat.shape[1]
    img = np.zeros((H, W, D)); alpha = np.zeros((H, W)); cnt = np.zeros((H, W), np.int64)
    order = {}
    for py in range(H):
        iny = keep & (fv >= py - 1) & (fv < py + 1)
        if not iny.any():
            continue
        cand = np.nonzero(iny)[0]
        for px in range(W):
            m = cand[(fu[cand] >= px - 1) & (fu[cand] < px + 1)]
            cnt[py, px] = len(m)
            if len(m) == 0:
                continue
            m = m[np.lexsort((m, zb[m]))]
            order[(py, px)] = m
            w = (1 - np.abs(fu[m] - px)) * (1 - np.abs(fv[m] - py))
            T = 1.0
            for k, i in enumerate(m):
                if T < t_min:
                    break
                a = float(op[i]) * w[k]
                img[py, px] += T * a * feat[i].astype(np.float64)
                alpha[py, px] += T * a
                T *= 1 - a
    return img, alpha, cnt, order


@pytest.mark.parametrize("pose", [False, True])
def test_brute_force_counts_order_image(pose):
    w = make_workload("tiny", n_points=1500)
    cam = Camera(fx=16.0, fy=16.0, cx=8.0, cy=8.0, width=16, height=16)   # dense: ~23 fragments / pixel
    if pose:
        cam = cam.with_pose(*second_pose())
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, cam)
    img, alpha, nb, _ = r.blend()
    bimg, balpha, bcnt, border = _brute_force(w.pos, w.opacity, w.feat, cam)
    np.testing.assert_array_equal(r.counts(), bcnt)
    off, idx, dep, _ = r.sorted_fragments()
    for (py, px), m in border.items():
        p = py * cam.width + px
        np.testing.assert_array_equal(idx[off[p]:off[p + 1]], m)
    np.testing.assert_allclose(img, bimg, rtol=0, atol=1e-12)
    np.testing.assert_allclose(alpha, balpha, rtol=0, atol=1e-12)
    assert r.total == 4 * r.kept - r.border_dropped            # count identity
    assert bcnt.max() > 32                                      # several pixels deeper than a warp


def test_tiny_counts_identity_and_strict_order():
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    assert r.counts().sum() == r.total == 4 * r.kept - r.border_dropped
    off, idx, dep, wgt = r.sorted_fragments()
    key = dep.astype(np.int64) << 32 | idx
    same_pixel = np.ones(len(key) - 1, bool)
    same_pixel[off[1:-1][(off[1:-1] > 0) & (off[1:-1] < len(key))] - 1] = False
    assert np.all(np.diff(key)[same_pixel] > 0)                 # total order, strictly increasing
    assert np.all((wgt >= 0) & (wgt <= 1))


def test_forced_depth_ties_break_by_point_index():
    # three coincident points (same depth bits) on a pixel centre: order must be 0,1,2 whatever the
    # input order of their attributes; result C = a0 f0 + (1-a0) a1 f1 + (1-a0)(1-a1) a2 f2.
    p = [0.53125, -0.46875, 4.0]
    a = np.array([0.25, 0.5, 0.75], np.float32)
    f = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float32)
    r = _one([p, p, p], a, f)
    off, idx, dep, _ = r.sorted_fragments()
    q = 24 * 64 + 40
    np.testing.assert_array_equal(idx[off[q]:off[q + 1]], [0, 1, 2])
    img, alpha, _, _ = r.blend()
    np.testing.assert_allclose(img[24, 40], [0.25, 0.75 * 0.5, 0.75 * 0.5 * 0.75, 0], atol=1e-12)
    np.testing.assert_allclose(alpha[24, 40], 1 - 0.75 * 0.5 * 0.25, atol=1e-12)
    # nearer point wins regardless of index
    r = _one([p, [0.53125 * 0.5, -0.46875 * 0.5, 2.0]], [0.25, 0.5], f[:2])
    off, idx, _, _ = r.sorted_fragments()
    np.testing.assert_array_equal(idx[off[q]:off[q + 1]], [1, 0])


# ---------------------------------------------------------------- Eq. 1 closed forms (S4)

def test_stacked_equal_opacity_cutoff_golden():
    p = [0.53125, -0.46875, 4.0]
    for n, blended, alpha_ref in _golden("stacked_half.txt"):
        n = int(n)
        r = _one([p] * n, [0.5] * n, [[1, 1, 1, 1]] * n)
        img, alpha, nb, margin = r.blend()
        assert nb[24, 40] == int(blended)
        assert alpha[24, 40] == alpha_ref                       # exact in binary
        assert img[24, 40, 0] == alpha_ref
    # cut-off disabled: alpha = 1 - prod(1-a), order independent
    r = _one([p] * 40, [0.5] * 40, [[1, 1, 1, 1]] * 40)
    _, alpha, nb, _ = r.blend(t_min=0.0)
    assert nb[24, 40] == 40 and abs(alpha[24, 40] - (1 - 0.5 ** 40)) < 1e-15


def test_margin_output_golden():
    """`margin` decides which pixels the GPU harness treats as termination-ambiguous: pinned to hand-derived
    values (tests/golden/stacked_margin.txt), not to the oracle's own formula."""
    p = [0.53125, -0.46875, 4.0]
    for a, n, blended, m_ref in _golden("stacked_margin.txt"):
        n = int(n)
        r = _one([p] * n, [a] * n, [[1, 1, 1, 1]] * n)
        _, _, nb, margin = r.blend()
        assert nb[24, 40] == int(blended)
        assert abs(margin[24, 40] - m_ref) <= 1e-7 * m_ref
        assert np.isinf(margin[0, 0])                            # a pixel without fragments tests nothing
    _, _, _, margin = r.blend(t_min=0.0)
    assert np.isinf(margin).all()                                # cut-off disabled


def test_forced_blend_count_and_sorted_T():
    """force_nb (harness aid, R7) replaces the termination test by a fixed count and nothing else:
    n stacked fragments of a = 0.5 forced to 20 give alpha = 1 - 2^-20; sorted_T lists 2^-k for the blended
    fragments and -1 behind them."""
    p = [0.53125, -0.46875, 4.0]
    r = _one([p] * 40, [0.5] * 40, [[1, 1, 1, 1]] * 40)
    force = np.full((64, 64), oracle.NO_FORCE, dtype=np.uint32)
    force[24, 40] = 20
    img, alpha, nb, margin = r.blend(force_nb=force)
    assert nb[24, 40] == 20 and alpha[24, 40] == 1 - 0.5 ** 20 and img[24, 40, 2] == 1 - 0.5 ** 20
    off, _, _, _ = r.sorted_fragments()
    q = 24 * 64 + 40
    T = r.sorted_T()[off[q]:off[q + 1]]
    np.testing.assert_array_equal(T[:20], 0.5 ** np.arange(20))
    np.testing.assert_array_equal(T[20:], -1.0)
    # unforced pixels keep the test: the same stack with NO_FORCE everywhere is the golden 14
    _, alpha, nb, _ = r.blend(force_nb=np.full((64, 64), oracle.NO_FORCE, dtype=np.uint32))
    assert nb[24, 40] == 14 and alpha[24, 40] == 0.99993896484375
    np.testing.assert_array_equal(r.sorted_T()[off[q]:off[q + 1]][14:], -1.0)
    # and the backward pass follows the forced state: d alpha / d a_k = prod_{j != k} (1 - a_j) over the 20
    r.blend(force_nb=force)
    _, d_op, _ = r.backward(np.zeros((64, 64, 4)), np.ones((64, 64)))
    np.testing.assert_allclose(d_op[:20], 0.5 ** 19, rtol=1e-12)
    np.testing.assert_array_equal(d_op[20:], 0.0)


def test_blend_weights_golden():
    """NEXT row f1 (Eq. 3 input): hand-derived values of tests/golden/blend_weight.txt."""
    gold = {}
    for line in open(os.path.join(GOLDEN, "blend_weight.txt")):
        if line.strip() and not line.startswith("#"):
            c, i, v = line.split()
            gold[(c, int(i))] = float(v)
    p = [0.53125, -0.46875, 4.0]                                   # u = 40.5, v = 24.5: a pixel centre
    n = 16
    z = 4.0 + 0.25 * np.arange(n)                                  # depth order = index order
    pos = np.stack([0.53125 / 4 * z, -0.46875 / 4 * z, z], 1)
    r = _one(pos, [0.5] * n, [[1, 1, 1, 1]] * n)
    r.blend()
    bw = r.blend_weights()
    for (c, i), v in gold.items():
        if c == "A":
            assert bw[i] == v, (i, bw[i], v)                       # powers of two: exact
    np.testing.assert_array_equal(bw[:14], 0.5 ** (np.arange(14) + 1))
    # case B: A on the centre of pixel (36, 28) at depth 3, B at (36.8, 28.8) depth 4
    A = [(36.5 - 32) / 64 * 3.0, (28.5 - 32) / 64 * 3.0, 3.0]
    B = [0.3, -0.2, 4.0]
    r = _one([A, B], [0.8, 0.5], [[1, 1, 1, 1]] * 2)
    r.blend()
    bw = r.blend_weights()
    # fp32 inputs: opacity 0.8f, and u = 36.8 carries an fp32 ulp of 3.8e-6 into tx = ty = 0.3
    assert abs(bw[0] - gold[("B", 0)]) < 1e-7 and abs(bw[1] - gold[("B", 1)]) < 2e-6
    # culled / zero-opacity points get exactly 0; a weight never exceeds the opacity
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    r.blend()
    bw = r.blend_weights()
    assert (bw >= 0).all() and (bw <= w.opacity.astype(np.float64) + 1e-15).all() and bw.max() > 0.3


def test_level_camera_golden_and_multisample_mean():
    """NEXT row f3: the level camera against a hand-derived footprint (tests/golden/level1_point.txt); the
    multisample image is the plain mean; the planar layout is a transposition."""
    cam = Camera(**TINY)
    c1 = oracle.level_camera(cam, 1)
    assert (c1.width, c1.height, float(c1.fx), float(c1.cx)) == (32, 32, 32.0, 16.0)
    c2 = oracle.level_camera(Camera(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840), 2)
    assert (c2.width, c2.height, float(c2.fx), float(c2.cx), float(c2.cy)) == (325, 210, 275.0, 162.125, 105.0)
    f = np.array([[0.25, 0.5, 0.75, 1.0]], np.float32)
    r0, r1 = oracle.rasterize_levels([[0.3, -0.2, 4.0]], [0.5], f, cam, 2)
    img, alpha, _, _ = r1.blend()
    assert img.shape == (32, 32, 4)
    total = 0.0
    for x, y, w in _golden("level1_point.txt"):
        assert abs(alpha[int(y), int(x)] - 0.5 * w) < 2e-6            # fp32 u carries an ulp of 2e-6 into tx
        np.testing.assert_allclose(img[int(y), int(x)], 0.5 * w * f[0], atol=2e-6)
        total += alpha[int(y), int(x)]
    assert abs(total - 0.5) < 1e-12 and abs(alpha.sum() - 0.5) < 1e-12
    # the same point at level 0 keeps the single_point.txt footprint
    a0 = r0.blend()[1]
    assert abs(a0[28, 36] - 0.5 * 0.49) < 2e-6
    # multisample: mean of the clouds' images; two single-point clouds on different pixels -> half of each
    A = ([[0.3, -0.2, 4.0]], [0.5], f)
    B = ([[-0.4, 0.1, 2.0]], [0.8], f * 0.5)
    (m_img, m_alpha), = oracle.multisample([A, B], cam)
    ia = oracle.Raster.from_points(*A, cam).blend()
    ib = oracle.Raster.from_points(*B, cam).blend()
    np.testing.assert_array_equal(m_img, (ia[0] + ib[0]) / 2)
    np.testing.assert_array_equal(m_alpha, (ia[1] + ib[1]) / 2)
    assert abs(m_alpha.sum() - (0.5 + float(np.float32(0.8))) / 2) < 1e-12       # opacities are fp32 inputs
    (s_img, s_alpha), = oracle.multisample([A, A, A, A], cam)            # identical clouds: the mean is the image
    np.testing.assert_allclose(s_img, ia[0], atol=1e-16)
    pl = oracle.to_planar(m_img)
    assert pl.shape == (4, 64, 64) and pl[2, 28, 36] == m_img[28, 36, 2]


def test_sh_basis_against_scipy_and_closed_forms():
    """NEXT row f2: the oracle's real SH basis (degree <= 2) against a LIBRARY routine -- the complex spherical
    harmonics of scipy.special -- and against closed forms on the axes."""
    from scipy import special
    rng = np.random.default_rng(11)
    d = rng.standard_normal((200, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    theta = np.arctan2(d[:, 1], d[:, 0])            # azimuth
    phi = np.arccos(d[:, 2])                        # polar angle
    if hasattr(special, "sph_harm_y"):
        Ylm = lambda l, m: special.sph_harm_y(l, m, phi, theta)
    else:
        Ylm = lambda l, m: special.sph_harm(m, l, theta, phi)
    ref = []
    for l in range(3):
        for m in range(-l, l + 1):
            if m == 0:
                ref.append(Ylm(l, 0).real)
            elif m > 0:
                ref.append(np.sqrt(2) * Ylm(l, m).real)       # scipy includes the Condon-Shortley phase: the real
            else:                                             # combination is sqrt(2) Re / Im of Y_l^|m|, no extra sign
                ref.append(np.sqrt(2) * Ylm(l, -m).imag)
    np.testing.assert_allclose(oracle.sh_basis(d), np.stack(ref, 1), atol=1e-12)
    # closed forms: +z sees Y = (C0, 0, C1, 0, 0, 0, 2 * 0.3154, 0, 0)
    np.testing.assert_allclose(oracle.sh_basis([0, 0, 1.0]), [0.28209479177387814, 0, 0.4886025119029199, 0, 0, 0,
                                                             0.6307831305050401, 0, 0], atol=1e-15)
    np.testing.assert_allclose(oracle.sh_basis([1.0, 0, 0]), [0.28209479177387814, 0, 0, -0.4886025119029199, 0, 0,
                                                             -0.31539156525252005, 0, 0.5462742152960396], atol=1e-15)
    # orthonormality on the sphere (Monte Carlo): (4 pi / n) sum Y_a Y_b ~ delta_ab
    dd = rng.standard_normal((400000, 3)); dd /= np.linalg.norm(dd, axis=1, keepdims=True)
    Y = oracle.sh_basis(dd)
    np.testing.assert_allclose(4 * np.pi * (Y.T @ Y) / len(dd), np.eye(9), atol=0.02)


def test_sh_features_and_adjoint():
    cam = Camera(**TINY)
    R, t = second_pose()
    cam = cam.with_pose(R, t)
    rng = np.random.default_rng(12)
    pos = rng.uniform(-1, 1, (50, 3)) + [0, 0, 4]
    coeff = rng.standard_normal((50, 36))
    f = oracle.sh_features(pos, coeff, cam)
    # a coefficient vector that is non-zero only in the constant term gives C0 * that term, whatever the direction
    c0 = np.zeros((50, 36)); c0[:, :4] = coeff[:, :4]
    np.testing.assert_allclose(oracle.sh_features(pos, c0, cam), 0.28209479177387814 * coeff[:, :4], atol=1e-15)
    # the camera centre is -R^T t: a point there sees the constant term only
    centre = -np.asarray(R, np.float64).T @ np.asarray(t, np.float64)
    np.testing.assert_allclose(oracle.sh_features([centre], coeff[:1], cam), 0.28209479177387814 * coeff[:1, :4], atol=1e-12)
    # linear in the coefficients; sh_backward is the exact adjoint
    g = rng.standard_normal((50, 4))
    assert abs((f * g).sum() - (oracle.sh_backward(pos, cam, g) * coeff).sum()) < 1e-10


def test_general_stack_formula():
    rng = np.random.default_rng(5)
    n = 12
    a = rng.uniform(0.05, 0.6, n).astype(np.float32)
    f = rng.uniform(0, 1, (n, 4)).astype(np.float32)
    z = np.sort(rng.uniform(2, 6, n)).astype(np.float32)
    pos = np.stack([0.53125 / 4 * z, -0.46875 / 4 * z, z], 1).astype(np.float32)
    # keep only those that land exactly on the pixel centre in fp32 (u = 40.5): all do if x/z exact
    u, v, _, _ = _project_np32(pos, Camera(**TINY))
    ok = (u == 40.5) & (v == 24.5)
    pos, a, f = pos[ok], a[ok], f[ok]
    assert ok.sum() >= 4
    perm = rng.permutation(len(a))
    r = _one(pos[perm], a[perm], f[perm])
    img, alpha, _, _ = r.blend()
    T = np.concatenate([[1.0], np.cumprod(1 - a.astype(np.float64))])
    np.testing.assert_allclose(img[24, 40], (T[:-1, None] * a[:, None] * f).sum(0), atol=1e-12)
    np.testing.assert_allclose(alpha[24, 40], 1 - T[-1], atol=1e-12)


# ---------------------------------------------------------------- invariants

def test_invariants_tiny():
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    img, alpha, nb, _ = r.blend()
    cnt = r.counts()
    assert np.all(alpha >= 0) and np.all(alpha <= 1)
    assert np.all(img[cnt == 0] == 0) and np.all(alpha[cnt == 0] == 0)
    assert np.all(nb <= cnt)
    # alpha <= sum of fragment opacities;  image linear in features
    r2 = oracle.Raster.from_points(w.pos, w.opacity, 2.0 * w.feat, w.cam)
    img2, alpha2, _, _ = r2.blend()
    np.testing.assert_allclose(img2, 2.0 * img, rtol=1e-12, atol=1e-12)
    np.testing.assert_array_equal(alpha2, alpha)
    # zero opacity => zero image, zero alpha, but same counts (A6)
    r0 = oracle.Raster.from_points(w.pos, 0 * w.opacity, w.feat, w.cam)
    img0, alpha0, _, _ = r0.blend()
    assert not img0.any() and not alpha0.any()
    np.testing.assert_array_equal(r0.counts(), cnt)
    # features == 1 => image channel == alpha
    r1 = oracle.Raster.from_points(w.pos, w.opacity, np.ones_like(w.feat), w.cam)
    img1, alpha1, _, _ = r1.blend()
    np.testing.assert_allclose(img1[..., 0], alpha1, atol=1e-14)


def test_transmittance_monotone_and_alpha_is_one_minus_T():
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    _, alpha_cut, nb, _ = r.blend()
    _, alpha_all, nb_all, _ = r.blend(t_min=0.0)
    assert np.all(nb_all == r.counts())
    assert np.all(alpha_all >= alpha_cut - 1e-15)                 # more fragments only add
    assert np.all(alpha_all - alpha_cut <= 1e-4 + 1e-12)          # what the cut-off drops is < t_min
    off, idx, dep, wgt = r.sorted_fragments()
    a = w.opacity[idx].astype(np.float64) * wgt
    for p in np.random.default_rng(0).integers(0, r.P, 200):
        seg = a[off[p]:off[p + 1]]
        T = np.cumprod(1 - seg)
        assert np.all(np.diff(np.concatenate([[1.0], T])) <= 0)    # monotone non-increasing
        np.testing.assert_allclose(alpha_all.reshape(-1)[p], 1 - (T[-1] if len(T) else 1.0), atol=1e-13)


def test_permutation_invariance():
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    _, _, dep, _ = r.sorted_fragments()
    img, alpha, _, _ = r.blend()
    perm = np.random.default_rng(1).permutation(w.N)
    rp = oracle.Raster.from_points(w.pos[perm], w.opacity[perm], w.feat[perm], w.cam)
    imgp, alphap, _, _ = rp.blend()
    # valid only when no pixel holds two fragments with equal depth bits (index tie-break otherwise)
    off, idx, dep, _ = r.sorted_fragments()
    inner = np.ones(len(dep) - 1, bool); inner[off[1:-1][off[1:-1] < len(dep)] - 1] = False
    assert not np.any((np.diff(dep.astype(np.int64)) == 0) & inner)
    np.testing.assert_array_equal(imgp, img)
    np.testing.assert_array_equal(alphap, alpha)
    np.testing.assert_array_equal(rp.counts(), r.counts())


def test_opaque_centre_points_is_zbuffer():
    # all points on pixel centres with opacity 1 => nearest point's feature, alpha 1 (textbook z-buffer)
    rng = np.random.default_rng(2)
    n = 300
    px = rng.integers(0, 8, n); py = rng.integers(0, 8, n)
    z = rng.choice(np.array([1.0, 2.0, 4.0, 8.0], np.float32), n)      # exact divisions
    cam = Camera(fx=8.0, fy=8.0, cx=4.0, cy=4.0, width=8, height=8)
    pos = np.stack([(px + 0.5 - 4.0) / 8.0 * z, (py + 0.5 - 4.0) / 8.0 * z, z], 1).astype(np.float32)
    feat = rng.uniform(0, 1, (n, 4)).astype(np.float32)
    r = oracle.Raster.from_points(pos, np.ones(n, np.float32), feat, cam)
    img, alpha, nb, _ = r.blend()
    for y in range(8):
        for x in range(8):
            m = np.nonzero((px == x) & (py == y))[0]
            if len(m) == 0:
                continue
            first = m[np.lexsort((m, z[m]))][0]
            np.testing.assert_array_equal(img[y, x], feat[first].astype(np.float64))
            assert alpha[y, x] == 1.0 and nb[y, x] >= 1      # zero-weight fragments of neighbours may sit in front (A6)


# ---------------------------------------------------------------- library reduction: grid_sample adjoint

@pytest.mark.parametrize("pose", [False, True])
def test_low_opacity_limit_is_grid_sample_adjoint(pose):
    """As opacity -> 0, img/eps -> sum_fragments w * alpha_h * f, which is the adjoint (VJP w.r.t. the
    input image) of bilinear sampling with zero padding and align_corners=False: pins the pixel-centre
    convention and the per-fragment border rule against torch, independently of the oracle's code."""
    w = make_workload("tiny", n_points=3000)
    cam = w.cam.with_pose(*second_pose()) if pose else w.cam
    eps = 1e-7
    op = (w.opacity.astype(np.float64) * eps).astype(np.float32)
    r = oracle.Raster.from_points(w.pos, op, w.feat, cam)
    img, _, _, _ = r.blend(t_min=0.0)
    u, v, _, keep = _project_np32(w.pos, cam)
    H, W = cam.height, cam.width
    gx = torch.tensor(2.0 * u[keep].astype(np.float64) / W - 1.0)
    gy = torch.tensor(2.0 * v[keep].astype(np.float64) / H - 1.0)
    grid = torch.stack([gx, gy], -1).view(1, 1, -1, 2)
    X = torch.zeros(1, 4, H, W, dtype=torch.float64, requires_grad=True)
    s = torch.nn.functional.grid_sample(X, grid, mode="bilinear", padding_mode="zeros", align_corners=False)
    cot = torch.tensor((op[keep].astype(np.float64)[:, None] * w.feat[keep].astype(np.float64)).T).view(1, 4, 1, -1)
    (adj,) = torch.autograd.grad(s, X, cot)
    ref = adj[0].permute(1, 2, 0).numpy()
    scale = np.abs(ref).max()
    assert scale > 0
    np.testing.assert_allclose(img, ref, rtol=0, atol=scale * 1e-5)   # O(eps * depth complexity) + fp32 grid rounding


# ---------------------------------------------------------------- gradients (S5, S6)

def _uv_problem(seed, n=48, W=6, H=5, D=3, dense=False):
    rng = np.random.default_rng(seed)
    # keep u, v at least 0.02 px away from pixel-centre kinks (where |.| is not differentiable)
    def coords(m, size):
        base = rng.integers(0, size + 1, m).astype(np.float64) - 0.5      # floor(f) in {-1..size-1}
        if dense:
            base = np.full(m, 0.5)             # every point between the same 2x2 centres: deep pixels
        return base + 0.5 + rng.uniform(0.02, 0.98, m)
    u, v = coords(n, W), coords(n, H)
    depth = rng.uniform(1, 9, n).astype(np.float32)
    op = rng.uniform(0.05, 0.9, n).astype(np.float32)
    feat = rng.uniform(0, 1, (n, D)).astype(np.float32)
    g_img = rng.standard_normal((H, W, D)); g_alpha = rng.standard_normal((H, W))
    return u, v, depth, op, feat, g_img, g_alpha, W, H


def _loss(u, v, depth, op, feat, g_img, g_alpha, W, H, t_min):
    r = oracle.Raster.from_uv(u, v, depth, op, feat, W, H)
    img, alpha, _, margin = r.blend(t_min)
    return float((img * g_img).sum() + (alpha * g_alpha).sum()), margin


@pytest.mark.parametrize("t_min", [0.0, 1e-4])
def test_gradients_central_finite_differences(t_min):
    u, v, depth, op, feat, g_img, g_alpha, W, H = _uv_problem(7)
    if t_min > 0:   # make the cut-off bite: many fairly opaque points on the same four pixels
        u, v, depth, op, feat, g_img, g_alpha, W, H = _uv_problem(8, n=80, W=3, H=3, dense=True)
        op = np.clip(op * 1.6, 0, 0.97).astype(np.float32)
    r = oracle.Raster.from_uv(u, v, depth, op, feat, W, H)
    _, _, nb, margin = r.blend(t_min)
    if t_min > 0:
        assert (nb < r.counts()).any(), "cut-off not exercised"
        assert margin.min() > 1e-3                                # far from the termination discontinuity
    d_feat, d_op, d_uv = r.backward(g_img, g_alpha)
    h = 1e-6
    args = (g_img, g_alpha, W, H, t_min)
    for i in range(len(u)):
        for arr, k in ((u, 0), (v, 1)):
            a1 = arr.copy(); a1[i] += h; a0 = arr.copy(); a0[i] -= h
            Lp = _loss(a1 if k == 0 else u, a1 if k == 1 else v, depth, op, feat, *args)[0]
            Lm = _loss(a0 if k == 0 else u, a0 if k == 1 else v, depth, op, feat, *args)[0]
            fd = (Lp - Lm) / (2 * h)
            assert abs(fd - d_uv[i, k]) <= 1e-5 * max(1.0, abs(fd)), (i, k, fd, d_uv[i, k])
    # opacity and features are float32 inputs: perturb by an exactly representable step
    ho = 2.0 ** -12
    for i in range(len(u)):
        o1 = op.copy(); o1[i] += ho; o0 = op.copy(); o0[i] -= ho
        step = float(o1[i]) - float(o0[i])
        fd = (_loss(u, v, depth, o1, feat, *args)[0] - _loss(u, v, depth, o0, feat, *args)[0]) / step
        assert abs(fd - d_op[i]) <= 2e-4 * max(1.0, abs(fd)), (i, fd, d_op[i])   # O(h^2) truncation
    for i in range(0, len(u), 5):
        for d in range(feat.shape[1]):
            f1 = feat.copy(); f1[i, d] += ho; f0 = feat.copy(); f0[i, d] -= ho
            step = float(f1[i, d]) - float(f0[i, d])
            fd = (_loss(u, v, depth, op, f1, *args)[0] - _loss(u, v, depth, op, f0, *args)[0]) / step
            assert abs(fd - d_feat[i, d]) <= 1e-8 * max(1.0, abs(fd))             # exactly linear in f


def test_feature_gradient_is_exact_adjoint():
    w = make_workload("tiny")
    r = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    img, alpha, _, _ = r.blend()
    d_feat, d_op, d_uv = r.backward(w.g_img, None)
    lhs = (img * w.g_img).sum()
    rhs = (d_feat * w.feat).sum()
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)                    # <g, img(F)> = <d_feat(g), F>
    # culled / unblended points get exactly zero everywhere
    z = np.zeros((w.cam.height, w.cam.width, 4))
    d0 = r.backward(z, np.zeros((w.cam.height, w.cam.width)))
    assert not d0[0].any() and not d0[1].any() and not d0[2].any()


def test_alpha_gradient_closed_form():
    # dA/da_k = prod_{j != k} (1 - a_j) for stacked fragments on one pixel centre, cut-off disabled
    p = [0.53125, -0.46875, 4.0]
    a = np.array([0.2, 0.4, 0.1, 0.3], np.float32)
    r = _one([p] * 4, a, np.ones((4, 4), np.float32))
    r.blend(t_min=0.0)
    g_alpha = np.zeros((64, 64)); g_alpha[24, 40] = 1.0
    _, d_op, _ = r.backward(np.zeros((64, 64, 4)), g_alpha)
    a64 = a.astype(np.float64)
    for k in range(4):
        ref = np.prod(np.delete(1 - a64, k))                     # weight w = 1 at the centre pixel
        assert abs(d_op[k] - ref) < 1e-14


def _torch_reference(u, v, depth, op, feat, g_img, g_alpha, W, H, t_min):
    """Independent restatement with torch autograd: dense tent weights, per-pixel lexsort + cumprod."""
    tu = torch.tensor(u, requires_grad=True); tv = torch.tensor(v, requires_grad=True)
    top = torch.tensor(op.astype(np.float64), requires_grad=True)
    tf = torch.tensor(feat.astype(np.float64), requires_grad=True)
    zb = depth.view(np.uint32).astype(np.int64)
    L = torch.zeros((), dtype=torch.float64)
    fu, fv = u - 0.5, v - 0.5
    for py in range(H):
        for px in range(W):
            m = np.nonzero((fu >= px - 1) & (fu < px + 1) & (fv >= py - 1) & (fv < py + 1))[0]
            if len(m) == 0:
                continue
            m = m[np.lexsort((m, zb[m]))]
            mi = torch.tensor(m)
            wgt = (1 - (tu[mi] - 0.5 - px).abs()) * (1 - (tv[mi] - 0.5 - py).abs())
            a = top[mi] * wgt
            T = torch.cat([torch.ones(1, dtype=torch.float64), torch.cumprod(1 - a, 0)[:-1]])
            keep = (T.detach() >= t_min).to(torch.float64)
            c = T * a * keep
            L = L + (c[:, None] * tf[mi] * torch.tensor(g_img[py, px])[None, :]).sum() + c.sum() * g_alpha[py, px]
    L.backward()
    return float(L.detach()), tf.grad.numpy(), top.grad.numpy(), torch.stack([tu.grad, tv.grad], 1).numpy()


@pytest.mark.parametrize("seed,t_min", [(11, 1e-4), (12, 0.0), (13, 1e-4)])
def test_backward_matches_torch_autograd(seed, t_min):
    u, v, depth, op, feat, g_img, g_alpha, W, H = _uv_problem(seed, n=400, W=7, H=6, D=4, dense=(seed == 13))
    if t_min > 0:
        op = np.clip(op * 1.5, 0, 0.95).astype(np.float32)
    r = oracle.Raster.from_uv(u, v, depth, op, feat, W, H)
    img, alpha, nb, margin = r.blend(t_min)
    d_feat, d_op, d_uv = r.backward(g_img, g_alpha)
    L, tf, to, tuv = _torch_reference(u, v, depth, op, feat, g_img, g_alpha, W, H, t_min)
    assert abs(L - ((img * g_img).sum() + (alpha * g_alpha).sum())) < 1e-10 * max(1, abs(L))
    np.testing.assert_allclose(d_feat, tf, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(d_op, to, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(d_uv, tuv, rtol=1e-9, atol=1e-11)
    if seed == 13:
        assert (nb < r.counts()).any()


def test_world_and_uv_entries_agree():
    """oracle_create (fp32 canonical projection) and oracle_create_uv (given u, v) agree when fed the
    same projected coordinates: ties the FD / autograd pins (uv entry) to the product entry."""
    w = make_workload("tiny")
    u, v, zc, keep = _project_np32(w.pos, w.cam)
    r1 = oracle.Raster.from_points(w.pos, w.opacity, w.feat, w.cam)
    r2 = oracle.Raster.from_uv(u[keep].astype(np.float64), v[keep].astype(np.float64), zc[keep],
                               w.opacity[keep], w.feat[keep], w.cam.width, w.cam.height)
    a1 = r1.blend(); a2 = r2.blend()
    np.testing.assert_array_equal(a1[0], a2[0]); np.testing.assert_array_equal(a1[1], a2[1])
    np.testing.assert_array_equal(r1.counts(), r2.counts())
    g1 = r1.backward(w.g_img, w.g_alpha); g2 = r2.backward(w.g_img, w.g_alpha)
    np.testing.assert_array_equal(g1[0][keep], g2[0]); np.testing.assert_array_equal(g1[2][keep], g2[2])


def test_fp64_projection_diagnostic_reports_small_fraction():
    w = make_workload("1m", n_points=200_000)
    ch = oracle.fp64_projection_changes(w.pos, w.cam)
    assert 0 <= ch < 200_000 * 1e-3      # ~1e-4 of points sit within an fp32 ulp of a pixel boundary
