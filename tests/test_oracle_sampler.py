"""CPU pins of the sampler oracle (NEXT row f4, oracle/sampler.py): hand-derived weights, the published SplitMix64
test vector, exact integer helpers, and the statistical / geometric properties the paper states for the sampler."""
import os

import numpy as np

from oracle import sampler
from paper_2403_16862_b200.workloads import Camera, make_octree, second_pose

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
CAM = Camera(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840)


def test_leaf_weight_golden():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "sampler_weights.txt")) if l.strip() and not l.startswith("#")]
    z = np.array([float(r[0]) for r in rows]); lv = np.array([int(r[1]) for r in rows]); p = np.array([float(r[2]) for r in rows])
    want = np.array([float(r[3]) for r in rows])
    centre = np.stack([np.zeros_like(z), np.zeros_like(z), z], 1)
    got = sampler.leaf_weights(centre, lv, p, 64.0, CAM)
    np.testing.assert_allclose(got, want, rtol=2e-7)              # z = 0.01 and p are fp32 inputs
    assert got[4] == 0.0


def test_splitmix64_published_vector_and_mulhi():
    # SplitMix64 (Steele, Lea, Flood 2014; Vigna's reference splitmix64.c) from state 0
    out = sampler.splitmix64(0, np.arange(3))
    assert [int(x) for x in out] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    rng = np.random.default_rng(3)
    a = rng.integers(0, 2 ** 64, 1000, dtype=np.uint64); b = rng.integers(0, 2 ** 64, 1000, dtype=np.uint64)
    assert [int(x) for x in sampler._mulhi64(a, b)] == [(int(x) * int(y)) >> 64 for x, y in zip(a, b)]


def test_integer_cdf_is_the_quantised_distribution():
    phat = np.array([0.0, 2.0, 1.0, 0.0, 4.0, 1e-12])
    cdf = sampler.integer_cdf(phat)
    w = np.diff(np.concatenate([[0], cdf.astype(np.int64)]))
    assert list(w) == [0, 2 ** 31, 2 ** 30, 0, 2 ** 32, 0]          # floor(p / max * 2^32); 1e-12 / 4 * 2^32 < 1
    assert sampler.integer_cdf(np.zeros(5)).sum() == 0


def test_samples_follow_eq4_and_stay_in_the_frustum():
    centre, level, prob, root = make_octree(4096, seed=9)
    N = 400_000
    for cam in (CAM, CAM.with_pose(*second_pose())):
        phat = sampler.leaf_weights(centre, level, prob, root, cam)
        assert (phat == 0).sum() > 100 and (phat > 0).sum() > 1000      # both kinds of leaves exist
        pos, leaf = sampler.sample_view(centre, level, prob, root, cam, seed=123, N=N)
        ok = leaf >= 0
        assert ok.mean() > 0.99
        # (1) no sample outside the view frustum, none from an invisible leaf
        assert sampler.inside_frustum(cam, pos[ok])[0].all()
        assert (phat[leaf[ok]] > 0).all()
        # every sample lies inside its leaf's cube (uniform offset of the centre)
        half = 0.5 * root / 2.0 ** level[leaf[ok]]
        assert (np.abs(pos[ok] - centre[leaf[ok]]) <= half[:, None] * (1 + 1e-6)).all()
        # multinomial with replacement ~ p^: re-drawing only re-distributes the mass of rejected positions, so AMONG the
        # leaves that lie entirely inside the frustum (never rejected) the counts are proportional to p^ (compare the
        # heaviest ones within 5 sigma)
        inner = np.ones(len(level), bool)
        for k in range(8):
            h = 0.5 * root / 2.0 ** level
            off = np.stack([np.where(k & 1, h, -h), np.where(k & 2, h, -h), np.where(k & 4, h, -h)], 1)
            inner &= sampler.inside_frustum(cam, (centre + off).astype(np.float32))[0]
        cnt = np.bincount(leaf[ok], minlength=len(level))
        assert inner.sum() > 500
        expect = cnt[inner].sum() * phat / phat[inner].sum()
        top = np.argsort(-expect * inner)[:50]
        sigma = np.sqrt(expect[top])
        assert (np.abs(cnt[top] - expect[top]) <= 5 * sigma + 0.02 * expect[top]).all()
        # the jitter is uniform: mean offset ~ 0, second moment ~ side^2 / 12
        i = top[0]
        rel = (pos[ok][leaf[ok] == i] - centre[i]) / (root / 2.0 ** level[i])
        assert np.abs(rel.mean(0)).max() < 0.02 and np.abs((rel ** 2).mean(0) - 1 / 12).max() < 0.01


def test_reweighting_properties_2_and_3():
    """(2) farther leaves get fewer samples, (3) leaves of a higher subdivision level get fewer."""
    z = np.array([2.0, 4.0, 8.0, 16.0]); c = np.stack([np.zeros(4), np.zeros(4), z], 1)
    w = sampler.leaf_weights(c, np.full(4, 6), np.full(4, 0.5), 64.0, CAM)
    assert (np.diff(w) < 0).all()
    w = sampler.leaf_weights(np.tile([[0, 0, 5.0]], (4, 1)), np.array([4, 5, 6, 7]), np.full(4, 0.5), 64.0, CAM)
    np.testing.assert_allclose(w[:-1] / w[1:], np.sqrt(2.0), rtol=1e-12)


def test_determinism_and_seed():
    centre, level, prob, root = make_octree(1024, seed=5)
    a = sampler.sample_view(centre, level, prob, root, CAM, seed=1, N=5000)
    b = sampler.sample_view(centre, level, prob, root, CAM, seed=1, N=5000)
    c = sampler.sample_view(centre, level, prob, root, CAM, seed=2, N=5000)
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[0], b[0], equal_nan=True)
    assert (a[1] != c[1]).mean() > 0.9
    # a prefix of the samples does not depend on N (counter-based)
    d = sampler.sample_view(centre, level, prob, root, CAM, seed=1, N=100)
    assert np.array_equal(d[1], a[1][:100])
    # no visible leaf: everything invalid
    e = sampler.sample_view(np.array([[0, 0, -5.0]], np.float32), [8], [1.0], 64.0, CAM, seed=1, N=10)
    assert (e[1] == -1).all() and np.isnan(e[0]).all()


def test_inside_frustum_golden_borders():
    """oracle.sampler.inside_frustum against hand-derived border points (tests/golden/frustum_points.txt): which of
    u = 0, u = W, v = 0, v = H, z = near, z = far belong to the frustum, under two poses."""
    poses = [(np.eye(3), np.zeros(3)), (np.array([[0, 0, -1.0], [0, 1, 0], [1, 0, 0]]), np.array([0, 0, 1.0]))]
    cam = Camera(fx=1024.0, fy=1024.0, cx=648.5, cy=420.0, width=1297, height=840)
    rows = [l.split() for l in open(os.path.join(GOLDEN, "frustum_points.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 18
    for r in rows:
        p = np.array([[float(r[1]), float(r[2]), float(r[3])]])
        assert np.array_equal(p.astype(np.float32).astype(np.float64), p), "fixture value is not an fp32 number"
        got = sampler.inside_frustum(cam.with_pose(*poses[int(r[0])]), p)[0][0]
        assert bool(got) == bool(int(r[4])), r


def _cube_meets_frustum_brute_force(cam, centre, side, n=40):
    """Does any point of a dense n^3 lattice of the cube (faces included) lie inside the frustum?  Plain fp64 pinhole
    projection, nothing shared with the oracle's plane test."""
    g = np.linspace(-0.5, 0.5, n)
    q = centre[None, :] + side * np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    R = np.asarray(cam.R, np.float64).reshape(3, 3); t = np.asarray(cam.t, np.float64)
    pc = q @ R.T + t
    z = pc[:, 2]
    ok = (z > cam.near_z) & (z < cam.far_z)
    with np.errstate(divide="ignore", invalid="ignore"):
        u = cam.fx * pc[:, 0] / z + cam.cx; v = cam.fy * pc[:, 1] / z + cam.cy
    return bool((ok & (u >= 0) & (u < cam.width) & (v >= 0) & (v < cam.height)).any())


def test_visibility_never_misses_a_leaf_the_frustum_enters():
    """Eq. 4's indicator must be 1 for every leaf whose volume intersects the frustum (PAPER.md:322 speaks of "leaves
    whose volume intersects the faces of the viewing frustum" as sampled leaves), also when neither the centre nor a
    corner is inside: a leaf that contains the camera, one the frustum crosses through a face.  Hand-built cases, then
    brute force on large random leaves; and one leaf behind each of the six frustum planes must get p^ = 0."""
    one = lambda c, l: sampler.leaf_weights(np.array([c], np.float64), [l], [1.0], 64.0, CAM)[0]
    # contains the frustum apex: cube [-32, 32]^3 around the camera; all corners project outside or lie behind
    assert not sampler.inside_frustum(CAM, np.array([[0, 0, 0.0]]))[0][0]
    assert one([0, 0, 0], 0) > 0
    # crossed through its face x = 4: cube [4,36] x [-16,16] x [-6,26]; the frustum point (4, 0, 26) is on that face,
    # the corners at z = 26 project to v = 420 +- 677 (above and below the image), the centre to u = 2848
    assert _cube_meets_frustum_brute_force(CAM, np.array([20.0, 0, 10]), 32.0)
    assert one([20, 0, 10], 1) > 0
    # side 8 cubes separated by exactly one plane each: left, right, top, bottom, near (behind the camera), far
    for c in ([-30, 0, 10], [30, 0, 10], [0, -30, 10], [0, 30, 10], [0, 0, -10], [0, 0, 120]):
        assert not _cube_meets_frustum_brute_force(CAM, np.array(c, np.float64), 8.0, n=12)
        assert one(c, 3) == 0.0, c
    # brute force: leaves of side 64 .. 8 scattered around both poses
    rng = np.random.default_rng(11)
    for cam in (CAM, CAM.with_pose(*second_pose())):
        centre = rng.uniform(-60, 60, (300, 3)); level = rng.integers(0, 4, 300)
        phat = sampler.leaf_weights(centre, level, np.ones(300), 64.0, cam)
        c32 = centre.astype(np.float32).astype(np.float64)
        meets = np.array([_cube_meets_frustum_brute_force(cam, c32[i], 64.0 / 2.0 ** level[i], n=24) for i in range(300)])
        assert (phat[meets] > 0).all()
        # the cases the centre-or-corner rule alone would lose exist in this draw, and the plane test is not "always visible"
        corner_rule = sampler.inside_frustum(cam, c32)[0]
        for k in range(8):
            off = np.array([(k & 1) - 0.5, ((k >> 1) & 1) - 0.5, ((k >> 2) & 1) - 0.5]) * (64.0 / 2.0 ** level)[:, None]
            corner_rule |= sampler.inside_frustum(cam, c32 + off)[0]
        assert (meets & ~corner_rule).sum() >= 5
        assert (phat == 0).sum() >= 30
        assert ((phat > 0) & ~meets).mean() < 0.15          # conservative, not sloppy: few cubes admitted that the lattice does not reach


def test_leaf_level_outside_0_30_is_never_sampled():
    w = sampler.leaf_weights(np.tile([[0, 0, 5.0]], (4, 1)), np.array([-1, 31, 200, 6]), np.ones(4), 64.0, CAM)
    assert list(w[:3]) == [0.0, 0.0, 0.0] and w[3] > 0


def test_no_resample_mode_is_the_first_attempt():
    """inference omits re-sampling.  attempts = 1 keeps exactly the samples whose first draw was inside the
    frustum (same bits as the re-sampling mode there) and returns NaN / -1 for the others -- which the re-sampling
    mode had re-drawn, so it has strictly more valid samples on a tree with leaves across the frustum's faces."""
    centre, level, prob, root = make_octree(4096, seed=9)
    N = 50_000
    p8, l8 = sampler.sample_view(centre, level, prob, root, CAM, seed=5, N=N)
    p1, l1 = sampler.sample_view(centre, level, prob, root, CAM, seed=5, N=N, attempts=1)
    ok1 = l1 >= 0
    assert 0.5 < ok1.mean() < 1.0 and (l8 >= 0).sum() > ok1.sum()
    assert np.array_equal(l1[ok1], l8[ok1]) and np.array_equal(p1[ok1], p8[ok1])
    assert np.isnan(p1[~ok1]).all()
    assert sampler.inside_frustum(CAM, p1[ok1])[0].all()
