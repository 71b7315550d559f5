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
