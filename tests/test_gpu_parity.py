"""GPU parity tests proper (-m gpu): the CUDA path, called through the C ABI, against the oracle.

Every test goes through harness.full_parity: whole-image, every-point, element-by-element comparison in
the three launch configurations (introspection dump, bench.py's fwd+bwd step flags, bench.py's forward-only
flags).  Sizes: Tiny, 1M and reduced draws of the octree / cluster samplers that still span many tiles,
ragged tile edges and the long-run path, then BASELINE.json's full sizes (8M / 16M / 33M points), which the
oracle finishes in tens of seconds.  The last test checks that every kernel instantiation bench.py launches
is one these tests compared with the oracle.
"""
import ctypes
import numpy as np
import pytest
import torch

import oracle
from paper_2403_16862_b200 import raster
from paper_2403_16862_b200.workloads import Camera, Workload, make_workload, second_pose

import bench
import harness
from harness import full_parity, gpu_backward, gpu_forward

pytestmark = pytest.mark.gpu

TINY = dict(fx=64.0, fy=64.0, cx=32.0, cy=32.0, width=64, height=64)


def _wl(pos, op, feat, cam, seed=0, name="custom"):
    pos = np.ascontiguousarray(pos, np.float32).reshape(-1, 3)
    n = pos.shape[0]
    feat = np.ascontiguousarray(feat, np.float32).reshape(n, -1)
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    g_img = rng.standard_normal((cam.height, cam.width, feat.shape[1])).astype(np.float32)
    g_alpha = rng.standard_normal((cam.height, cam.width)).astype(np.float32)
    return Workload(name, pos, np.ascontiguousarray(op, np.float32).reshape(n), feat, cam, g_img, g_alpha, True, seed)


# ------------------------------------------------------------------------------ BASELINE configs

def test_tiny_full_parity():
    rep = full_parity(make_workload("tiny"))
    assert rep["stats"]["n_fragments"] > 4 * 4096 * 0.9


def test_tiny_second_pose_and_no_alpha_grad():
    wl = make_workload("tiny")
    R, t = second_pose()
    wl.cam = wl.cam.with_pose(R, t)
    full_parity(wl, g_alpha=False)


def test_tiny_d8():
    full_parity(make_workload("tiny", D=8))


def test_1m_full_parity():
    rep = full_parity(make_workload("1m"))
    assert rep["stats"]["n_kept"] == 1 << 20


def test_1m_second_pose():
    wl = make_workload("1m", n_points=1 << 18)
    R, t = second_pose()
    wl.cam = wl.cam.with_pose(R, t)
    full_parity(wl)


def test_train_sampler_reduced():
    # octree sampler, 1M draws: same camera / structure as config 3, deep enough to split tiles
    rep = full_parity(make_workload("train", n_points=1 << 20))
    assert rep["stats"]["n_tile_items"] > 0


def test_infer_sampler_reduced_d8():
    full_parity(make_workload("infer", n_points=1 << 20), backward=False)


def test_infer_sampler_reduced_d8_backward():
    full_parity(make_workload("infer", n_points=1 << 18, D=8), backward=True)


def test_stress_sampler_reduced_hits_long_run_path():
    rep = full_parity(make_workload("stress", n_points=1 << 20))
    assert rep["stats"]["n_big_pixels"] > 0, "the reduced stress draw must exercise the long-run path"


# ------------------------------------------------------------------------------ full sizes (BASELINE.json configs 3-5)
# The oracle finishes these in tens of seconds, so the whole image / every gradient is compared, in the launch
# configurations bench.py times (harness runs B and C) as well as in the introspection one (run A).

def test_train_full_size():
    rep = full_parity(make_workload("train"))
    assert rep["stats"]["n_kept"] == 1 << 23


def test_infer_full_size_forward_d8():
    rep = full_parity(make_workload("infer"), backward=False)
    assert rep["stats"]["n_kept"] == 1 << 25


def test_stress_full_size():
    rep = full_parity(make_workload("stress"))
    assert rep["stats"]["n_big_pixels"] > 0


# ------------------------------------------------------------------------------ edge cases

def test_empty_input_gives_zero_image():
    cam = Camera(**TINY)
    pos = torch.zeros((0, 3), device="cuda"); op = torch.zeros((0,), device="cuda"); feat = torch.zeros((0, 4), device="cuda")
    img, alpha, ws = raster.inpc_raster_forward(pos, op, feat, cam)
    torch.cuda.synchronize()
    assert img.shape == (64, 64, 4) and float(img.abs().max()) == 0.0 and float(alpha.abs().max()) == 0.0
    assert int(raster.inpc_raster_get_counts(ws, 64, 64).sum()) == 0
    g = torch.ones((64, 64, 4), device="cuda")
    d_feat, d_op, d_uv = raster.inpc_raster_backward(pos, op, feat, cam, g, None, ws)
    torch.cuda.synchronize()
    assert d_feat.numel() == 0 and d_op.numel() == 0 and d_uv.numel() == 0


def test_all_points_culled():
    cam = Camera(**TINY)
    rng = np.random.Generator(np.random.PCG64(5))
    pos = rng.uniform(-1, 1, (1000, 3)).astype(np.float32)
    pos[:500, 2] = -3.0              # behind the camera
    pos[500:800, 2] = 200.0          # beyond far
    pos[800:900] = np.nan
    pos[900:, 0] = 1e6; pos[900:, 2] = 1.0     # far outside the image
    wl = _wl(pos, rng.uniform(0, 1, 1000), rng.uniform(0, 1, (1000, 4)), cam)
    rep = full_parity(wl)
    assert rep["stats"]["n_fragments"] == 0 and rep["stats"]["n_kept"] == 0


def test_forced_depth_ties_and_duplicates():
    cam = Camera(**TINY)
    rng = np.random.Generator(np.random.PCG64(6))
    base = np.stack([rng.uniform(-0.9, 0.9, 64), rng.uniform(-0.9, 0.9, 64), rng.uniform(2, 6, 64)], axis=1)
    pos = np.repeat(base, 40, axis=0)            # 40 exact duplicates of each point: every key ties 40-fold
    perm = rng.permutation(len(pos))
    pos = pos[perm]
    n = len(pos)
    full_parity(_wl(pos, rng.uniform(0, 0.3, n), rng.uniform(0, 1, (n, 4)), cam))


def test_points_on_pixel_centres_and_borders():
    cam = Camera(**TINY)
    rng = np.random.Generator(np.random.PCG64(7))
    # pixel centres (u = i + 0.5): weights 1,0,0,0 with four counted fragments
    i = rng.integers(0, 64, 500); j = rng.integers(0, 64, 500)
    z = rng.uniform(2, 6, 500)
    centres = np.stack([(i + 0.5 - 32.0) / 64.0 * z, (j + 0.5 - 32.0) / 64.0 * z, z], axis=1)
    # image border: u in [-0.6, 0.6] and [63.4, 64.6] -> one or two in-image fragments
    ub = np.concatenate([rng.uniform(-0.6, 0.6, 250), rng.uniform(63.4, 64.6, 250)])
    vb = rng.uniform(-0.6, 64.6, 500)
    zb = rng.uniform(2, 6, 500)
    border = np.stack([(ub - 32.0) / 64.0 * zb, (vb - 32.0) / 64.0 * zb, zb], axis=1)
    pos = np.concatenate([centres, border, border[:, [1, 0, 2]]], axis=0)
    n = len(pos)
    op = rng.uniform(0, 1, n)
    op[:100] = 1.0                                # opaque points on pixel centres: a = 1 exactly
    op[100:150] = 0.0
    full_parity(_wl(pos, op, rng.uniform(0, 1, (n, 4)), cam))


def test_one_very_deep_pixel_50k_fragments():
    cam = Camera(**TINY)
    rng = np.random.Generator(np.random.PCG64(8))
    n = 50_000
    z = rng.uniform(2, 6, n)
    u = rng.uniform(20.0, 21.0, n); v = rng.uniform(30.0, 31.0, n)      # all inside one 2x2 pixel block
    pos = np.stack([(u - 32.0) / 64.0 * z, (v - 32.0) / 64.0 * z, z], axis=1)
    op = rng.uniform(0, 2e-4, n)                  # tiny opacities: nothing is cut off, every fragment is blended
    rep = full_parity(_wl(pos, op, rng.uniform(0, 1, (n, 4)), cam))
    assert rep["stats"]["n_big_pixels"] >= 4 and rep["stats"]["n_big_fragments"] > 100_000


def test_deep_pixel_with_cutoff():
    cam = Camera(**TINY)
    rng = np.random.Generator(np.random.PCG64(9))
    n = 30_000
    z = rng.uniform(2, 6, n)
    u = rng.uniform(10.0, 14.0, n); v = rng.uniform(40.0, 43.0, n)
    pos = np.stack([(u - 32.0) / 64.0 * z, (v - 32.0) / 64.0 * z, z], axis=1)
    full_parity(_wl(pos, rng.uniform(0, 0.2, n), rng.uniform(0, 1, (n, 4)), cam))


def test_ragged_image_size_not_multiple_of_tile():
    cam = Camera(fx=50.0, fy=50.0, cx=18.5, cy=11.5, width=37, height=23)
    rng = np.random.Generator(np.random.PCG64(10))
    n = 20_000
    pos = np.stack([rng.uniform(-1.6, 1.6, n), rng.uniform(-1.0, 1.0, n), rng.uniform(1, 5, n)], axis=1)
    full_parity(_wl(pos, rng.uniform(0, 1, n), rng.uniform(0, 1, (n, 4)), cam))


def test_single_pixel_image():
    cam = Camera(fx=2.0, fy=2.0, cx=0.5, cy=0.5, width=1, height=1)
    rng = np.random.Generator(np.random.PCG64(11))
    n = 300
    pos = np.stack([rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(1, 5, n)], axis=1)
    full_parity(_wl(pos, rng.uniform(0, 0.05, n), rng.uniform(0, 1, (n, 4)), cam))


# ------------------------------------------------------------------------------ NEXT row f3: levels, multisampling, [D,H,W]

def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _reference_with_gpu_counts(ref, ws, W, H):
    """Oracle image / alpha with the termination-ambiguous pixels resolved by harness.resolve_ambiguous (the one rule:
    counts equal outside the ambiguous pixels, inside them bounded by the cut-off moved by -+2 MARGIN, then forced)."""
    nb = raster.inpc_raster_get_blended_counts(ws, W, H).cpu().numpy().view(np.uint32)
    img_r, alpha_r, _, _ = harness.resolve_ambiguous(ref, nb, W, H, check_bound=False)
    return img_r, alpha_r


@pytest.mark.parametrize("name,kw,planar", [("tiny", {}, False), ("tiny", {"D": 8}, True),
                                            ("train", {"n_points": 1 << 19}, True), ("1m", {}, False)])
def test_three_resolution_levels_forward_and_backward(name, kw, planar):
    """One cloud at three resolution levels, each level against the oracle run with that
    level's camera -- forward, and backward through inpc_raster_backward_ex with the level's own gradient images;
    [D,H,W] layout on request."""
    wl = make_workload(name, **kw)
    D = wl.D
    flags = raster.SAVE_FOR_BACKWARD | (raster.OUT_PLANAR if planar else 0)
    pos, op, feat = _dev(wl.pos), _dev(wl.opacity), _dev(wl.feat)
    imgs, alphas, wss, cams = raster.inpc_raster_forward_levels(pos, op, feat, wl.cam, 3, flags=flags)
    torch.cuda.synchronize()
    refs = oracle.rasterize_levels(wl.pos, wl.opacity, wl.feat, wl.cam, 3)
    rng = np.random.Generator(np.random.PCG64(77))
    for l in range(3):
        oc = oracle.level_camera(wl.cam, l)
        W, H = cams[l].width, cams[l].height
        assert (W, H) == (oc.width, oc.height) and cams[l].fx == float(oc.fx) and cams[l].cx == float(oc.cx)
        cnt = raster.inpc_raster_get_counts(wss[l], W, H).cpu().numpy().view(np.uint32)
        assert np.array_equal(cnt, refs[l].counts()), f"level {l}: per-pixel counts differ"
        img_r, alpha_r = _reference_with_gpu_counts(refs[l], wss[l], W, H)
        img = imgs[l].cpu().numpy().astype(np.float64)
        if planar:
            assert img.shape == (D, H, W)
            img_cmp = oracle.to_planar(img_r)
        else:
            img_cmp = img_r
        assert np.abs(img - img_cmp).max() <= harness.FWD_ATOL, f"level {l}"
        assert np.abs(alphas[l].cpu().numpy() - alpha_r).max() <= harness.FWD_ATOL
        # backward of this level
        g_img = rng.standard_normal((H, W, D)).astype(np.float32)
        g_alpha = rng.standard_normal((H, W)).astype(np.float32)
        g_dev = _dev(oracle.to_planar(g_img) if planar else g_img)
        out = raster.inpc_raster_backward(pos, op, feat, cams[l], g_dev, _dev(g_alpha), wss[l],
                                          flags=raster.OUT_PLANAR if planar else 0, grad_scale=0.5, blend_weight=True)
        torch.cuda.synchronize()
        assert raster.inpc_raster_get_status(wss[l]) == 0
        rf, ro, ru = refs[l].backward(0.5 * g_img.astype(np.float64), 0.5 * g_alpha.astype(np.float64))
        harness.check_grads(f"level {l} grad_feat", out[0], rf)
        harness.check_grads(f"level {l} grad_opacity", out[1], ro)
        harness.check_grads(f"level {l} grad_uv", out[2], ru)
        assert np.abs(out[3].cpu().numpy() - refs[l].blend_weights()).max() <= harness.BW_ATOL


@pytest.mark.parametrize("planar", [False, True])
def test_multisample_average_of_four_clouds(planar):
    """Inference multisampling: four independently drawn clouds, per-pixel mean, two levels."""
    clouds_np, clouds = [], []
    for s in range(4):
        wl = make_workload("train", n_points=1 << 18, seed=40 + s)
        clouds_np.append((wl.pos, wl.opacity, wl.feat))
        clouds.append((_dev(wl.pos), _dev(wl.opacity), _dev(wl.feat)))
    cam = wl.cam
    imgs, alphas = raster.inpc_raster_forward_multisample(clouds, cam, n_levels=2, flags=raster.OUT_PLANAR if planar else 0)
    torch.cuda.synchronize()
    ref = oracle.multisample(clouds_np, cam, n_levels=2)
    for l in range(2):
        img = imgs[l].cpu().numpy().astype(np.float64)
        img_r = oracle.to_planar(ref[l][0]) if planar else ref[l][0]
        # each cloud's image is within 1e-4 (termination-ambiguous pixels included: one fragment more or less at
        # T ~ 1e-4 moves a pixel by < 1e-4), so is their mean
        assert np.abs(img - img_r).max() <= harness.FWD_ATOL
        assert np.abs(alphas[l].cpu().numpy() - ref[l][1]).max() <= harness.FWD_ATOL
    # bit-reproducible, and equal to accumulating by hand through inpc_raster_forward_ex
    imgs2, alphas2 = raster.inpc_raster_forward_multisample(clouds, cam, n_levels=2, flags=raster.OUT_PLANAR if planar else 0)
    assert torch.equal(imgs[0], imgs2[0]) and torch.equal(alphas[1], alphas2[1])
    fl = raster.OUT_PLANAR if planar else 0
    out_f, out_a, ws = raster.inpc_raster_forward(*clouds[0], cam, flags=fl, out_scale=0.25)
    for c in clouds[1:]:
        raster.inpc_raster_forward(*c, cam, out_feat=out_f, out_alpha=out_a, workspace=ws, flags=fl | raster.ACCUMULATE,
                                   out_scale=0.25)
    assert torch.equal(out_f, imgs[0]) and torch.equal(out_a, alphas[0])


def test_forward_ex_defaults_are_bit_identical_to_forward():
    wl = make_workload("tiny")
    pos, op, feat = _dev(wl.pos), _dev(wl.opacity), _dev(wl.feat)
    a = raster.inpc_raster_forward(pos, op, feat, wl.cam, flags=raster.SAVE_FOR_BACKWARD)
    lib = raster.load()
    img = torch.empty_like(a[0]); alpha = torch.empty_like(a[1])
    cs = raster.camera_struct(wl.cam)
    rc = lib.inpc_raster_forward_ex(pos.data_ptr(), op.data_ptr(), feat.data_ptr(), wl.N, 4, ctypes.byref(cs), img.data_ptr(),
                                    alpha.data_ptr(), a[2].data_ptr(), a[2].numel(), raster.SAVE_FOR_BACKWARD, 1.0, None)
    torch.cuda.synchronize()
    assert rc == 0 and torch.equal(img, a[0]) and torch.equal(alpha, a[1])
    with pytest.raises(raster.InpcError) as e:                  # the plain entry point refuses the layout flags
        lib2 = raster.load()
        rc = lib2.inpc_raster_forward(pos.data_ptr(), op.data_ptr(), feat.data_ptr(), wl.N, 4, ctypes.byref(cs), img.data_ptr(),
                                      alpha.data_ptr(), a[2].data_ptr(), a[2].numel(), raster.OUT_PLANAR, None)
        if rc != 0:
            raise raster.InpcError(rc, "inpc_raster_forward")
    assert e.value.status == -1


# ------------------------------------------------------------------------------ NEXT row f2: fused spherical harmonics

@pytest.mark.parametrize("name,kw,pose", [("tiny", {}, False), ("tiny", {}, True), ("train", {"n_points": 1 << 20}, False)])
def test_fused_sh_forward_and_backward(name, kw, pose):
    """36 SH coefficients per point instead of a feature: forward image / alpha and the gradients
    w.r.t. the coefficients, opacity and screen position against the oracle (numpy SH in fp64 + the plain oracle)."""
    wl = make_workload(name, **kw)
    if pose:
        R, t = second_pose()
        wl.cam = wl.cam.with_pose(R, t)
    W, H, N = wl.cam.width, wl.cam.height, wl.N
    rng = np.random.Generator(np.random.PCG64(123))
    coeff = (rng.standard_normal((N, 36)) * 0.5).astype(np.float32)
    pos, op, cf = _dev(wl.pos), _dev(wl.opacity), _dev(coeff)
    img, alpha, ws = raster.inpc_raster_forward_sh(pos, op, cf, wl.cam, flags=raster.SAVE_FOR_BACKWARD)
    torch.cuda.synchronize()
    feat_r = oracle.sh_features(wl.pos, coeff, wl.cam)
    ref = oracle.Raster.from_points(wl.pos, wl.opacity, feat_r.astype(np.float32), wl.cam)
    cnt = raster.inpc_raster_get_counts(ws, W, H).cpu().numpy().view(np.uint32)
    assert np.array_equal(cnt, ref.counts())
    img_r, alpha_r = _reference_with_gpu_counts(ref, ws, W, H)
    scale = max(1.0, float(np.abs(feat_r).max()))              # the image is linear in the features
    assert np.abs(img.cpu().numpy() - img_r).max() <= harness.FWD_ATOL * scale
    assert np.abs(alpha.cpu().numpy() - alpha_r).max() <= harness.FWD_ATOL
    g_c, g_o, g_uv, bw = raster.inpc_raster_backward_sh(pos, op, cf, wl.cam, _dev(wl.g_img), _dev(wl.g_alpha), ws,
                                                        blend_weight=True)
    torch.cuda.synchronize()
    assert raster.inpc_raster_get_status(ws) == 0
    rf, ro, ru = ref.backward(wl.g_img, wl.g_alpha)
    harness.check_grads("grad_sh_coeff", g_c, oracle.sh_backward(wl.pos, wl.cam, rf))
    # opacity / uv gradients carry the feature magnitude: same relative tolerance, the absolute floor scaled with it
    for name_, got, want in (("grad_opacity", g_o, ro), ("grad_uv", g_uv, ru)):
        got = got.cpu().numpy().astype(np.float64).reshape(want.shape)
        tol = np.maximum(harness.GRAD_RTOL * np.abs(want), harness.GRAD_ATOL * scale)
        assert (np.abs(got - want) <= tol).all(), name_
    assert np.abs(bw.cpu().numpy() - ref.blend_weights()).max() <= harness.BW_ATOL
    # culled points: exact zeros in all 36 coefficient gradients
    dead = ~np.isin(np.arange(N), ref.sorted_fragments()[1])
    if dead.any():
        assert float(g_c.cpu().numpy()[dead].__abs__().max()) == 0.0


# ------------------------------------------------------------------------------ NEXT row f4: view-specific sampler

@pytest.mark.parametrize("n_leaves,N,pose", [(4096, 100_000, False), (1 << 16, 1 << 20, True), (1 << 20, 1 << 22, False)])
def test_view_specific_sampler_is_bit_exact(n_leaves, N, pose):
    """Eq. 4 re-weighting, multinomial with replacement, in-leaf jitter, frustum re-sampling:
    the drawn leaf indices and the fp32 positions against oracle/sampler.py, bit for bit."""
    from oracle import sampler as osampler
    from paper_2403_16862_b200.workloads import make_octree
    centre, level, prob, root = make_octree(n_leaves, seed=21)
    cam = make_workload("tiny").cam.__class__(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840)
    if pose:
        cam = cam.with_pose(*second_pose())
    pos, leaf, ws = raster.inpc_sample_view(_dev(centre), _dev(level), _dev(prob), root, cam, seed=2024, N=N)
    torch.cuda.synchronize()
    rpos, rleaf = osampler.sample_view(centre, level, prob, root, cam, seed=2024, N=N)
    assert np.array_equal(leaf.cpu().numpy(), rleaf), "drawn leaf indices differ"
    assert np.array_equal(pos.cpu().numpy().view(np.uint32)[rleaf >= 0], rpos.view(np.uint32)[rleaf >= 0]), "positions differ"
    assert np.isnan(pos.cpu().numpy()[rleaf < 0]).all()
    st = raster.inpc_sample_get_stats(ws)
    cdf = osampler.integer_cdf(osampler.leaf_weights(centre, level, prob, root, cam))
    assert st["n_valid"] == int((rleaf >= 0).sum()) and st["cdf_total"] == int(cdf[-1])
    assert st["max_weight"] == float(osampler.leaf_weights(centre, level, prob, root, cam).max())
    # the sampled cloud goes straight into the rasterizer: every valid sample lands in the image
    n = min(N, 1 << 20)
    op = torch.full((n,), 0.3, device="cuda"); feat = torch.rand((n, 4), device="cuda")
    _, alpha, rws = raster.inpc_raster_forward(pos[:n].contiguous(), op, feat, cam, flags=0)
    assert raster.inpc_raster_get_stats(rws)["n_kept"] == int((rleaf[:n] >= 0).sum())


def test_sampler_sees_leaves_the_frustum_only_crosses():
    """Leaves with neither centre nor corner inside the frustum (one contains the camera, one is entered through a face,
    large ones around the frustum) and leaf levels outside [0, 30]: same visible set, leaves and positions as the oracle."""
    from oracle import sampler as osampler
    cam = Camera(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840)
    rng = np.random.default_rng(5)
    centre = np.concatenate([[[0, 0, 0], [20, 0, 10], [0, 0, 5], [0, 0, 6]], rng.uniform(-60, 60, (2000, 3))]).astype(np.float32)
    level = np.concatenate([[0, 1, -3, 31], rng.integers(0, 5, 2000)]).astype(np.int32)
    prob = np.ones(len(level), np.float32)
    for c in (cam, cam.with_pose(*second_pose())):
        phat = osampler.leaf_weights(centre, level, prob, 64.0, c)
        if c is cam:
            assert phat[0] > 0 and phat[1] > 0 and phat[2] == 0 and phat[3] == 0
        N = 200_000
        pos, leaf, ws = raster.inpc_sample_view(_dev(centre), _dev(level), _dev(prob), 64.0, c, seed=99, N=N)
        torch.cuda.synchronize()
        rpos, rleaf = osampler.sample_view(centre, level, prob, 64.0, c, seed=99, N=N)
        assert np.array_equal(leaf.cpu().numpy(), rleaf)
        assert np.array_equal(pos.cpu().numpy().view(np.uint32)[rleaf >= 0], rpos.view(np.uint32)[rleaf >= 0])
        st = raster.inpc_sample_get_stats(ws)
        assert st["cdf_total"] == int(osampler.integer_cdf(phat)[-1]) and st["max_weight"] == float(phat.max())
        assert not np.isin(rleaf, [2, 3]).any()


def test_sampler_without_resampling_is_bit_exact():
    """INPC_SAMPLE_NO_RESAMPLE (inference): one draw per sample, against the oracle's attempts = 1."""
    from oracle import sampler as osampler
    from paper_2403_16862_b200.workloads import make_octree
    centre, level, prob, root = make_octree(1 << 14, seed=3)
    cam = Camera(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840).with_pose(*second_pose())
    N = 300_001
    pos, leaf, ws = raster.inpc_sample_view(_dev(centre), _dev(level), _dev(prob), root, cam, seed=77, N=N,
                                            flags=raster.SAMPLE_NO_RESAMPLE)
    torch.cuda.synchronize()
    rpos, rleaf = osampler.sample_view(centre, level, prob, root, cam, seed=77, N=N, attempts=1)
    assert np.array_equal(leaf.cpu().numpy(), rleaf)
    assert np.array_equal(pos.cpu().numpy().view(np.uint32)[rleaf >= 0], rpos.view(np.uint32)[rleaf >= 0])
    assert np.isnan(pos.cpu().numpy()[rleaf < 0]).all() and (rleaf < 0).any()
    assert raster.inpc_sample_get_stats(ws)["n_valid"] == int((rleaf >= 0).sum())
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_sample_view(_dev(centre), _dev(level), _dev(prob), root, cam, seed=77, N=N, flags=2)
    assert e.value.status == -1


def test_sampler_edge_cases():
    from paper_2403_16862_b200.workloads import make_octree
    cam = make_workload("tiny").cam
    centre = torch.tensor([[0.0, 0.0, -5.0]], device="cuda"); level = torch.tensor([8], dtype=torch.int32, device="cuda")
    prob = torch.tensor([1.0], device="cuda")
    pos, leaf, ws = raster.inpc_sample_view(centre, level, prob, 64.0, cam, seed=1, N=100)      # nothing visible
    torch.cuda.synchronize()
    assert (leaf == -1).all() and torch.isnan(pos).all() and raster.inpc_sample_get_stats(ws)["cdf_total"] == 0
    pos, leaf, ws = raster.inpc_sample_view(centre, level, prob, 64.0, cam, seed=1, N=0)        # N = 0
    assert pos.shape == (0, 3)
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_sample_view(centre, level, prob, -1.0, cam, seed=1, N=10)
    assert e.value.status == -1


# ------------------------------------------------------------------------------ API behaviour

def test_forward_is_repeatable_and_workspace_reusable():
    wl = make_workload("tiny")
    st = gpu_forward(wl)
    img0, a0 = st["img"].clone(), st["alpha"].clone()
    for _ in range(3):
        raster.inpc_raster_forward(st["pos"], st["op"], st["feat"], wl.cam, out_feat=st["img"], out_alpha=st["alpha"],
                                   workspace=st["ws"], flags=raster.SAVE_FOR_BACKWARD | raster.SAVE_SORTED)
    torch.cuda.synchronize()
    # no atomics in the value path: results are bit-reproducible run to run
    assert torch.equal(img0, st["img"]) and torch.equal(a0, st["alpha"])
    g1 = gpu_backward(wl, st)
    g2 = gpu_backward(wl, st)
    for a, b in zip(g1, g2):
        assert torch.equal(a, b)


def test_backward_twice_on_split_tiles_and_large_cells():
    """The backward pass walks the blend order the forward pass saved (ord[], one block per tile item) and hands
    k_combine's large units through a device-side queue: both must leave the saved state intact and be re-entrant.
    The reduced stress draw has split tiles, long-run pixels and cells of thousands of points."""
    wl = make_workload("stress", n_points=1 << 18)
    st = gpu_forward(wl, flags=raster.SAVE_FOR_BACKWARD)
    g1 = [g.clone() for g in gpu_backward(wl, st, weights=True)]
    g2 = gpu_backward(wl, st, weights=True)
    for a, b in zip(g1, g2):
        assert torch.equal(a, b)
    # and a second forward into the same workspace reproduces the saved state the backward reads
    raster.inpc_raster_forward(st["pos"], st["op"], st["feat"], wl.cam, out_feat=st["img"], out_alpha=st["alpha"],
                               workspace=st["ws"], flags=raster.SAVE_FOR_BACKWARD)
    g3 = gpu_backward(wl, st, weights=True)
    for a, b in zip(g1, g3):
        assert torch.equal(a, b)


def _carve(nbytes, canary=0xA5, pad=1 << 16):
    """A buffer of nbytes in the middle of a larger canary-filled allocation (256-byte aligned start)."""
    whole = torch.full((nbytes + 2 * pad,), canary, dtype=torch.uint8, device="cuda")
    return whole, whole[pad:pad + nbytes]


def _intact(whole, nbytes, canary=0xA5, pad=1 << 16):
    return bool((whole[:pad] == canary).all()) and bool((whole[pad + nbytes:] == canary).all())


@pytest.mark.parametrize("name,kw", [("tiny", {}), ("tiny", {"D": 8}), ("stress", {"n_points": 1 << 18})])
def test_guard_bands_around_every_buffer(name, kw):
    """Stand-in for compute-sanitizer memcheck (closed on this pool, profiles/r02_sanitizer.md): nothing outside
    the caller's buffers -- and nothing beyond inpc_raster_workspace_bytes -- is written."""
    wl = make_workload(name, **kw)
    N, D, W, H = wl.N, wl.D, wl.cam.width, wl.cam.height
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    pos, op, feat, g_img, g_alpha = t(wl.pos), t(wl.opacity), t(wl.feat), t(wl.g_img), t(wl.g_alpha)
    for flags in (raster.SAVE_FOR_BACKWARD | raster.SAVE_SORTED, raster.SAVE_FOR_BACKWARD, 0):
        sizes = dict(ws=raster.inpc_raster_workspace_bytes(N, D, W, H, flags), img=H * W * D * 4, alpha=H * W * 4,
                     d_feat=N * D * 4, d_op=N * 4, d_uv=N * 8)
        bufs = {k: _carve(v) for k, v in sizes.items()}
        view = lambda k, shape: bufs[k][1].view(torch.float32).view(shape)
        raster.inpc_raster_forward(pos, op, feat, wl.cam, out_feat=view("img", (H, W, D)), out_alpha=view("alpha", (H, W)),
                                   workspace=bufs["ws"][1], flags=flags)
        if flags & raster.SAVE_FOR_BACKWARD:
            raster.inpc_raster_backward(pos, op, feat, wl.cam, g_img, g_alpha, bufs["ws"][1],
                                        grad_feat=view("d_feat", (N, D)), grad_opacity=view("d_op", (N,)),
                                        grad_uv=view("d_uv", (N, 2)))
        torch.cuda.synchronize()
        for k, (whole, _) in bufs.items():
            assert _intact(whole, sizes[k]), f"{k}: bytes outside the buffer were written (flags {flags})"


def test_results_do_not_depend_on_workspace_contents():
    """Stand-in for compute-sanitizer initcheck: whatever the workspace held before the call, the results are
    bit-identical (no read of memory the call itself has not written reaches a result)."""
    wl = make_workload("stress", n_points=1 << 18)
    N, D, W, H = wl.N, wl.D, wl.cam.width, wl.cam.height
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    pos, op, feat, g_img, g_alpha = t(wl.pos), t(wl.opacity), t(wl.feat), t(wl.g_img), t(wl.g_alpha)
    nbytes = raster.inpc_raster_workspace_bytes(N, D, W, H, raster.SAVE_FOR_BACKWARD)
    results = []
    for fill in ("zero", "ff", "random"):
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        if fill == "zero":
            ws.zero_()
        elif fill == "ff":
            ws.fill_(0xFF)
        else:
            ws.copy_(torch.randint(0, 256, (nbytes,), dtype=torch.uint8, device="cuda"))
        img, alpha, _ = raster.inpc_raster_forward(pos, op, feat, wl.cam, workspace=ws, flags=raster.SAVE_FOR_BACKWARD)
        nb = raster.inpc_raster_get_blended_counts(ws, W, H)
        grads = raster.inpc_raster_backward(pos, op, feat, wl.cam, g_img, g_alpha, ws)
        torch.cuda.synchronize()
        results.append((img, alpha, nb) + tuple(grads))
    for other in results[1:]:
        for a, b in zip(results[0], other):
            assert torch.equal(a, b)


def test_null_gradient_outputs_are_skipped():
    """Any of grad_feat / grad_opacity / grad_uv may be NULL: the others come out bit-identical, a buffer that was not
    passed is not touched, and all-NULL is a valid (if pointless) call."""
    wl = make_workload("1m", n_points=1 << 17)
    st = gpu_forward(wl)
    g_img, g_a = torch.from_numpy(wl.g_img).cuda(), torch.from_numpy(wl.g_alpha).cuda()
    full = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"], check=True)
    for skip in range(3):
        kw = {("grad_feat", "grad_opacity", "grad_uv")[skip]: False}
        got = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"], check=True, **kw)
        for k in range(3):
            if k == skip:
                assert got[k] is None
            else:
                assert torch.equal(got[k], full[k])
    only_uv = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"], grad_feat=False,
                                          grad_opacity=False, check=True)
    assert only_uv[0] is None and only_uv[1] is None and torch.equal(only_uv[2], full[2])
    none = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"], grad_feat=False,
                                       grad_opacity=False, grad_uv=False, blend_weight=True, check=True)
    bw = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"], blend_weight=True)[3]
    assert none[:3] == (None, None, None) and torch.equal(none[3], bw)


def test_two_host_threads_on_two_streams():
    """The library keeps one side stream per device and a process-wide mutex around the enqueue of calls that use it
    (deviations).  Two host threads that rasterise different clouds on their own streams at the
    same time must neither deadlock nor disturb each other: every result equals the one the same call gives alone."""
    import threading
    wls = [make_workload("1m", n_points=1 << 17), make_workload("train", n_points=1 << 17)]
    alone = []
    for wl in wls:
        st = gpu_forward(wl, flags=raster.SAVE_FOR_BACKWARD)
        g = gpu_backward(wl, st)
        alone.append((st["img"].clone(), st["alpha"].clone(), [x.clone() for x in g]))
    errors, results = [], [None, None]

    def work(k):
        try:
            wl = wls[k]
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                pos, op, feat = _dev(wl.pos), _dev(wl.opacity), _dev(wl.feat)
                g_img, g_a = _dev(wl.g_img), _dev(wl.g_alpha)
                for _ in range(20):
                    img, alpha, ws = raster.inpc_raster_forward(pos, op, feat, wl.cam, flags=raster.SAVE_FOR_BACKWARD, stream=stream)
                    grads = raster.inpc_raster_backward(pos, op, feat, wl.cam, g_img, g_a, ws, stream=stream)
                stream.synchronize()
                assert raster.inpc_raster_get_status(ws, stream=stream) == 0
                results[k] = (img, alpha, grads)
        except Exception as e:                                   # noqa: BLE001 -- reported by the main thread
            errors.append(e)

    threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
        assert not t.is_alive(), "a rasterising thread did not finish: deadlock on the side stream?"
    assert not errors, errors
    for k in range(2):
        img, alpha, grads = results[k]
        assert torch.equal(img, alone[k][0]) and torch.equal(alpha, alone[k][1])
        for a, b in zip(grads, alone[k][2]):
            assert torch.equal(a, b)


def test_error_codes():
    wl = make_workload("tiny")
    st = gpu_forward(wl, flags=0)
    g = torch.zeros((64, 64, 4), device="cuda")
    with pytest.raises(raster.InpcError) as e:     # a forward without INPC_SAVE_FOR_BACKWARD leaves a smaller workspace
        raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g, None, st["ws"])
    assert e.value.status == -2
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_raster_get_sorted(st["ws"], 64, 64)
    assert e.value.status == -4
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_raster_get_blended_counts(st["ws"], 64, 64)
    assert e.value.status == -4
    # a workspace that is large enough but holds no saving forward: the backward's device-side header check
    # refuses (gradient buffers untouched) and inpc_raster_get_status reports why
    big = raster.alloc_workspace(wl.N, 4, 64, 64, raster.SAVE_FOR_BACKWARD)
    raster.inpc_raster_forward(st["pos"], st["op"], st["feat"], wl.cam, workspace=big, flags=0)
    sentinel = torch.full((wl.N, 4), 7.0, device="cuda")
    raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g, None, big, grad_feat=sentinel)
    assert raster.inpc_raster_get_status(big) == -4
    assert float(sentinel.min()) == 7.0 and float(sentinel.max()) == 7.0
    # ... a saving forward of ANOTHER shape: INVALID_ARG
    raster.inpc_raster_forward(st["pos"][:100], st["op"][:100], st["feat"][:100], wl.cam, workspace=big,
                               flags=raster.SAVE_FOR_BACKWARD)
    raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g, None, big, grad_feat=sentinel)
    assert raster.inpc_raster_get_status(big) == -1
    assert float(sentinel.min()) == 7.0
    # ... never written by any forward (zeroed, then garbage)
    big.zero_()
    raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g, None, big, grad_feat=sentinel)
    assert raster.inpc_raster_get_status(big) == -4 and float(sentinel.min()) == 7.0
    with pytest.raises(raster.InpcError) as e:     # the binding's checked mode reads the device's verdict back and raises
        raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g, None, big, grad_feat=sentinel, check=True)
    assert e.value.status == -4 and float(sentinel.min()) == 7.0
    ok = gpu_forward(wl)                            # ... and stays silent on a matching workspace
    raster.inpc_raster_backward(ok["pos"], ok["op"], ok["feat"], wl.cam, g, None, ok["ws"], check=True)
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_raster_get_counts(big, 64, 64)
    assert e.value.status == -4
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_raster_forward(st["pos"], st["op"], st["feat"], wl.cam, workspace=small)
    assert e.value.status == -2
    feat3 = torch.zeros((wl.N, 3), device="cuda")
    with pytest.raises(ValueError):
        raster.alloc_workspace(wl.N, 3, 64, 64)
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_raster_forward(st["pos"], st["op"], feat3, wl.cam, workspace=st["ws"])
    assert e.value.status == -5


def test_launch_counter_counts_kernels():
    wl = make_workload("tiny")
    before = raster.inpc_raster_launch_count()
    st = gpu_forward(wl, flags=raster.SAVE_FOR_BACKWARD)
    mid = raster.inpc_raster_launch_count()
    gpu_backward(wl, st)
    after = raster.inpc_raster_launch_count()
    assert mid - before >= 5 and after - mid >= 1


def test_workspace_may_be_copied_between_forward_and_backward():
    """The state lives in the workspace, not in the library (include/inpc_raster.h): a bitwise copy of the
    workspace at another address serves the backward pass and the introspection calls."""
    wl = make_workload("tiny")
    st = gpu_forward(wl, flags=raster.SAVE_FOR_BACKWARD)
    g1 = gpu_backward(wl, st)
    moved = dict(st)
    moved["ws"] = st["ws"].clone()
    st["ws"].zero_()
    g2 = gpu_backward(wl, moved)
    for a, b in zip(g1, g2):
        assert torch.equal(a, b)
    assert raster.inpc_raster_get_stats(moved["ws"])["n_points"] == wl.N


def test_raw_ctypes_forward_backward_without_the_binding():
    """Drive the C ABI directly (no raster.py): the binding adds nothing but marshalling."""
    wl = make_workload("tiny")
    lib = ctypes.CDLL(raster.LIB_PATH)
    vp, i64, i32, u32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_uint32
    lib.inpc_raster_workspace_bytes.restype = ctypes.c_size_t
    lib.inpc_raster_workspace_bytes.argtypes = [i64, i32, i32, i32, u32]
    lib.inpc_raster_forward.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp, vp, ctypes.c_size_t, u32, vp]
    lib.inpc_raster_backward.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, ctypes.c_size_t, vp]
    cam = (ctypes.c_float * 18)(64, 64, 32, 32, 1, 0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0, 0.01, 100.0)
    cam_bytes = bytes(cam) + (ctypes.c_int32 * 2)(64, 64)
    cam_buf = ctypes.create_string_buffer(bytes(cam_bytes), len(cam_bytes))
    N, D, W, H = wl.N, 4, 64, 64
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    pos, op, feat, g_img, g_alpha = t(wl.pos), t(wl.opacity), t(wl.feat), t(wl.g_img), t(wl.g_alpha)
    nbytes = lib.inpc_raster_workspace_bytes(N, D, W, H, 1)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    img = torch.empty((H, W, D), device="cuda"); alpha = torch.empty((H, W), device="cuda")
    d_feat = torch.empty((N, D), device="cuda"); d_op = torch.empty((N,), device="cuda"); d_uv = torch.empty((N, 2), device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    p = lambda x: ctypes.c_void_p(x.data_ptr())
    assert lib.inpc_raster_forward(p(pos), p(op), p(feat), N, D, ctypes.cast(cam_buf, vp), p(img), p(alpha), p(ws), nbytes,
                                   1, ctypes.c_void_p(stream)) == 0
    assert lib.inpc_raster_backward(p(pos), p(op), p(feat), N, D, ctypes.cast(cam_buf, vp), p(g_img), p(g_alpha), p(d_feat),
                                    p(d_op), p(d_uv), p(ws), nbytes, ctypes.c_void_p(stream)) == 0
    torch.cuda.synchronize()
    ref = oracle.Raster.from_points(wl.pos, wl.opacity, wl.feat, wl.cam)
    img_r, alpha_r, _, margin = ref.blend()
    assert (margin >= harness.MARGIN).all(), "tiny has no termination-ambiguous pixel at this seed"
    harness.check_image(dict(img=img, alpha=alpha), img_r, alpha_r, "raw ctypes")
    rf, ro, ru = ref.backward(wl.g_img, wl.g_alpha)
    harness.check_grads("grad_feat", d_feat, rf); harness.check_grads("grad_opacity", d_op, ro)
    harness.check_grads("grad_uv", d_uv, ru)


def test_zz_bench_kernels_are_the_parity_tested_ones():
    """Every kernel template instantiation bench.py launches (its fwd+bwd step and its forward-only figure, for
    D = 4 and D = 8, tile path and long-run path) must be one that full_parity compared with the oracle."""
    harness.PARITY_KERNELS.clear()
    wls = [make_workload("tiny"), make_workload("tiny", D=8), make_workload("stress", n_points=1 << 18),
           make_workload("infer", n_points=1 << 16)]
    for wl in wls:
        full_parity(wl)
    tested = set(harness.PARITY_KERNELS)
    raster.inpc_raster_launched_kernels(reset=True)
    for wl in wls:                                          # bench.py's own step functions, same flags
        fwd, bwd, _ = bench.make_step_functions(raster, wl, torch.device("cuda"))
        fwd(bench.FLAGS_STEP); bwd(); fwd(bench.FLAGS_FWD)
    torch.cuda.synchronize()
    launched = raster.inpc_raster_launched_kernels()
    assert {"k_blend<4,1,0>", "k_blend<4,0,0>", "k_blend<8,1,0>", "k_blend<8,0,0>", "k_big<4,0>", "k_big<4,2>", "k_back<4>", "k_back<8>"} <= launched
    assert launched <= tested, f"bench.py launches kernels no parity test ran: {sorted(launched - tested)}"
