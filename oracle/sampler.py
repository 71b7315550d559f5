"""ORACLE -- TEST INFRASTRUCTURE ONLY.  NEXT row f4: viewpoint-specific sampling of the implicit point cloud
(Sec. 3.2 Eq. 4; Eq. 9; re-sampling PAPER.md:322), plain numpy, step by step in
the paper's order.  It shares no code with paper_2403_16862_b200/csrc/sampler.cuh; both follow the arithmetic that
DESIGN.md section 3 (reading R19) fixes so that the drawn leaves and positions are reproducible bit for bit:

  1. per leaf: z_view by the canonical fp32 projection; visible <=> the leaf's cube can intersect the frustum: centre or
     one of the 8 corners inside it, or no frustum plane with all 8 corners on its outer side (box_outside_a_plane);
     d = max(|z_view - near| / (far - near), 1e-8) (Eq. 9) and p^ = p / (d * 2^(level / 2)) (Eq. 4, lambda_l = 0.5)
     in fp64, one rounded operation per step;
  2. integer weights w = floor(p^ / max p^ * 2^32), inclusive prefix sums in u64 = the CDF;
  3. sample j, attempt a: four SplitMix64 numbers with counters ((j * 8 + a) * 4 + k); k = 0 picks the leaf,
     r = floor(rng * total / 2^64), leaf = first i with CDF_i > r; k = 1..3 give u = top 24 bits * 2^-24 and the
     position c + (u - 0.5) * side in fp32; the first attempt (of 8) inside the frustum is kept, else NaN / -1.
"""
from __future__ import annotations

import numpy as np

ATTEMPTS = 8
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)


def splitmix64(seed, counter):
    """Counter-based SplitMix64: mix(seed + (counter + 1) * golden gamma); numpy uint64 arithmetic wraps mod 2^64."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (np.asarray(counter, dtype=np.uint64) + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def _mulhi64(a, b):
    """floor(a * b / 2^64) for uint64 arrays, by 32-bit limbs."""
    a = np.asarray(a, dtype=np.uint64); b = np.asarray(b, dtype=np.uint64)
    m = np.uint64(0xFFFFFFFF); s = np.uint64(32)
    al, ah, bl, bh = a & m, a >> s, b & m, b >> s
    with np.errstate(over="ignore"):
        ll, lh, hl, hh = al * bl, al * bh, ah * bl, ah * bh
        mid = (ll >> s) + (lh & m) + (hl & m)
        return hh + (lh >> s) + (hl >> s) + (mid >> s)


def _project32(cam, p):
    """Canonical fp32 projection (the rasterizer's S1): -> zc, u, v as float32 arrays (each operation rounded)."""
    f = np.float32
    R = np.asarray(cam.R, dtype=np.float32).reshape(9); t = np.asarray(cam.t, dtype=np.float32).reshape(3)
    x, y, z = p[:, 0].astype(f), p[:, 1].astype(f), p[:, 2].astype(f)
    xc = ((R[0] * x + R[1] * y) + R[2] * z) + t[0]
    yc = ((R[3] * x + R[4] * y) + R[5] * z) + t[1]
    zc = ((R[6] * x + R[7] * y) + R[8] * z) + t[2]
    with np.errstate(divide="ignore", invalid="ignore"):
        u = (f(cam.fx) * xc) / zc + f(cam.cx)
        v = (f(cam.fy) * yc) / zc + f(cam.cy)
    return zc, u, v


def inside_frustum(cam, p):
    zc, u, v = _project32(cam, np.asarray(p, dtype=np.float32).reshape(-1, 3))
    with np.errstate(invalid="ignore"):
        return (zc > np.float32(cam.near_z)) & (zc < np.float32(cam.far_z)) & (u >= 0) & (u < np.float32(cam.width)) & \
               (v >= 0) & (v < np.float32(cam.height)), zc


MAX_LEVEL = 30      # a leaf_level outside [0, 30] never gets a sample (2^-level must be a normal fp32; the paper stops at 8)


def box_outside_a_plane(cam, corners):
    """corners[8][L,3] float32 (world).  True where ONE of the six frustum planes has all eight corners on its outer
    side -- then the cube cannot meet the frustum (PAPER.md:92 property (1): such a leaf must get no samples).  The
    planes in camera space, fp32, one rounded operation at a time: near z_c > near, far z_c < far, and the four side
    planes through the camera centre in the division-free form of 0 <= u < W, 0 <= v < H:
        fx x_c + cx z_c >= 0,  fx x_c + (cx - W) z_c < 0,  fy y_c + cy z_c >= 0,  fy y_c + (cy - H) z_c < 0.
    A corner is outside a plane when the inequality is NOT satisfied (so NaN is outside of everything)."""
    f = np.float32
    R = np.asarray(cam.R, dtype=np.float32).reshape(9); t = np.asarray(cam.t, dtype=np.float32).reshape(3)
    all_out = None
    for p in corners:
        x, y, z = p[:, 0].astype(f), p[:, 1].astype(f), p[:, 2].astype(f)
        with np.errstate(invalid="ignore", over="ignore"):
            xc = ((R[0] * x + R[1] * y) + R[2] * z) + t[0]
            yc = ((R[3] * x + R[4] * y) + R[5] * z) + t[1]
            zc = ((R[6] * x + R[7] * y) + R[8] * z) + t[2]
            fxx, fyy = f(cam.fx) * xc, f(cam.fy) * yc
            inside = np.stack([zc > f(cam.near_z), zc < f(cam.far_z),
                               fxx + f(cam.cx) * zc >= 0, fxx + (f(cam.cx) - f(cam.width)) * zc < 0,
                               fyy + f(cam.cy) * zc >= 0, fyy + (f(cam.cy) - f(cam.height)) * zc < 0], 1)
        all_out = ~inside if all_out is None else (all_out & ~inside)
    return all_out.any(axis=1)


def leaf_weights(centre, level, prob, root_side, cam):
    """Eq. 4 / Eq. 9 -> p^[L] in fp64 (0 for invisible leaves)."""
    centre = np.asarray(centre, dtype=np.float32).reshape(-1, 3)
    level = np.asarray(level, dtype=np.int64)
    level_ok = (level >= 0) & (level <= MAX_LEVEL)
    level = np.where(level_ok, level, 0)
    half = np.float32(0.5) * (np.float32(root_side) * np.exp2(-level).astype(np.float32))
    vis, zc = inside_frustum(cam, centre)
    corners = []
    for k in range(8):
        off = np.stack([np.where(k & 1, half, -half), np.where(k & 2, half, -half), np.where(k & 4, half, -half)], 1)
        corners.append(centre + off.astype(np.float32))
        vis = vis | inside_frustum(cam, corners[-1])[0]
    vis = (vis | ~box_outside_a_plane(cam, corners)) & level_ok
    near, far = np.float64(np.float32(cam.near_z)), np.float64(np.float32(cam.far_z))
    d = np.maximum(np.abs(zc.astype(np.float64) - near) / (far - near), 1e-8)              # Eq. 9
    f = np.ldexp(np.where(level & 1, 1.4142135623730951, 1.0), level >> 1)                 # 2^(level * 0.5)
    with np.errstate(invalid="ignore", divide="ignore"):
        p = np.asarray(prob, dtype=np.float32).astype(np.float64) / (d * f)                # Eq. 4
    p = np.where(vis & (p > 0) & np.isfinite(p), p, 0.0)
    return p


def integer_cdf(phat):
    m = phat.max() if len(phat) else 0.0
    if not m > 0:
        return np.zeros(len(phat), dtype=np.uint64)
    w = np.floor((phat / m) * 4294967296.0).astype(np.uint64)
    return np.cumsum(w, dtype=np.uint64)


def sample_view(centre, level, prob, root_side, cam, seed: int, N: int, attempts: int = ATTEMPTS):
    """-> pos[N,3] float32 (NaN where all attempts failed), leaf[N] int32 (-1 there).
    attempts = 1 is the inference mode of PAPER.md:322 ("omit resampling"): one draw, outside the frustum -> NaN."""
    centre = np.asarray(centre, dtype=np.float32).reshape(-1, 3)
    level = np.asarray(level, dtype=np.int64)
    cdf = integer_cdf(leaf_weights(centre, level, prob, root_side, cam))
    total = cdf[-1] if len(cdf) else np.uint64(0)
    pos = np.full((N, 3), np.nan, dtype=np.float32)
    leaf = np.full(N, -1, dtype=np.int32)
    if total == 0:
        return pos, leaf
    todo = np.arange(N, dtype=np.uint64)
    for a in range(attempts):
        if len(todo) == 0:
            break
        c0 = (todo * np.uint64(ATTEMPTS) + np.uint64(a)) * np.uint64(4)
        r = _mulhi64(splitmix64(seed, c0), np.full(len(todo), total, dtype=np.uint64))
        i = np.searchsorted(cdf, r, side="right")                                          # first i with cdf[i] > r
        side = np.float32(root_side) * np.exp2(-level[i]).astype(np.float32)
        q = np.empty((len(todo), 3), dtype=np.float32)
        for k in range(3):
            u = (splitmix64(seed, c0 + np.uint64(1 + k)) >> np.uint64(40)).astype(np.float32) * np.float32(2.0 ** -24)
            q[:, k] = centre[i, k] + (u - np.float32(0.5)) * side
        ok = inside_frustum(cam, q)[0]
        j = todo[ok].astype(np.int64)
        pos[j] = q[ok]
        leaf[j] = i[ok].astype(np.int32)
        todo = todo[~ok]
    return pos, leaf
