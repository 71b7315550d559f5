"""Seeded synthetic inputs for the INPC bilinear point rasterizer (BASELINE.json `configs`).

This module is the ONLY code shared by the oracle side (`oracle/`, tests) and the CUDA side
(`bench.py`, GPU tests).  It holds none of the method's arithmetic (no rasterizer projection, no
bilinear weights, no sorting, no blending): it only draws point clouds, cameras and output
gradients.  The recipe is the one SURVEY.md section 8(d) makes concrete and DESIGN.md section 4 repeats.

The inputs are synthetic stand-ins for the paper's real-scene workloads (public
benchmarks that are not in the container): they take the workload's *shape* -- sampled points in
the view frustum, unordered multinomial sampler output, near/far
0.01/100, 4-D features, opacities in [0,1].

Everything is numpy, `Generator(PCG64(seed))`, returned as contiguous float32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np


@dataclass
class Camera:
    """Pinhole camera. Pixel (i, j) has its centre at (i+0.5, j+0.5); +z forward, +y down.

    p_c = R p_w + t (R row-major 3x3).  near/far follow PAPER.md:310 (0.01 / 100)."""
    fx: float
    fy: float
    cx: float
    cy: float
    width: int
    height: int
    R: np.ndarray = field(default_factory=lambda: np.eye(3, dtype=np.float32))
    t: np.ndarray = field(default_factory=lambda: np.zeros(3, dtype=np.float32))
    near_z: float = 0.01
    far_z: float = 100.0

    def with_pose(self, R, t) -> "Camera":
        return Camera(self.fx, self.fy, self.cx, self.cy, self.width, self.height,
                      np.ascontiguousarray(R, dtype=np.float32).reshape(3, 3),
                      np.ascontiguousarray(t, dtype=np.float32).reshape(3),
                      self.near_z, self.far_z)


@dataclass
class Workload:
    name: str
    pos: np.ndarray        # [N,3] f32 world positions
    opacity: np.ndarray    # [N]   f32 in [0,1]
    feat: np.ndarray       # [N,D] f32
    cam: Camera
    g_img: np.ndarray      # [H,W,D] f32  dL/d(feature image)
    g_alpha: np.ndarray    # [H,W]   f32  dL/d(alpha)
    backward: bool
    seed: int

    @property
    def N(self) -> int:
        return int(self.pos.shape[0])

    @property
    def D(self) -> int:
        return int(self.feat.shape[1])


CAM_TINY = dict(fx=64.0, fy=64.0, cx=32.0, cy=32.0, width=64, height=64)
CAM_1297 = dict(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840)
CAM_1080 = dict(fx=1628.0, fy=1628.0, cx=960.0, cy=540.0, width=1920, height=1080)

# name -> (N, camera, D, backward?, seed, position sampler)
CONFIGS = {
    "tiny":   dict(N=4096,    cam=CAM_TINY, D=4, backward=True,  seed=0, sampler="box"),
    "1m":     dict(N=1 << 20, cam=CAM_1297, D=4, backward=True,  seed=1, sampler="surface"),
    "train":  dict(N=1 << 23, cam=CAM_1297, D=4, backward=True,  seed=2, sampler="octree"),
    "infer":  dict(N=1 << 25, cam=CAM_1080, D=8, backward=False, seed=3, sampler="octree"),
    "stress": dict(N=1 << 24, cam=CAM_1297, D=4, backward=True,  seed=4, sampler="clusters"),
}

_PLANES = (  # (depth on the optical axis, un-normalised normal)
    (2.0, (0.3, 0.0, -1.0)),
    (6.0, (-0.2, 0.4, -1.0)),
    (15.0, (0.0, -0.3, -1.0)),
)


def _pixel_rays(rng, n, cam, lo=0.0, hi=1.0):
    """Ray directions (x/z, y/z, 1) through n uniformly drawn image positions."""
    u = rng.uniform(lo * cam["width"], hi * cam["width"], n)
    v = rng.uniform(lo * cam["height"], hi * cam["height"], n)
    return np.stack([(u - cam["cx"]) / cam["fx"], (v - cam["cy"]) / cam["fy"], np.ones(n)], axis=1)


def _inside(p, cam, zlo, zhi):
    z = p[:, 2]
    with np.errstate(divide="ignore", invalid="ignore"):
        u = cam["fx"] * p[:, 0] / z + cam["cx"]
        v = cam["fy"] * p[:, 1] / z + cam["cy"]
    return (z >= zlo) & (z <= zhi) & (u >= 0) & (u <= cam["width"]) & (v >= 0) & (v <= cam["height"])


def _surface_once(rng, n, cam):
    """25 % on each of three tilted planes (noisy), 25 % background shell.  No rejection here."""
    which = rng.integers(0, 4, n)
    d = _pixel_rays(rng, n, cam)
    p = np.empty((n, 3))
    noise = rng.standard_normal(n)
    zshell = rng.uniform(30.0, 50.0, n)
    for k, (depth, nrm) in enumerate(_PLANES):
        nrm = np.asarray(nrm, dtype=np.float64)
        nrm = nrm / np.linalg.norm(nrm)
        m = which == k
        t = (nrm[2] * depth) / (d[m] @ nrm)          # ray/plane intersection, plane through (0,0,depth)
        q = d[m] * t[:, None]
        q = q + nrm[None, :] * (noise[m] * 0.01 * q[:, 2])[:, None]
        p[m] = q
    m = which == 3
    p[m] = d[m] * zshell[m][:, None]
    return p


def _rejection(draw, rng, n, cam, zlo, zhi):
    out = np.empty((n, 3))
    filled = 0
    while filled < n:
        need = n - filled
        cand = draw(rng, int(need * 1.15) + 64, cam)
        cand = cand[_inside(cand, cam, zlo, zhi)][:need]
        out[filled:filled + len(cand)] = cand
        filled += len(cand)
    return out


def sample_box(rng, n, cam):
    return np.stack([rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(2, 6, n)], axis=1)


def sample_surface(rng, n, cam):
    return _rejection(_surface_once, rng, n, cam, 0.5, 50.0)


def sample_octree(rng, n, cam, n_leaves=1 << 20):
    """Synthetic stand-in for the paper's view-specific octree sampler:
    leaves of levels 4..12 of the root cube [-32,32]^2 x [0,64] placed on the surface generator,
    leaf probability proportional to 1/volume, multinomial with replacement (inverse CDF),
    uniform jitter inside the leaf, out-of-frustum samples re-drawn."""
    n_leaves = min(n_leaves, max(16, n))
    s = _rejection(_surface_once, rng, n_leaves, cam, 0.5, 50.0)
    level = rng.integers(4, 13, n_leaves)
    side = 64.0 / np.exp2(level)
    origin = np.array([-32.0, -32.0, 0.0])
    centre = (np.floor((s - origin) / side[:, None]) + 0.5) * side[:, None] + origin
    cdf = np.cumsum(np.power(8.0, level - 12.0))
    cdf /= cdf[-1]

    def draw(rng_, m, cam_):
        leaf = np.minimum(np.searchsorted(cdf, rng_.uniform(0, 1, m), side="right"), n_leaves - 1)
        return centre[leaf] + rng_.uniform(-0.5, 0.5, (m, 3)) * side[leaf][:, None]

    return _rejection(draw, rng, n, cam, 0.5, 50.0)


def sample_clusters(rng, n, cam, n_clusters=64, sigma=0.02):
    """90 %: tight isotropic Gaussian clusters (depth complexity 0 .. >10k per pixel); 10 % uniform.
    Cluster tails that leave the frustum are NOT re-drawn (exercises culling)."""
    n_cl = (n * 9) // 10
    zc = rng.uniform(1.0, 10.0, n_clusters)
    mean = _pixel_rays(rng, n_clusters, cam, 0.1, 0.9) * zc[:, None]
    which = rng.integers(0, n_clusters, n_cl)
    p_cl = mean[which] + sigma * rng.standard_normal((n_cl, 3))
    n_bg = n - n_cl
    p_bg = _pixel_rays(rng, n_bg, cam) * rng.uniform(0.5, 50.0, n_bg)[:, None]
    p = np.concatenate([p_cl, p_bg], axis=0)
    return p[rng.permutation(n)]


_SAMPLERS = dict(box=sample_box, surface=sample_surface, octree=sample_octree, clusters=sample_clusters)


def second_pose():
    """A non-identity pose (about 20 degrees about y, plus a translation) used for parity only."""
    a = np.deg2rad(20.0)
    R = np.array([[np.cos(a), 0.0, np.sin(a)], [0.0, 1.0, 0.0], [-np.sin(a), 0.0, np.cos(a)]])
    t = np.array([0.3, -0.1, 0.5])
    return R.astype(np.float32), t.astype(np.float32)


def make_workload(name: str, n_points: int | None = None, seed: int | None = None,
                  D: int | None = None, grads: bool = True) -> Workload:
    """Build one of the five configs.  `n_points` overrides N (same sampler and camera: a smaller
    or larger draw from the same distribution), `seed` and `D` likewise."""
    cfg = CONFIGS[name]
    n = int(cfg["N"] if n_points is None else n_points)
    seed = int(cfg["seed"] if seed is None else seed)
    D = int(cfg["D"] if D is None else D)
    camd = cfg["cam"]
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = _SAMPLERS[cfg["sampler"]](rng, n, camd)
    opacity = 1.0 / (1.0 + np.exp(-rng.normal(0.0, 1.5, n)))      # sigmoid(N(0, 1.5))
    feat = rng.uniform(0.0, 1.0, (n, D))
    H, W = camd["height"], camd["width"]
    if grads:
        g_img = rng.standard_normal((H, W, D)).astype(np.float32)
        g_alpha = rng.standard_normal((H, W)).astype(np.float32)
    else:
        g_img = np.zeros((0, 0, D), dtype=np.float32)
        g_alpha = np.zeros((0, 0), dtype=np.float32)
    cam = Camera(**camd)
    return Workload(name=name,
                    pos=np.ascontiguousarray(pos, dtype=np.float32),
                    opacity=np.ascontiguousarray(opacity, dtype=np.float32),
                    feat=np.ascontiguousarray(feat, dtype=np.float32),
                    cam=cam, g_img=g_img, g_alpha=g_alpha,
                    backward=bool(cfg["backward"]), seed=seed)


def leaf_coherent_order(wl: Workload, bits: int = 10) -> Workload:
    """The same cloud with its points stored in a leaf-coherent order (the secondary measurement; the
    headline is the unordered multinomial sampler output): a stable sort by the 3-D Morton code of the
    position on the 2^bits grid of the octree's root cube [-32,32]^2 x [0,64] -- points of one leaf become contiguous,
    leaves follow a z-order curve.  Only the storage order changes; no value does."""
    q = np.clip(((wl.pos.astype(np.float64) - np.array([-32.0, -32.0, 0.0])) / 64.0 * (1 << bits)).astype(np.int64), 0, (1 << bits) - 1)
    code = np.zeros(wl.N, dtype=np.int64)
    for b in range(bits):
        for a in range(3):
            code |= ((q[:, a] >> b) & 1) << (3 * b + a)
    order = np.argsort(code, kind="stable")
    return Workload(name=wl.name + "+leaf-coherent", pos=np.ascontiguousarray(wl.pos[order]),
                    opacity=np.ascontiguousarray(wl.opacity[order]), feat=np.ascontiguousarray(wl.feat[order]),
                    cam=wl.cam, g_img=wl.g_img, g_alpha=wl.g_alpha, backward=wl.backward, seed=wl.seed)


def make_octree(n_leaves: int = 1 << 16, seed: int = 7, cam: dict = CAM_1297, root_side: float = 64.0):
    """Synthetic probability octree for the view-specific sampler (NEXT row f4; PAPER.md:62-84 describes the real
    one, which needs the optimisation loop): leaves of levels 4..12 of the root cube [-32,32]^2 x [0,64] placed on
    the surface generator (so most are in front of the camera), a tenth of them mirrored behind the camera or pushed
    out of the frustum (to exercise the visibility indicator), probabilities U[0.02, 1].
    -> (centre[L,3] f32, level[L] i32, prob[L] f32, root_side)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    s = _rejection(_surface_once, rng, n_leaves, cam, 0.5, 50.0)
    out = rng.uniform(0, 1, n_leaves) < 0.1
    s[out, 2] *= np.where(rng.uniform(0, 1, out.sum()) < 0.5, -1.0, 1.0)      # behind the camera ...
    s[out, 0] += np.where(s[out, 2] > 0, 40.0, 0.0)                            # ... or far off to the side
    level = rng.integers(4, 13, n_leaves)
    side = root_side / np.exp2(level)
    origin = np.array([-root_side / 2, -root_side / 2, 0.0])
    centre = (np.floor((s - origin) / side[:, None]) + 0.5) * side[:, None] + origin
    prob = rng.uniform(0.02, 1.0, n_leaves)
    return (np.ascontiguousarray(centre, dtype=np.float32), np.ascontiguousarray(level, dtype=np.int32),
            np.ascontiguousarray(prob, dtype=np.float32), float(root_side))
