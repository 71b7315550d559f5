"""ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle/oracle.cpp header).

ctypes wrapper around the plain fp64 CPU implementation in oracle/oracle.cpp.  Imported only by
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg.  Nothing in
paper_2403_16862_b200 (the product) imports this package, and this package imports nothing from
the product except nothing at all: inputs arrive as numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB_OMP = os.path.join(_HERE, "liboracle_omp.so")
_lib = None

T_MIN = 1e-4   # transmittance cut-off (BASELINE.json north_star; not in the paper)
NO_FORCE = 0xFFFFFFFF   # force_nb value meaning "use the termination test"


def build(force: bool = False, openmp: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (the canonical fp32 projection must not be contracted to FMA).
    openmp=True builds the SAME source a second time with -fopenmp (liboracle_omp.so): only bench.py's
    all-cores baseline leg uses it (use_openmp); every test runs the single-threaded build."""
    lib = _LIB_OMP if openmp else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c++17"] +
                              (["-fopenmp"] if openmp else []) + ["-shared", "-fPIC", "-o", lib, _SRC])
    return lib


def use_openmp(on: bool) -> int:
    """Switch this process to the -fopenmp build (bench.py only) or back; returns the threads it will use."""
    global _lib
    _lib = None
    _load(openmp=on)
    return int(_lib.oracle_threads())


class _Camera(C.Structure):
    _fields_ = [("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("near_z", C.c_float), ("far_z", C.c_float),
                ("width", C.c_int32), ("height", C.c_int32)]


def _load(openmp: bool = False):
    global _lib
    if _lib is None:
        lib = C.CDLL(build(openmp=openmp))
        lib.oracle_threads.restype = C.c_int
        lib.oracle_create.restype = C.c_void_p
        lib.oracle_create.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p]
        lib.oracle_create_uv.restype = C.c_void_p
        lib.oracle_create_uv.argtypes = [C.c_void_p] * 5 + [C.c_int64, C.c_int32, C.c_int32, C.c_int32]
        lib.oracle_free.argtypes = [C.c_void_p]
        for name in ("oracle_total", "oracle_kept", "oracle_border_dropped"):
            getattr(lib, name).restype = C.c_int64
            getattr(lib, name).argtypes = [C.c_void_p]
        lib.oracle_counts.argtypes = [C.c_void_p, C.c_void_p]
        lib.oracle_sorted.argtypes = [C.c_void_p] * 5
        lib.oracle_blend.argtypes = [C.c_void_p, C.c_double] + [C.c_void_p] * 5
        lib.oracle_sorted_T.restype = C.c_int
        lib.oracle_sorted_T.argtypes = [C.c_void_p, C.c_void_p]
        lib.oracle_blend_weights.restype = C.c_int
        lib.oracle_blend_weights.argtypes = [C.c_void_p, C.c_void_p]
        lib.oracle_backward.restype = C.c_int
        lib.oracle_backward.argtypes = [C.c_void_p] * 6
        lib.oracle_count_fp64_projection_changes.restype = C.c_int64
        lib.oracle_count_fp64_projection_changes.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        _lib = lib
    return _lib


def _cam_struct(cam) -> _Camera:
    c = _Camera()
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    R = np.asarray(cam.R, dtype=np.float32).reshape(9)
    t = np.asarray(cam.t, dtype=np.float32).reshape(3)
    for i in range(9):
        c.R[i] = float(R[i])
    for i in range(3):
        c.t[i] = float(t[i])
    c.near_z, c.far_z = float(cam.near_z), float(cam.far_z)
    c.width, c.height = int(cam.width), int(cam.height)
    return c


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class Raster:
    """One rasterisation problem held by the oracle: buckets built and sorted at construction."""

    def __init__(self, handle, N, D, W, H):
        self._h, self.N, self.D, self.W, self.H = handle, N, D, W, H
        self.P = W * H

    @classmethod
    def from_points(cls, pos, opacity, feat, cam) -> "Raster":
        lib = _load()
        pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
        opacity = np.ascontiguousarray(opacity, dtype=np.float32).reshape(-1)
        feat = np.ascontiguousarray(feat, dtype=np.float32)
        N, D = pos.shape[0], (feat.shape[1] if feat.ndim == 2 else 0)
        assert opacity.shape[0] == N and feat.shape[0] == N
        cs = _cam_struct(cam)
        h = lib.oracle_create(_p(pos), _p(opacity), _p(feat), N, D, C.byref(cs))
        return cls(h, N, D, int(cam.width), int(cam.height))

    @classmethod
    def from_uv(cls, u, v, depth, opacity, feat, W, H) -> "Raster":
        lib = _load()
        u = np.ascontiguousarray(u, dtype=np.float64)
        v = np.ascontiguousarray(v, dtype=np.float64)
        depth = np.ascontiguousarray(depth, dtype=np.float32)
        opacity = np.ascontiguousarray(opacity, dtype=np.float32)
        feat = np.ascontiguousarray(feat, dtype=np.float32)
        N, D = u.shape[0], feat.shape[1]
        h = lib.oracle_create_uv(_p(u), _p(v), _p(depth), _p(opacity), _p(feat), N, D, int(W), int(H))
        return cls(h, N, D, int(W), int(H))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.oracle_free(self._h)
            self._h = None

    @property
    def total(self) -> int:
        return int(_lib.oracle_total(self._h))

    @property
    def kept(self) -> int:
        return int(_lib.oracle_kept(self._h))

    @property
    def border_dropped(self) -> int:
        return int(_lib.oracle_border_dropped(self._h))

    def counts(self) -> np.ndarray:
        c = np.empty(self.P, dtype=np.uint32)
        _lib.oracle_counts(self._h, _p(c))
        return c.reshape(self.H, self.W)

    def sorted_fragments(self):
        """offsets[P+1], point_idx[total], depth_bits[total], weight[total] in pixel-major sorted order."""
        tot = self.total
        off = np.empty(self.P + 1, dtype=np.int64)
        idx = np.empty(tot, dtype=np.int64)
        dep = np.empty(tot, dtype=np.uint32)
        w = np.empty(tot, dtype=np.float64)
        _lib.oracle_sorted(self._h, _p(off), _p(idx), _p(dep), _p(w))
        return off, idx, dep, w

    def blend(self, t_min: float = T_MIN, force_nb=None):
        """-> img[H,W,D] f64, alpha[H,W] f64, nb[H,W] u32, margin[H,W] f64.
        force_nb[H,W] u32 (harness aid): where it is not NO_FORCE the pixel blends exactly that many fragments."""
        img = np.empty((self.H, self.W, self.D), dtype=np.float64)
        alpha = np.empty((self.H, self.W), dtype=np.float64)
        nb = np.empty((self.H, self.W), dtype=np.uint32)
        margin = np.empty((self.H, self.W), dtype=np.float64)
        if force_nb is not None:
            force_nb = np.ascontiguousarray(force_nb, dtype=np.uint32).reshape(self.H, self.W)
        _lib.oracle_blend(self._h, float(t_min), None if force_nb is None else _p(force_nb),
                          _p(img), _p(alpha), _p(nb), _p(margin))
        return img, alpha, nb, margin

    def sorted_T(self) -> np.ndarray:
        """Per fragment (order of sorted_fragments): the transmittance in front of it if the last blend()
        composited it, -1 otherwise."""
        T = np.empty(self.total, dtype=np.float64)
        if _lib.oracle_sorted_T(self._h, _p(T)) != 0:
            raise RuntimeError("oracle_sorted_T: blend() has not been called")
        return T

    def blend_weights(self) -> np.ndarray:
        """Per-point blending weight b = max over the point's blended fragments of alpha T (Eq. 3's input); call
        blend() first.  -> [N] f64."""
        bw = np.empty(self.N, dtype=np.float64)
        if _lib.oracle_blend_weights(self._h, _p(bw)) != 0:
            raise RuntimeError("oracle_blend_weights: blend() has not been called")
        return bw

    def backward(self, g_img, g_alpha=None):
        """Gradients of <g_img, img> + <g_alpha, alpha>; call blend() first (same t_min).
        -> d_feat[N,D], d_opacity[N], d_uv[N,2], all f64."""
        g_img = np.ascontiguousarray(g_img, dtype=np.float64).reshape(self.H, self.W, self.D)
        ga = None if g_alpha is None else np.ascontiguousarray(g_alpha, dtype=np.float64).reshape(self.H, self.W)
        d_feat = np.empty((self.N, self.D), dtype=np.float64)
        d_op = np.empty(self.N, dtype=np.float64)
        d_uv = np.empty((self.N, 2), dtype=np.float64)
        rc = _lib.oracle_backward(self._h, _p(g_img), None if ga is None else _p(ga),
                                  _p(d_feat), _p(d_op), _p(d_uv))
        if rc != 0:
            raise RuntimeError("oracle_backward: blend() has not been called")
        return d_feat, d_op, d_uv


def fp64_projection_changes(pos, cam) -> int:
    lib = _load()
    pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
    cs = _cam_struct(cam)
    return int(lib.oracle_count_fp64_projection_changes(_p(pos), pos.shape[0], C.byref(cs)))


# ---------------------------------------------------------------------------------------------------
# NEXT row f3 -- the paper's call pattern, as plain compositions of the oracle above (test infrastructure):
# several resolution levels of one cloud, the per-pixel average of several clouds
# ("multisampling"), and the [D,H,W] layout the CNN reads.

class _LevelCamera:
    pass


def level_camera(cam, level: int):
    """Camera of resolution level l: the image halved l times.  width_l = ceil(width / 2^l), likewise height;
    fx, fy, cx, cy times 2^-l (a power of two: exact in fp32), so (u, v) becomes (u, v) / 2^l and pixel centres stay
    at (i + 0.5, j + 0.5).  Reading: the paper only says "progressively lower resolution"; halving
    matches the 2x average pooling between the U-Net's levels."""
    c = _LevelCamera()
    s = np.float32(1.0) / np.float32(2 ** level)
    c.fx, c.fy = np.float32(cam.fx) * s, np.float32(cam.fy) * s
    c.cx, c.cy = np.float32(cam.cx) * s, np.float32(cam.cy) * s
    c.R, c.t, c.near_z, c.far_z = cam.R, cam.t, cam.near_z, cam.far_z
    c.width = -(-int(cam.width) // 2 ** level)
    c.height = -(-int(cam.height) // 2 ** level)
    return c


def rasterize_levels(pos, opacity, feat, cam, n_levels: int):
    """-> [Raster of level 0, ..., Raster of level n_levels - 1]."""
    return [Raster.from_points(pos, opacity, feat, level_camera(cam, l)) for l in range(n_levels)]


def multisample(clouds, cam, n_levels: int = 1):
    """clouds: list of (pos, opacity, feat).  -> per level (img[H,W,D], alpha[H,W]): the plain per-pixel mean of the
    clouds' images ("rasterize multiple point clouds ... and average the results")."""
    out = []
    for l in range(n_levels):
        cl = level_camera(cam, l)
        imgs, alphas = [], []
        for pos, op, feat in clouds:
            img, alpha, _, _ = Raster.from_points(pos, op, feat, cl).blend()
            imgs.append(img); alphas.append(alpha)
        out.append((np.mean(imgs, axis=0), np.mean(alphas, axis=0)))
    return out


def to_planar(img):
    """[H,W,D] -> [D,H,W]."""
    return np.ascontiguousarray(np.transpose(img, (2, 0, 1)))


# ---------------------------------------------------------------------------------------------------
# NEXT row f2 -- view-dependent features from spherical harmonics (SH of degree 2, 4-D output,
# M = 36 coefficients per point; "fused into this pipeline").  Plain numpy, fp64.

SH_C0 = 0.28209479177387814      # 1 / (2 sqrt(pi))
SH_C1 = 0.4886025119029199       # sqrt(3 / (4 pi))
SH_C2 = (1.0925484305920792,     # sqrt(15 / (4 pi))
         0.31539156525252005,    # sqrt(5 / (16 pi))
         0.5462742152960396)     # sqrt(15 / (16 pi))


def sh_basis(d):
    """Real SH basis of degree 0..2 at unit directions d[...,3] -> [...,9], in the order (l, m) = (0,0), (1,-1), (1,0),
    (1,1), (2,-2), (2,-1), (2,0), (2,1), (2,2), with the Condon-Shortley phase (-1)^m (reading R18: the paper names no
    convention; this is the one of the common graphics code bases).  Pinned against scipy.special in the tests."""
    d = np.asarray(d, dtype=np.float64)
    x, y, z = d[..., 0], d[..., 1], d[..., 2]
    return np.stack([np.full_like(x, SH_C0), -SH_C1 * y, SH_C1 * z, -SH_C1 * x,
                     SH_C2[0] * x * y, -SH_C2[0] * y * z, SH_C2[1] * (2 * z * z - x * x - y * y),
                     -SH_C2[0] * x * z, SH_C2[2] * (x * x - y * y)], axis=-1)


def view_directions(pos, cam):
    """Unit vectors from the camera centre (-R^T t) to the points (zero vector for a point on the centre)."""
    R = np.asarray(cam.R, dtype=np.float64).reshape(3, 3)
    t = np.asarray(cam.t, dtype=np.float64).reshape(3)
    v = np.asarray(pos, dtype=np.float64).reshape(-1, 3) - (-R.T @ t)
    n = np.linalg.norm(v, axis=1, keepdims=True)
    return np.divide(v, n, out=np.zeros_like(v), where=n > 0)


def sh_features(pos, coeff, cam):
    """coeff[N,36] (basis-major: coefficient 4 b + d belongs to basis b, channel d) -> feat[N,4] f64."""
    Y = sh_basis(view_directions(pos, cam))                                   # [N,9]
    Y = np.where(np.linalg.norm(view_directions(pos, cam), axis=1, keepdims=True) > 0, Y, np.array([SH_C0] + [0.0] * 8))
    c = np.asarray(coeff, dtype=np.float64).reshape(-1, 9, 4)
    return np.einsum("nb,nbd->nd", Y, c)


def sh_backward(pos, cam, d_feat):
    """dL/dcoeff[N,36] = Y_b dL/dfeat[d] (the feature is linear in the coefficients)."""
    dirs = view_directions(pos, cam)
    Y = sh_basis(dirs)
    Y = np.where(np.linalg.norm(dirs, axis=1, keepdims=True) > 0, Y, np.array([SH_C0] + [0.0] * 8))
    return np.einsum("nb,nd->nbd", Y, np.asarray(d_feat, dtype=np.float64)).reshape(-1, 36)
