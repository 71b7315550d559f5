"""Thin ctypes binding over the C ABI in include/inpc_raster.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libinpc_raster.so is missing (run
`python -m paper_2403_16862_b200.build` or `__graft_entry__.build()`), loading raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libinpc_raster.so")

SAVE_FOR_BACKWARD = 1
SAVE_SORTED = 2
OUT_PLANAR = 4          # _ex / _levels / _multisample entry points: feature image as [D][H][W]
ACCUMULATE = 8          # _ex: add to the image already in the output buffers
FUSED_SH = 16           # workspace sizing of the _sh entry points
SAMPLE_NO_RESAMPLE = 1  # inpc_sample_view_ex: one draw per sample (inference mode)
SH_COEFFS = 36          # M: 9 basis functions x 4 channels, basis-major

EXPORTS = (
    "inpc_raster_workspace_bytes", "inpc_raster_forward", "inpc_raster_backward", "inpc_raster_backward_weights",
    "inpc_raster_forward_ex", "inpc_raster_backward_ex", "inpc_raster_level_camera", "inpc_raster_forward_levels",
    "inpc_raster_forward_multisample", "inpc_raster_forward_sh", "inpc_raster_backward_sh",
    "inpc_sample_workspace_bytes", "inpc_sample_view", "inpc_sample_get_stats",
    "inpc_sample_static_max_leaves", "inpc_sample_view_static", "inpc_sample_view_ex",
    "inpc_raster_get_counts", "inpc_raster_get_blended_counts", "inpc_raster_get_sorted", "inpc_raster_get_stats",
    "inpc_raster_get_status",
    "inpc_raster_strerror", "inpc_raster_last_cuda_error", "inpc_raster_launch_count", "inpc_raster_launched_kernels",
    "inpc_raster_set_kernel_timing", "inpc_raster_kernel_count", "inpc_raster_kernel_name",
    "inpc_raster_get_kernel_times",
)


class InpcCamera(C.Structure):
    _fields_ = [("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("near_z", C.c_float), ("far_z", C.c_float),
                ("width", C.c_int32), ("height", C.c_int32)]


class InpcStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("n_points", "n_kept", "n_fragments", "n_tile_items",
                                          "n_big_pixels", "n_big_fragments", "n_big_cells")]


class InpcError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = load()
        msg = lib.inpc_raster_strerror(status).decode()
        if status == -3:
            msg += ": " + lib.inpc_raster_last_cuda_error().decode()
        super().__init__(f"{where} failed ({status}): {msg}")
        self.status = status


_lib = None


def load() -> C.CDLL:
    """dlopen libinpc_raster.so; raises (loudly) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: the CUDA library has not been built "
                              "(python -m paper_2403_16862_b200.build); there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        vp, i64, i32, u32 = C.c_void_p, C.c_int64, C.c_int32, C.c_uint32
        lib.inpc_raster_workspace_bytes.restype = C.c_size_t
        lib.inpc_raster_workspace_bytes.argtypes = [i64, i32, i32, i32, u32]
        lib.inpc_raster_forward.restype = C.c_int
        lib.inpc_raster_forward.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), vp, vp, vp, C.c_size_t, u32, vp]
        lib.inpc_raster_backward.restype = C.c_int
        lib.inpc_raster_backward.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
        lib.inpc_raster_forward_ex.restype = C.c_int
        lib.inpc_raster_forward_ex.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), vp, vp, vp, C.c_size_t, u32, C.c_float, vp]
        lib.inpc_raster_backward_ex.restype = C.c_int
        lib.inpc_raster_backward_ex.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), vp, vp, vp, vp, vp, vp, vp, C.c_size_t, u32, C.c_float, vp]
        lib.inpc_raster_forward_sh.restype = C.c_int
        lib.inpc_raster_forward_sh.argtypes = [vp, vp, vp, i64, C.POINTER(InpcCamera), vp, vp, vp, C.c_size_t, u32, C.c_float, vp]
        lib.inpc_raster_backward_sh.restype = C.c_int
        lib.inpc_raster_backward_sh.argtypes = [vp, vp, vp, i64, C.POINTER(InpcCamera), vp, vp, vp, vp, vp, vp, vp, C.c_size_t, u32, C.c_float, vp]
        lib.inpc_sample_workspace_bytes.restype = C.c_size_t
        lib.inpc_sample_workspace_bytes.argtypes = [i64]
        lib.inpc_sample_view.restype = C.c_int
        lib.inpc_sample_view.argtypes = [vp, vp, vp, i64, C.c_float, C.POINTER(InpcCamera), C.c_uint64, i64, vp, vp, vp, C.c_size_t, vp]
        lib.inpc_sample_static_max_leaves.restype = C.c_int64
        lib.inpc_sample_static_max_leaves.argtypes = []
        lib.inpc_sample_view_static.restype = C.c_int
        lib.inpc_sample_view_static.argtypes = [vp, vp, vp, i64, C.c_float, C.POINTER(InpcCamera), C.c_uint64, i64, vp, vp, vp]
        lib.inpc_sample_view_ex.restype = C.c_int
        lib.inpc_sample_view_ex.argtypes = [vp, vp, vp, i64, C.c_float, C.POINTER(InpcCamera), C.c_uint64, i64, vp, vp, vp, C.c_size_t, u32, vp]
        lib.inpc_sample_get_stats.restype = C.c_int
        lib.inpc_sample_get_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_double), vp]
        lib.inpc_raster_level_camera.restype = C.c_int
        lib.inpc_raster_level_camera.argtypes = [C.POINTER(InpcCamera), i32, C.POINTER(InpcCamera)]
        lib.inpc_raster_forward_levels.restype = C.c_int
        lib.inpc_raster_forward_levels.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), i32, C.POINTER(vp), C.POINTER(vp),
                                                   C.POINTER(vp), C.POINTER(C.c_size_t), u32, C.c_float, vp]
        lib.inpc_raster_forward_multisample.restype = C.c_int
        lib.inpc_raster_forward_multisample.argtypes = [i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(i64), i32,
                                                        C.POINTER(InpcCamera), i32, C.POINTER(vp), C.POINTER(vp), vp, C.c_size_t, u32, vp]
        lib.inpc_raster_backward_weights.restype = C.c_int
        lib.inpc_raster_backward_weights.argtypes = [vp, vp, vp, i64, i32, C.POINTER(InpcCamera), vp, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
        lib.inpc_raster_get_counts.restype = C.c_int
        lib.inpc_raster_get_counts.argtypes = [vp, i32, i32, vp, vp]
        lib.inpc_raster_get_blended_counts.restype = C.c_int
        lib.inpc_raster_get_blended_counts.argtypes = [vp, i32, i32, vp, vp]
        lib.inpc_raster_get_status.restype = C.c_int
        lib.inpc_raster_get_status.argtypes = [vp, vp]
        lib.inpc_raster_get_sorted.restype = C.c_int
        lib.inpc_raster_get_sorted.argtypes = [vp, i32, i32, vp, vp, vp, vp, C.POINTER(C.c_uint64), vp]
        lib.inpc_raster_get_stats.restype = C.c_int
        lib.inpc_raster_get_stats.argtypes = [vp, C.POINTER(InpcStats), vp]
        lib.inpc_raster_strerror.restype = C.c_char_p
        lib.inpc_raster_strerror.argtypes = [C.c_int]
        lib.inpc_raster_last_cuda_error.restype = C.c_char_p
        lib.inpc_raster_launch_count.restype = C.c_uint64
        lib.inpc_raster_launched_kernels.restype = C.c_size_t
        lib.inpc_raster_launched_kernels.argtypes = [C.c_char_p, C.c_size_t, C.c_int]
        lib.inpc_raster_set_kernel_timing.argtypes = [C.c_int]
        lib.inpc_raster_kernel_name.restype = C.c_char_p
        lib.inpc_raster_kernel_name.argtypes = [C.c_int]
        lib.inpc_raster_get_kernel_times.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.c_int]
        _lib = lib
    return _lib


def camera_struct(cam) -> InpcCamera:
    """cam: any object with fx, fy, cx, cy, R (3x3), t (3), near_z, far_z, width, height."""
    c = InpcCamera()
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    R = [float(x) for row in cam.R for x in (row if hasattr(row, "__len__") else [row])]
    t = [float(x) for x in cam.t]
    for i in range(9):
        c.R[i] = R[i]
    for i in range(3):
        c.t[i] = t[i]
    c.near_z, c.far_z = float(cam.near_z), float(cam.far_z)
    c.width, c.height = int(cam.width), int(cam.height)
    return c


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check(t, dtype, name):
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise ValueError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")


def inpc_raster_workspace_bytes(N: int, D: int, W: int, H: int, flags: int = SAVE_FOR_BACKWARD) -> int:
    return int(load().inpc_raster_workspace_bytes(N, D, W, H, flags))


def alloc_workspace(N: int, D: int, W: int, H: int, flags: int = SAVE_FOR_BACKWARD, device="cuda") -> torch.Tensor:
    nbytes = inpc_raster_workspace_bytes(N, D, W, H, flags)
    if nbytes == 0:
        raise ValueError("unsupported problem size / D")
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def _img_shape(H, W, D, flags):
    return (D, H, W) if flags & OUT_PLANAR else (H, W, D)


def inpc_raster_level_camera(cam, level: int) -> InpcCamera:
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    out = InpcCamera()
    rc = load().inpc_raster_level_camera(C.byref(cs), level, C.byref(out))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_level_camera")
    return out


def _ptr_array(tensors):
    return (C.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


def inpc_raster_forward_levels(pos, opacity, feat, cam, n_levels: int, flags: int = SAVE_FOR_BACKWARD, out_scale: float = 1.0,
                               stream=None, outs=None):
    """One cloud at n_levels resolution levels -> (list of out_feat, list of out_alpha, list of workspaces, list of
    level cameras)."""
    lib = load()
    _check(pos, torch.float32, "pos"); _check(opacity, torch.float32, "opacity"); _check(feat, torch.float32, "feat")
    N, D = int(pos.shape[0]), int(feat.shape[1])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    cams = [inpc_raster_level_camera(cs, l) for l in range(n_levels)]
    dev = pos.device
    if outs is not None:                        # (imgs, alphas, workspaces) of an earlier call: nothing is allocated
        imgs, alphas, wss = outs
    else:
        imgs = [torch.empty(_img_shape(c.height, c.width, D, flags), dtype=torch.float32, device=dev) for c in cams]
        alphas = [torch.empty((c.height, c.width), dtype=torch.float32, device=dev) for c in cams]
        wss = [alloc_workspace(N, D, c.width, c.height, flags & 3, dev) for c in cams]
    sizes = (C.c_size_t * n_levels)(*[w.numel() for w in wss])
    rc = lib.inpc_raster_forward_levels(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), n_levels, _ptr_array(imgs),
                                        _ptr_array(alphas), _ptr_array(wss), sizes, flags, out_scale, _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_forward_levels")
    return imgs, alphas, wss, cams


def inpc_raster_forward_multisample(clouds, cam, n_levels: int = 1, flags: int = 0, stream=None, outs=None, workspace=None):
    """clouds: list of (pos, opacity, feat) device tensors.  -> (list of averaged out_feat per level, list of alpha)."""
    lib = load()
    D = int(clouds[0][2].shape[1])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    cams = [inpc_raster_level_camera(cs, l) for l in range(n_levels)]
    dev = clouds[0][0].device
    if outs is not None:
        imgs, alphas = outs
    else:
        imgs = [torch.empty(_img_shape(c.height, c.width, D, flags), dtype=torch.float32, device=dev) for c in cams]
        alphas = [torch.empty((c.height, c.width), dtype=torch.float32, device=dev) for c in cams]
    Ns = [int(c[0].shape[0]) for c in clouds]
    ws = workspace if workspace is not None else alloc_workspace(max(Ns), D, cs.width, cs.height, 0, dev)
    S = len(clouds)
    rc = lib.inpc_raster_forward_multisample(S, _ptr_array([c[0] for c in clouds]), _ptr_array([c[1] for c in clouds]),
                                             _ptr_array([c[2] for c in clouds]), (C.c_int64 * S)(*Ns), D, C.byref(cs),
                                             n_levels, _ptr_array(imgs), _ptr_array(alphas), _ptr(ws), ws.numel(), flags,
                                             _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_forward_multisample")
    return imgs, alphas


def inpc_sample_view(leaf_centre, leaf_level, leaf_prob, root_side: float, cam, seed: int, N: int, workspace=None, stream=None,
                     flags: int = 0):
    """View-specific sampling (Eq. 4): -> (pos[N,3] float32, leaf[N] int32, workspace).  No sync.
    flags = SAMPLE_NO_RESAMPLE: one draw per sample (inpc_sample_view_ex)."""
    lib = load()
    _check(leaf_centre, torch.float32, "leaf_centre"); _check(leaf_level, torch.int32, "leaf_level")
    _check(leaf_prob, torch.float32, "leaf_prob")
    L = int(leaf_level.shape[0])
    dev = leaf_centre.device
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    if workspace is None:
        workspace = torch.empty(int(lib.inpc_sample_workspace_bytes(L)), dtype=torch.uint8, device=dev)
    pos = torch.empty((N, 3), dtype=torch.float32, device=dev)
    leaf = torch.empty((N,), dtype=torch.int32, device=dev)
    if flags:
        rc = lib.inpc_sample_view_ex(_ptr(leaf_centre), _ptr(leaf_level), _ptr(leaf_prob), L, float(root_side), C.byref(cs),
                                     C.c_uint64(seed), N, _ptr(pos), _ptr(leaf), _ptr(workspace), workspace.numel(), flags,
                                     _stream(stream))
    else:
        rc = lib.inpc_sample_view(_ptr(leaf_centre), _ptr(leaf_level), _ptr(leaf_prob), L, float(root_side), C.byref(cs),
                                  C.c_uint64(seed), N, _ptr(pos), _ptr(leaf), _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_sample_view")
    return pos, leaf, workspace


def inpc_sample_static_max_leaves() -> int:
    return int(load().inpc_sample_static_max_leaves())


def inpc_sample_view_static(leaf_centre, leaf_level, leaf_prob, root_side: float, cam, seed: int, N: int, pos=None, leaf=None,
                            stream=None):
    """inpc_sample_view without a workspace, for callers that cannot allocate device memory (a plugin under a host
    application's memory pool, a frame loop that may not touch cudaMalloc): the scratch is a fixed 4.25 MiB array inside
    the library, good for up to inpc_sample_static_max_leaves() = 2^18 leaves (InpcError -6 beyond that).  Pass
    pre-allocated pos[N,3] float32 / leaf[N] int32 and the call allocates nothing at all; without them this wrapper
    makes the two output tensors (the C entry point never does).  All calls on a device share the one array: keep them
    on one stream, or otherwise ordered -- two that overlap on the GPU corrupt each other.  The first call on a device
    looks up the array's address; make it before any stream capture.  -> (pos, leaf).  No sync."""
    lib = load()
    _check(leaf_centre, torch.float32, "leaf_centre"); _check(leaf_level, torch.int32, "leaf_level")
    _check(leaf_prob, torch.float32, "leaf_prob")
    dev = leaf_centre.device
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    if pos is None:
        pos = torch.empty((N, 3), dtype=torch.float32, device=dev)
    if leaf is None:
        leaf = torch.empty((N,), dtype=torch.int32, device=dev)
    _check(pos, torch.float32, "pos"); _check(leaf, torch.int32, "leaf")
    if pos.numel() != 3 * N or leaf.numel() != N:
        raise ValueError("pos must hold N x 3 and leaf N elements")
    rc = lib.inpc_sample_view_static(_ptr(leaf_centre), _ptr(leaf_level), _ptr(leaf_prob), int(leaf_level.shape[0]),
                                     float(root_side), C.byref(cs), C.c_uint64(seed), N, _ptr(pos), _ptr(leaf), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_sample_view_static")
    return pos, leaf


def inpc_sample_get_stats(workspace, stream=None) -> dict:
    nv, tot, mx = C.c_uint64(0), C.c_uint64(0), C.c_double(0.0)
    rc = load().inpc_sample_get_stats(_ptr(workspace), C.byref(nv), C.byref(tot), C.byref(mx), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_sample_get_stats")
    return {"n_valid": int(nv.value), "cdf_total": int(tot.value), "max_weight": float(mx.value)}


def inpc_raster_forward_sh(pos, opacity, sh_coeff, cam, flags: int = SAVE_FOR_BACKWARD, out_scale: float = 1.0, stream=None,
                           out_feat=None, out_alpha=None, workspace=None):
    """Forward with the SH evaluation fused in: sh_coeff[N,36] instead of feat.  -> (out_feat, out_alpha, workspace);
    the three are allocated here unless passed in."""
    lib = load()
    _check(pos, torch.float32, "pos"); _check(opacity, torch.float32, "opacity"); _check(sh_coeff, torch.float32, "sh_coeff")
    N = int(pos.shape[0])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    W, H = cs.width, cs.height
    ws = workspace if workspace is not None else alloc_workspace(N, 4, W, H, (flags & 3) | FUSED_SH, pos.device)
    if out_feat is None:
        out_feat = torch.empty(_img_shape(H, W, 4, flags), dtype=torch.float32, device=pos.device)
    if out_alpha is None:
        out_alpha = torch.empty((H, W), dtype=torch.float32, device=pos.device)
    rc = lib.inpc_raster_forward_sh(_ptr(pos), _ptr(opacity), _ptr(sh_coeff), N, C.byref(cs), _ptr(out_feat), _ptr(out_alpha),
                                    _ptr(ws), ws.numel(), flags, out_scale, _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_forward_sh")
    return out_feat, out_alpha, ws


def _raise_on_device_status(workspace, stream, where: str):
    """The backward pass validates the workspace ON THE DEVICE (does it hold the forward these arguments describe?); on
    a mismatch its kernels do nothing and leave the gradient buffers untouched.  check=True reads that verdict back
    (inpc_raster_get_status; synchronises the stream) and raises instead of returning uninitialised gradients."""
    st = inpc_raster_get_status(workspace, stream)
    if st != 0:
        raise InpcError(st, where + " (device-side workspace check)")


def inpc_raster_backward_sh(pos, opacity, sh_coeff, cam, grad_out_feat, grad_out_alpha, workspace, flags: int = 0,
                            grad_scale: float = 1.0, blend_weight: bool = False, stream=None, check: bool = False,
                            grads=None):
    """-> (grad_sh_coeff[N,36], grad_opacity[N], grad_uv[N,2][, blend_weight[N]]).  check=True: see inpc_raster_backward."""
    lib = load()
    N = int(pos.shape[0])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    dev = pos.device
    if grads is not None:                       # (grad_sh_coeff, grad_opacity, grad_uv) of the caller
        g_c, g_o, g_uv = grads
    else:
        g_c = torch.empty((N, SH_COEFFS), dtype=torch.float32, device=dev)
        g_o = torch.empty((N,), dtype=torch.float32, device=dev)
        g_uv = torch.empty((N, 2), dtype=torch.float32, device=dev)
    bw = torch.empty((N,), dtype=torch.float32, device=dev) if blend_weight else None
    rc = lib.inpc_raster_backward_sh(_ptr(pos), _ptr(opacity), _ptr(sh_coeff), N, C.byref(cs), _ptr(grad_out_feat),
                                     _ptr(grad_out_alpha), _ptr(g_c), _ptr(g_o), _ptr(g_uv), _ptr(bw), _ptr(workspace),
                                     workspace.numel(), flags, grad_scale, _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_backward_sh")
    if check:
        _raise_on_device_status(workspace, stream, "inpc_raster_backward_sh")
    return (g_c, g_o, g_uv) + ((bw,) if blend_weight else ())


def inpc_raster_forward(pos, opacity, feat, cam, out_feat=None, out_alpha=None, workspace=None,
                        flags: int = SAVE_FOR_BACKWARD, stream=None, out_scale: float = 1.0):
    """-> (out_feat[H,W,D] ([D,H,W] with OUT_PLANAR), out_alpha[H,W], workspace).  Enqueues on the current stream;
    no sync.  OUT_PLANAR / ACCUMULATE / out_scale != 1 go through inpc_raster_forward_ex."""
    lib = load()
    _check(pos, torch.float32, "pos"); _check(opacity, torch.float32, "opacity"); _check(feat, torch.float32, "feat")
    N, D = int(pos.shape[0]), int(feat.shape[1])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    W, H = cs.width, cs.height
    if workspace is None:
        workspace = alloc_workspace(N, D, W, H, flags & 3, pos.device)
    if out_feat is None:
        out_feat = torch.empty(_img_shape(H, W, D, flags), dtype=torch.float32, device=pos.device)
    if out_alpha is None:
        out_alpha = torch.empty((H, W), dtype=torch.float32, device=pos.device)
    if (flags & ~3) or out_scale != 1.0:
        rc = lib.inpc_raster_forward_ex(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), _ptr(out_feat),
                                        _ptr(out_alpha), _ptr(workspace), workspace.numel(), flags, out_scale, _stream(stream))
    else:
        rc = lib.inpc_raster_forward(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), _ptr(out_feat),
                                     _ptr(out_alpha), _ptr(workspace), workspace.numel(), flags, _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_forward")
    return out_feat, out_alpha, workspace


def inpc_raster_backward(pos, opacity, feat, cam, grad_out_feat, grad_out_alpha, workspace,
                         grad_feat=None, grad_opacity=None, grad_uv=None, stream=None, blend_weight=None,
                         flags: int = 0, grad_scale: float = 1.0, check: bool = False):
    """-> (grad_feat[N,D], grad_opacity[N], grad_uv[N,2]).  Enqueues on the current stream; no sync.
    With blend_weight (True, or a float32 tensor [N]) the fused per-point blending weights (Eq. 3) come back
    as a fourth result (inpc_raster_backward_weights).
    check=True synchronises and raises InpcError when the device-side check found that `workspace` does not hold the
    forward pass these arguments describe (the host call returns INPC_OK in that case and the gradients are left as
    they were); the default stays asynchronous -- query inpc_raster_get_status yourself."""
    lib = load()
    N, D = int(pos.shape[0]), int(feat.shape[1])
    cs = cam if isinstance(cam, InpcCamera) else camera_struct(cam)
    _check(grad_out_feat, torch.float32, "grad_out_feat")
    if grad_out_alpha is not None:
        _check(grad_out_alpha, torch.float32, "grad_out_alpha")
    dev = pos.device
    # None = allocate it; False = "not wanted": NULL goes to the library, which skips that gradient's stores
    if grad_feat is None:
        grad_feat = torch.empty((N, D), dtype=torch.float32, device=dev)
    if grad_opacity is None:
        grad_opacity = torch.empty((N,), dtype=torch.float32, device=dev)
    if grad_uv is None:
        grad_uv = torch.empty((N, 2), dtype=torch.float32, device=dev)
    grad_feat = None if grad_feat is False else grad_feat
    grad_opacity = None if grad_opacity is False else grad_opacity
    grad_uv = None if grad_uv is False else grad_uv
    if blend_weight is True:
        blend_weight = torch.empty((N,), dtype=torch.float32, device=dev)
    elif blend_weight is False:
        blend_weight = None
    if flags or grad_scale != 1.0:
        rc = lib.inpc_raster_backward_ex(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), _ptr(grad_out_feat),
                                         _ptr(grad_out_alpha), _ptr(grad_feat), _ptr(grad_opacity), _ptr(grad_uv),
                                         _ptr(blend_weight), _ptr(workspace), workspace.numel(), flags, grad_scale,
                                         _stream(stream))
        if rc != 0:
            raise InpcError(rc, "inpc_raster_backward_ex")
        if check:
            _raise_on_device_status(workspace, stream, "inpc_raster_backward_ex")
        return (grad_feat, grad_opacity, grad_uv) + ((blend_weight,) if blend_weight is not None else ())
    if blend_weight is not None:
        rc = lib.inpc_raster_backward_weights(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), _ptr(grad_out_feat),
                                              _ptr(grad_out_alpha), _ptr(grad_feat), _ptr(grad_opacity), _ptr(grad_uv),
                                              _ptr(blend_weight), _ptr(workspace), workspace.numel(), _stream(stream))
        if rc != 0:
            raise InpcError(rc, "inpc_raster_backward_weights")
        if check:
            _raise_on_device_status(workspace, stream, "inpc_raster_backward_weights")
        return grad_feat, grad_opacity, grad_uv, blend_weight
    rc = lib.inpc_raster_backward(_ptr(pos), _ptr(opacity), _ptr(feat), N, D, C.byref(cs), _ptr(grad_out_feat),
                                  _ptr(grad_out_alpha), _ptr(grad_feat), _ptr(grad_opacity), _ptr(grad_uv),
                                  _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_backward")
    if check:
        _raise_on_device_status(workspace, stream, "inpc_raster_backward")
    return grad_feat, grad_opacity, grad_uv


def inpc_raster_get_counts(workspace, W: int, H: int, stream=None) -> torch.Tensor:
    counts = torch.empty((H, W), dtype=torch.int32, device=workspace.device)
    rc = load().inpc_raster_get_counts(_ptr(workspace), W, H, _ptr(counts), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_counts")
    return counts


def inpc_raster_get_blended_counts(workspace, W: int, H: int, stream=None) -> torch.Tensor:
    nb = torch.empty((H, W), dtype=torch.int32, device=workspace.device)
    rc = load().inpc_raster_get_blended_counts(_ptr(workspace), W, H, _ptr(nb), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_blended_counts")
    return nb


def inpc_raster_get_status(workspace, stream=None) -> int:
    """Sticky status of the device-side checks (0 = ok); synchronises."""
    return int(load().inpc_raster_get_status(_ptr(workspace), _stream(stream)))


def inpc_raster_get_sorted(workspace, W: int, H: int, stream=None, transmittance: bool = False):
    """-> offsets[H*W+1], point_idx[total], depth_bits[total] (int32 tensors holding the u32 bit patterns)
    [, transmittance[total] float32 when asked for]."""
    lib = load()
    total = C.c_uint64(0)
    rc = lib.inpc_raster_get_sorted(_ptr(workspace), W, H, None, None, None, None, C.byref(total), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_sorted")
    n = int(total.value)
    dev = workspace.device
    offsets = torch.empty(W * H + 1, dtype=torch.int32, device=dev)
    idx = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    depth = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    tr = torch.empty(max(n, 1), dtype=torch.float32, device=dev) if transmittance else None
    rc = lib.inpc_raster_get_sorted(_ptr(workspace), W, H, _ptr(offsets), _ptr(idx), _ptr(depth), _ptr(tr),
                                    C.byref(total), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_sorted")
    return (offsets, idx[:n], depth[:n], tr[:n]) if transmittance else (offsets, idx[:n], depth[:n])


def inpc_raster_get_stats(workspace, stream=None) -> dict:
    st = InpcStats()
    rc = load().inpc_raster_get_stats(_ptr(workspace), C.byref(st), _stream(stream))
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_stats")
    return {n: int(getattr(st, n)) for n, _ in InpcStats._fields_}


def inpc_raster_launch_count() -> int:
    return int(load().inpc_raster_launch_count())


def inpc_raster_launched_kernels(reset: bool = False) -> set:
    """Distinct kernel template instantiations launched by this process since the last reset."""
    lib = load()
    n = lib.inpc_raster_launched_kernels(None, 0, 0)
    buf = C.create_string_buffer(int(n) + 1)
    lib.inpc_raster_launched_kernels(buf, len(buf), 1 if reset else 0)
    return {k for k in buf.value.decode().split(";") if k}


def inpc_raster_set_kernel_timing(enable: bool) -> None:
    load().inpc_raster_set_kernel_timing(1 if enable else 0)


def inpc_raster_get_kernel_times(reset: bool = True) -> dict:
    """-> {stage name: (summed device ms, timed launches)} since the last reset (waits for the events)."""
    lib = load()
    n = lib.inpc_raster_kernel_count()
    ms = (C.c_double * n)()
    cnt = (C.c_uint64 * n)()
    rc = lib.inpc_raster_get_kernel_times(ms, cnt, 1 if reset else 0)
    if rc != 0:
        raise InpcError(rc, "inpc_raster_get_kernel_times")
    return {lib.inpc_raster_kernel_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(n)}
