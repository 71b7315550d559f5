"""Parity harness: run the CUDA path (through the C-ABI binding) and the oracle on the same seeded
inputs and compare them element by element (BASELINE.json north_star tolerances).

  counts, sorted (pixel, depth_bits, point_idx) lists : bit-exact
  feature image, alpha                                 : max abs error <= 1e-4
  gradients                                            : |gpu - ref| <= max(1e-3 |ref|, 1e-5)

Termination-ambiguous pixels (reading R7): the cut-off `T >= 1e-4` is decided in
fp32 on the GPU (the kernel's precision) and in fp64 by the oracle; where some transmittance the test
looked at lies within MARGIN (relative) of 1e-4 the two may legitimately blend one fragment more or
less.  Such pixels are accepted if they match the oracle re-run with the cut-off moved just below /
just above the ambiguous value; the points with a fragment in such a pixel are left out of the
gradient comparison.  Their number is reported and bounded.
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2403_16862_b200 import raster

FWD_ATOL = 1e-4
GRAD_RTOL = 1e-3
GRAD_ATOL = 1e-5
MARGIN = 2e-3          # relative distance of a transmittance to the cut-off below which a pixel is ambiguous


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_forward(wl, flags=raster.SAVE_FOR_BACKWARD | raster.SAVE_SORTED):
    pos, op, feat = to_dev(wl.pos), to_dev(wl.opacity), to_dev(wl.feat)
    img, alpha, ws = raster.inpc_raster_forward(pos, op, feat, wl.cam, flags=flags)
    torch.cuda.synchronize()
    return dict(pos=pos, op=op, feat=feat, img=img, alpha=alpha, ws=ws)


def gpu_backward(wl, st, g_alpha=True):
    g_img = to_dev(wl.g_img)
    g_a = to_dev(wl.g_alpha) if g_alpha else None
    out = raster.inpc_raster_backward(st["pos"], st["op"], st["feat"], wl.cam, g_img, g_a, st["ws"])
    torch.cuda.synchronize()
    return out


def check_counts_and_order(wl, st, ref, window=None):
    W, H = wl.cam.width, wl.cam.height
    cnt = raster.inpc_raster_get_counts(st["ws"], W, H).cpu().numpy().view(np.uint32)
    rc = ref.counts()
    off, idx, dep = raster.inpc_raster_get_sorted(st["ws"], W, H)
    off = off.cpu().numpy().view(np.uint32).astype(np.int64)
    idx = idx.cpu().numpy().view(np.uint32).astype(np.int64)
    dep = dep.cpu().numpy().view(np.uint32)
    assert np.array_equal(np.diff(off), cnt.reshape(-1).astype(np.int64)), "offsets are not the exclusive sum of counts"
    stats = raster.inpc_raster_get_stats(st["ws"])
    assert stats["n_fragments"] == int(cnt.sum(dtype=np.int64))
    roff, ridx, rdep, _ = ref.sorted_fragments()
    if window is None:
        assert np.array_equal(cnt, rc), f"per-pixel counts differ at {np.argwhere(cnt != rc)[:5]}"
        assert stats["n_kept"] == ref.kept
        assert np.array_equal(off, roff)
        assert np.array_equal(dep, rdep), "sorted depth keys differ"
        assert np.array_equal(idx, ridx), "sorted point indices differ"
    else:
        x0, y0, x1, y1 = window
        assert np.array_equal(cnt[y0:y1, x0:x1], rc[y0:y1, x0:x1]), "per-pixel counts differ inside the window"
        for y in range(y0, y1):          # pixel rows of the window are contiguous runs in both lists
            p0, p1 = y * W + x0, y * W + x1
            a, b = off[p0], off[p1]
            ra, rb = roff[p0], roff[p1]
            assert b - a == rb - ra
            assert np.array_equal(dep[a:b], rdep[ra:rb]), f"sorted depth keys differ in row {y}"
            assert np.array_equal(idx[a:b], ridx[ra:rb]), f"sorted point indices differ in row {y}"
    return stats


def _ambiguous(ref, margin):
    return margin < MARGIN


def check_forward(wl, st, ref, window=None, report=None):
    img_r, alpha_r, nb_r, margin = ref.blend()
    amb = _ambiguous(ref, margin)
    img = st["img"].cpu().numpy().astype(np.float64)
    alpha = st["alpha"].cpu().numpy().astype(np.float64)
    err = np.maximum(np.abs(img - img_r).max(axis=2), np.abs(alpha - alpha_r))
    if window is not None:
        x0, y0, x1, y1 = window
        mask = np.zeros_like(amb)
        mask[y0:y1, x0:x1] = True
    else:
        mask = np.ones_like(amb)
    bad = (err > FWD_ATOL) & mask & ~amb
    assert not bad.any(), f"forward error {err[bad].max():.3e} > {FWD_ATOL} at {np.argwhere(bad)[:5]}"
    n_amb = int((amb & mask).sum())
    if n_amb:
        # ambiguous pixels: accept the oracle with the cut-off just below / above the ambiguous transmittance
        lo = ref.blend(oracle.T_MIN * (1 - 2 * MARGIN))
        hi = ref.blend(oracle.T_MIN * (1 + 2 * MARGIN))
        ref.blend()   # restore the saved per-fragment state for the backward pass
        e_alt = err.copy()
        for im2, al2, _, _ in (lo, hi):
            e_alt = np.minimum(e_alt, np.maximum(np.abs(img - im2).max(axis=2), np.abs(alpha - al2)))
        bad = (e_alt > FWD_ATOL) & mask & amb
        assert not bad.any(), f"ambiguous-pixel forward error {e_alt[bad].max():.3e} at {np.argwhere(bad)[:5]}"
    # flagged pixels are still compared (against the oracle re-blended with the cut-off moved by +-2 MARGIN); the
    # bound only guards against the flag swallowing the test.  Deep workloads reach the cut-off in ~10 % of
    # their pixels and each of those has a ~3 % chance of a T_k inside the +-MARGIN band => 0.3 % (train) to 0.8 % (infer) flagged.
    assert n_amb <= max(8, int(0.02 * mask.sum())), f"too many termination-ambiguous pixels: {n_amb}"
    if report is not None:
        report.update(fwd_max_err=float(err[mask & ~amb].max()) if (mask & ~amb).any() else 0.0, n_ambiguous=n_amb)
    return amb


def points_touching(ref, amb):
    """Indices of the points that have a fragment in an ambiguous pixel."""
    if not amb.any():
        return np.zeros(0, dtype=np.int64)
    off, idx, _, _ = ref.sorted_fragments()
    pix = np.flatnonzero(amb.reshape(-1))
    return np.unique(np.concatenate([idx[off[p]:off[p + 1]] for p in pix])) if len(pix) else np.zeros(0, np.int64)


def check_grads(name, got, want, skip_rows=None):
    got = got.cpu().numpy().astype(np.float64).reshape(want.shape)
    tol = np.maximum(GRAD_RTOL * np.abs(want), GRAD_ATOL)
    diff = np.abs(got - want)
    bad = diff > tol
    if skip_rows is not None and len(skip_rows):
        bad[skip_rows] = False
    if bad.any():
        i = np.argwhere(bad)[0]
        raise AssertionError(f"{name}: {int(bad.sum())} elements out of tolerance; first at {tuple(i)}: "
                             f"gpu {got[tuple(i)]:.8g} ref {want[tuple(i)]:.8g}")
    return float((diff / np.maximum(np.abs(want), GRAD_ATOL / GRAD_RTOL)).max())


def check_backward(wl, st, ref, amb, g_alpha=True, point_mask=None, report=None):
    """ref.blend() must have been called (check_forward does).  point_mask: rows to compare (window runs)."""
    d_feat, d_op, d_uv = gpu_backward(wl, st, g_alpha)
    rf, ro, ru = ref.backward(wl.g_img, wl.g_alpha if g_alpha else None)
    skip = points_touching(ref, amb)
    if point_mask is not None:
        skip = np.union1d(skip, np.flatnonzero(~point_mask))
    e1 = check_grads("grad_feat", d_feat, rf, skip)
    e2 = check_grads("grad_opacity", d_op, ro, skip)
    e3 = check_grads("grad_uv", d_uv, ru, skip)
    if report is not None:
        report.update(grad_rel_err=max(e1, e2, e3), n_points_skipped=int(len(skip)))
    return d_feat, d_op, d_uv


def full_parity(wl, backward=True, g_alpha=True):
    """Whole-image parity of one workload; returns a small report dict."""
    report = {}
    st = gpu_forward(wl)
    ref = oracle.Raster.from_points(wl.pos, wl.opacity, wl.feat, wl.cam)
    report["stats"] = check_counts_and_order(wl, st, ref)
    amb = check_forward(wl, st, ref, report=report)
    if backward:
        check_backward(wl, st, ref, amb, g_alpha=g_alpha, report=report)
    return report
