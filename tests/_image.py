"""Helpers shared by the image tests: shower-like synthetic charge images (no
method arithmetic: only inputs) and the device-vs-oracle comparison with the
tolerances DESIGN.md section 7 derives for the fp32 event parameters."""
from __future__ import annotations

import numpy as np

import dl0gen

F32 = np.float32


def blob_images(E, P, seed, pitch=0.05):
    """Elliptical Gaussian blobs on a hex camera plus noise: shower-like test images."""
    rng = np.random.default_rng(seed)
    x, y, nbr = dl0gen.hex_camera(P, pitch)
    R = float(np.hypot(x, y).max())
    q = rng.normal(0, 1.5, (E, P))
    t = rng.normal(15, 3, (E, P))
    for e in range(E):
        cx, cy = rng.uniform(-0.5 * R, 0.5 * R, 2)
        L, Wd = rng.uniform(2, 6) * pitch, rng.uniform(0.7, 2) * pitch
        a = rng.uniform(-np.pi / 2, np.pi / 2)
        u = (x - cx) * np.cos(a) + (y - cy) * np.sin(a)
        v = -(x - cx) * np.sin(a) + (y - cy) * np.cos(a)
        q[e] += rng.uniform(30, 300) * np.exp(-0.5 * ((u / L) ** 2 + (v / Wd) ** 2))
    return q.astype(F32), t.astype(F32), x, y, nbr


def assert_image_parity(got, want, pix_x, pix_y, what=""):
    """got / want = (n_pix int32[E], params float32[E][8], mask uint8[E][P] or None).

    Exact: n_pix, mask, q_max, and which events are empty. The sums are fp64 on
    both sides, accumulated in a different order and rounded once to fp32, so
    (DESIGN.md section 7): size, t_mean relative 1e-6; cog absolute 1e-6 of the
    camera extent; length relative 1e-6; width absolute 1e-6 * length (the
    difference of two nearly equal numbers under a square root); psi absolute
    1e-6 rad modulo pi, checked where the image has a defined axis
    (length^2 - width^2 > 1e-6 * length^2)."""
    gn, gp, gm = got
    wn, wp, wm = want
    assert np.array_equal(gn, wn), what + ": n_pix differs"
    if gm is not None and wm is not None:
        assert np.array_equal(gm.astype(bool), wm.astype(bool)), what + ": mask differs"
        assert set(np.unique(gm).tolist()) <= {0, 1}, what + ": mask values are 0/1"
    gp = gp.astype(np.float64)
    wp = wp.astype(np.float64)
    # an infinite charge in the mask makes size infinite and the ratios NaN on
    # both sides (IEEE): such events must agree on being non-finite, no more
    fin = np.isfinite(wp).all(1)
    assert np.array_equal(np.isfinite(gp).all(1), fin), what + ": non-finite events differ"
    gp, wp = gp[fin], wp[fin]
    assert np.array_equal(gp[:, 7], wp[:, 7]), what + ": q_max differs"
    empty = (wp == 0).all(1)
    assert np.array_equal((gp == 0).all(1), empty), what + ": empty events differ"
    ext = float(max(np.abs(pix_x).max(), np.abs(pix_y).max(), 1e-30))
    rel = lambda a, b: np.abs(a - b) <= 1e-6 * np.abs(b)
    assert rel(gp[:, 0], wp[:, 0]).all(), what + ": size outside rel 1e-6"
    assert (np.abs(gp[:, 1:3] - wp[:, 1:3]) <= 1e-6 * ext).all(), what + ": cog outside 1e-6 of the extent"
    assert rel(gp[:, 3], wp[:, 3]).all(), what + ": length outside rel 1e-6"
    assert (np.abs(gp[:, 4] - wp[:, 4]) <= 1e-6 * wp[:, 3]).all(), what + ": width outside 1e-6 * length"
    tm_ok = rel(gp[:, 6], wp[:, 6]) | (np.abs(gp[:, 6] - wp[:, 6]) <= 1e-6)
    assert tm_ok.all(), what + ": t_mean outside 1e-6"
    L2, W2 = wp[:, 3] ** 2, wp[:, 4] ** 2
    axis = ~empty & (L2 - W2 > 1e-6 * L2)
    dpsi = (gp[axis, 5] - wp[axis, 5] + np.pi / 2) % np.pi - np.pi / 2
    assert (np.abs(dpsi) <= 1e-6).all(), what + ": psi outside 1e-6 rad"
    return int(axis.sum())
