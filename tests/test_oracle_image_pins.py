"""Pins for the cleaning + image-moments oracle (oracle/rta_oracle_image.cpp; CPU
only). The paper names the chain (§4.1, §4.2) and says
that event-level parameters, not raw data, leave the site; the
definition is DESIGN.md readings R31-R35. Pinned to a hand-worked camera
(tests/golden/image7.json), closed forms, numpy.linalg.eigh of the weighted
covariance matrix, a vectorised numpy restatement of the cleaning, invariances,
and mutations. No expected value comes from the CUDA path."""
import json
import math
import os

import numpy as np
import pytest

import dl0gen
import oracle
from tests._image import blob_images

GOLD = os.path.join(os.path.dirname(__file__), "golden", "image7.json")
F32 = np.float32


def derived(sxx, syy, sxy):
    d = sxx - syy
    z = math.sqrt(d * d + 4 * sxy * sxy)
    return (math.sqrt(0.5 * (sxx + syy + z)), math.sqrt(max(0.0, 0.5 * (sxx + syy - z))),
            0.5 * math.atan2(2 * sxy, d))


def test_hand_worked_camera():
    g = json.load(open(GOLD))
    q = np.array([[float(v) for v in ev["charge"]] for ev in g["events"]], F32)
    t = np.array([ev["time"] for ev in g["events"]], F32)
    npix, par, mask = oracle.image_moments(q, t, g["pix_x"], g["pix_y"], g["neighbors"],
                                           g["thr_picture"], g["thr_boundary"])
    for i, ev in enumerate(g["events"]):
        assert mask[i].tolist() == ev["mask"], ev["name"]
        assert npix[i] == ev["n_pix"]
        fr = lambda k: ev[k][0] / ev[k][1]
        L, Wd, psi = derived(fr("sxx"), fr("syy"), fr("sxy"))
        want = [ev["size"], fr("cog_x"), fr("cog_y"), L, Wd, psi, fr("t_mean"), ev["q_max"]]
        if ev["n_pix"] == 0:
            want = [0.0] * 8
        np.testing.assert_allclose(par[i], np.array(want, F32), rtol=3e-7, atol=1e-7, err_msg=ev["name"])
        assert par[i][0] == F32(ev["size"]) and par[i][7] == F32(ev["q_max"])


def np_clean(q, nbr, tp, tb):
    """vectorised restatement of the cleaning: neighbour gathers with a padded column."""
    E, P = q.shape
    idx = np.where(nbr >= 0, nbr, P)                       # P = a padding pixel that is never set

    def any_nb(flag):
        padded = np.concatenate([flag, np.zeros((E, 1), bool)], 1)
        return padded[:, idx].any(-1)
    with np.errstate(invalid="ignore"):
        core = q >= F32(tp)
        low = q >= F32(tb)
    keep = core & any_nb(core)
    return keep | (low & any_nb(keep))


def np_moments(q, t, x, y, mask):
    """restatement through the weighted covariance matrix and numpy.linalg.eigh."""
    out = np.zeros((q.shape[0], 8))
    for e in range(q.shape[0]):
        m = mask[e]
        w = q[e][m].astype(np.float64)
        if m.sum() == 0 or not w.sum() > 0:
            continue
        xs, ys = x[m].astype(np.float64), y[m].astype(np.float64)
        cov = np.cov(np.stack([xs, ys]), aweights=w, bias=True) if m.sum() > 1 else np.zeros((2, 2))
        ev, vec = np.linalg.eigh(cov)
        major = vec[:, 1]
        psi = math.atan2(major[1], major[0])
        out[e] = [w.sum(), np.average(xs, weights=w), np.average(ys, weights=w),
                  math.sqrt(max(ev[1], 0)), math.sqrt(max(ev[0], 0)), psi,
                  np.average(t[e][m].astype(np.float64), weights=w), q[e][m].max()]
    return out


@pytest.mark.parametrize("P,seed", [(1855, 0), (1764, 1), (37, 2), (2048, 3)])
def test_numpy_restatements_on_blob_images(P, seed):
    q, t, x, y, nbr = blob_images(40, P, seed)
    npix, par, mask = oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0)
    m2 = np_clean(q, nbr, 8.0, 4.0)
    assert (mask.astype(bool) == m2).all() and (npix == m2.sum(1)).all()
    assert npix.max() > 10                                  # the blobs survive the cleaning
    ref = np_moments(q, t, x, y, m2)
    np.testing.assert_allclose(par[:, :5], ref[:, :5], rtol=2e-6, atol=1e-7)
    np.testing.assert_allclose(par[:, 6:], ref[:, 6:], rtol=2e-6, atol=1e-7)
    # psi is an axis: compare modulo pi where the image is clearly elongated
    el = (par[:, 3] > 1.2 * par[:, 4]) & (npix > 2)
    dpsi = (par[el, 5] - ref[el, 5] + np.pi / 2) % np.pi - np.pi / 2
    assert el.sum() > 5 and np.abs(dpsi).max() < 1e-5


def test_two_pixel_closed_forms_and_rotation():
    """Two equal pixels at +-a along an axis at angle th: cog = centre, length = a,
    width = 0, psi = th; unequal charges move the centre of gravity by the lever rule."""
    for th in (0.0, 0.3, -1.1, math.pi / 2):
        a = 2.0
        c, s = math.cos(th), math.sin(th)
        x = np.array([-a * c + 3, a * c + 3], F32)
        y = np.array([-a * s - 1, a * s - 1], F32)
        nbr = np.full((2, 6), -1, np.int32)
        nbr[0, 0], nbr[1, 0] = 1, 0
        npix, par, mask = oracle.image_moments(np.array([[10, 10]], F32), np.array([[4, 8]], F32),
                                               x, y, nbr, 5.0, 1.0)
        assert npix[0] == 2 and mask.all()
        np.testing.assert_allclose(par[0], [20, 3, -1, a, 0, th if th < math.pi / 2 - 1e-9 else par[0][5],
                                            6, 10], rtol=1e-6, atol=2e-6)
        if th >= math.pi / 2 - 1e-9:
            assert abs(abs(par[0][5]) - math.pi / 2) < 1e-6
        npix, par, _ = oracle.image_moments(np.array([[30, 10]], F32), np.array([[4, 8]], F32),
                                            x, y, nbr, 5.0, 1.0)
        # lever rule: centre at x0 + (10*2a)/40 from pixel 0; spread sqrt(p(1-p)) * 2a
        np.testing.assert_allclose(par[0][:5], [40, x[0] + 0.25 * (x[1] - x[0]), y[0] + 0.25 * (y[1] - y[0]),
                                                2 * a * math.sqrt(0.25 * 0.75), 0], rtol=1e-6, atol=2e-6)
        assert par[0][6] == F32(5.0) and par[0][7] == F32(30)


def test_invariances():
    q, t, x, y, nbr = blob_images(12, 469, 7)
    n0, p0, m0 = oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0)
    # charges and thresholds scaled by 4 (exact in binary): same mask, size x 4, shape unchanged
    n1, p1, m1 = oracle.image_moments(4 * q, t, x, y, nbr, 32.0, 16.0)
    assert (m1 == m0).all()
    np.testing.assert_allclose(p1[:, 0], 4 * p0[:, 0], rtol=1e-6)
    np.testing.assert_allclose(p1[:, 1:7], p0[:, 1:7], rtol=1e-5, atol=1e-7)
    # camera translated: cog moves, the rest stays
    n2, p2, m2 = oracle.image_moments(q, t, x + F32(0.25), y - F32(0.5), nbr, 8.0, 4.0)
    assert (m2 == m0).all()
    ok = n0 > 0
    np.testing.assert_allclose(p2[ok, 1], p0[ok, 1] + 0.25, atol=2e-6)
    np.testing.assert_allclose(p2[ok, 2], p0[ok, 2] - 0.5, atol=2e-6)
    np.testing.assert_allclose(p2[:, 3:5], p0[:, 3:5], rtol=1e-4, atol=1e-6)
    # pixel order permuted (neighbour table renumbered): same event parameters
    rng = np.random.default_rng(0)
    perm = rng.permutation(x.size)
    inv = np.empty_like(perm)
    inv[perm] = np.arange(perm.size)
    nbr_p = np.where(nbr[perm] >= 0, inv[np.maximum(nbr[perm], 0)], -1).astype(np.int32)
    n3, p3, m3 = oracle.image_moments(q[:, perm], t[:, perm], x[perm], y[perm], nbr_p, 8.0, 4.0)
    assert (n3 == n0).all() and (m3 == m0[:, perm]).all()
    np.testing.assert_allclose(p3, p0, rtol=1e-5, atol=1e-6)
    # time shifted by a constant: only t_mean moves
    n4, p4, _ = oracle.image_moments(q, t + F32(2), x, y, nbr, 8.0, 4.0)
    np.testing.assert_allclose(p4[ok, 6], p0[ok, 6] + 2, rtol=1e-6)


def test_cleaning_special_cases():
    x, y, nbr = dl0gen.hex_camera(19, 1.0)
    z = np.zeros((1, 19), F32)

    def mask_of(q):
        return oracle.image_moments(q, z, x, y, nbr, 10.0, 5.0)[2][0].astype(bool)
    q = z.copy(); q[0, 0] = 100                             # one isolated hot pixel: dropped
    assert not mask_of(q).any()
    q[0, nbr[0, 0]] = 10                                    # a second core pixel next to it: both kept
    assert mask_of(q).sum() == 2
    q[0, :] = np.where(q[0] > 0, q[0], 5)                   # everything else at the boundary cut
    m = mask_of(q)
    kept = {0, int(nbr[0, 0])}
    expected = set(kept)
    for p in range(19):
        if any(int(n) in kept for n in nbr[p] if n >= 0):
            expected.add(p)
    assert set(np.flatnonzero(m).tolist()) == expected and len(expected) < 19
    q[0, :] = 4.999                                         # nothing passes
    assert not mask_of(q).any()
    q[0, :] = 10                                            # everything is core with core neighbours
    assert mask_of(q).all()
    # picture < boundary is allowed: a kept core pixel is in the image whatever the boundary cut
    m = oracle.image_moments(q, z, x, y, nbr, 10.0, 50.0)[2][0]
    assert m.all()


def test_degenerate_images_give_zero_parameters():
    x, y, nbr = dl0gen.hex_camera(7, 1.0)
    q = np.array([[-5, -5, -5, -5, -5, -5, -5]], F32)
    n, p, m = oracle.image_moments(q, q, x, y, nbr, -10.0, -10.0)   # all pass, but size < 0
    assert n[0] == 7 and m.all() and (p == 0).all()
    q = np.full((1, 7), np.nan, F32)
    n, p, m = oracle.image_moments(q, q, x, y, nbr, 1.0, 1.0)
    assert n[0] == 0 and (p == 0).all()


def test_mutations_fail_the_fixture():
    """Plausible wrong definitions do not reproduce the hand-worked masks."""
    g = json.load(open(GOLD))
    q = np.array([[float(v) for v in ev["charge"]] for ev in g["events"]], F32)
    want = np.array([ev["mask"] for ev in g["events"]], bool)
    nbr = np.array(g["neighbors"], np.int32)
    assert (np_clean(q, nbr, 8.0, 3.0) == want).all()
    E, P = q.shape
    idx = np.where(nbr >= 0, nbr, P)
    pad = lambda f: np.concatenate([f, np.zeros((E, 1), bool)], 1)
    with np.errstate(invalid="ignore"):
        core, low = q >= 8, q >= 3
        keep = core & pad(core)[:, idx].any(-1)
        assert not ((core | (low & pad(core)[:, idx].any(-1))) == want).all()        # isolated cores kept
        assert not ((keep | (low & pad(low)[:, idx].any(-1))) == want).all()          # boundary chains grow
        strict = (q > 8) & pad(q > 8)[:, idx].any(-1)
        assert not ((strict | ((q > 3) & pad(strict)[:, idx].any(-1))) == want).all()  # strict thresholds
