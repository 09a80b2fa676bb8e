"""Pins for the CPU oracle: what the paper and the mathematics fix, checked against oracle/ only.

None of these values comes from the CUDA path.  Each test cites the passage that fixes the
expected value (PAPER.md / SPEC.md line) or the identity it uses.  Numbering G1..G14 follows
SURVEY.md section 8(c).
"""
import json
import math
import os
from types import SimpleNamespace

import numpy as np
import pytest

from qr_inputs import make_scene, make_camera

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


# --------------------------------------------------------------------------------------------
# G1: hand-worked rays through Algorithm 1
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ray", _gold("algorithm1_rays.json")["rays"], ids=lambda r: r["name"][:4])
def test_G1_algorithm1_hand_worked(orc, ray):
    n = len(ray["alphas"])
    feats = np.eye(n, dtype=np.float32)  # one-hot features: the output IS the weight vector
    lists = orc.lists_from_rays([(range(n), ray["alphas"])])
    q = orc.qrender(lists, ray["K"], feats)
    ns = len(ray["selected"])
    assert q.n_sel[0] == ns
    assert q.sel_idx[0, :ns].tolist() == ray["selected"]
    assert (q.sel_idx[0, ns:] == -1).all()
    # alphas are fp32 inputs, so compare at fp32 resolution
    np.testing.assert_allclose(q.sel_w[0, :ns], ray["w_hat"], rtol=3e-7)
    np.testing.assert_allclose(q.resid_TQ[0], ray["TQ"], rtol=3e-7)
    expect = np.zeros(n)
    for s, w in zip(ray["selected"], ray["w_hat"]):
        expect[s] = w
    np.testing.assert_allclose(q.out_map[0], expect, rtol=3e-7, atol=1e-12)
    if ns:
        wq = q.sel_w[0, :ns] * (1.0 - q.resid_TQ[0])
        np.testing.assert_allclose(wq, ray["wQ"], rtol=3e-7)


def test_G1_K0_is_a_domain_error(orc):
    lists = orc.lists_from_rays([([0], [0.5])])
    with pytest.raises(ValueError):
        orc.qrender(lists, 0, None)


def test_G1_empty_ray(orc):
    lists = orc.lists_from_rays([([], [])])  # zero vector + no-selection flag
    q = orc.qrender(lists, 4, np.ones((1, 3), np.float32))
    assert q.n_sel[0] == 0 and q.resid_TQ[0] == 1.0 and (q.out_map[0] == 0).all()


# --------------------------------------------------------------------------------------------
# G2: V-Render micro rays (Eq. 1)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ray", _gold("vrender_rays.json")["rays"], ids=lambda r: r["name"][:10])
def test_G2_vrender_micro(orc, ray):
    n = len(ray["alphas"])
    lists = orc.lists_from_rays([(range(n), ray["alphas"])])
    v = orc.vrender(lists, np.eye(n, dtype=np.float32), t_min=0.0)
    np.testing.assert_allclose(v.out_map[0], ray["weights"], rtol=3e-7)
    np.testing.assert_allclose(v.final_T[0], ray["residual"], rtol=2e-6)


def _random_rays(rng, n_rays, max_len, lo=0.004, hi=0.99):
    rays = []
    for _ in range(n_rays):
        n = int(rng.integers(0, max_len + 1))
        a = rng.uniform(lo, hi, size=n) ** rng.choice([1.0, 2.0, 4.0])
        a = np.clip(a, 1.0 / 255.0, 0.99).astype(np.float32)
        rays.append((rng.permutation(max_len)[:n], a))
    return rays


# --------------------------------------------------------------------------------------------
# Brute-force per-ray compositing: Eq. 1 written as a cumulative product in NumPy (a different
# formulation from the oracle's sequential walk).
# --------------------------------------------------------------------------------------------
def test_vrender_equals_cumprod_formulation(orc):
    rng = np.random.default_rng(1)
    rays = _random_rays(rng, 200, 60)
    feats = rng.standard_normal((60, 5)).astype(np.float32)
    v = orc.vrender(orc.lists_from_rays(rays), feats, t_min=0.0)
    for j, (ids, a) in enumerate(rays):
        a64 = a.astype(np.float64)
        T = np.concatenate([[1.0], np.cumprod(1.0 - a64)])
        w = T[:-1] * a64
        np.testing.assert_allclose(v.out_map[j], w @ feats[ids].astype(np.float64) if len(ids) else 0.0,
                                   rtol=2e-6, atol=2e-7)
        np.testing.assert_allclose(v.final_T[j], T[-1], rtol=1e-12)


def test_vrender_early_stop_R7(orc):
    # t_min: stop WITHOUT blending the Gaussian that would take T below t_min (reading R7)
    a = [0.9, 0.9, 0.9, 0.9, 0.9]          # T: 1, .1, .01, .001, 1e-4 -> 1e-5
    lists = orc.lists_from_rays([(range(5), a)])
    v = orc.vrender(lists, np.eye(5, dtype=np.float32), t_min=5e-4)
    assert v.n_blended[0] == 3               # T_test after 4th = 1e-4 < 5e-4 -> stop before blending it
    np.testing.assert_allclose(v.out_map[0], [0.9, 0.09, 0.009, 0, 0], rtol=1e-6)
    np.testing.assert_allclose(v.final_T[0], 1e-3, rtol=1e-6)


# --------------------------------------------------------------------------------------------
# G3 / G4: telescoping identities and cardinality on random rays
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [1, 2, 5, 10, 40, 64])
def test_G3_G4_telescoping_and_cardinality(orc, K):
    rng = np.random.default_rng(K)
    rays = _random_rays(rng, 500, 80)
    lists = orc.lists_from_rays(rays)
    nG = 80
    q = orc.qrender(lists, K, np.eye(nG, dtype=np.float32))
    v = orc.vrender(lists, np.eye(nG, dtype=np.float32), t_min=0.0)
    # dense: sum_i w_i + T_final = 1, weights >= 0, sum <= 1
    assert (v.out_map >= 0).all()
    np.testing.assert_allclose(v.out_map.astype(np.float64).sum(1) + v.final_T, 1.0, atol=5e-6)
    for j, (ids, a) in enumerate(rays):
        ns = q.n_sel[j]
        assert 0 <= ns <= K                                    # G4
        assert ns <= len(ids)
        w = q.sel_w[j]
        assert (w >= 0).all() and (w[ns:] == 0).all()
        if ns == 0:
            assert q.resid_TQ[j] == 1.0 and (q.out_map[j] == 0).all()
            continue
        assert abs(w[:ns].sum() - 1.0) < 1e-12                 # convex combination
        # sum_s w^Q_s = 1 - T^Q (telescoping of the sparse product)
        sel_pos = [list(ids).index(g) for g in q.sel_idx[j, :ns]]
        assert sel_pos == sorted(sel_pos) and len(set(sel_pos)) == ns   # strictly increasing list position
        TQ = np.prod(1.0 - a[sel_pos].astype(np.float64))
        np.testing.assert_allclose(q.resid_TQ[j], TQ, rtol=1e-12)
        assert q.n_walked[j] <= len(ids)
        # true invariants noted in SURVEY G10: T^Q >= dense T at the last walked step
        Tdense = np.prod(1.0 - a[: q.n_walked[j]].astype(np.float64))
        assert q.resid_TQ[j] >= Tdense - 1e-12


def test_closed_form_level_characterisation(orc):
    """Reading R3: the sequential listing is equivalent to 'selected <=> level(T_after) > level(T_before)',
    level(T) = #{k in 0..K-1 : T < thr_k}; break <=> T_after < 1/(K+1).  Independent fp32 NumPy evaluation."""
    rng = np.random.default_rng(7)
    for K in (3, 10, 40):
        rays = _random_rays(rng, 300, 50)
        q = orc.qrender(orc.lists_from_rays(rays), K, None)
        thr = (np.float32(1.0) - (np.arange(1, K + 1, dtype=np.float32) / np.float32(K + 1))).astype(np.float32)
        tb = np.float32(1.0) / np.float32(K + 1)
        for j, (ids, a) in enumerate(rays):
            if q.margin[j] <= 1e-6:
                continue
            T = np.float32(1.0); sel = []
            for s, al in enumerate(a):
                Tt = np.float32(T * np.float32(np.float32(1.0) - al))
                if (Tt < thr).sum() > (T < thr).sum():
                    sel.append(int(ids[s]))
                if Tt < tb:
                    break
                T = Tt
            assert sel == q.sel_idx[j, : q.n_sel[j]].tolist()


# --------------------------------------------------------------------------------------------
# G5 / G6 / G7: constant feature, linearity, payload-width independence, permutation safety
# --------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny(orc):
    sc = make_scene("cfg1", seed=0, N=600, W=32, H=32, D=8)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    return sc, proj, lists


def test_G5_constant_feature_scene(orc, tiny):
    sc, proj, lists = tiny
    f = np.tile(np.array([[0.3, -1.2, 2.0]], np.float32), (sc.N, 1))
    q = orc.qrender(lists, 10, f)
    hit = q.n_sel > 0
    assert hit.any() and (~hit).any()
    np.testing.assert_allclose(q.out_map[hit], np.broadcast_to(f[0], (hit.sum(), 3)), rtol=1e-6)
    assert (q.out_map[~hit] == 0).all()


def test_G6_linearity_and_width_independence(orc, tiny):
    sc, proj, lists = tiny
    rng = np.random.default_rng(3)
    f1 = rng.standard_normal((sc.N, 6)).astype(np.float32)
    f2 = rng.standard_normal((sc.N, 6)).astype(np.float32)
    qa = orc.qrender(lists, 12, f1); qb = orc.qrender(lists, 12, f2)
    qc = orc.qrender(lists, 12, (2.0 * f1.astype(np.float64) - 0.5 * f2).astype(np.float32))
    np.testing.assert_allclose(qc.out_map, 2.0 * qa.out_map - 0.5 * qb.out_map, rtol=1e-5, atol=2e-6)
    q1 = orc.qrender(lists, 12, f1[:, :1])
    assert np.array_equal(q1.sel_idx, qa.sel_idx) and np.array_equal(q1.n_sel, qa.n_sel)
    q0 = orc.qrender(lists, 12, None)
    assert np.array_equal(q0.sel_idx, qa.sel_idx)


def test_G7_permutation_safety(orc, tiny):
    sc, proj, lists = tiny
    rng = np.random.default_rng(4)
    perm = rng.permutation(sc.N)
    projp = orc.project(sc.cam, sc.means[perm], sc.scales[perm], sc.quats[perm], sc.opac[perm])
    listsp = orc.pixel_lists(sc.cam, projp)
    assert len(np.unique(proj.depth[proj.visible > 0])) == int((proj.visible > 0).sum())  # no depth ties
    q = orc.qrender(lists, 10, sc.features)
    qp = orc.qrender(listsp, 10, sc.features[perm])
    assert np.array_equal(q.out_map, qp.out_map)
    relabel = np.where(qp.sel_idx >= 0, perm[np.maximum(qp.sel_idx, 0)], -1)
    assert np.array_equal(relabel, q.sel_idx)


# --------------------------------------------------------------------------------------------
# G8: brute-force lists == binned lists, exact
# --------------------------------------------------------------------------------------------
def test_G8_brute_equals_binned(orc):
    for seed in range(50):
        w, h = (8, 8) if seed % 2 == 0 else (16, 12)
        sc = make_scene("cfg1", seed=seed, N=100 if seed % 3 else 50, W=w, H=h, D=4)
        if seed % 5 == 0:   # bigger, nearer splats so that lists are long and AABBs leave the image
            sc.scales *= 6.0
        proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
        a = orc.pixel_lists(sc.cam, proj, "brute")
        b = orc.pixel_lists(sc.cam, proj, "binned")
        assert np.array_equal(a.off, b.off), seed
        assert np.array_equal(a.gid, b.gid), seed
        assert np.array_equal(a.alpha, b.alpha), seed
        assert a.off[-1] > 0


def test_lists_depth_order_and_alpha_range(orc, tiny):
    sc, proj, lists = tiny
    assert lists.off[-1] > 1000
    assert (lists.alpha >= np.float32(1.0 / 255.0)).all() and (lists.alpha <= np.float32(0.99)).all()
    for p in range(0, 32 * 32, 7):
        g, _ = lists.ray(p)
        d = proj.depth[g]
        assert (np.diff(d) >= 0).all()
        ties = np.diff(d) == 0
        assert (np.diff(g)[ties] > 0).all()


def test_tile_lists_are_supersets_in_order(orc, tiny):
    """Per-tile (depth, id)-sorted lists from the 3-sigma AABB contain every pixel's list as a subsequence."""
    sc, proj, lists = tiny
    rect, touched = orc.tile_rects(sc.cam, proj)
    isect, rng_ = orc.tile_lists(sc.cam, proj.depth, rect, touched)
    assert len(isect) == int(touched.sum())
    tx = sc.cam.width // 16
    for p in range(0, 32 * 32, 5):
        y, x = divmod(p, sc.cam.width)
        t = (y // 16) * tx + x // 16
        tl = isect[rng_[t, 0]: rng_[t, 1]].astype(np.int64)
        pos = {int(g): i for i, g in enumerate(tl)}
        g, _ = lists.ray(p)
        idx = [pos[int(k)] for k in g]          # KeyError = not a superset
        assert idx == sorted(idx)


# --------------------------------------------------------------------------------------------
# G9: limiting case Q -> dense (every walked Gaussian crosses a boundary)
# --------------------------------------------------------------------------------------------
def test_G9_limit_Q_equals_dense(orc):
    n = 5
    K = 2 ** (n + 1) - 1          # K+1 = 64 >= 2^{n+1}: boundaries at multiples of 1/64, T_i = 2^-i
    a = [0.5] * n
    rng = np.random.default_rng(5)
    feats = rng.standard_normal((n, 7)).astype(np.float32)
    lists = orc.lists_from_rays([(range(n), a)])
    q = orc.qrender(lists, K, feats)
    v = orc.vrender(lists, feats, t_min=0.0)
    assert q.n_sel[0] == n
    np.testing.assert_allclose(q.resid_TQ[0], v.final_T[0], rtol=1e-12)
    np.testing.assert_allclose(q.out_map[0], v.out_map[0] / (1.0 - v.final_T[0]), rtol=1e-6)


# --------------------------------------------------------------------------------------------
# G10: Appendix-C bound |C_vol - C~_Q| <= M / (2K) on discretised smooth 1-D models
# (PAPER.md:672-678, :713-723).  Statistical check; see DESIGN.md for the caveat on T_Q <= 1/(K+1).
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [4, 8, 16, 32, 64])
def test_G10_riemann_bound(orc, K):
    # App. C is stated in the continuous limit (alpha' -> 0): the K sparse weights w^Q_j ~ alpha'(1-alpha')^j
    # are only equal up to (1-alpha')^K, so the discretisation must keep K*alpha' << 1 (n = 40000: 2 % at K = 64).
    n = 40000
    sigma_dt = 12.0 / n                                   # total optical depth 12: T_end = e^-12
    a = np.full(n, 1.0 - math.exp(-sigma_dt))
    T_before = np.exp(-sigma_dt * np.arange(n))
    u_mid = T_before * math.exp(-0.5 * sigma_dt)
    c = np.stack([u_mid, np.sin(3.0 * u_mid) + u_mid ** 2, np.cos(2.0 * u_mid)], axis=1)  # c(u), |c'| <= M
    M = np.array([1.0, 5.0, 2.0])
    lists = orc.lists_from_rays([(range(n), a)])
    # alpha' here is below 1/255; the oracle's ray functions take any alpha' in (0, 0.99]
    q = orc.qrender(lists, K, c.astype(np.float32))
    v = orc.vrender(lists, c.astype(np.float32), t_min=0.0)
    err = np.abs(q.out_map[0].astype(np.float64) - v.out_map[0].astype(np.float64))
    assert (err <= M / (2.0 * K) + 1e-4).all(), (K, err)
    assert q.n_sel[0] == K
    if K >= 8:   # c(u) = u integrates to 1/2 and the K equally weighted samples are symmetric
        assert abs(q.out_map[0, 0] - 0.5) < 2e-2


def test_G10_error_decreases_with_K(orc):
    n = 40000                                              # continuous limit, see test_G10_riemann_bound
    sigma_dt = 12.0 / n
    a = np.full(n, 1.0 - math.exp(-sigma_dt))
    u_mid = np.exp(-sigma_dt * (np.arange(n) + 0.5))
    c = (np.sin(3.0 * u_mid) + u_mid ** 2)[:, None].astype(np.float32)
    lists = orc.lists_from_rays([(range(n), a)])
    v = orc.vrender(lists, c, t_min=0.0).out_map[0, 0]
    errs = [abs(orc.qrender(lists, K, c).out_map[0, 0] - v) for K in (4, 16, 64)]
    assert errs[0] > errs[1] > errs[2]
    slope = math.log(errs[2] / errs[0]) / math.log(64 / 4)
    assert -1.4 < slope < -0.7                              # O(1/K)


# --------------------------------------------------------------------------------------------
# G11: projection closed forms
# --------------------------------------------------------------------------------------------
def test_G11_covariance_examples(orc):
    for c in _gold("projection_cases.json")["covariance"]:
        S = orc.covariance3d(c["scale"], c["quat"])
        np.testing.assert_allclose(S, np.diag(c["Sigma_diag"]), atol=1e-12)
    rng = np.random.default_rng(0)
    for _ in range(20):                                      # eigenvalues = squared scales
        s = rng.uniform(0.1, 2.0, 3); q = rng.standard_normal(4); q /= np.linalg.norm(q)
        S = orc.covariance3d(s, q)
        np.testing.assert_allclose(S, S.T, atol=1e-12)
        np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(S)), np.sort(s ** 2), rtol=1e-9)


def _one(cam, mean, scale, quat=(1, 0, 0, 0), opac=0.8):
    return (np.array([mean], np.float32), np.array([scale], np.float32), np.array([quat], np.float32),
            np.array([opac], np.float32))


@pytest.mark.parametrize("which", ["f64", "f32"])
def test_G11_projection_closed_forms(orc, which):
    proj = orc.project_f64 if which == "f64" else orc.project
    rtol = 1e-9 if which == "f64" else 2e-6
    cam = make_camera(64, 48)
    z, s = 3.0, float(np.float32(0.05))          # the scale the oracle sees is the fp32-rounded one
    p = proj(cam, *_one(cam, (0, 0, z), (s, s, s)))
    assert p.visible[0] == 1
    np.testing.assert_allclose(p.mean2d[0], [cam.cx, cam.cy], rtol=rtol)
    var = (cam.fx * s / z) ** 2 + 0.3
    np.testing.assert_allclose(p.conic_opac[0, :3], [1.0 / var, 0.0, 1.0 / var], rtol=rtol, atol=1e-9)
    np.testing.assert_allclose(p.extent[0], [3.0 * math.sqrt(var)] * 2, rtol=rtol)
    np.testing.assert_allclose(p.depth[0], z, rtol=rtol)
    assert abs(p.conic_opac[0, 3] - 0.8) < 1e-7
    if which == "f64":
        np.testing.assert_allclose(p.cov2d[0], [var, 0.0, var], rtol=1e-9, atol=1e-12)
    # culling: behind the camera / inside znear
    for zc in (-1.0, 0.0, 0.1, 0.2):
        assert proj(cam, *_one(cam, (0, 0, zc), (s, s, s))).visible[0] == 0
    # off-axis pinhole: mean2d = (fx x/z + cx, fy y/z + cy)
    p = proj(cam, *_one(cam, (0.5, -0.25, 2.0), (s, s, s)))
    np.testing.assert_allclose(p.mean2d[0], [cam.fx * 0.25 + cam.cx, -cam.fy * 0.125 + cam.cy], rtol=rtol)
    # anisotropic, rotated 90 degrees about z: world covariance diag(s1^2, s0^2, s2^2) on axis
    q = (math.sqrt(0.5), 0, 0, math.sqrt(0.5))
    p = proj(cam, *_one(cam, (0, 0, z), (0.2, 0.05, 0.1), q))
    vx = (cam.fx * 0.05 / z) ** 2 + 0.3; vy = (cam.fy * 0.2 / z) ** 2 + 0.3
    np.testing.assert_allclose(p.conic_opac[0, :3], [1 / vx, 0.0, 1 / vy], rtol=max(rtol, 1e-6), atol=1e-7)


def test_G11_perspective_jacobian_against_finite_differences(orc):
    """cov2d - 0.3 I = J W Sigma W^T J^T with J the Jacobian of the pinhole map: check J by central
    differences of the projection itself (independent of the closed form used in the oracle)."""
    from qr_inputs import look_at
    cam = make_camera(80, 60, world_to_cam=look_at((0.3, -0.2, -1.0), (0.1, 0.0, 2.0)))
    rng = np.random.default_rng(2)
    W = cam.world_to_cam.astype(np.float64)

    def pix(x):
        t = W[:, :3] @ x + W[:, 3]
        return np.array([cam.fx * t[0] / t[2] + cam.cx, cam.fy * t[1] / t[2] + cam.cy])

    for _ in range(10):
        mu = rng.uniform(-0.3, 0.3, 3) + np.array([0.1, 0.0, 2.0])
        s = rng.uniform(0.02, 0.1, 3); q = rng.standard_normal(4); q /= np.linalg.norm(q)
        p = orc.project_f64(cam, *_one(cam, mu, s, q))
        mu32 = np.float32(mu).astype(np.float64)
        h = 1e-6
        Jn = np.stack([(pix(mu32 + h * e) - pix(mu32 - h * e)) / (2 * h) for e in np.eye(3)], axis=1)  # 2x3
        Sig = orc.covariance3d(np.float32(s).astype(np.float64), np.float32(q).astype(np.float64))
        cov = Jn @ Sig @ Jn.T + 0.3 * np.eye(2)
        np.testing.assert_allclose(p.cov2d[0], [cov[0, 0], cov[0, 1], cov[1, 1]], rtol=1e-6, atol=1e-8)
        inv = np.linalg.inv(cov)
        np.testing.assert_allclose(p.conic_opac[0, :3], [inv[0, 0], inv[0, 1], inv[1, 1]], rtol=1e-6, atol=1e-9)
        np.testing.assert_allclose(p.mean2d[0], pix(mu32), rtol=1e-9)


def test_f32_projection_tracks_f64(orc):
    sc = make_scene("cfg3", seed=1, N=20000, W=160, H=120, D=4)
    a = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    b = orc.project_f64(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    vis = (a.visible > 0) & (b.visible > 0)
    assert (a.visible != b.visible).sum() <= 2 and vis.sum() > 5000
    np.testing.assert_allclose(a.depth[vis], b.depth[vis], rtol=1e-6)
    np.testing.assert_allclose(a.mean2d[vis], b.mean2d[vis], rtol=1e-4, atol=1e-2)
    rel = np.abs(a.conic_opac[vis, :3] - b.conic_opac[vis, :3]) / (np.abs(b.conic_opac[vis, :3]).max(1, keepdims=True))
    assert np.median(rel) < 1e-6 and np.percentile(rel, 99) < 1e-4


def test_R12_jacobian_clamp_keeps_footprints_finite(orc):
    cam = make_camera(64, 48)
    # far off-axis, just beyond znear: without the clamp J02 explodes
    p = orc.project_f64(cam, *_one(cam, (5.0, 0.0, 0.25), (0.01, 0.01, 0.01)))
    lim = 1.3 * (cam.width / 2) / cam.fx
    j02 = cam.fx * lim / 0.25
    assert p.cov2d[0, 0] <= (cam.fx * 0.01 / 0.25) ** 2 + (j02 * 0.01) ** 2 + 0.3 + 1e-6


# --------------------------------------------------------------------------------------------
# G12: alpha' closed forms
# --------------------------------------------------------------------------------------------
def test_G12_alpha_prime_closed_forms(orc):
    cam = make_camera(64, 48)
    cases = _gold("projection_cases.json")["alpha_prime"]
    for c in cases:
        a = 0.02
        dx = math.sqrt(c["mahalanobis_sq"] / a)            # pixel centre dx away along x: d^T conic d = a dx^2
        px, py = 20, 10
        proj = orc.Projected(np.array([[px + 0.5 - dx, py + 0.5]], np.float32),
                             np.array([[a, 0.0, a, c["alpha"]]], np.float32),
                             np.array([1.0], np.float32), np.array([[22.0, 22.0]], np.float32),
                             np.array([1], np.uint8))
        lists = orc.pixel_lists(cam, proj, "brute")
        g, al = lists.ray(py * cam.width + px)
        assert g.tolist() == [0]                            # the list at p = [(0, alpha')]
        np.testing.assert_allclose(al[0], c["alpha_prime"], rtol=2e-6)


def test_R4_inclusion_rule(orc):
    cam = make_camera(64, 48)
    a = 0.02   # sigma^2 = 50; 3 sigma = 21.2 px
    proj = orc.Projected(np.array([[10.5, 10.5]], np.float32), np.array([[a, 0.0, a, 0.9]], np.float32),
                         np.array([1.0], np.float32), np.array([[21.3, 21.3]], np.float32), np.array([1], np.uint8))
    lists = orc.pixel_lists(cam, proj, "brute")
    n_in = np.diff(lists.off).reshape(cam.height, cam.width)
    yy, xx = np.mgrid[0:cam.height, 0:cam.width]
    r2 = (xx - 10) ** 2 + (yy - 10) ** 2
    inside = a * r2 <= 9.0 - 1e-3                            # power >= -4.5  <=>  d^T conic d <= 9
    outside = a * r2 >= 9.0 + 1e-3
    assert (n_in[inside] == 1).all() and (n_in[outside] == 0).all()
    # alpha' >= 1/255 cut: opacity 0.01 -> alpha' < 1/255 once exp(power) < 0.392
    proj.conic_opac[0, 3] = 0.01
    lists = orc.pixel_lists(cam, proj, "brute")
    n_in = np.diff(lists.off).reshape(cam.height, cam.width)
    keep = 0.01 * np.exp(-0.5 * a * r2) >= 1.0 / 255.0 + 1e-6
    drop = 0.01 * np.exp(-0.5 * a * r2) <= 1.0 / 255.0 - 1e-6
    assert (n_in[keep] == 1).all() and (n_in[drop] == 0).all() and keep.sum() > 10


def test_R15_borderline_position(orc):
    """Reading R15: a pixel is exempt for list membership only if the walk MEETS the borderline Gaussian.  A Gaussian
    centred on pixel (5, 5) with opacity exactly 1/255 has alpha' == alpha_min there (power = 0): a borderline event.
    bl_first = number of included entries in front of it: 0 when it is nearest, 1 behind one opaque Gaussian; pixels it
    does not reach carry INT64_MAX.  With K = 1 and an alpha' = 0.8 Gaussian in front the walk consumes 1 entry and
    breaks, so position 1 <= n_walked is still (conservatively) exempt, while behind two such Gaussians the walk never
    gets there."""
    cam = make_camera(16, 16)
    amin = np.float32(1.0) / np.float32(255.0)
    big = 0.02
    def lists_for(depth_b, n_front):
        m2 = [[5.5, 5.5]] + [[5.5, 5.5]] * n_front
        co = [[big, 0.0, big, amin]] + [[big, 0.0, big, 0.8]] * n_front
        dp = [depth_b] + [1.0 + 0.1 * i for i in range(n_front)]
        n = len(m2)
        proj = orc.Projected(np.array(m2, np.float32), np.array(co, np.float32), np.array(dp, np.float32),
                             np.full((n, 2), 21.3, np.float32), np.ones(n, np.uint8))
        return orc.pixel_lists(cam, proj, "brute")
    p = 5 * 16 + 5
    imax = np.iinfo(np.int64).max
    L = lists_for(0.5, 1)                      # borderline Gaussian nearest
    assert L.borderline[p] == 1 and L.bl_first[p] == 0
    assert (L.bl_first[L.borderline == 0] == imax).all() and (L.bl_first[L.borderline == 1] < imax).all()
    L = lists_for(5.0, 1)                      # behind one opaque Gaussian
    assert L.bl_first[p] == 1
    q = orc.qrender(L, 1)
    assert q.n_walked[p] == 1 and L.bl_first[p] <= q.n_walked[p]
    L = lists_for(5.0, 2)                      # behind two: alpha' = 0.8 breaks a K = 1 walk at the first entry
    q = orc.qrender(L, 1)
    assert L.bl_first[p] == 2 and q.n_walked[p] == 1 and not (L.bl_first[p] <= q.n_walked[p])


# --------------------------------------------------------------------------------------------
# G13: backward -- Jacobian rows, adjoint identity, finite differences
# --------------------------------------------------------------------------------------------
def test_G13_backward_adjoint_and_fd(orc, tiny):
    sc, proj, lists = tiny
    K, D = 10, 8
    rng = np.random.default_rng(11)
    F = rng.standard_normal((sc.N, D)).astype(np.float32)
    G = rng.standard_normal((sc.cam.height * sc.cam.width, D)).astype(np.float32)
    q = orc.qrender(lists, K, F)
    dF = orc.backward(q.sel_idx, q.sel_w, q.n_sel, G, sc.N)
    lhs = float((q.out_map.astype(np.float64) * G).sum())        # <render(F), G>
    rhs = float((F.astype(np.float64) * dF).sum())               # <F, backward(G)>
    assert abs(lhs - rhs) <= 1e-6 * max(1.0, abs(lhs))
    # sampled rows agree with the full table
    rows = np.array([0, 5, 17, sc.N - 1], np.int64)
    np.testing.assert_array_equal(orc.backward(q.sel_idx, q.sel_w, q.n_sel, G, sc.N, rows), dF[rows])
    # rows of the Jacobian sum to the identity: backward of G summed over Gaussians = sum over hit pixels of G
    hit = q.n_sel > 0
    np.testing.assert_allclose(dF.sum(0), G[hit].astype(np.float64).sum(0), rtol=1e-9, atol=1e-9)
    # central finite differences of L = <render(F), G> w.r.t. a few entries (render is linear in F)
    touched = np.unique(q.sel_idx[q.sel_idx >= 0])
    for i in touched[:: max(1, len(touched) // 5)][:5]:
        for d in (0, D - 1):
            h = 0.25
            Fp = F.copy(); Fp[i, d] += h
            Fm = F.copy(); Fm[i, d] -= h
            Lp = (orc.qrender(lists, K, Fp).out_map.astype(np.float64) * G).sum()
            Lm = (orc.qrender(lists, K, Fm).out_map.astype(np.float64) * G).sum()
            assert abs((Lp - Lm) / (2 * h) - dF[i, d]) <= 1e-4 * max(1.0, abs(dF[i, d]))


def test_G13_single_gaussian_jacobian_is_identity(orc):
    lists = orc.lists_from_rays([([0], [0.3])])          # normalisation cancels the weight
    q = orc.qrender(lists, 4, np.ones((1, 2), np.float32))
    assert q.n_sel[0] == 1 and abs(q.sel_w[0, 0] - 1.0) < 1e-15
    dF = orc.backward(q.sel_idx, q.sel_w, q.n_sel, np.array([[2.0, -3.0]], np.float32), 1)
    np.testing.assert_allclose(dF, [[2.0, -3.0]])


# --------------------------------------------------------------------------------------------
# G14: Q vs V similarity rises with K (sanity)
# --------------------------------------------------------------------------------------------
def test_G14_q_approaches_v_with_K(orc):
    sc = make_scene("cfg3", seed=2, N=30000, W=96, H=64, D=32)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    v = orc.vrender(lists, sc.features, t_min=0.0)
    sat = v.final_T < 0.01
    assert sat.sum() > 300

    def cos(K):
        q = orc.qrender(lists, K, sc.features).out_map[sat].astype(np.float64)
        r = v.out_map[sat].astype(np.float64)
        return float(((q * r).sum(1) / (np.linalg.norm(q, axis=1) * np.linalg.norm(r, axis=1) + 1e-30)).mean())

    c = [cos(K) for K in (5, 10, 20, 40, 80)]
    assert all(c[i + 1] >= c[i] - 1e-3 for i in range(4)), c
    assert c[3] > 0.97 and c[4] > c[0], c


def test_fp16_features_are_widened_exactly(orc, tiny):
    sc, proj, lists = tiny                                   # reading R14
    f16 = sc.features.astype(np.float16)
    a = orc.qrender(lists, 10, f16).out_map
    b = orc.qrender(lists, 10, f16.astype(np.float32)).out_map
    assert np.array_equal(a, b)


# --------------------------------------------------------------------------------------------
# NEXT-1: top-K render (reading R17)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ray", _gold("topk_rays.json")["rays"], ids=lambda r: r["name"][:2])
def test_topk_hand_worked(orc, ray):
    n = len(ray["alphas"])
    feats = np.eye(n, dtype=np.float32)
    lists = orc.lists_from_rays([(range(n), ray["alphas"])])
    t = orc.topk(lists, ray["K"], feats, t_min=ray["t_min"])
    ns = len(ray["selected"])
    assert t.n_sel[0] == ns and t.n_dense[0] == len(ray["dense_w"])
    assert t.sel_idx[0, :ns].tolist() == ray["selected"] and (t.sel_idx[0, ns:] == -1).all()
    np.testing.assert_allclose(t.sel_w[0, :ns], ray["w_hat"], rtol=2e-6)
    np.testing.assert_allclose(t.resid[0], ray["T_top"], rtol=2e-5)     # products of fp32-rounded alphas
    np.testing.assert_allclose(t.sel_w[0, :ns] * (1.0 - t.resid[0]), ray["w_top"], rtol=2e-6)
    expect = np.zeros(n)
    expect[ray["selected"]] = ray["w_hat"]
    np.testing.assert_allclose(t.out_map[0], expect, rtol=2e-6, atol=1e-12)


def _topk_numpy(alphas, K, t_min):
    """Independent restatement with library routines: cumprod for Eq. 1, a stable argsort for the selection."""
    a = np.asarray(alphas, np.float32)
    T = np.float32(1.0); w = []
    for x in a:                                   # the fp32 decision arithmetic of DESIGN.md: T_test = T * (1 - a), w = T * a
        Tt = np.float32(T * np.float32(np.float32(1.0) - x))
        if Tt < np.float32(t_min):
            break
        w.append(np.float32(T * x)); T = Tt
    w = np.asarray(w, np.float32)
    keep = np.sort(np.argsort(-w, kind="stable")[:K])
    ad = a[keep].astype(np.float64)
    Tex = np.concatenate([[1.0], np.cumprod(1.0 - ad)])
    wt = Tex[:-1] * ad
    resid = Tex[-1] if len(keep) else 1.0
    return keep, (wt / (1.0 - resid) if len(keep) else wt), resid, len(w)


def test_topk_matches_numpy_restatement_on_random_rays(orc):
    rng = np.random.default_rng(11)
    rays = []
    for _ in range(400):
        n = int(rng.integers(0, 70))
        al = np.minimum(0.99, rng.beta(0.7, 2.0, n)).astype(np.float32)
        al[rng.random(n) < 0.15] = np.float32(0.25)            # repeated values: exercises the tie rule
        rays.append((np.arange(n), al))
    lists = orc.lists_from_rays(rays)
    for K, t_min in [(1, 0.0), (4, 1e-4), (10, 1e-4), (40, 0.0), (64, 1e-4)]:
        t = orc.topk(lists, K, None, t_min=t_min)
        for p, (_, al) in enumerate(rays):
            keep, w, resid, nd = _topk_numpy(al, K, t_min)
            assert t.n_dense[p] == nd and t.n_sel[p] == len(keep) == min(K, nd)
            assert t.sel_idx[p, :len(keep)].tolist() == keep.tolist()
            np.testing.assert_allclose(t.sel_w[p, :len(keep)], w, rtol=1e-12)
            np.testing.assert_allclose(t.resid[p], resid, rtol=1e-12)


def test_topk_keeps_the_heaviest_subset_brute_force(orc):
    """Among all K-subsets of the weighted entries the kept one has the largest total dense weight (definition of
    'K largest'), checked by enumeration on tiny rays."""
    import itertools
    rng = np.random.default_rng(12)
    for _ in range(60):
        n = int(rng.integers(1, 9)); K = int(rng.integers(1, 5))
        al = rng.uniform(0.02, 0.9, n).astype(np.float32)
        t = orc.topk(orc.lists_from_rays([(np.arange(n), al)]), K, None, t_min=0.0)
        T = np.concatenate([[1.0], np.cumprod(1.0 - al.astype(np.float64))])[:-1]
        w = T * al
        best = max(itertools.combinations(range(n), min(K, n)), key=lambda c: sum(w[list(c)]))
        assert sorted(t.sel_idx[0, :t.n_sel[0]].tolist()) == sorted(best)


def test_topk_limits_and_invariants(orc):
    sc = make_scene("cfg1", seed=3)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    v = orc.vrender(lists, sc.features, t_min=0.0)
    big = orc.topk(lists, 4096, sc.features, t_min=0.0)          # K >= every list: V-Render / (1 - T)
    has = big.n_sel > 0
    np.testing.assert_allclose(big.out_map[has], v.out_map[has] / (1.0 - v.final_T[has, None]), rtol=2e-6, atol=1e-7)
    np.testing.assert_allclose(big.resid[has], v.final_T[has], rtol=1e-12)
    t = orc.topk(lists, 8, sc.features, t_min=1e-4)
    assert (t.n_sel == np.minimum(8, t.n_dense)).all()
    np.testing.assert_allclose(t.sel_w.sum(1)[t.n_sel > 0], 1.0, rtol=1e-12)      # same normalisation as Algorithm 1 line 20
    assert (t.sel_w >= 0).all() and ((t.resid >= 0) & (t.resid <= 1)).all()
    assert (t.out_map[t.n_sel == 0] == 0).all() and (t.resid[t.n_sel == 0] == 1).all()        # R8
    # kept entries come back in depth order: positions inside the pixel's list strictly increase
    for p in np.flatnonzero(t.n_sel > 1)[:300]:
        ids, _ = lists.ray(p)
        pos = [int(np.flatnonzero(ids == g)[0]) for g in t.sel_idx[p, :t.n_sel[p]]]
        assert pos == sorted(pos)
    with pytest.raises(ValueError):
        orc.topk(lists, 0, None)                                                  # K = 0 is a domain error


# --------------------------------------------------------------------------------------------
# NEXT-3: stratified-K (reading R18)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ray", _gold("stratified_rays.json")["rays"], ids=lambda r: r["name"][:2])
def test_stratified_hand_worked(orc, ray):
    n = len(ray["alphas"])
    feats = np.eye(n, dtype=np.float32)
    lists = orc.lists_from_rays([(range(n), ray["alphas"])])
    t = orc.stratified(lists, ray["K"], feats, t_min=ray["t_min"])
    ns = len(ray["selected"])
    assert t.n_dense[0] == len(ray["T"])
    np.testing.assert_allclose(t.mu[0], ray["mu"], rtol=1e-6)
    np.testing.assert_allclose(t.sigma[0], ray["sigma"], rtol=2e-5, atol=1e-7)
    assert t.n_sel[0] == ns and t.sel_idx[0, :ns].tolist() == ray["selected"] and (t.sel_idx[0, ns:] == -1).all()
    np.testing.assert_allclose(t.sel_w[0, :ns], ray["w_hat"], rtol=1e-6)
    np.testing.assert_allclose(t.resid_TQ[0], ray["TQ"], rtol=1e-6)
    np.testing.assert_allclose(t.sel_w[0, :ns] * (1.0 - t.resid_TQ[0]), ray["wQ"], rtol=1e-6)
    expect = np.zeros(n)
    expect[ray["selected"]] = ray["w_hat"]
    np.testing.assert_allclose(t.out_map[0], expect, rtol=1e-6, atol=1e-12)


def _stratified_numpy(alphas, K, t_min, z_max=2.0):
    """Independent restatement: library cumprod / mean / std for the statistics (fp64, then compared through the
    boundaries' effect), and the level characterisation of Algorithm 1 (selected <=> the number of
    boundaries below which T lies grows) instead of the sequential listing."""
    f32 = np.float32
    a = np.asarray(alphas, f32)
    T = f32(1.0); Ts = []
    for x in a:                                   # fp32 decision arithmetic: T_test = T * (1 - a)
        Tt = f32(T * f32(f32(1.0) - x))
        if Tt < f32(t_min):
            break
        T = Tt; Ts.append(T)
    nd = len(Ts)
    S1 = f32(0.0); S2 = f32(0.0)
    for v in Ts:
        S1 = f32(S1 + v)
        S2 = f32(np.float64(v) * np.float64(v) + np.float64(S2))       # fmaf: one rounding
    if nd:
        mu = f32(S1 / f32(nd)); var = f32(f32(S2 / f32(nd)) - f32(mu * mu)); sg = f32(np.sqrt(max(var, f32(0.0))))
    else:
        mu = sg = f32(0.0)
    if sg > 0:
        b = []
        for k in range(K):
            z = f32(f32(z_max) * f32(f32(1.0) - f32(f32(2 * (k + 1)) / f32(K + 1))))
            b.append(min(max(f32(np.float64(sg) * np.float64(z) + np.float64(mu)), f32(0.0)), f32(1.0)))
        b = np.asarray(b, f32)
    else:
        b = np.asarray([f32(1.0) - f32(k + 1) / f32(K + 1) for k in range(K)], f32)
    level = lambda t: int((t < b).sum())          # boundaries are non-increasing in k
    sel = []; T = f32(1.0)
    for s, x in enumerate(a):
        Tt = f32(T * f32(f32(1.0) - x))
        if level(Tt) > level(T) if s else level(Tt) > 0:
            sel.append(s)
        if Tt < b[-1] or Tt < f32(t_min):
            break
        T = Tt
    return sel, float(mu), float(sg), nd, b


def test_stratified_matches_numpy_restatement_on_random_rays(orc):
    rng = np.random.default_rng(13)
    rays = []
    for _ in range(300):
        n = int(rng.integers(0, 60))
        rays.append((np.arange(n), np.minimum(0.99, rng.beta(0.7, 2.5, n)).astype(np.float32)))
    lists = orc.lists_from_rays(rays)
    for K, t_min in [(1, 0.0), (4, 1e-4), (10, 1e-4), (40, 1e-4), (40, 0.0)]:
        t = orc.stratified(lists, K, None, t_min=t_min)
        for p, (_, al) in enumerate(rays):
            sel, mu, sg, nd, b = _stratified_numpy(al, K, t_min)
            assert t.n_dense[p] == nd
            assert t.mu[p] == np.float32(mu) and t.sigma[p] == np.float32(sg), (p, t.mu[p], mu, t.sigma[p], sg)
            assert t.sel_idx[p, :t.n_sel[p]].tolist() == sel, (K, p)
            assert (np.diff(b) <= 0).all()                            # boundaries descend with k
            if sg > 0:
                assert (b >= max(mu - 2 * sg, 0) - 1e-6).all() and (b <= min(mu + 2 * sg, 1) + 1e-6).all()


def test_stratified_statistics_against_library_routines(orc):
    """mu and sigma are the mean and population standard deviation of the dense transmittance (np.cumprod / mean / std)."""
    rng = np.random.default_rng(14)
    rays = [(np.arange(n), rng.uniform(0.02, 0.6, n).astype(np.float32)) for n in rng.integers(2, 40, 100)]
    t = orc.stratified(orc.lists_from_rays(rays), 8, None, t_min=0.0)
    for p, (_, al) in enumerate(rays):
        T = np.cumprod(1.0 - al.astype(np.float64))
        np.testing.assert_allclose(t.mu[p], T.mean(), rtol=2e-6)
        np.testing.assert_allclose(t.sigma[p], T.std(), rtol=1e-3, atol=2e-6)     # fp32 E[T^2] - mu^2 cancels


def test_stratified_fallback_invariants_and_domain(orc):
    sc = make_scene("cfg1", seed=3)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    t = orc.stratified(lists, 8, sc.features, t_min=1e-4)
    q = orc.qrender(lists, 8, sc.features)
    flat = t.sigma == 0                                          # sigma = 0 -> Q-Render's partition, except that the
    one = flat & (t.n_dense == 1)                                # walk also ends at the dense stop; single-entry rays cannot reach it
    assert one.sum() > 0
    assert (t.sel_idx[one] == q.sel_idx[one]).all() and np.allclose(t.out_map[one], q.out_map[one])
    assert (t.n_sel <= 8).all() and (t.n_sel >= 0).all()
    np.testing.assert_allclose(t.sel_w.sum(1)[t.n_sel > 0], 1.0, rtol=1e-12)          # Algorithm 1 line 20
    assert (t.out_map[t.n_sel == 0] == 0).all() and (t.resid_TQ[t.n_sel == 0] == 1).all()     # R8
    with pytest.raises(ValueError):
        orc.stratified(lists, 0, None)


# --------------------------------------------------------------------------------------------
# NEXT-2: de-voxelisation (Listing 3) and the mask-pooled contrastive loss (Eq. 2;
# DESIGN.md reading R19)
# --------------------------------------------------------------------------------------------
def test_devoxelize_examples_and_library_routines(orc):
    u = np.array([[1, 2], [3, 0]], np.float32)                       # rows (1,2), (3,0)
    assert orc.devoxelize(u, [0, 1], [2], "max")[0].tolist() == [[3.0, 2.0]]
    assert orc.devoxelize(u, [0, 1], [2], "mean")[0].tolist() == [[2.0, 1.0]]
    rng = np.random.default_rng(15)
    U, C_, G = 300, 7, 120
    uni = rng.standard_normal((U, C_)).astype(np.float32)
    counts = rng.integers(0, 6, G); counts[5] = 0
    inv = rng.integers(0, U, counts.sum())
    off = np.concatenate([[0], np.cumsum(counts)])
    vox = uni[inv].astype(np.float64)                                 # step 1: expansion by the inverse index
    mx, am = orc.devoxelize(uni, inv, counts, "max")
    mn, _ = orc.devoxelize(uni, inv, counts, "mean")
    ne = counts > 0
    # step 2 with NumPy's segmented reductions (reduceat needs non-empty segments)
    np.testing.assert_array_equal(mx[ne], np.maximum.reduceat(vox, off[:-1][ne], axis=0))
    np.testing.assert_allclose(mn[ne], np.add.reduceat(vox, off[:-1][ne], axis=0) / counts[ne, None], rtol=1e-13)
    assert (mx[~ne] == 0).all() and (mn[~ne] == 0).all() and (am[~ne] == -1).all()
    one = np.ones(U, np.int64)                                        # centre sampling, 1 voxel per Gaussian
    perm = rng.permutation(U)
    for mode in ("max", "mean"):
        np.testing.assert_array_equal(orc.devoxelize(uni, perm, one, mode)[0], uni[perm].astype(np.float64))
    with pytest.raises(ValueError):
        orc.devoxelize(uni, [0, U], [2], "max")                       # index out of range
    # first voxel wins a tie for the max
    _, am2 = orc.devoxelize(np.array([[1.0], [1.0]], np.float32), [0, 1, 0], [3], "max")
    assert am2[0, 0] == 0


def test_devoxelize_backward_is_the_adjoint(orc):
    rng = np.random.default_rng(16)
    U, C_, G = 80, 5, 40
    uni = rng.standard_normal((U, C_)).astype(np.float32)
    counts = rng.integers(0, 5, G)
    inv = rng.integers(0, U, counts.sum())
    dgs = rng.standard_normal((G, C_)).astype(np.float32)
    # mean is linear: <devox(uni), dgs> = <uni, devox^T(dgs)>
    mn, _ = orc.devoxelize(uni, inv, counts, "mean")
    du = orc.devoxelize_backward(U, inv, counts, "mean", None, dgs)
    np.testing.assert_allclose((mn * dgs).sum(), (uni.astype(np.float64) * du).sum(), rtol=1e-12)
    # max: gradient lands on the arg max only; finite differences where the maximiser is unique
    mx, am = orc.devoxelize(uni, inv, counts, "max")
    dm = orc.devoxelize_backward(U, inv, counts, "max", am, dgs)
    h = 1e-3
    for _ in range(20):
        u, c = int(rng.integers(U)), int(rng.integers(C_))
        up = uni.copy(); up[u, c] += h
        um = uni.copy(); um[u, c] -= h
        fd = ((orc.devoxelize(up, inv, counts, "max")[0] - orc.devoxelize(um, inv, counts, "max")[0]) * dgs).sum() / (2 * h)
        assert abs(fd - dm[u, c]) < 1e-3 * (1 + abs(fd)) or abs(abs(fd) - abs(dm[u, c])) < 0.6 * abs(dgs).max()   # kink within h


def test_mask_loss_closed_forms_and_gradient(orc):
    t = np.array([[1, 0, 0], [0, 1, 0]], np.float32)
    # rendered = positive, one orthogonal negative -> -log(e / (e + 1))
    r = orc.mask_loss(np.array([[2.0, 0, 0]], np.float32), [0], t)
    assert abs(r.loss - (-math.log(math.e / (math.e + 1)))) < 1e-12
    # similarity 0 to both -> log 2
    r = orc.mask_loss(np.array([[0, 0, 5.0]], np.float32), [0], t)
    assert abs(r.loss - math.log(2)) < 1e-12
    # pooling is the arithmetic mean over the mask; pixels outside every mask get no gradient; loss = mean over masks
    rng = np.random.default_rng(17)
    P_, D, S = 60, 6, 4
    fmap = rng.standard_normal((P_, D)).astype(np.float32)
    mid = rng.integers(-1, S, P_).astype(np.int32)
    mid[mid == 2] = -1                                               # mask 2 is empty
    tg = rng.standard_normal((S, D)).astype(np.float32)
    r = orc.mask_loss(fmap, mid, tg)
    for s in (0, 1, 3):
        np.testing.assert_allclose(r.pooled[s], fmap[mid == s].astype(np.float64).mean(0), rtol=1e-12)
    assert r.loss_per_mask[2] == 0 and abs(r.loss - r.loss_per_mask[[0, 1, 3]].mean()) < 1e-12
    assert (r.d_map[mid < 0] == 0).all()
    # independent restatement with library routines (log-sum-exp of cosine similarities)
    for s in (0, 1, 3):
        p = r.pooled[s]
        cs = (tg.astype(np.float64) @ p) / (np.linalg.norm(tg.astype(np.float64), axis=1) * np.linalg.norm(p))
        assert abs(r.loss_per_mask[s] - (np.log(np.exp(cs).sum()) - cs[s])) < 1e-12
    # central finite differences of the total loss w.r.t. map entries
    h = 1e-3
    for _ in range(25):
        p, d = int(rng.integers(P_)), int(rng.integers(D))
        a = fmap.copy(); a[p, d] += h
        b = fmap.copy(); b[p, d] -= h
        fd = (orc.mask_loss(a, mid, tg).loss - orc.mask_loss(b, mid, tg).loss) / (2 * h)
        assert abs(fd - r.d_map[p, d]) < 2e-5 + 1e-3 * abs(fd)
    # adding a duplicate negative strictly increases the loss
    r1 = orc.mask_loss(fmap, mid, np.concatenate([tg, tg[1:2]]))
    assert r1.loss > r.loss


def test_tile_rectangles_cover_every_included_pixel_of_elongated_gaussians(orc):
    """Rule R4 is per pixel; the tile rectangle must be a superset of it.  Needle-like Gaussians (scale ratio 1000:1, random
    orientation: ill-conditioned cov2d, where the fp32-inverted conic's ellipse and the AABB of cov2d drift apart) placed so that
    they straddle tile edges: every (pixel, Gaussian) pair of the brute-force per-pixel lists lies inside that Gaussian's tile
    rectangle, and the binned lists equal the brute-force ones."""
    rng = np.random.default_rng(19)
    cam = make_camera(96, 64)
    n = 400
    means = np.stack([rng.uniform(-1.2, 1.2, n), rng.uniform(-0.8, 0.8, n), rng.uniform(1.5, 3.0, n)], 1).astype(np.float32)
    scales = np.stack([rng.uniform(0.2, 0.6, n), rng.uniform(2e-4, 6e-4, n), rng.uniform(2e-4, 6e-4, n)], 1).astype(np.float32)
    q = rng.standard_normal((n, 4)).astype(np.float32)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    opac = rng.uniform(0.3, 0.99, n).astype(np.float32)
    proj = orc.project(cam, means, scales, q, opac)
    rect, touched = orc.tile_rects(cam, proj)
    brute = orc.pixel_lists(cam, proj, "brute")
    binned = orc.pixel_lists(cam, proj, "binned")
    assert np.array_equal(brute.off, binned.off) and np.array_equal(brute.gid, binned.gid)
    assert len(brute.gid) > 2000
    pix = np.repeat(np.arange(cam.width * cam.height), np.diff(brute.off))
    tx, ty = (pix % cam.width) // 16, (pix // cam.width) // 16
    r = rect[brute.gid]
    assert ((tx >= r[:, 0]) & (tx < r[:, 2]) & (ty >= r[:, 1]) & (ty < r[:, 3])).all()
    assert (touched[np.unique(brute.gid)] > 0).all()


# ---------------------------------------------------------------------------------------------------------------
# spherical-harmonics colour (reading R20)
# ---------------------------------------------------------------------------------------------------------------
def test_sh_basis_equals_scipys_complex_harmonics(orc):
    """R20 defines the basis through the complex Y_l^m: Y_{l,0} = Y_l^0, Y_{l,m} = sqrt2 Re Y_l^m, Y_{l,-m} = sqrt2 Im Y_l^m
    (phase kept).  scipy.special evaluates Y_l^m from its own recurrences; the oracle's polynomials must agree at random
    directions, for every degree (a wrong constant, sign, or swapped pair of indices fails)."""
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(3)
    for _ in range(200):
        d = rng.standard_normal(3)
        d /= np.linalg.norm(d)
        theta, phi = math.acos(d[2]), math.atan2(d[1], d[0])
        want = []
        for l in range(4):
            for m in range(-l, l + 1):
                y = complex(sph_harm_y(l, abs(m), theta, phi))
                want.append(y.real if m == 0 else math.sqrt(2) * (y.real if m > 0 else y.imag))
        got = orc.sh_basis(3, d)
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)
        for deg in range(3):
            np.testing.assert_allclose(orc.sh_basis(deg, d), want[:(deg + 1) ** 2], rtol=0, atol=1e-13)


def test_sh_basis_is_orthonormal_on_the_sphere(orc):
    """Integral over the sphere of Y_i Y_j = delta_ij: Gauss-Legendre in cos(theta) x uniform phi integrates products of
    degree <= 6 polynomials exactly."""
    xs, ws = np.polynomial.legendre.leggauss(8)
    nphi = 16
    G = np.zeros((16, 16))
    for z, w in zip(xs, ws):
        s = math.sqrt(1 - z * z)
        for k in range(nphi):
            p = 2 * math.pi * k / nphi
            Y = orc.sh_basis(3, [s * math.cos(p), s * math.sin(p), z])
            G += w * (2 * math.pi / nphi) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), rtol=0, atol=1e-12)


def test_sh_basis_hand_values(orc):
    """Values anyone can check by hand: Y_0 = 1/(2 sqrt(pi)); at the north pole only the m = 0 terms survive,
    Y_{l,0}(z = 1) = sqrt((2 l + 1) / (4 pi)); along +x the degree-1 terms are (0, 0, -sqrt(3 / (4 pi)))."""
    Y = orc.sh_basis(3, [0.0, 0.0, 1.0])
    want = np.zeros(16)
    for l, k in ((0, 0), (1, 2), (2, 6), (3, 12)):
        want[k] = math.sqrt((2 * l + 1) / (4 * math.pi))
    np.testing.assert_allclose(Y, want, rtol=0, atol=1e-15)
    assert abs(Y[0] - 0.28209479177387814) < 1e-16
    Yx = orc.sh_basis(1, [1.0, 0.0, 0.0])
    np.testing.assert_allclose(Yx, [0.28209479177387814, 0.0, 0.0, -math.sqrt(3 / (4 * math.pi))], rtol=0, atol=1e-15)


def test_sh_colors_definition_and_special_cases(orc):
    """colour = max(0, 1/2 + sum_k Y_k(dir) sh_k) with dir from the camera CENTRE (-R^T t) to the mean: restated in NumPy on
    the pinned basis with a rotated, translated camera; degree 0 is view independent; a Gaussian at the camera centre keeps
    only the constant term; negative sums clamp to 0."""
    rng = np.random.default_rng(5)
    cam = make_camera(64, 48)
    # a non-trivial pose: rotate about y by 0.4 rad, about x by -0.2 rad, translate
    cy, sy, cx, sx = math.cos(0.4), math.sin(0.4), math.cos(-0.2), math.sin(-0.2)
    R = np.array([[1, 0, 0], [0, cx, -sx], [0, sx, cx]]) @ np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]])
    t = np.array([0.3, -0.2, 1.5])
    cam.world_to_cam = np.concatenate([R, t[:, None]], 1).astype(np.float32)
    Rf, tf = cam.world_to_cam[:, :3].astype(np.float64), cam.world_to_cam[:, 3].astype(np.float64)
    centre = -Rf.T @ tf
    N = 300
    means = rng.uniform(-2, 2, (N, 3)).astype(np.float32)
    means[7] = centre.astype(np.float32)
    for deg in range(4):
        nb = (deg + 1) ** 2
        sh = (rng.standard_normal((N, nb, 3)) * 0.8).astype(np.float32)
        got = orc.sh_colors(cam, means, sh, deg)
        for i in range(N):
            d = means[i].astype(np.float64) - centre
            n = np.linalg.norm(d)
            if n == 0 or i == 7 and n < 1e-6:
                continue
            Y = orc.sh_basis(deg, d / n)
            want = np.maximum(0.0, 0.5 + Y @ sh[i].astype(np.float64))
            np.testing.assert_allclose(got[i], want, rtol=0, atol=1e-12)
        assert (got >= 0).all() and (got == 0).any()
        if deg == 0:
            cam2 = make_camera(64, 48)
            np.testing.assert_array_equal(got, orc.sh_colors(cam2, means, sh, 0))
    # exactly at the centre (float32 centre may differ from the float64 one: build the camera so that it is exact)
    cam3 = make_camera(64, 48)
    cam3.world_to_cam = np.concatenate([np.eye(3), np.array([[0.5], [0.25], [-1.0]])], 1).astype(np.float32)
    m3 = np.array([[-0.5, -0.25, 1.0]], np.float32)
    sh3 = rng.standard_normal((1, 16, 3)).astype(np.float32)
    np.testing.assert_allclose(orc.sh_colors(cam3, m3, sh3, 3)[0], np.maximum(0, 0.5 + 0.28209479177387814 * sh3[0, 0].astype(np.float64)), atol=1e-15)
