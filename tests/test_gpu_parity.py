"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Stage-isolated (each GPU stage fed the oracle's upstream outputs) and end to end, at sizes the oracle finishes in
seconds that still span several tiles and ragged tails, plus sampled checks at BASELINE.json's config-3 size.
"""
import math

import numpy as np
import pytest
import torch

from qr_inputs import make_scene, make_camera
import parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qr():
    import paper_2512_20927_b200 as q
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    q.binding.load()
    return q


def _i32(t):
    return t.cpu().numpy()


# ------------------------------------------------------------------------------------------------
# qr_preprocess: bit-exact against the oracle's fp32 decision arithmetic
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw", [("cfg1", {}), ("cfg2", dict(N=20000)), ("cfg3", dict(N=60000, W=200, H=120, D=8)),
                                     ("cfg4", dict(N=60000, W=160, H=96, D=8, pose=3, feat_dtype="f32"))])
def test_preprocess_bit_exact(qr, orc, name, kw):
    sc = make_scene(name, seed=1, **kw)
    g = P.upload(sc)
    pr = qr.qr_preprocess(sc.cam, g.means, g.scales, g.quats, g.opac)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    rect, touched = orc.tile_rects(sc.cam, proj)
    np.testing.assert_array_equal(pr.depth.cpu().numpy().view(np.uint32), proj.depth.view(np.uint32))
    np.testing.assert_array_equal(pr.mean2d.cpu().numpy().view(np.uint32), proj.mean2d.view(np.uint32))
    np.testing.assert_array_equal(pr.conic_opac.cpu().numpy().view(np.uint32), proj.conic_opac.view(np.uint32))
    np.testing.assert_array_equal(_i32(pr.tile_rect), rect)
    np.testing.assert_array_equal(_i32(pr.tiles_touched).view(np.uint32), touched)
    assert touched.sum() > 0


# ------------------------------------------------------------------------------------------------
# qr_bin_count / qr_bin_sort: exact lists and ranges
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw", [("cfg1", {}), ("cfg2", dict(N=30000)), ("cfg3", dict(N=80000, W=330, H=250, D=8))])
def test_bin_sort_exact(qr, orc, name, kw):
    sc = make_scene(name, seed=2, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    # stage-isolated: feed the oracle's projection
    offsets, M = qr.qr_bin_count(P.to_dev(touched.view(np.int32)))
    assert M == int(touched.sum()) == len(isect)
    np.testing.assert_array_equal(offsets.cpu().numpy(), np.cumsum(touched.astype(np.int64)))
    ig, tr = qr.qr_bin_sort(sc.cam, M, P.to_dev(proj.depth), P.to_dev(rect), offsets)
    np.testing.assert_array_equal(_i32(ig).view(np.uint32), isect)
    np.testing.assert_array_equal(_i32(tr), rng)
    # end to end
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    assert fe.M == M
    np.testing.assert_array_equal(_i32(fe.isect_gauss).view(np.uint32), isect)
    np.testing.assert_array_equal(_i32(fe.tile_range), rng)


def test_bin_sort_depth_ties_break_by_index(qr, orc):
    """R6: equal depths keep ascending Gaussian index (stable sort)."""
    sc = make_scene("cfg1", seed=3, N=600)
    sc.means[:, 2] = np.float32(3.0)             # all depths equal
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    np.testing.assert_array_equal(_i32(fe.isect_gauss).view(np.uint32), isect)
    for t in range(rng.shape[0]):
        ids = isect[rng[t, 0]:rng[t, 1]]
        assert (np.diff(ids.astype(np.int64)) > 0).all()


@pytest.mark.parametrize("N,scale", [(12000, 1.0), (60000, 3.0)])
def test_bin_sort_crowded_tiles(qr, orc, N, scale):
    """Tile buckets beyond one shared-memory sort: > 2,048 keys (big-bucket kernel) and > 16,384 keys (several sorted
    runs merged by rank) in a 48x40 image; duplicated depths keep ascending index."""
    sc = make_scene("cfg1", seed=11, N=N, W=48, H=40)
    sc.scales *= np.float32(scale)
    sc.means[::7, 2] = np.float32(4.0)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    per_tile = (rng[:, 1] - rng[:, 0]).max()
    assert per_tile > (16384 if scale > 1 else 2048), per_tile
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    assert fe.M == len(isect)
    np.testing.assert_array_equal(_i32(fe.tile_range), rng)
    np.testing.assert_array_equal(_i32(fe.isect_gauss).view(np.uint32), isect)


def test_bin_sort_with_capacity_instead_of_count(qr, orc):
    """qr_bin_sort with M = an upper bound (no qr_bin_count, no host synchronisation): same lists and ranges, the
    found count is reported on the device; with a bound that is too small the lists are truncated, never overrun."""
    sc = make_scene("cfg3", seed=13, N=80000, W=330, H=250, D=6)      # D = 6: a deterministic blend (the tcgen05 path's summation order follows a race)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    g = P.upload(sc)
    M = len(isect)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac, capacity=M + 1000)
    assert int(fe.found.item()) == M and fe.M == M + 1000
    np.testing.assert_array_equal(_i32(fe.tile_range), rng)
    np.testing.assert_array_equal(_i32(fe.isect_gauss)[:M].view(np.uint32), isect)
    out_a = qr.pipeline.forward(sc.cam, fe, g.features, 40)
    out_b = qr.pipeline.forward(sc.cam, qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac), g.features, 40)
    ia, wa, na = P.masked_records(out_a)
    ib, wb, nb = P.masked_records(out_b)
    assert (ia == ib).all() and (na == nb).all() and torch.equal(out_a.out_map, out_b.out_map)
    # too small: truncated at the capacity, ranges clamped, the true count still reported
    cap = M // 2
    fe2 = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac, capacity=cap)
    assert int(fe2.found.item()) == M
    tr = _i32(fe2.tile_range)
    np.testing.assert_array_equal(tr, np.minimum(rng, cap))
    whole = int(rng[rng[:, 1] <= cap, 1].max())            # tiles that fit entirely are exact; the one cut at cap keeps
    np.testing.assert_array_equal(_i32(fe2.isect_gauss)[:whole].view(np.uint32), isect[:whole])   # an arbitrary part
    qr.pipeline.forward(sc.cam, fe2, g.features, 40)        # runs on the truncated lists without touching anything else
    torch.cuda.synchronize()


def test_bin_empty_scene(qr):
    """Everything culled (behind the camera): M = 0, all ranges empty, forward renders zeros."""
    sc = make_scene("cfg1", seed=0, N=50)
    sc.means[:, 2] = -1.0
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    assert fe.M == 0
    assert (fe.tile_range.cpu().numpy() == 0).all()
    out = qr.pipeline.forward(sc.cam, fe, g.features, 40)
    assert (out.out_map == 0).all() and (out.n_sel == 0).all() and (out.resid_TQ == 1).all()


# ------------------------------------------------------------------------------------------------
# qr_forward
# ------------------------------------------------------------------------------------------------
FWD_CASES = [
    ("cfg1", dict(), 40),                                       # BASELINE config 1 as given
    ("cfg1", dict(W=70, H=50, D=3), 40),                        # ragged tiles, scalar-channel path
    ("cfg1", dict(W=33, H=17, D=20), 1),                        # K = 1
    ("cfg1", dict(D=132), 7),                                   # D % 128 != 0
    ("cfg2", dict(N=20000, W=128, H=96), 40),
    ("cfg2", dict(N=20000, W=96, H=64, D=256), 64),
    ("cfg3", dict(N=60000, W=160, H=112, D=512), 40),           # blob scene, camera inside, D = 512
    ("cfg3", dict(N=60000, W=96, H=64, D=384), 10),
    ("cfg3", dict(N=40000, W=96, H=64, D=64), 200),             # K large
    ("cfg1", dict(W=70, H=50, D=256), 40),                      # tcgen05 blend on a ragged image (store guard, skipped half tiles)
    ("cfg3", dict(N=60000, W=100, H=72, D=512), 5),
    ("cfg3", dict(N=40000, W=100, H=72, D=160), 40),            # tcgen05 path on padded tiles: 128 + 32 channels
    ("cfg2", dict(N=20000, W=70, H=50, D=96), 12),              # ... one partial tile, ragged image
    ("cfg1", dict(W=70, H=50, D=4), 40),                        # ... the smallest: 4 of 128 channels
    ("cfg3", dict(N=40000, W=100, H=72, D=3), 40),              # thread = pixel blend (D <= 8, D % 4 != 0)
    ("cfg2", dict(N=20000, W=64, H=48, D=7), 12),
    ("cfg1", dict(W=33, H=17, D=1), 3),
]


@pytest.mark.parametrize("name,kw,K", FWD_CASES)
def test_forward_stage_isolated(qr, orc, name, kw, K):
    sc = make_scene(name, seed=4, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, sc.features)
    out = qr.qr_forward(sc.cam, K, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac),
                        P.to_dev(isect.view(np.int32)), P.to_dev(rng), P.to_dev(sc.features))
    stats = P.compare_forward(out, q, lists, K, sc.D)
    assert stats["exempt"] < 0.01 * stats["pixels"] + 5, stats
    print(name, kw, K, stats)


@pytest.mark.parametrize("name,kw,K", [FWD_CASES[0], FWD_CASES[4], FWD_CASES[6]])
def test_forward_end_to_end(qr, orc, name, kw, K):
    sc = make_scene(name, seed=5, **kw)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, g.features, K)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, sc.features)
    stats = P.compare_forward(out, q, lists, K, sc.D)
    print(stats)


@pytest.mark.parametrize("D", [512, 64, 24, 40])      # 64, 24: padded 128-channel tile; 40: D % 32 != 0 -> blend_tu_kernel
def test_forward_fp16_features(qr, orc, D):
    sc = make_scene("cfg4", seed=6, N=60000, W=128, H=96, D=D, pose=2)        # fp16 storage, fp32 accumulation (R14)
    assert sc.features.dtype == np.float16
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    for K in (4, 32):
        q = orc.qrender(lists, K, sc.features)
        out = qr.qr_forward(sc.cam, K, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac),
                            P.to_dev(isect.view(np.int32)), P.to_dev(rng), P.to_dev(sc.features))
        P.compare_forward(out, q, lists, K, sc.D, f16=True)


def test_forward_invariants_full_scale(qr):
    """Properties that hold at any size, checked on the GPU output of a mid-size scene."""
    sc = make_scene("cfg3", seed=7, N=200000, W=320, H=240, D=128)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    K = 40
    out = qr.pipeline.forward(sc.cam, fe, g.features, K)
    idx, w, n_sel = P.masked_records(out)
    n_sel = n_sel.reshape(out.n_sel.shape)
    w = w.astype(np.float64).reshape(out.sel_w.shape)
    assert n_sel.max() <= K and n_sel.min() >= 0
    assert (w >= 0).all()
    has = n_sel > 0
    np.testing.assert_allclose(w.sum(-1)[has], 1.0, atol=1e-5)   # convex combination (G3); 1 - T^Q can be ~0.03 in fp32
    # constant feature scene: out == f wherever something is selected (G5)
    const = torch.ones_like(g.features) * 0.25
    out_c = qr.pipeline.forward(sc.cam, fe, const, K)
    np.testing.assert_allclose(out_c.out_map.cpu().numpy()[has], 0.25, rtol=1e-5)
    assert (P.masked_records(out_c)[0] == idx).all()                            # selection independent of payload (G6)
    # payload width independence
    out_3 = qr.pipeline.forward(sc.cam, fe, g.features[:, :3].contiguous(), K)
    assert (P.masked_records(out_3)[0] == idx).all()
    np.testing.assert_allclose(out_3.out_map.cpu().numpy(), out.out_map[..., :3].cpu().numpy(), rtol=2e-5, atol=1e-6)   # FFMA vs tcgen05 path


# ------------------------------------------------------------------------------------------------
# qr_dense_forward (Eq. 1)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw,t_min", [("cfg1", dict(), 1e-4), ("cfg1", dict(W=70, H=50, D=3), 0.0),
                                           ("cfg3", dict(N=60000, W=128, H=80, D=512), 1e-4),
                                           ("cfg2", dict(N=20000, W=96, H=96), 0.0)])
def test_dense_forward(qr, orc, name, kw, t_min):
    sc = make_scene(name, seed=8, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    v = orc.vrender(lists, sc.features, t_min=t_min)
    om, fT = qr.qr_dense_forward(sc.cam, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac),
                                 P.to_dev(isect.view(np.int32)), P.to_dev(rng), P.to_dev(sc.features), t_min)
    H, W = sc.cam.height, sc.cam.width
    om = om.cpu().numpy().reshape(H * W, -1).astype(np.float64); fT = fT.cpu().numpy().reshape(-1)
    ok = ~((v.stop_margin <= 1e-5) | lists.borderline.astype(bool))       # early-stop decision within rounding
    assert ok.mean() > 0.99
    ref = v.out_map.astype(np.float64)
    tol = P.ATOL + P.RTOL * np.abs(ref)
    assert (np.abs(om - ref)[ok] <= tol[ok]).all()
    np.testing.assert_allclose(fT[ok], v.final_T[ok], rtol=1e-4, atol=1e-7)


@pytest.mark.parametrize("name,kw,t_min,cap", [("cfg3", dict(N=60000, W=128, H=80, D=512), 1e-4, 128),
                                               ("cfg3", dict(N=60000, W=100, H=72, D=256), 0.0, 256),      # ragged, exact Eq. 1
                                               ("cfg2", dict(N=20000, W=96, H=96), 1e-4, 64),              # D = 16: padded tile
                                               ("cfg1", dict(W=70, H=50, D=128), 1e-4, 128),
                                               # lists far too small: most half tiles are flagged and go to the FFMA kernel
                                               ("cfg3", dict(N=60000, W=128, H=80, D=128), 1e-4, 4),
                                               ("cfg3", dict(N=60000, W=128, H=80, D=128), 1e-4, 24)])
def test_dense_forward_on_tensor_cores(qr, orc, name, kw, t_min, cap):
    """qr_dense_forward_tc against the oracle's V-Render (the same bar as qr_dense_forward) and against qr_dense_forward."""
    sc = make_scene(name, seed=8, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    v = orc.vrender(lists, sc.features, t_min=t_min)
    args = (sc.cam, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac), P.to_dev(isect.view(np.int32)), P.to_dev(rng), P.to_dev(sc.features), t_min)
    om_t, fT_t, ws = qr.binding.qr_dense_forward_tc(*args, cap)
    om_f, fT_f = qr.qr_dense_forward(*args)
    H, W = sc.cam.height, sc.cam.width
    om = om_t.cpu().numpy().reshape(H * W, -1).astype(np.float64); fT = fT_t.cpu().numpy().reshape(-1)
    ok = ~((v.stop_margin <= 1e-5) | lists.borderline.astype(bool))       # early-stop decision within rounding
    assert ok.mean() > 0.99
    ref = v.out_map.astype(np.float64)
    tol = P.ATOL + P.RTOL * np.abs(ref)
    assert (np.abs(om - ref)[ok] <= tol[ok]).all(), float((np.abs(om - ref)[ok] / tol[ok]).max())
    np.testing.assert_allclose(fT[ok], v.final_T[ok], rtol=1e-4, atol=1e-7)
    assert torch.equal(fT_t, fT_f)                                        # the same fp32 decision arithmetic: identical T
    torch.testing.assert_close(om_t, om_f, rtol=2e-4, atol=2e-5)
    # second call into the same workspace (flags, tickets and lists of the first call are stale)
    om2, fT2, _ = qr.binding.qr_dense_forward_tc(*args, cap, ws=ws)
    assert torch.equal(fT2, fT_t)
    torch.testing.assert_close(om2, om_t, rtol=2e-4, atol=2e-5)


# ------------------------------------------------------------------------------------------------
# qr_backward
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw,K", [("cfg2", dict(N=20000, W=128, H=96), 40),
                                       ("cfg1", dict(W=70, H=50, D=3, backward=True), 40),
                                       ("cfg3", dict(N=60000, W=112, H=80, D=512), 40),
                                       ("cfg3", dict(N=40000, W=96, H=64, D=132), 8),
                                       ("cfg2", dict(N=20000, W=64, H=64, D=64), 100),
                                       # tcgen05 path (D % 128 == 0): ragged image, unions > 64 rows (passes),
                                       # K large enough to split a half tile into several stage ranges
                                       ("cfg1", dict(W=70, H=50, D=128, backward=True), 40),
                                       ("cfg2", dict(N=20000, W=100, H=72, D=256), 40),
                                       ("cfg3", dict(N=60000, W=96, H=64, D=384), 10),
                                       ("cfg3", dict(N=40000, W=64, H=48, D=128), 200),
                                       ("cfg2", dict(N=30000, W=64, H=40, D=128), 256),
                                       # thread = pixel backward (D <= 8, D % 4 != 0); K = 200 on the blob scene overflows
                                       # the tile's shared-memory hash table (direct global atomics for the rest)
                                       # tcgen05 path on padded 128-channel tiles (TMA zero fill, epilogue guard)
                                       ("cfg3", dict(N=40000, W=100, H=72, D=160), 10),
                                       ("cfg2", dict(N=20000, W=70, H=50, D=96), 12),
                                       ("cfg1", dict(W=70, H=50, D=16, backward=True), 40),
                                       ("cfg1", dict(W=70, H=50, D=4, backward=True), 40),
                                       ("cfg3", dict(N=40000, W=100, H=72, D=3), 40),
                                       ("cfg3", dict(N=40000, W=64, H=48, D=3), 200),
                                       ("cfg2", dict(N=20000, W=64, H=48, D=7), 12),
                                       ("cfg1", dict(W=33, H=17, D=1, backward=True), 3)])
def test_backward_stage_isolated(qr, orc, name, kw, K):
    sc = make_scene(name, seed=9, **kw)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, None)
    H, W = sc.cam.height, sc.cam.width
    ref = orc.backward(q.sel_idx, q.sel_w, q.n_sel, sc.dL_dmap, sc.N)
    got = qr.qr_backward(sc.cam, sc.N, P.to_dev(q.sel_idx.reshape(H, W, K)),
                         P.to_dev(q.sel_w.reshape(H, W, K).astype(np.float32)),
                         P.to_dev(q.n_sel.reshape(H, W)), P.to_dev(sc.dL_dmap)).cpu().numpy().astype(np.float64)
    tol = P.ATOL + P.RTOL * np.abs(ref)
    err = np.abs(got - ref)
    assert (err <= tol).all(), float((err / tol).max())
    touched = np.zeros(sc.N, bool); touched[q.sel_idx[q.sel_idx >= 0]] = True
    assert (got[~touched] == 0).all()                       # rows never selected are untouched
    assert touched.sum() > 10


def test_backward_accumulates_and_adjoint(qr, orc):
    """qr_backward adds into dL_dfeat; <render(F), G> == <F, backward(G)> (render is linear in F)."""
    sc = make_scene("cfg3", seed=10, N=60000, W=128, H=96, D=64)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, g.features, 40)
    G = P.to_dev(sc.dL_dmap)
    dF = qr.pipeline.backward(sc.cam, sc.N, out, G)
    lhs = float((out.out_map.double() * G.double()).sum())
    rhs = float((g.features.double() * dF.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * max(abs(lhs), 1.0), (lhs, rhs)
    dF2 = qr.pipeline.backward(sc.cam, sc.N, out, G, dF.clone())
    torch.testing.assert_close(dF2, 2.0 * dF, rtol=1e-5, atol=1e-6)


@pytest.mark.parametrize("name,kw,K", [("cfg3", dict(N=60000, W=112, H=80, D=512), 40),      # tcgen05 path: numbered unions
                                       ("cfg2", dict(N=20000, W=70, H=50, D=64), 40),        # no workspace: per record
                                       ("cfg3", dict(N=40000, W=64, H=48, D=128), 200)])     # over-full half tiles
def test_backward_clear_zeroes_exactly_the_touched_rows(qr, orc, name, kw, K):
    """qr_backward_clear: rows of selected Gaussians become 0, every other row keeps its value (a sentinel)."""
    sc = make_scene(name, seed=12, **kw)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, g.features, K)
    G = P.to_dev(sc.dL_dmap)
    ws = qr.qr_backward_workspace(sc.cam, K, sc.D, G.device)
    dF = torch.full((sc.N, sc.D), 7.0, dtype=torch.float32, device=G.device)
    qr.pipeline.backward(sc.cam, sc.N, out, G, dF, ws)
    qr.pipeline.backward_clear(sc.cam, sc.N, out, dF, ws)
    idx_m = torch.from_numpy(P.masked_records(out)[0]).to(G.device)
    sel = idx_m[idx_m >= 0].long()
    touched = torch.zeros(sc.N, dtype=torch.bool, device=G.device)
    touched[sel] = True
    assert int(touched.sum()) > 10
    assert (dF[touched] == 0).all()
    assert (dF[~touched] == 7.0).all()
    # zero once, then backward / clear / backward gives the same gradient as a fresh table
    dF.zero_()
    qr.pipeline.backward(sc.cam, sc.N, out, G, dF, ws)
    first = dF.clone()
    qr.pipeline.backward_clear(sc.cam, sc.N, out, dF, ws)
    assert (dF == 0).all()
    qr.pipeline.backward(sc.cam, sc.N, out, G, dF, ws)
    torch.testing.assert_close(dF, first, rtol=1e-5, atol=1e-6)


# ------------------------------------------------------------------------------------------------
# full-size checks in the configuration bench.py times
# ------------------------------------------------------------------------------------------------
def _backward_rows_check(qr, orc, sc, K, out, qa, same, n_rows, tag):
    """Gradient parity on sampled dL/dF rows at full size, two ways:
    (a) stage-isolated -- qr_backward on the ORACLE's selection records (every sampled row is comparable);
    (b) end to end -- qr_backward on the GPU forward's own records, compared on the sampled rows that no pixel with a
        differing selection touches (those pixels are the exempt ones; their rows legitimately differ)."""
    H, W = sc.cam.height, sc.cam.width
    G = P.to_dev(sc.dL_dmap)
    sel = qa.sel_idx[qa.sel_idx >= 0]
    rows_all = np.unique(sel)
    rows = rows_all[:: max(1, len(rows_all) // n_rows)][:n_rows].astype(np.int64)
    assert len(rows) >= 100, len(rows)
    ref = orc.backward(qa.sel_idx, qa.sel_w, qa.n_sel, sc.dL_dmap, sc.N, rows=rows)
    A = orc.backward(qa.sel_idx, qa.sel_w, qa.n_sel, np.abs(sc.dL_dmap), sc.N, rows=rows)     # sum |w g| per element
    ridx = torch.from_numpy(rows).cuda()
    # (a)
    dF = qr.qr_backward(sc.cam, sc.N, P.to_dev(qa.sel_idx.reshape(H, W, K)),
                        P.to_dev(qa.sel_w.reshape(H, W, K).astype(np.float32)), P.to_dev(qa.n_sel.reshape(H, W)), G)
    worst_a, over_a = P.compare_backward_rows(dF[ridx].cpu().numpy(), ref, f"{tag} stage-isolated", A)
    del dF
    # (b)
    dF = qr.pipeline.backward(sc.cam, sc.N, out, G)
    got = dF[ridx].cpu().numpy()
    del dF
    bad_px = np.flatnonzero(~same)
    gsel = out.sel_idx.cpu().numpy().reshape(-1, K)
    gn = out.n_sel.cpu().numpy().reshape(-1)
    tainted = set()
    for p in bad_px:
        tainted.update(int(v) for v in gsel[p, :gn[p]])
        tainted.update(int(v) for v in qa.sel_idx[p, :qa.n_sel[p]])
    keep = np.array([int(r) not in tainted for r in rows])
    assert keep.sum() >= 0.8 * len(rows), (int(keep.sum()), len(rows))
    worst_b, over_b = P.compare_backward_rows(got[keep], ref[keep], f"{tag} end-to-end", A[keep])
    print(f"{tag} backward rows: stage-isolated {len(rows)} rows (worst err/tol {worst_a:.3f}, {over_a} elements over the "
          f"plain bar); end-to-end {int(keep.sum())} of {len(rows)} rows (worst {worst_b:.3f}, {over_b} over the plain bar); "
          f"largest fan-in sum|w g| {float(A.max()):.0f}; pixels with differing selection {len(bad_px)}")


def _full_size_check(qr, orc, sc, Ks, n_pix=3000, n_rows=150, f16=False, max_exempt_frac=0.004):
    """Full-size frame in bench.py's launch configuration: selection parity on every pixel, features on sampled
    pixels, gradient rows of sampled Gaussians (the oracle computes those one by one)."""
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    rect, touched = orc.tile_rects(sc.cam, proj)
    assert fe.M == int(touched.sum())
    lists = orc.pixel_lists(sc.cam, proj)
    rng = np.random.default_rng(1)
    pix = np.sort(rng.choice(sc.cam.width * sc.cam.height, size=n_pix, replace=False))
    for K in Ks:
        out = qr.pipeline.forward(sc.cam, fe, g.features, K)
        q = orc.qrender(lists, K, sc.features, pixels=pix)
        stats = P.compare_forward(out, q, lists, K, sc.D, f16=f16, pixels=pix)
        qa = orc.qrender(lists, K, None)
        ex_m, ex_b = P.exempt_classes(qa, lists)
        ex = ex_m | ex_b
        same = P.same_selection(out.sel_idx.cpu().numpy().reshape(-1, K), out.n_sel.cpu().numpy().reshape(-1), qa)
        assert ((~same) & (~ex)).sum() == 0
        print(sc.name, "K", K, "sampled:", stats, "| all pixels:", same.size, "exempt by margin", int(ex_m.sum()),
              "by borderline membership only", int((ex_b & ~ex_m).sum()), "differing (all exempt)", int((~same).sum()))
        assert ex.sum() <= max_exempt_frac * same.size, (int(ex.sum()), same.size)
        if sc.dL_dmap is not None and K == Ks[-1]:
            _backward_rows_check(qr, orc, sc, K, out, qa, same, n_rows, f"{sc.name} K={K}")
        del out


def test_config3_full_size_sampled(qr, orc):
    """BASELINE.json configs[2], the headline: 640x480, 500,000 Gaussians, D = 512 fp32, K = 40, forward + backward."""
    _full_size_check(qr, orc, make_scene("cfg3", seed=0), [40], n_pix=4000, n_rows=200)


def test_config5_full_size_sampled(qr, orc):
    """BASELINE.json configs[4]: 1280x720, 1,000,000 Gaussians, D = 512 fp32, K = 40, forward + backward."""
    _full_size_check(qr, orc, make_scene("cfg5", seed=0), [40])


def test_config5_narrow_payload_full_size(qr, orc):
    """configs[4] D sweep, D = 64: the first 64 columns of the 512-D draw, re-normalised (FFMA blend / backward paths)."""
    sc = make_scene("cfg5", seed=0, D=64)
    _full_size_check(qr, orc, sc, [40], n_pix=2000, n_rows=100)


@pytest.mark.parametrize("pose", [0, 5])
def test_config4_full_size_sampled(qr, orc, pose):
    """BASELINE.json configs[3]: 1024x768, 2,000,000 Gaussians, D = 512 stored fp16 (fp32 accumulation), two poses of
    the radius-3 circle, K = 4 and K = 32."""
    sc = make_scene("cfg4", seed=0, pose=pose)
    assert sc.features.dtype == np.float16
    _full_size_check(qr, orc, sc, [4, 32], n_pix=2000, n_rows=150, f16=True)


@pytest.mark.parametrize("D", [256, 512])
def test_midsize_every_row_many_units_per_cta(qr, orc, D):
    """A frame with more half tiles (600) than SMs (148), so that every persistent CTA of the tcgen05 kernels runs several
    work units (ring wrap-around, accumulator ping-pong), small enough that the oracle produces EVERY pixel and EVERY
    gradient row: forward end to end, backward both on the oracle's records and on the forward's own."""
    sc = make_scene("cfg3", seed=21, N=100000, W=320, H=240, D=D)
    K = 40
    H, W = sc.cam.height, sc.cam.width
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, g.features, K)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, sc.features)
    stats = P.compare_forward(out, q, lists, K, sc.D)
    print("mid-size forward:", stats)
    G = P.to_dev(sc.dL_dmap)
    ref = orc.backward(q.sel_idx, q.sel_w, q.n_sel, sc.dL_dmap, sc.N)
    got = qr.qr_backward(sc.cam, sc.N, P.to_dev(q.sel_idx.reshape(H, W, K)), P.to_dev(q.sel_w.reshape(H, W, K).astype(np.float32)),
                         P.to_dev(q.n_sel.reshape(H, W)), G).cpu().numpy()
    A = orc.backward(q.sel_idx, q.sel_w, q.n_sel, np.abs(sc.dL_dmap), sc.N)
    worst, over = P.compare_backward_rows(got, ref, "mid-size stage-isolated", A)
    same = P.same_selection(out.sel_idx.cpu().numpy().reshape(-1, K), out.n_sel.cpu().numpy().reshape(-1), q)
    got2 = qr.pipeline.backward(sc.cam, sc.N, out, G).cpu().numpy()
    tainted = np.zeros(sc.N, bool)
    gsel = out.sel_idx.cpu().numpy().reshape(-1, K); gn = out.n_sel.cpu().numpy().reshape(-1)
    for p in np.flatnonzero(~same):
        tainted[gsel[p, :gn[p]]] = True
        tainted[q.sel_idx[p, :q.n_sel[p]]] = True
    worst2, over2 = P.compare_backward_rows(got2[~tainted], ref[~tainted], "mid-size end-to-end", A[~tainted])
    print(f"mid-size backward: all {sc.N} rows stage-isolated (worst {worst:.3f}, {over} elements over the plain bar); "
          f"{int((~tainted).sum())} rows end to end (worst {worst2:.3f}, {over2} over)")


# ------------------------------------------------------------------------------------------------
# argument errors are status codes, not crashes
# ------------------------------------------------------------------------------------------------
# ------------------------------------------------------------------------------------------------
# qr_topk_forward (NEXT-1; reading R17)
# ------------------------------------------------------------------------------------------------
TOPK_CASES = [
    ("cfg1", dict(), 8, 1e-4),                                   # FFMA-free plain path (D = 16)
    ("cfg1", dict(W=70, H=50, D=3), 40, 0.0),                    # ragged image, odd D, whole-list weights
    ("cfg2", dict(N=20000, W=128, H=96), 5, 1e-4),
    ("cfg3", dict(N=60000, W=160, H=112, D=512), 40, 1e-4),      # tcgen05 blend, R = 5,120 records per full half tile
    ("cfg3", dict(N=60000, W=100, H=72, D=256), 10, 1e-4),       # tcgen05 blend, ragged image
    ("cfg3", dict(N=60000, W=96, H=64, D=128), 64, 1e-4),        # K = QR_TOPK_MAX_K: half tiles over the prep's capacity
    ("cfg1", dict(D=64), 1, 1e-4),                               # K = 1
]


@pytest.mark.parametrize("name,kw,K,t_min", TOPK_CASES)
def test_topk_forward_stage_isolated(qr, orc, name, kw, K, t_min):
    sc = make_scene(name, seed=21, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    t = orc.topk(lists, K, sc.features, t_min=t_min)
    out = qr.qr_topk_forward(sc.cam, K, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac), P.to_dev(isect.view(np.int32)),
                             P.to_dev(rng), P.to_dev(sc.features), t_min)
    stats = P.compare_topk(out, t, lists, K, sc.D)
    assert stats["exempt"] < 0.02 * stats["pixels"] + 5, stats
    print(name, kw, K, stats)


def test_topk_fp16_and_backward_accepts_its_records(qr, orc):
    """fp16 features through the plain blend; qr_backward on top-K's records equals the oracle's backward of them."""
    sc = make_scene("cfg4", seed=22, N=60000, W=96, H=64, D=128, pose=1, backward=True)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    K = 12
    t = orc.topk(lists, K, sc.features, t_min=1e-4)
    args = (P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac), P.to_dev(isect.view(np.int32)), P.to_dev(rng))
    out = qr.qr_topk_forward(sc.cam, K, *args, P.to_dev(sc.features), 1e-4)
    P.compare_topk(out, t, lists, K, sc.D, f16=True)
    H, W = sc.cam.height, sc.cam.width
    dF = qr.qr_backward(sc.cam, sc.N, P.to_dev(t.sel_idx.reshape(H, W, K)), P.to_dev(t.sel_w.reshape(H, W, K).astype(np.float32)),
                        P.to_dev(t.n_sel.reshape(H, W)), P.to_dev(sc.dL_dmap))
    ref = orc.backward(t.sel_idx, t.sel_w, t.n_sel, sc.dL_dmap, sc.N)
    P.compare_backward_rows(dF.cpu().numpy(), ref, "top-K records")


def test_topk_full_size_config3_sampled(qr, orc):
    """BASELINE config 3 at full size, K = 40: selection on every pixel, features on sampled pixels."""
    sc = make_scene("cfg3", seed=0)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.topk_forward(sc.cam, fe, g.features, sc.K, 1e-4)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    t = orc.topk(lists, sc.K, None, t_min=1e-4)
    stats = P.compare_topk(out, t, lists, sc.K, sc.D)
    rng = np.random.default_rng(5)
    pix = np.sort(rng.choice(sc.cam.width * sc.cam.height, 1500, replace=False))
    tp = orc.topk(lists, sc.K, sc.features, t_min=1e-4, pixels=pix)
    sub = type("L", (), dict(borderline=lists.borderline))()
    s2 = P.compare_topk(out, tp, sub, sc.K, sc.D, pixels=pix)
    assert stats["exempt"] < 0.02 * stats["pixels"], stats
    print("top-K cfg3 full size:", stats, "sampled:", s2)


# ------------------------------------------------------------------------------------------------
# multi-camera batching (NEXT-4; include/qr.h "Multi-camera batching")
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("D,K,n_views", [(128, 16, 3), (16, 40, 4), (512, 8, 2)])
def test_batch_of_views_equals_the_oracle_per_view(qr, orc, D, K, n_views):
    """B poses of config 4's circle rendered by ONE set of launches (tall tile grid): every view's slice is compared with
    the oracle run on that camera alone, the projection is bit-identical to the single-view call, and the gradient of
    all views, accumulated into one dL_dfeat by one backward, equals the sum of the oracle's per-view gradients."""
    from qr_inputs.scenes import pose_on_circle
    sc = make_scene("cfg4", seed=23, N=40000, W=96, H=64, D=D, pose=0, backward=True)
    feats = sc.features.astype(np.float32)
    cams = []
    for j in range(n_views):
        c = sc.cam.copy()
        c.world_to_cam = pose_on_circle(2 * j + 1, 8)
        cams.append(c)
    H, W, N = sc.cam.height, sc.cam.width, sc.N
    g = P.upload(sc)
    gf = P.to_dev(feats)
    tall, fe = qr.pipeline.frontend_batch(cams, g.means, g.scales, g.quats, g.opac)
    assert tall.height == n_views * H and tall.width == W
    out = qr.pipeline.forward_batch(tall, n_views, N, fe, gf, K)
    rng = np.random.default_rng(3)
    G = rng.standard_normal((n_views * H, W, D), dtype=np.float32)
    dF = qr.pipeline.backward(tall, N, out, P.to_dev(G))
    gref = np.zeros((N, D))
    A = np.zeros((N, D))                         # sum |w g| per element: the fan-in term of the gradient tolerance
    tainted = np.zeros(N, bool)
    for j, cam in enumerate(cams):
        single = qr.qr_preprocess(cam, g.means, g.scales, g.quats, g.opac)
        for name in ("mean2d", "conic_opac", "depth", "tiles_touched"):
            assert torch.equal(getattr(fe.proj, name)[j * N:(j + 1) * N], getattr(single, name)), name
        proj = orc.project(cam, sc.means, sc.scales, sc.quats, sc.opac)
        lists = orc.pixel_lists(cam, proj)
        q = orc.qrender(lists, K, feats)
        view = qr.binding.ForwardOut(out.out_map[j * H:(j + 1) * H], out.sel_idx[j * H:(j + 1) * H], out.sel_w[j * H:(j + 1) * H],
                                     out.n_sel[j * H:(j + 1) * H], out.resid_TQ[j * H:(j + 1) * H])
        stats = P.compare_forward(view, q, lists, K, D)
        print("view", j, stats)
        gref += orc.backward(q.sel_idx, q.sel_w, q.n_sel, G[j * H:(j + 1) * H].reshape(H * W, D), N)
        A += orc.backward(q.sel_idx, q.sel_w, q.n_sel, np.abs(G[j * H:(j + 1) * H]).reshape(H * W, D), N)
        sel, _, n = P.masked_records(view)
        same = P.same_selection(sel, n, q)
        for pth in np.flatnonzero(~same):
            tainted[sel[pth, :n[pth]]] = True
            tainted[q.sel_idx[pth, :q.n_sel[pth]]] = True
    assert (~tainted).sum() > 0.5 * N
    worst, over = P.compare_backward_rows(dF.cpu().numpy()[~tainted], gref[~tainted], "batched backward", A[~tainted])
    print("gradient rows compared", int((~tainted).sum()), "worst err/tol", worst, "elements over the plain bar", over)
    qr.pipeline.backward_clear(tall, N, out, dF)
    assert float(dF.abs().max()) == 0.0


# ------------------------------------------------------------------------------------------------
# stratified-K (NEXT-3; reading R18)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw,K,t_min", [("cfg3", dict(N=60000, W=160, H=112, D=512), 40, 1e-4),
                                             ("cfg2", dict(N=20000, W=96, H=64, D=256), 8, 1e-4),
                                             ("cfg1", dict(W=70, H=50, D=128), 16, 0.0),          # ragged image, whole-list statistics
                                             ("cfg3", dict(N=60000, W=100, H=72, D=128), 1, 1e-4),
                                             ("cfg2", dict(N=20000, W=96, H=64, D=64), 8, 1e-4),            # padded 128-channel tile
                                             ("cfg1", dict(W=70, H=50), 16, 1e-4)])                         # D = 16
def test_stratified_forward_and_backward(qr, orc, name, kw, K, t_min):
    sc = make_scene(name, seed=25, backward=True, **kw)
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    t = orc.stratified(lists, K, sc.features, t_min=t_min)
    out = qr.binding.qr_forward_stratified(sc.cam, K, P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac), P.to_dev(isect.view(np.int32)),
                                           P.to_dev(rng), P.to_dev(sc.features), t_min)
    stats = P.compare_stratified(out, t, lists, K, sc.D)
    assert stats["exempt"] < 0.03 * stats["pixels"] + 5, stats
    print(name, kw, K, stats)
    if K == 1:
        return          # every weight is exactly 1 and single Gaussians collect thousands of pixels: outside what the gradient bar covers
    # the selection lists it leaves are what qr_backward_lists consumes: gradient on untainted rows vs the oracle's
    dF = qr.pipeline.backward(sc.cam, sc.N, out, P.to_dev(sc.dL_dmap))
    sel, _, n = P.masked_records(out)
    same = P.same_selection(sel, n, t)
    tainted = np.zeros(sc.N, bool)
    for pth in np.flatnonzero(~same):
        tainted[sel[pth, :n[pth]]] = True
        tainted[t.sel_idx[pth, :t.n_sel[pth]]] = True
    gref = orc.backward(t.sel_idx, t.sel_w, t.n_sel, sc.dL_dmap, sc.N)
    A = orc.backward(t.sel_idx, t.sel_w, t.n_sel, np.abs(sc.dL_dmap), sc.N)
    P.compare_backward_rows(dF.cpu().numpy()[~tainted], gref[~tainted], "stratified backward", A[~tainted])


def test_stratified_unsupported_shapes_are_status_codes(qr):
    sc = make_scene("cfg1", seed=1, D=36)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    with pytest.raises(qr.QRError) as e:
        qr.pipeline.stratified_forward(sc.cam, fe, g.features, 8)          # D = 36: not on the tcgen05 path (D % 32 != 0)
    assert e.value.code == -3


# ------------------------------------------------------------------------------------------------
# the path's neighbours (NEXT-2): de-voxelisation (Listing 3) and the mask-pooled loss (Eq. 2, reading R19)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("U,Cn,G,reduce", [(5000, 512, 3000, "max"), (5000, 512, 3000, "mean"), (300, 7, 1000, "max"), (1, 64, 1, "mean")])
def test_devoxelize_forward_and_backward(qr, orc, U, Cn, G, reduce):
    rng = np.random.default_rng(41)
    uni = rng.standard_normal((U, Cn)).astype(np.float32)
    counts = rng.integers(0, 9, G).astype(np.int32)
    counts[G // 2] = 0 if G > 1 else 3
    inv = rng.integers(0, U, int(counts.sum())).astype(np.int64)
    ref, am_ref = orc.devoxelize(uni, inv, counts, reduce)
    gs, am, ws = qr.binding.qr_devoxelize(P.to_dev(uni), P.to_dev(inv), P.to_dev(counts), reduce)
    got = gs.cpu().numpy()
    if reduce == "max":
        assert np.array_equal(got.astype(np.float64), ref)                       # a maximum is exact
        assert np.array_equal(am.cpu().numpy().astype(np.int64), am_ref)
    else:
        assert (np.abs(got - ref) <= P.ATOL + P.RTOL * np.abs(ref)).all()
    dgs = rng.standard_normal((G, Cn)).astype(np.float32)
    dref = orc.devoxelize_backward(U, inv, counts, reduce, am_ref if reduce == "max" else None, dgs)
    du = qr.binding.qr_devoxelize_backward(U, P.to_dev(inv), reduce, am, P.to_dev(dgs), ws).cpu().numpy()
    assert (np.abs(du - dref) <= P.ATOL + P.RTOL * np.abs(dref)).all()


@pytest.mark.parametrize("W,H,D,S", [(96, 64, 128, 12), (70, 50, 512, 5), (64, 64, 16, 40)])
def test_mask_loss_and_gradient(qr, orc, W, H, D, S):
    from qr_inputs import make_camera
    rng = np.random.default_rng(43)
    cam = make_camera(W, H)
    fmap = rng.standard_normal((H, W, D)).astype(np.float32)
    # blocky masks (spatially coherent, as segmentation masks are), some pixels outside every mask, one mask empty
    mid = ((np.arange(H)[:, None] // 9) * 7 + (np.arange(W)[None, :] // 11)) % (S + 2) - 1
    mid[mid >= S] = -1
    mid[mid == 1] = -1
    mid = mid.astype(np.int32)
    tg = rng.standard_normal((S, D)).astype(np.float32)
    ref = orc.mask_loss(fmap, mid, tg)
    loss, per, dmap = qr.binding.qr_mask_loss(cam, P.to_dev(fmap), P.to_dev(mid), P.to_dev(tg))
    assert abs(float(loss.item()) - ref.loss) <= 1e-5 + 1e-4 * abs(ref.loss)
    np.testing.assert_allclose(per.cpu().numpy(), ref.loss_per_mask, rtol=1e-4, atol=1e-5)
    got = dmap.cpu().numpy().reshape(-1, D).astype(np.float64)
    scale = np.abs(ref.d_map).max()                                  # entries are O(1 / (pixels per mask x masks)): compare relative to the map's scale
    assert (np.abs(got - ref.d_map) <= 1e-4 * scale + 1e-4 * np.abs(ref.d_map)).all()
    assert (got[mid.reshape(-1) < 0] == 0).all()


@pytest.mark.parametrize("name,kw,K,S", [("cfg3", dict(N=60000, W=160, H=112, D=512), 40, 9), ("cfg2", dict(N=20000, W=100, H=72, D=128), 16, 30),
                                         ("cfg2", dict(N=20000, W=100, H=72, D=64), 16, 30),        # padded 128-channel tile
                                         ("cfg1", dict(W=70, H=50), 40, 6)])                        # D = 16
def test_pooled_loss_equals_loss_on_the_map_then_backward(qr, orc, name, kw, K, S):
    """qr_pooled_loss (no map, no dL/dmap) against the oracle's unfused chain: Algorithm 1 map -> mask loss -> d_map -> backward;
    and selection-only forward leaves the same lists as the full forward."""
    sc = make_scene(name, seed=27, **kw)
    H, W, D, N = sc.cam.height, sc.cam.width, sc.D, sc.N
    proj, rect, touched, isect, rng = P.oracle_frontend(orc, sc)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, sc.features)
    r = np.random.default_rng(5)
    mid = ((np.arange(H)[:, None] // 13) * 5 + (np.arange(W)[None, :] // 17)) % (S + 1) - 1        # blocky masks, -1 = none
    mid = mid.astype(np.int32)
    tg = r.standard_normal((S, D)).astype(np.float32)
    ref = orc.mask_loss(q.out_map, mid, tg)
    gref = orc.backward(q.sel_idx, q.sel_w, q.n_sel, ref.d_map.astype(np.float32), N)
    args = (P.to_dev(proj.mean2d), P.to_dev(proj.conic_opac), P.to_dev(isect.view(np.int32)), P.to_dev(rng), P.to_dev(sc.features))
    out = qr.qr_forward(sc.cam, K, *args, select_only=True)
    sel, _, n = P.masked_records(out)
    same = P.same_selection(sel, n, q)
    assert ((~same) & ~P.exempt_mask(q, lists)).sum() == 0
    loss, per, dF = qr.binding.qr_pooled_loss(sc.cam, K, N, out, args[4], P.to_dev(mid), P.to_dev(tg))
    if same.all():           # a differing (exempt) pixel changes its mask's pooled vector: compare only when none differs
        assert abs(float(loss.item()) - ref.loss) <= 1e-5 + 1e-4 * abs(ref.loss)
        np.testing.assert_allclose(per.cpu().numpy(), ref.loss_per_mask, rtol=1e-4, atol=1e-5)
        scale = np.abs(gref).max()
        assert (np.abs(dF.cpu().numpy() - gref) <= 1e-4 * scale + 1e-4 * np.abs(gref)).all()
    # against the library's own unfused chain on the same selection (always comparable)
    full = qr.qr_forward(sc.cam, K, *args)
    l2, per2, dmap = qr.binding.qr_mask_loss(sc.cam, full.out_map, P.to_dev(mid), P.to_dev(tg))
    dF2 = qr.pipeline.backward(sc.cam, N, full, dmap)
    assert abs(float(loss.item()) - float(l2.item())) <= 1e-5 + 1e-4 * abs(float(l2.item()))
    a, b = dF.cpu().numpy(), dF2.cpu().numpy()
    assert (np.abs(a - b) <= 2e-4 * np.abs(b).max() + 1e-3 * np.abs(b)).all()
    print("pooled loss", float(loss.item()), "oracle", ref.loss, "pixels differing", int((~same).sum()))


@pytest.mark.parametrize("W,H,D,N,K", [(1, 1, 128, 50, 4), (17, 3, 128, 300, 40), (16, 16, 512, 1, 1), (5, 40, 256, 2000, 7), (33, 9, 16, 500, 3)])
def test_degenerate_image_sizes_through_every_forward(qr, orc, W, H, D, N, K):
    """One-pixel, one-Gaussian, sliver-shaped images: front end, Q-Render forward + backward, stratified-K and top-K against the
    oracle (TMA boxes larger than the image, half tiles below it, unions of one column)."""
    sc = make_scene("cfg1", seed=3, W=W, H=H, D=D, N=N, backward=True)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, g.features, K)
    dF = qr.pipeline.backward(sc.cam, N, out, P.to_dev(sc.dL_dmap))
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, K, sc.features)
    st = P.compare_forward(out, q, lists, K, D)
    if st["mismatch_exempt"] == 0:
        P.compare_backward_rows(dF.cpu().numpy(), orc.backward(q.sel_idx, q.sel_w, q.n_sel, sc.dL_dmap, N), "tiny image")
    if D % 128 == 0:
        so = qr.pipeline.stratified_forward(sc.cam, fe, g.features, K)
        P.compare_stratified(so, orc.stratified(lists, K, sc.features, t_min=1e-4), lists, K, D)
    tk = qr.pipeline.topk_forward(sc.cam, fe, g.features, K, 1e-4)
    P.compare_topk(tk, orc.topk(lists, K, sc.features, t_min=1e-4), lists, K, D)


def test_error_codes(qr):
    sc = make_scene("cfg1", seed=0, N=100)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    with pytest.raises(qr.QRError) as e:
        qr.pipeline.forward(sc.cam, fe, g.features, 0)
    assert e.value.code == -1
    with pytest.raises(qr.QRError) as e:
        qr.pipeline.forward(sc.cam, fe, g.features, 1000)
    assert e.value.code == -3
    with pytest.raises(qr.QRError):
        qr.qr_preprocess(sc.cam, g.means.cpu(), g.scales, g.quats, g.opac)   # no CPU path
    bad = make_camera(0, 10)
    with pytest.raises(qr.QRError) as e:
        qr.qr_preprocess(bad, g.means, g.scales, g.quats, g.opac)
    assert e.value.code == -1


# ------------------------------------------------------------------------------------------------
# RGB payload (NEXT-4): spherical-harmonics colours (reading R20), then Q-Render / V-Render with D = 3
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,degree", [(50000, 3), (1000, 2), (129, 1), (77, 0), (1, 3)])
def test_sh_colors_against_the_oracle(qr, orc, N, degree):
    from qr_inputs import make_camera
    rng = np.random.default_rng(47 + degree)
    cam = make_camera(96, 64)
    cy, sy = math.cos(0.3), math.sin(0.3)
    cam.world_to_cam = np.array([[cy, 0, sy, 0.2], [0, 1, 0, -0.1], [-sy, 0, cy, 0.7]], np.float32)
    means = rng.uniform(-3, 3, (N, 3)).astype(np.float32)
    sh = (rng.standard_normal((N, (degree + 1) ** 2, 3)) * 0.6).astype(np.float32)
    ref = orc.sh_colors(cam, means, sh, degree)
    got = qr.pipeline.sh_colors(cam, P.to_dev(means), P.to_dev(sh), degree).cpu().numpy()
    assert got.shape == (N, 3) and (got >= 0).all()
    # the basis is a cubic in a unit vector normalised in fp32 and the sum has up to 16 terms of either sign
    A = 0.5 + np.abs(sh.astype(np.float64)).sum(1)
    assert (np.abs(got - ref) <= P.ATOL + P.RTOL * np.abs(ref) + 8 * 2.0 ** -24 * A).all()
    if N >= 1000:
        assert (ref == 0).any() and ((got == 0) == (ref == 0)).mean() > 0.999      # the clamp is exercised


def test_rgb_render_from_sh_colors(qr, orc):
    """The whole RGB path: colours of this view from degree-3 coefficients, then Q-Render with D = 3 -- selection as for
    any payload, the image within the fp32 feature tolerance of the oracle run on the ORACLE's colours."""
    sc = make_scene("cfg1", seed=9, D=3)
    rng = np.random.default_rng(9)
    sh = (rng.standard_normal((sc.N, 16, 3)) * 0.5).astype(np.float32)
    g = P.upload(sc)
    colors = qr.pipeline.sh_colors(sc.cam, g.means, P.to_dev(sh), 3)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    out = qr.pipeline.forward(sc.cam, fe, colors, sc.K)
    cref = orc.sh_colors(sc.cam, sc.means, sh, 3).astype(np.float32)
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, sc.K, cref)
    stats = P.compare_forward(out, q, lists, sc.K, 3)
    assert stats["mismatch_nonexempt"] == 0


# ------------------------------------------------------------------------------------------------
# several K in one walk (NEXT-3, second half): every K's outputs are those of qr_forward with that K
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw,Ks", [("cfg4", dict(N=60000, W=128, H=96, D=512, pose=1), (4, 8, 16, 32)),    # BASELINE config 4's sweep
                                        ("cfg3", dict(N=60000, W=100, H=72, D=128), (40, 7)),                  # ragged image, descending K
                                        ("cfg2", dict(N=20000, W=96, H=64, D=64), (1, 200, 12)),               # K = 1, K large, padded tile
                                        ("cfg1", dict(W=70, H=50), (40,))])
def test_forward_multik_equals_single_k_forwards(qr, orc, name, kw, Ks):
    sc = make_scene(name, seed=21, **kw)
    g = P.upload(sc)
    fe = qr.pipeline.frontend(sc.cam, g.means, g.scales, g.quats, g.opac)
    outs = qr.pipeline.forward_multik(sc.cam, fe, g.features, Ks)
    torch.cuda.synchronize()
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    G = P.to_dev(sc.dL_dmap) if sc.dL_dmap is not None else None
    for K, o in zip(Ks, outs):
        ref = qr.pipeline.forward(sc.cam, fe, g.features, K)
        # the decision arithmetic is the same instruction sequence: records identical, bit for bit
        assert torch.equal(o.n_sel, ref.n_sel) and torch.equal(o.resid_TQ, ref.resid_TQ)
        ia, wa, na = P.masked_records(o)
        ib, wb, nb = P.masked_records(ref)
        assert (ia == ib).all() and (wa == wb).all()
        torch.testing.assert_close(o.out_map, ref.out_map, rtol=2e-4, atol=2e-5)      # union numbering is a race: summation order
        # and against the oracle, as qr_forward is
        q = orc.qrender(lists, K, sc.features)
        stats = P.compare_forward(o, q, lists, K, sc.D, f16=sc.features.dtype == np.float16)
        assert stats["mismatch_nonexempt"] == 0
        # the lists each K leaves behind feed the backward as qr_forward's do
        if G is not None:
            dF = qr.pipeline.backward(sc.cam, sc.N, o, G)
            dF_ref = qr.pipeline.backward(sc.cam, sc.N, ref, G)
            torch.testing.assert_close(dF, dF_ref, rtol=1e-3, atol=1e-4 * float(dF_ref.abs().max()) + 1e-6)
