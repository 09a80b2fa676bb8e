"""qr_mask_loss_static: the entry point that allocates nothing (include/qr.h).  Its scratch is a static device array inside
the library, shared by every call and never cleared between them, so the checks are: same results as qr_mask_loss (the
existing path with a caller-provided workspace) on TWO calls in a row with different inputs -- the second would inherit the
first call's sums if the array were not cleared -- and a clear error beyond the array's size.

Collected last on purpose (file name): the suite runs with pytest -x, and a failure here must not hide other tests."""
import numpy as np
import pytest
import torch

from qr_inputs import make_camera

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4          # north_star's fp32 tolerance, as tests/parity.py


@pytest.fixture(scope="module")
def qr():
    import paper_2512_20927_b200 as q
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    q.binding.load()
    return q


def _case(seed, W, H, D, S):
    rng = np.random.default_rng(seed)
    cam = make_camera(W, H)
    fmap = rng.standard_normal((H, W, D)).astype(np.float32)
    # blocky masks, some pixels outside every mask, the last mask empty
    ys, xs = np.arange(H)[:, None] // max(H // 4, 1), np.arange(W)[None, :] // max(W // 4, 1)
    mid = ((ys * 4 + xs + seed) % max(S - 1, 1)).astype(np.int32)
    mid[rng.random((H, W)) < 0.05] = -1
    tg = rng.standard_normal((S, D)).astype(np.float32)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return cam, dev(fmap), dev(mid), dev(tg)


def _close(a, b, what):
    a, b = a.double().cpu().numpy(), b.double().cpu().numpy()
    assert np.isfinite(a).all(), what
    assert (np.abs(a - b) <= ATOL + RTOL * np.abs(b)).all(), (what, float(np.abs(a - b).max()))


def test_static_scratch_matches_the_workspace_path_twice_in_a_row(qr):
    B = qr.binding
    # two different problems back to back on the one array: big first, then a smaller one whose sums must not see the first's
    cases = [_case(1, 96, 64, 512, 200), _case(2, 70, 50, 128, 7), _case(3, 96, 64, 512, 200)]
    refs = [B.qr_mask_loss(cam, fmap, mid, tg) for cam, fmap, mid, tg in cases]
    torch.cuda.synchronize()
    for (cam, fmap, mid, tg), (l_ref, per_ref, dm_ref) in zip(cases, refs):
        S, D = tg.shape
        loss = torch.full((1,), float("nan"), device="cuda")
        per = torch.full((S,), float("nan"), device="cuda")
        dm = torch.full((cam.height, cam.width, D), float("nan"), device="cuda")
        B.qr_mask_loss_static(cam, fmap, mid, tg, loss, per, dm)
        torch.cuda.synchronize()
        _close(loss, l_ref, "loss")
        _close(per, per_ref, "loss_per_mask")
        _close(dm, dm_ref, "d_map")
        assert float(dm.abs().max()) > 0 and float(loss) > 0
    # the very same call twice: identical inputs, results inside the tolerance of each other
    cam, fmap, mid, tg = cases[0]
    a = B.qr_mask_loss_static(cam, fmap, mid, tg)
    b = B.qr_mask_loss_static(cam, fmap, mid, tg)
    torch.cuda.synchronize()
    for x, y, what in zip(a, b, ("loss", "loss_per_mask", "d_map")):
        _close(x, y, what + " (repeat)")


def test_static_scratch_rejects_sizes_beyond_the_array(qr):
    B = qr.binding
    cam, fmap, mid, tg = _case(4, 32, 32, 512, 257)           # 257 masks at D = 512: one more than the array holds
    with pytest.raises(qr.QRError) as e:
        B.qr_mask_loss_static(cam, fmap, mid, tg)
    assert e.value.code == -3 and "static array" in str(e.value) and "257" in str(e.value)
    cam, fmap, mid, tg = _case(5, 32, 32, 512, 256)           # exactly the limit works, and so do more masks at a smaller D
    l, per, dm = B.qr_mask_loss_static(cam, fmap, mid, tg)
    l2, per2, dm2 = B.qr_mask_loss(cam, fmap, mid, tg)
    _close(l, l2, "loss at the limit"); _close(dm, dm2, "d_map at the limit")
    cam, fmap, mid, tg = _case(6, 32, 32, 64, 1500)
    l, per, dm = B.qr_mask_loss_static(cam, fmap, mid, tg)
    l2, per2, dm2 = B.qr_mask_loss(cam, fmap, mid, tg)
    _close(l, l2, "loss, 1500 masks at D = 64"); _close(per, per2, "per mask")
