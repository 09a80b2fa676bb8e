"""Red-zone checks of every C-ABI call (compute-sanitizer is closed on this GPU pool: its wrapper refuses to run, see
profiles/README.md, so out-of-bounds writes are looked for with canaries instead).

Every output array and every workspace of a call is carved out of a larger device buffer with 4 KB guard bands filled
with a byte pattern on both sides; after the call the bands must be untouched and every INPUT array must be bit-identical
to what went in ("Inputs are never modified", include/qr.h).  Scenes: BASELINE config 1 (FFMA kernels), a ragged image,
and the D = 512 blob scene of smoke() (tcgen05 kernels, TMA tensor stores, workspace lists)."""
import numpy as np
import pytest
import torch

from qr_inputs import make_scene

pytestmark = pytest.mark.gpu



@pytest.fixture(scope="module")
def qr():
    import paper_2512_20927_b200 as q
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    q.binding.load()
    return q


GUARD = 4096
PATTERN = 0xA5


class Zones:
    def __init__(self):
        self.bufs = []

    def alloc(self, shape, dtype):
        n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        n_al = (n + 255) // 256 * 256
        raw = torch.full((GUARD + n_al + GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
        view = raw[GUARD:GUARD + n].view(dtype).reshape(shape)
        self.bufs.append((raw, n))
        return view

    def check(self, what):
        torch.cuda.synchronize()
        for i, (raw, n) in enumerate(self.bufs):
            assert bool((raw[:GUARD] == PATTERN).all()), f"{what}: buffer {i}: write BEFORE the array"
            assert bool((raw[GUARD + n:] == PATTERN).all()), f"{what}: buffer {i}: write PAST the array"


@pytest.mark.parametrize("name,kw,K", [("cfg1", dict(backward=True), 40),
                                       ("cfg1", dict(W=70, H=50, D=20, backward=True), 7),
                                       ("cfg3", dict(N=60000, W=160, H=112, D=512), 40),
                                       ("cfg3", dict(N=30000, W=100, H=72, D=128), 64)])
def test_no_call_writes_outside_its_arrays(qr, name, kw, K):
    B = qr.binding
    sc = make_scene(name, seed=31, **kw)
    cam, N, D = sc.cam, sc.N, sc.D
    H, W = cam.height, cam.width
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    inputs = {k: dev(getattr(sc, k)) for k in ("means", "scales", "quats", "opac", "features", "dL_dmap")}
    before = {k: v.clone() for k, v in inputs.items()}
    lib = B.load()
    import ctypes as C
    c = B.make_camera(cam)
    st = B._stream()
    T = B.qr_num_tiles(cam)
    z = Zones()
    ptr = lambda t: t.data_ptr()

    # qr_preprocess
    mean2d, conic = z.alloc((N, 2), torch.float32), z.alloc((N, 4), torch.float32)
    depth, rect, touched = z.alloc((N,), torch.float32), z.alloc((N, 4), torch.int32), z.alloc((N,), torch.int32)
    B._check(lib.qr_preprocess(C.byref(c), N, ptr(inputs["means"]), ptr(inputs["scales"]), ptr(inputs["quats"]), ptr(inputs["opac"]),
                               ptr(mean2d), ptr(conic), ptr(depth), ptr(rect), ptr(touched), st))
    z.check("qr_preprocess")
    # qr_bin_count / qr_bin_sort (exact size, then a too-small capacity: truncation must stay in bounds)
    offsets = z.alloc((N,), torch.int64)
    cws = z.alloc((max(B.qr_bin_workspace_bytes(N, 0, 0), 16),), torch.uint8)
    M = C.c_int64(0)
    B._check(lib.qr_bin_count(N, ptr(touched), ptr(offsets), C.byref(M), ptr(cws), cws.numel(), st))
    M = int(M.value)
    for cap in (M, max(M // 3, 1)):
        isect, rng = z.alloc((max(cap, 1),), torch.int32), z.alloc((T, 2), torch.int32)
        bws = z.alloc((max(B.qr_bin_workspace_bytes(N, cap, T), 16),), torch.uint8)
        B._check(lib.qr_bin_sort(C.byref(c), N, cap, ptr(depth), ptr(rect), None, ptr(isect), ptr(rng), ptr(bws), bws.numel(), st))
        z.check(f"qr_bin_sort(capacity {cap} of {M})")
    isect, rng = z.alloc((max(M, 1),), torch.int32), z.alloc((T, 2), torch.int32)
    bws = z.alloc((max(B.qr_bin_workspace_bytes(N, M, T), 16),), torch.uint8)
    B._check(lib.qr_bin_sort(C.byref(c), N, M, ptr(depth), ptr(rect), None, ptr(isect), ptr(rng), ptr(bws), bws.numel(), st))
    z.check("qr_bin_sort")

    def records(kk):
        return (z.alloc((H, W, D), torch.float32), z.alloc((H, W, kk), torch.int32), z.alloc((H, W, kk), torch.float32),
                z.alloc((H, W), torch.int32), z.alloc((H, W), torch.float32))

    # qr_forward
    out_map, sel_idx, sel_w, n_sel, resid = records(K)
    fws = z.alloc((max(B.qr_forward_workspace_bytes(cam, K, D), 256),), torch.uint8)
    B._check(lib.qr_forward(C.byref(c), K, D, 0, ptr(mean2d), ptr(conic), ptr(isect), ptr(rng), ptr(inputs["features"]),
                            ptr(out_map), ptr(sel_idx), ptr(sel_w), ptr(n_sel), ptr(resid), ptr(fws), fws.numel(), st))
    z.check("qr_forward")
    # qr_backward (own workspace), qr_backward_lists (the forward's, where supported), qr_backward_clear
    dF = z.alloc((N, D), torch.float32)
    dF.zero_()
    kws = z.alloc((max(B.qr_backward_workspace_bytes(cam, K, D), 256),), torch.uint8)
    B._check(lib.qr_backward(C.byref(c), K, D, N, ptr(sel_idx), ptr(sel_w), ptr(n_sel), ptr(inputs["dL_dmap"]), ptr(dF),
                             ptr(kws), kws.numel(), st))
    z.check("qr_backward")
    B._check(lib.qr_backward_clear(C.byref(c), K, D, N, ptr(sel_idx), ptr(n_sel), ptr(dF), ptr(kws), kws.numel(), st))
    z.check("qr_backward_clear")
    assert float(dF.abs().max()) == 0.0, "qr_backward_clear left a touched row"
    if B.lists_supported(torch.float32, D):
        B._check(lib.qr_backward_lists(C.byref(c), K, D, N, ptr(fws), fws.numel(), ptr(inputs["dL_dmap"]), ptr(dF), st))
        z.check("qr_backward_lists")
        B._check(lib.qr_backward_clear(C.byref(c), K, D, N, ptr(sel_idx), ptr(n_sel), ptr(dF), ptr(fws), fws.numel(), st))
        z.check("qr_backward_clear (forward workspace)")
        assert float(dF.abs().max()) == 0.0
    # qr_dense_forward, qr_topk_forward
    dmap, dT = z.alloc((H, W, D), torch.float32), z.alloc((H, W), torch.float32)
    B._check(lib.qr_dense_forward(C.byref(c), D, 0, C.c_float(1e-4), ptr(mean2d), ptr(conic), ptr(isect), ptr(rng),
                                  ptr(inputs["features"]), ptr(dmap), ptr(dT), st))
    z.check("qr_dense_forward")
    if B.lists_supported(torch.float32, D):
        for cap in (64, 2):              # roomy lists; lists so small that the walk must stop emitting (flagged half tiles)
            dws = z.alloc((int(lib.qr_dense_workspace_bytes(C.byref(c), cap)),), torch.uint8)
            B._check(lib.qr_dense_forward_tc(C.byref(c), D, 0, C.c_float(1e-4), cap, ptr(mean2d), ptr(conic), ptr(isect), ptr(rng),
                                             ptr(inputs["features"]), ptr(dmap), ptr(dT), ptr(dws), dws.numel(), st))
            z.check(f"qr_dense_forward_tc(cap {cap})")
    kt = min(K, 64)
    t_map, t_idx, t_w, t_n, t_r = records(kt)
    tws = z.alloc((max(int(lib.qr_topk_workspace_bytes(C.byref(c), kt, D)), 256),), torch.uint8)
    B._check(lib.qr_topk_forward(C.byref(c), kt, D, 0, C.c_float(1e-4), ptr(mean2d), ptr(conic), ptr(isect), ptr(rng),
                                 ptr(inputs["features"]), ptr(t_map), ptr(t_idx), ptr(t_w), ptr(t_n), ptr(t_r), ptr(tws), tws.numel(), st))
    z.check("qr_topk_forward")
    # qr_sh_colors (every degree: the staging loops have a different row length each)
    for deg in range(4):
        shc = z.alloc((N, (deg + 1) ** 2, 3), torch.float32)
        shc.normal_()
        keep = shc.clone()
        col = z.alloc((N, 3), torch.float32)
        B._check(lib.qr_sh_colors(C.byref(c), N, deg, ptr(inputs["means"]), ptr(shc), ptr(col), st))
        z.check(f"qr_sh_colors(degree {deg})")
        assert torch.equal(shc, keep), "sh was modified"
    for k, v in inputs.items():
        assert torch.equal(v, before[k]), f"input {k} was modified"


@pytest.mark.parametrize("W,H,D,S,K", [(96, 64, 128, 12, 16), (70, 50, 512, 5, 40)])
def test_neighbour_calls_write_inside_their_arrays(qr, W, H, D, S, K):
    """The same canaries around the outputs and workspaces of the path's neighbours and variants: qr_forward_stratified,
    qr_pooled_loss, qr_mask_loss, qr_mask_loss_static, qr_devoxelize / qr_devoxelize_backward, qr_sh_colors is covered above."""
    import ctypes as C
    B = qr.binding
    lib = B.load()
    sc = make_scene("cfg2", seed=33, N=20000, W=W, H=H, D=D)
    cam, N = sc.cam, sc.N
    c = B.make_camera(cam)
    st = B._stream()
    ptr = lambda t: t.data_ptr()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = {k: dev(getattr(sc, k)) for k in ("means", "scales", "quats", "opac", "features")}
    fe = qr.pipeline.frontend(cam, g["means"], g["scales"], g["quats"], g["opac"])
    rng = np.random.default_rng(5)
    z = Zones()
    # qr_forward_stratified
    out_map, sel_idx, sel_w = z.alloc((H, W, D), torch.float32), z.alloc((H, W, K), torch.int32), z.alloc((H, W, K), torch.float32)
    n_sel, resid = z.alloc((H, W), torch.int32), z.alloc((H, W), torch.float32)
    sws = z.alloc((int(lib.qr_stratified_workspace_bytes(C.byref(c), K, D)),), torch.uint8)
    B._check(lib.qr_forward_stratified(C.byref(c), K, D, 0, C.c_float(1e-4), C.c_float(2.0), ptr(fe.proj.mean2d), ptr(fe.proj.conic_opac),
                                       ptr(fe.isect_gauss), ptr(fe.tile_range), ptr(g["features"]), ptr(out_map), ptr(sel_idx), ptr(sel_w),
                                       ptr(n_sel), ptr(resid), ptr(sws), sws.numel(), st))
    z.check("qr_forward_stratified")
    # qr_forward_multik: three K, guarded outputs and workspaces each
    Ks = (K, 3, 2 * K)
    mo = [(z.alloc((H, W, D), torch.float32), z.alloc((H, W, k_), torch.int32), z.alloc((H, W, k_), torch.float32),
           z.alloc((H, W), torch.int32), z.alloc((H, W), torch.float32), z.alloc((int(B.qr_forward_workspace_bytes(cam, k_, D)),), torch.uint8))
          for k_ in Ks]
    pa = lambda i: (C.c_void_p * 3)(*[ptr(t[i]) for t in mo])
    B._check(lib.qr_forward_multik(C.byref(c), 3, (C.c_int32 * 3)(*Ks), D, 0, ptr(fe.proj.mean2d), ptr(fe.proj.conic_opac), ptr(fe.isect_gauss),
                                   ptr(fe.tile_range), ptr(g["features"]), pa(0), pa(1), pa(2), pa(3), pa(4), pa(5),
                                   (C.c_size_t * 3)(*[t[5].numel() for t in mo]), st))
    z.check("qr_forward_multik")
    # qr_forward (lists in its workspace) -> qr_pooled_loss
    fws = z.alloc((int(B.qr_forward_workspace_bytes(cam, K, D)),), torch.uint8)
    B._check(lib.qr_forward(C.byref(c), K, D, 0, ptr(fe.proj.mean2d), ptr(fe.proj.conic_opac), ptr(fe.isect_gauss), ptr(fe.tile_range),
                            ptr(g["features"]), ptr(out_map), ptr(sel_idx), ptr(sel_w), ptr(n_sel), ptr(resid), ptr(fws), fws.numel(), st))
    mid = dev(((np.arange(H)[:, None] // 16) * 3 + np.arange(W)[None, :] // 32).astype(np.int32) % S)
    tg = dev(rng.standard_normal((S, D)).astype(np.float32))
    loss, per = z.alloc((1,), torch.float32), z.alloc((S,), torch.float32)
    dF = z.alloc((N, D), torch.float32); dF.zero_()
    mws = z.alloc((int(lib.qr_mask_loss_workspace_bytes(S, D)),), torch.uint8)
    B._check(lib.qr_pooled_loss(C.byref(c), K, D, N, ptr(fws), fws.numel(), ptr(g["features"]), ptr(mid), S, ptr(tg), ptr(loss), ptr(per),
                                ptr(dF), ptr(mws), mws.numel(), st))
    z.check("qr_pooled_loss")
    # qr_mask_loss with a workspace, and with the library's static scratch
    d_map = z.alloc((H, W, D), torch.float32)
    B._check(lib.qr_mask_loss(C.byref(c), D, S, ptr(out_map), ptr(mid), ptr(tg), ptr(loss), ptr(per), ptr(d_map), ptr(mws), mws.numel(), st))
    z.check("qr_mask_loss")
    B._check(lib.qr_mask_loss_static(C.byref(c), D, S, ptr(out_map), ptr(mid), ptr(tg), ptr(loss), ptr(per), ptr(d_map), st))
    z.check("qr_mask_loss_static")
    # qr_devoxelize / qr_devoxelize_backward, both reductions
    U, G = 3000, 2000
    uni = dev(rng.standard_normal((U, D)).astype(np.float32))
    counts = dev(rng.integers(0, 6, G).astype(np.int32))
    inv = dev(rng.integers(0, U, int(counts.sum().item())).astype(np.int64))
    for reduce in (0, 1):
        gs, am = z.alloc((G, D), torch.float32), z.alloc((G, D), torch.int32)
        dws = z.alloc((int(lib.qr_devoxelize_workspace_bytes(G)),), torch.uint8)
        B._check(lib.qr_devoxelize(U, D, G, ptr(uni), ptr(inv), ptr(counts), reduce, ptr(gs), ptr(am), ptr(dws), dws.numel(), st))
        z.check(f"qr_devoxelize(reduce {reduce})")
        d_uni = z.alloc((U, D), torch.float32); d_uni.zero_()
        B._check(lib.qr_devoxelize_backward(U, D, G, ptr(inv), reduce, ptr(am), ptr(gs), ptr(d_uni), ptr(dws), dws.numel(), st))
        z.check(f"qr_devoxelize_backward(reduce {reduce})")
