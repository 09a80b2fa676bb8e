"""CPU-side (-m "not gpu") checks of the boundary: libqr.so builds/loads without a GPU, exports every symbol that
include/qr.h declares, and rejects bad arguments with status codes before touching CUDA."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2512_20927_b200 import binding
    return binding.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "qr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qr_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2512_20927_b200 import binding
    names = _declared()
    assert set(names) == set(binding.SYMBOLS), (names, binding.SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_version_and_tiles(lib):
    from paper_2512_20927_b200 import binding
    from qr_inputs import make_camera
    assert lib.qr_version() == 200
    assert binding.qr_num_tiles(make_camera(640, 480)) == 1200
    assert binding.qr_num_tiles(make_camera(70, 50)) == 5 * 4
    assert lib.qr_num_tiles(None) == 0


def test_bad_arguments_are_status_codes(lib):
    from paper_2512_20927_b200 import binding
    from qr_inputs import make_camera
    cam = binding.make_camera(make_camera(64, 64))
    p = C.c_void_p(16)      # non-NULL, never dereferenced: every check below fails before any CUDA call
    z = C.c_void_p(0)
    # K = 0 is a domain error, K > QR_MAX_K unsupported
    assert lib.qr_forward(C.byref(cam), 0, 16, 0, p, p, p, p, p, p, p, p, p, p, p, 1 << 20, None) == -1
    assert b"K = 0" in lib.qr_last_error()
    assert lib.qr_forward(C.byref(cam), 1000, 16, 0, p, p, p, p, p, p, p, p, p, p, p, 1 << 20, None) == -3
    # D limits and fp16 alignment
    assert lib.qr_forward(C.byref(cam), 40, 0, 0, p, p, p, p, p, p, p, p, p, p, p, 1 << 20, None) == -1
    assert lib.qr_forward(C.byref(cam), 40, 1024, 0, p, p, p, p, p, p, p, p, p, p, p, 1 << 20, None) == -3
    assert lib.qr_forward(C.byref(cam), 40, 12, 1, p, p, p, p, p, p, p, p, p, p, p, 1 << 20, None) == -3
    # NULL outputs, too-small workspace
    assert lib.qr_forward(C.byref(cam), 40, 36, 0, p, p, p, p, p, z, p, p, p, p, p, 1 << 20, None) == -2      # D = 36: not a tcgen05 shape,
    assert lib.qr_forward(C.byref(cam), 40, 16, 0, p, p, p, p, p, p, z, p, p, p, p, 1 << 20, None) == -2      # where out_map = NULL is legal
    need = lib.qr_forward_workspace_bytes(C.byref(cam), 40, 16)
    assert need > 0
    assert lib.qr_forward(C.byref(cam), 40, 16, 0, p, p, p, p, p, p, p, p, p, p, p, need - 1, None) == -4
    # zero-area image, NULL camera
    bad = binding.make_camera(make_camera(64, 64)); bad.width = 0
    assert lib.qr_preprocess(C.byref(bad), 10, p, p, p, p, p, p, p, p, p, None) == -1
    assert lib.qr_preprocess(None, 10, p, p, p, p, p, p, p, p, p, None) == -2
    assert lib.qr_preprocess(C.byref(cam), -1, p, p, p, p, p, p, p, p, p, None) == -1
    assert lib.qr_preprocess(C.byref(cam), 0, z, z, z, z, z, z, z, z, z, None) == 0      # N = 0 is legal
    assert lib.qr_dense_forward(C.byref(cam), 16, 0, C.c_float(-1.0), p, p, p, p, p, p, p, None) == -1
    dtc = lambda D, t, cap, wsb: lib.qr_dense_forward_tc(C.byref(cam), D, 0, C.c_float(t), cap, p, p, p, p, p, p, p, p, wsb, None)
    assert dtc(128, -1.0, 64, 1 << 30) == -1 and dtc(128, 1e-4, 0, 1 << 30) == -1 and dtc(128, 1e-4, 257, 1 << 30) == -1
    assert dtc(36, 1e-4, 64, 1 << 30) == -3                    # not a shape of the tcgen05 path
    assert dtc(128, 1e-4, 64, 1024) == -4 and lib.qr_dense_workspace_bytes(C.byref(cam), 64) > 1024
    assert lib.qr_dense_workspace_bytes(C.byref(cam), 0) == 0
    assert lib.qr_backward(C.byref(cam), 0, 16, 10, p, p, p, p, p, None, 0, None) == -1
    # top-K comparator: K = 0 domain error, K > QR_TOPK_MAX_K unsupported, t_min < 0, NULL, small workspace
    tk = lambda K, D, t, out, wsb: lib.qr_topk_forward(C.byref(cam), K, D, 0, C.c_float(t), p, p, p, p, p, out, p, p, p, p, p, wsb, None)
    assert tk(0, 16, 1e-4, p, 1 << 20) == -1
    assert tk(65, 16, 1e-4, p, 1 << 20) == -3
    assert tk(8, 16, -1.0, p, 1 << 20) == -1
    assert tk(8, 16, 1e-4, z, 1 << 20) == -2
    assert lib.qr_forward_stratified(C.byref(cam), 8, 128, 0, C.c_float(-1.0), C.c_float(2.0), p, p, p, p, p, p, p, p, p, p, p, 1 << 30, None) == -1
    assert lib.qr_forward_stratified(C.byref(cam), 8, 36, 0, C.c_float(1e-4), C.c_float(2.0), p, p, p, p, p, p, p, p, p, p, p, 1 << 30, None) == -3
    assert lib.qr_stratified_workspace_bytes(C.byref(cam), 8, 128) == lib.qr_forward_workspace_bytes(C.byref(cam), 8, 128) + 64 * 64 * 8
    # batching: B out of range, unequal sizes, height % 16 != 0
    two = (binding.qr_camera * 2)(binding.make_camera(make_camera(64, 64)), binding.make_camera(make_camera(64, 48)))
    tall = binding.qr_camera()
    assert lib.qr_batch_camera(two, 0, C.byref(tall)) == -1 and lib.qr_batch_camera(two, 2, C.byref(tall)) == -1
    odd = (binding.qr_camera * 1)(binding.make_camera(make_camera(64, 50)))
    assert lib.qr_batch_camera(odd, 1, C.byref(tall)) == -1
    assert lib.qr_batch_camera(two, 1, C.byref(tall)) == 0 and tall.height == 64
    assert lib.qr_topk_workspace_bytes(C.byref(cam), 8, 16) > 0 and lib.qr_topk_workspace_bytes(C.byref(cam), 0, 16) == 0
    assert lib.qr_bin_sort(C.byref(cam), 10, 1 << 31, p, p, p, p, p, p, 1 << 20, None) == -5
    # spherical-harmonics colour: degree outside [0, 3], NULL arrays, N = 0
    assert lib.qr_sh_colors(C.byref(cam), 10, 4, p, p, p, None) == -1 and lib.qr_sh_colors(C.byref(cam), 10, -1, p, p, p, None) == -1
    assert lib.qr_sh_colors(C.byref(cam), 10, 3, p, z, p, None) == -2 and lib.qr_sh_colors(None, 10, 3, p, p, p, None) == -2
    assert lib.qr_sh_colors(C.byref(cam), 0, 3, z, z, z, None) == 0
    # the entry point with static scratch: sizes beyond the array are refused before anything touches CUDA
    assert lib.qr_mask_loss_static(C.byref(cam), 512, 257, p, p, p, p, p, p, None) == -3 and b"static array" in lib.qr_last_error()
    assert lib.qr_mask_loss_static(C.byref(cam), 512, 0, p, p, p, p, p, p, None) == -1
    assert lib.qr_mask_loss_static(C.byref(cam), 512, 256, p, z, p, p, p, p, None) == -2
    assert lib.qr_mask_loss_workspace_bytes(256, 512) == 256 * 512 * 4 + 3 * 1024
    # several K in one walk: nK out of range, NULL arrays, a shape outside the tcgen05 path, a bad K, a workspace that is too small
    ks = (C.c_int32 * 2)(8, 0)
    arr = (C.c_void_p * 2)(16, 16)
    szs = (C.c_size_t * 2)(1 << 30, 1 << 30)
    mk = lambda n, D, K_, a_, s_: lib.qr_forward_multik(C.byref(cam), n, K_, D, 0, p, p, p, p, p, a_, a_, a_, a_, a_, a_, s_, None)
    assert mk(0, 128, ks, arr, szs) == -1 and mk(5, 128, ks, arr, szs) == -1
    assert mk(2, 128, None, arr, szs) == -2 and mk(2, 128, ks, None, szs) == -2
    assert mk(1, 36, ks, arr, szs) == -3
    assert mk(2, 128, ks, arr, szs) == -1 and b"K[1] = 0" in lib.qr_last_error()
    ks[1] = 16
    assert mk(2, 128, ks, arr, szs) == -1 and b"share a workspace" in lib.qr_last_error()
    arr2 = (C.c_void_p * 2)(16, 32)
    small = (C.c_size_t * 2)(1 << 30, 64)
    assert lib.qr_forward_multik(C.byref(cam), 2, ks, 128, 0, p, p, p, p, p, arr, arr, arr, arr, arr, arr2, small, None) == -4
    m = C.c_int64(-1)
    assert lib.qr_bin_count(0, z, z, C.byref(m), z, 0, None) == 0 and m.value == 0
    assert lib.qr_bin_workspace_bytes(1000, 5000, 16) >= 5000 * 16 + 16 * 16 * 4      # keys + scratch + bucket cursors


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_2512_20927_b200 import binding
    from qr_inputs import make_camera
    t = torch.zeros((4, 3))
    with pytest.raises(binding.QRError):
        binding.qr_preprocess(make_camera(32, 32), t, t, torch.zeros((4, 4)), torch.zeros(4))


def test_product_never_imports_oracle():
    """The CUDA package and the oracle share no code and neither imports the other."""
    pkg = os.path.join(ROOT, "paper_2512_20927_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "qr_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2512" not in txt and "from paper_2512" not in txt and "libqr.so" not in txt, f
            assert not re.search(r'#include\s+"[^"]*(csrc|qr\.h|qr_common)', txt), f
