"""Boundary behaviour of the C ABI on the GPU box (SURVEY.md test group T8, include/hdc.h
conventions): argument errors are reported with the documented code BEFORE anything is enqueued
(the launch counter does not move), hdc_last_error carries a message, empty inputs succeed without
touching the outputs, and the workspace contract (too small => HDC_ERR_WORKSPACE) holds."""
from __future__ import annotations

import ctypes as C

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hd():
    import paper_2606_26547_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def h(hd):
    hh = hd.Handle(0)
    yield hh
    hh.close()


def _expect(hd, h, code, fn):
    before = h.launch_count()
    with pytest.raises(hd.HdcError) as ei:
        fn()
    assert ei.value.code == code, (ei.value.code, str(ei.value))
    assert h.launch_count() == before, "an argument error must not enqueue any kernel"
    assert len(h.last_error()) > 0


def test_knob_errors_are_invalid_arg(hd, h):
    H = torch.zeros((8, 4), dtype=torch.int32, device="cuda")
    Cc = torch.ones((3, 128), dtype=torch.float32, device="cuda")
    bad = [hd.knobs(129, hv_bits=1, sim=hd.HDC_SIM_HAMMING),          # D_eff > D
           hd.knobs(0, hv_bits=1, sim=hd.HDC_SIM_HAMMING),            # D_eff < 1
           hd.knobs(128, hv_bits=4, sim=hd.HDC_SIM_COS),              # hv_bits not in {32,16,8,1}
           hd.knobs(128, hv_bits=32, sim=hd.HDC_SIM_HAMMING),         # Hamming needs sign bits
           hd.knobs(128, hv_bits=32, sim=7)]                          # unknown similarity
    for kn in bad:
        _expect(hd, h, hd.HDC_ERR_INVALID_ARG, lambda kn=kn: h.hdc_classify(H, Cc, kn))
        _expect(hd, h, hd.HDC_ERR_INVALID_ARG, lambda kn=kn: h.hdc_similarity(H, Cc, kn))
    y = torch.zeros(8, dtype=torch.int32, device="cuda")
    _expect(hd, h, hd.HDC_ERR_INVALID_ARG, lambda: h.hdc_train_epoch(9, H, y, Cc, hd.knobs(128)))
    _expect(hd, h, hd.HDC_ERR_INVALID_ARG,
            lambda: h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, H, y, Cc, hd.knobs(128), batch=-1))
    X = torch.zeros((8, 16), dtype=torch.float32, device="cuda")
    P = torch.zeros((128, 16), dtype=torch.float32, device="cuda")
    _expect(hd, h, hd.HDC_ERR_INVALID_ARG, lambda: h.hdc_encode_rp(X, P, hd.knobs(129)))
    _expect(hd, h, hd.HDC_ERR_INVALID_ARG, lambda: h.hdc_encode_rp(X, P, hd.knobs(128, precision=9)))


def test_null_pointers_and_bad_sizes_through_the_raw_abi(hd, h):
    L, hh = h._L, h._h
    kn = hd.knobs(128, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    H = torch.zeros((8, 4), dtype=torch.int32, device="cuda")
    Cc = torch.ones((3, 128), dtype=torch.float32, device="cuda")
    lab = torch.empty(8, dtype=torch.int32, device="cuda")
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    vp = lambda t: C.c_void_p(t.data_ptr())  # noqa: E731
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    before = h.launch_count()

    def classify(Hp, Cp, K, ldc, knp, labp, N=8, ldh=4, wsp=vp(ws), wsb=ws.numel()):
        return L.hdc_classify(hh, Hp, N, ldh, Cp, K, ldc, 128, knp, labp, None, None, wsp, wsb, st)

    assert classify(None, vp(Cc), 3, 128, C.byref(kn), vp(lab)) == hd.HDC_ERR_INVALID_ARG      # H NULL
    assert classify(vp(H), None, 3, 128, C.byref(kn), vp(lab)) == hd.HDC_ERR_INVALID_ARG       # C NULL
    assert classify(vp(H), vp(Cc), 0, 128, C.byref(kn), vp(lab)) == hd.HDC_ERR_INVALID_ARG     # K = 0
    assert classify(vp(H), vp(Cc), 3, 64, C.byref(kn), vp(lab)) == hd.HDC_ERR_INVALID_ARG      # ldc < D
    assert classify(vp(H), vp(Cc), 3, 128, None, vp(lab)) == hd.HDC_ERR_INVALID_ARG            # knobs NULL
    assert classify(vp(H), vp(Cc), 3, 128, C.byref(kn), vp(lab), N=-1) == hd.HDC_ERR_INVALID_ARG
    assert L.hdc_classify(None, vp(H), 8, 4, vp(Cc), 3, 128, 128, C.byref(kn), vp(lab), None, None, vp(ws),
                          ws.numel(), st) == hd.HDC_ERR_INVALID_ARG                              # handle NULL
    # workspace too small (classify at hv_bits = 1 needs K*W sign words)
    assert classify(vp(H), vp(Cc), 3, 128, C.byref(kn), vp(lab), wsp=None, wsb=0) == hd.HDC_ERR_WORKSPACE
    assert classify(vp(H), vp(Cc), 3, 128, C.byref(kn), vp(lab), wsb=4) == hd.HDC_ERR_WORKSPACE
    assert h.launch_count() == before
    assert b"workspace" in L.hdc_last_error(hh)
    # the same call with a sufficient workspace succeeds
    assert classify(vp(H), vp(Cc), 3, 128, C.byref(kn), vp(lab)) == hd.HDC_OK
    torch.cuda.synchronize()
    assert h.launch_count() > before


def test_misaligned_bit_matrix_is_alignment_error(hd, h):
    L, hh = h._L, h._h
    kn = hd.knobs(64)
    lv = torch.zeros((4, 8), dtype=torch.uint8, device="cuda")
    raw = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    Hb = torch.zeros((4, 2), dtype=torch.int32, device="cuda")
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    before = h.launch_count()
    rc = L.hdc_encode_levelid(hh, C.c_void_p(lv.data_ptr()), 4, 8, 8, C.c_void_p(raw.data_ptr() + 1), 2,
                              C.c_void_p(raw.data_ptr() + 1024), 4, 2, 64, C.byref(kn),
                              C.c_void_p(Hb.data_ptr()), 2, None, 0, st)
    assert rc == hd.HDC_ERR_ALIGNMENT
    assert h.launch_count() == before


def test_empty_inputs_succeed_and_touch_nothing(hd, h):
    D, K, F = 256, 4, 16
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    H0 = torch.zeros((0, D // 32), dtype=torch.int32, device="cuda")
    Cc = torch.full((K, D), 3.0, dtype=torch.float32, device="cuda")
    before = h.launch_count()
    assert h.hdc_classify(H0, Cc, kn).shape == (0,)
    assert h.hdc_similarity(H0, Cc, kn).shape == (0, K)
    y0 = torch.zeros(0, dtype=torch.int32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, H0, y0, Cc, kn)
    h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, H0, y0, Cc, kn, lr=0.5)
    X0 = torch.zeros((0, F), dtype=torch.float32, device="cuda")
    P = torch.randn((D, F), device="cuda")
    assert h.hdc_encode_rp(X0, P, hd.knobs(D)).shape == (0, D // 32)
    lv0 = torch.zeros((0, F), dtype=torch.uint8, device="cuda")
    tab = torch.zeros((F, D // 32), dtype=torch.int32, device="cuda")
    assert h.hdc_encode_levelid(lv0, tab, tab[:4], D, hd.knobs(D)).shape == (0, D // 32)
    torch.cuda.synchronize()
    assert h.launch_count() == before
    assert np.array_equal(Cc.cpu().numpy(), np.full((K, D), 3.0, dtype=np.float32))


def test_wrong_device_generation_is_refused_by_create(hd):
    """hdc_create succeeds here (compute capability 10.x) and reports the version; a second handle is
    independent (handles share no mutable state)."""
    a, b = hd.Handle(0), hd.Handle(0)
    assert hd.lib().hdc_version() > 0
    assert a.launch_count() == 0 and b.launch_count() == 0
    H = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    Cc = torch.ones((2, 128), dtype=torch.float32, device="cuda")
    a.hdc_classify(H, Cc, hd.knobs(128, hv_bits=1, sim=hd.HDC_SIM_HAMMING))
    assert a.launch_count() > 0 and b.launch_count() == 0
    a.close()
    b.close()
