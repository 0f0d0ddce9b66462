"""Prepared model (include/hdc.h): hdc_model_prepare converts the query-independent operands once; the *_m
entry points must then return exactly what the plain entry points return (which the other `-m gpu` files hold
against the oracle), and -- checked here directly -- what the oracle says.  Also: two handles in one process,
the device guard, and the observable kernel choice (hdc_stat)."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O

from gpu_util import dev, dev_bits, host_bits

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


def rng(*key):
    return np.random.default_rng([4242, *[int(k) for k in key]])


def _inputs(N, F, D, K, key):
    r = rng(*key)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = (21 - 2 * r.binomial(21, 0.5, size=(K, D))).astype(np.float32) * np.float32(0.75)
    return X, P, C


CASES = [  # precision, flags, hv_bits, sim, K, perf (begin, stride), enc_perf (begin, stride)
    ("F32", 0, 32, "COS", 26, (0, 1), (0, 1)), ("F32", 8, 32, "COS", 26, (0, 1), (0, 1)),
    ("F32", 1, 32, "DOT", 6, (0, 1), (0, 1)), ("BF16", 0, 16, "COS", 26, (0, 1), (0, 1)),
    ("F16", 0, 17, "COS", 10, (0, 1), (0, 1)), ("I8", 0, 8, "COS", 6, (0, 1), (0, 1)),
    ("I8", 1, 8, "COS", 6, (0, 1), (0, 1)), ("B1", 0, 1, "HAMMING", 10, (0, 1), (0, 1)),
    ("B1", 0, 1, "HAMMING", 70, (0, 1), (0, 1)), ("B1", 0, 1, "HAMMING", 10, (5, 3), (0, 1)),
    ("BF16", 0, 8, "COS", 26, (3, 8), (0, 1)), ("BF16", 0, 32, "COS", 26, (0, 1), (1, 2)),
    ("I8", 0, 1, "DOT", 200, (0, 1), (0, 1)), ("BF16", 1, 1, "DOT", 5, (0, 1), (0, 1)),
    ("BF16", 0, 18, "COS", 26, (0, 1), (0, 1)), ("I8", 0, 18, "DOT", 200, (2, 3), (0, 1)),   # 18 = HDC_HV_I16
    ("I8", 1, 18, "COS", 6, (0, 1), (0, 1)),
    ("BF16", 0, 19, "COS", 26, (0, 1), (0, 1)), ("I8", 0, 20, "DOT", 200, (2, 3), (0, 1)),   # 19 / 20 = HDC_HV_I32 / _I64
]


@pytest.mark.parametrize("prec,flags,hv_bits,sim,K,perf,eperf", CASES)
@pytest.mark.parametrize("N,F,D,D_eff", [(300, 72, 1000, 1000), (1559, 617, 700, 515)])
def test_prepared_model_equals_plain_calls_and_the_oracle(hd, h, prec, flags, hv_bits, sim, K, perf, eperf, N, F, D, D_eff):
    X, P, C = _inputs(N, F, D, K, (1, N, F, D_eff, K, hv_bits))
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim),
                  flags=flags, perf_begin=perf[0], perf_stride=perf[1], enc_perf_begin=eperf[0], enc_perf_stride=eperf[1])
    Xd, Pd, Cd = dev(X), dev(P), dev(C)
    H0 = h.hdc_encode_rp(Xd, Pd, kn)
    lab0, b0, s0 = h.hdc_classify(H0, Cd, kn, want_scores=True)
    l0 = h.launch_count()
    m = h.hdc_model_prepare(Pd, Cd, kn)
    n_prep = h.launch_count() - l0
    # the workspace is scribbled over between the calls: nothing the *_m calls need may live in it
    h._ws.fill_(0xA5) if h._ws is not None else None
    l0 = h.launch_count()
    H1 = h.hdc_encode_rp_m(Xd, m)
    lab1, b1, s1 = h.hdc_classify_m(H1, m, want_scores=True)
    n_run = h.launch_count() - l0
    assert torch.equal(H1, H0) and torch.equal(lab1, lab0) and torch.equal(b1, b0) and torch.equal(s1, s0)
    h._ws.fill_(0x5A) if h._ws is not None else None
    lab2, b2, s2 = h.hdc_infer_rp_m(Xd, m, want_scores=True)
    assert torch.equal(lab2, lab0) and torch.equal(b2, b0) and torch.equal(s2, s0)
    # the preparation kernels left the per-query path (the plain pair of calls launches n_prep + n_run kernels)
    l0 = h.launch_count()
    h.hdc_encode_rp(Xd, Pd, kn)
    h.hdc_classify(H0, Cd, kn)
    assert h.launch_count() - l0 == n_prep + n_run
    assert n_prep >= 1 or (flags & 1)            # (the CUDA-core kernels of HDC_FLAG_SIMT read fp32 operands in place)
    # and the oracle: exact-arithmetic encode, then its similarity stage on those bits
    bits_or, _, _ = O.encode_rp(X, P, D_eff, getattr(O, prec), f_begin=eperf[0], f_stride=eperf[1])
    assert np.array_equal(host_bits(H1, D_eff), bits_or)
    S_or = O.similarity(bits_or, C, D_eff, getattr(O, "SIM_" + sim), hv_bits, perf[0], perf[1])
    lab_or, best_or, _ = O.classify(S_or, getattr(O, "SIM_" + sim))
    margin = np.abs(np.sort(S_or, axis=1)[:, -1] - np.sort(S_or, axis=1)[:, -2]) if K > 1 else np.ones(N)
    if sim == "HAMMING":
        margin = np.abs(np.sort(S_or, axis=1)[:, 0] - np.sort(S_or, axis=1)[:, min(1, K - 1)]) if K > 1 else np.ones(N)
    clear = margin > 1e-3 * np.maximum(np.abs(best_or), 1e-30) if hv_bits not in (20, 19, 18, 8, 1) else np.ones(N, dtype=bool)
    assert np.array_equal(lab1.cpu().numpy()[clear], lab_or[clear])


def test_model_with_one_half_only_and_argument_errors(hd, h):
    X, P, C = _inputs(200, 64, 512, 7, (2,))
    kn = hd.knobs(512, precision=hd.HDC_BF16, hv_bits=16, sim=hd.HDC_SIM_COS)
    Xd, Pd, Cd = dev(X), dev(P), dev(C)
    H0 = h.hdc_encode_rp(Xd, Pd, kn)
    lab0 = h.hdc_classify(H0, Cd, kn)
    mp = h.hdc_model_prepare(Pd, None, kn)
    mc = h.hdc_model_prepare(None, Cd, kn)
    assert torch.equal(h.hdc_encode_rp_m(Xd, mp), H0)
    assert torch.equal(h.hdc_classify_m(H0, mc), lab0)
    with pytest.raises(hd.HdcError) as e:
        h.hdc_classify_m(H0, mp)
    assert e.value.code == hd.HDC_ERR_INVALID_ARG
    with pytest.raises(hd.HdcError) as e:
        h.hdc_infer_rp_m(Xd, mc)
    assert e.value.code == hd.HDC_ERR_INVALID_ARG
    with pytest.raises(hd.HdcError) as e:
        h.hdc_classify_m(H0, hd.Model(hd.hdc_model_t(), None, kn))          # never prepared
    assert e.value.code == hd.HDC_ERR_INVALID_ARG


def test_fused_model(hd, h):
    N, F, D, K = 12288 + 5, 64, 1000, 26
    X, P, C = _inputs(N, F, D, K, (3,))
    kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=8, sim=hd.HDC_SIM_COS, flags=hd.HDC_FLAG_FUSED_INFER)
    Xd, Pd, Cd = dev(X), dev(P), dev(C)
    lab0, b0, s0 = h.hdc_infer_rp(Xd, Pd, Cd, kn, want_scores=True)
    m = h.hdc_model_prepare(Pd, Cd, kn)
    f0 = h.stat(hd.HDC_STAT_INFER_FUSED)
    lab1, b1, s1 = h.hdc_infer_rp_m(Xd, m, want_scores=True)
    assert h.stat(hd.HDC_STAT_INFER_FUSED) == f0 + 1
    assert torch.equal(lab1, lab0) and torch.equal(b1, b0) and torch.equal(s1, s0)
    # the same model serves a pass too small for the fused kernel (two kernels) and a plain classify
    u0 = h.stat(hd.HDC_STAT_INFER_UNFUSED)
    lab_small = h.hdc_infer_rp_m(Xd[:100], m)
    assert h.stat(hd.HDC_STAT_INFER_UNFUSED) == u0 + 1
    assert torch.equal(lab_small, h.hdc_infer_rp(Xd[:100], Pd, Cd, kn))
    H = h.hdc_encode_rp_m(Xd[:300], m)
    assert torch.equal(h.hdc_classify_m(H, m), h.hdc_classify(H, Cd, kn))


def test_two_handles_interleaved_and_a_foreign_current_stream(hd, h):
    """Handles are independent (no process-wide kernel state): a second handle created later launches every
    large-shared-memory kernel too, interleaved with the first, on its own stream."""
    h2 = hd.Handle(0)
    try:
        X, P, C = _inputs(600, 617, 1200, 26, (4,))
        kn = hd.knobs(1200, precision=hd.HDC_F32, hv_bits=32, sim=hd.HDC_SIM_COS)
        kh = hd.knobs(1200, precision=hd.HDC_I8, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
        Xd, Pd, Cd = dev(X), dev(P), dev(C)
        side = torch.cuda.Stream()
        outs = []
        for hh in (h, h2, h, h2):
            with torch.cuda.stream(side if hh is h2 else torch.cuda.current_stream()):
                H = hh.hdc_encode_rp(Xd, Pd, kn)
                lab = hh.hdc_classify(H, Cd, kn)
                Hi = hh.hdc_encode_rp(Xd, Pd, kh)
                labh = hh.hdc_classify(Hi, Cd, kh)
                outs.append((H, lab, Hi, labh))
        torch.cuda.synchronize()
        for o in outs[1:]:
            for a, b in zip(o, outs[0]):
                assert torch.equal(a, b)
    finally:
        h2.close()


def test_unaligned_inputs_still_take_the_tensor_path(hd, h):
    """A leading dimension / base address TMA cannot take is staged, not demoted to the CUDA-core kernel:
    HDC_STAT_SIMT_FALLBACKS stays put and the tcgen05 contraction is counted."""
    r = rng(5)
    N, F, D = 400, 617, 1024
    Xbig = torch.from_numpy(r.standard_normal((N, F + 3)).astype(np.float32)).cuda()
    Pbig = torch.from_numpy(r.standard_normal((D, F + 5)).astype(np.float32)).cuda()
    X, P = Xbig[:, 1:F + 1], Pbig[:, 3:F + 3]            # odd element offsets, odd leading dimensions
    Xb = Xbig.to(torch.bfloat16)[:, 1:F + 1]
    for prec, x in (("F32", X), ("BF16", X), ("BF16", Xb), ("I8", X), ("F16", X)):
        kn = hd.knobs(D, precision=getattr(hd, "HDC_" + prec))
        t0, s0 = h.stat(hd.HDC_STAT_TC_LAUNCHES), h.stat(hd.HDC_STAT_SIMT_FALLBACKS)
        H = h.hdc_encode_rp(x, P, kn)
        assert h.stat(hd.HDC_STAT_TC_LAUNCHES) == t0 + 1 and h.stat(hd.HDC_STAT_SIMT_FALLBACKS) == s0
        Href = h.hdc_encode_rp(x.contiguous(), P.contiguous(), kn)
        assert torch.equal(H, Href)
    kn = hd.knobs(D, precision=hd.HDC_F32, flags=hd.HDC_FLAG_SIMT)     # asked for: not a fallback
    t0, s0 = h.stat(hd.HDC_STAT_TC_LAUNCHES), h.stat(hd.HDC_STAT_SIMT_FALLBACKS)
    h.hdc_encode_rp(X, P, kn)
    assert h.stat(hd.HDC_STAT_TC_LAUNCHES) == t0 and h.stat(hd.HDC_STAT_SIMT_FALLBACKS) == s0


def test_levelid_feature_count_beyond_shared_memory_is_refused_on_the_host(hd, h):
    N, F, Q, D = 8, 9000, 4, 64
    lv = torch.zeros((N, F), dtype=torch.uint8, device="cuda")
    ID = torch.zeros((F, 2), dtype=torch.int32, device="cuda")
    LV = torch.zeros((Q, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(hd.HdcError) as e:
        h.hdc_encode_levelid(lv, ID, LV, D, hd.knobs(D))
    assert e.value.code == hd.HDC_ERR_UNSUPPORTED
    torch.cuda.synchronize()                                   # nothing was enqueued, nothing faulted
