"""Per-function parity of the CUDA path (through the C ABI) against the CPU oracle -- `-m gpu`.
Integer / bit paths: bit-exact.  Float paths: the agreement rules of DESIGN.md."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O
from workloads import gen

from gpu_util import (check_labels_float, check_scores, check_sign_band, dev, dev_bits, host_bits,
                      host_words)

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
    return np.random.default_rng([26547, *key])


# ------------------------------------------------------------------------------------ Hamming
@pytest.mark.parametrize("N,K,D,D_eff", [(1, 1, 32, 32), (300, 4, 2048, 2048), (300, 4, 2048, 1024),
                                         (257, 26, 10000, 10000), (129, 10, 10000, 4099),
                                         (77, 40, 4500, 33), (64, 3, 100, 1), (50, 70, 2100, 2047),
                                         (40, 5, 64, 31), (200, 70, 8192, 8000), (300, 100, 16384, 16384)])
def test_hamming_similarity_and_classify(hd, h, N, K, D, D_eff):
    r = rng(1, N, K, D_eff)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.standard_normal((K, D)).astype(np.float32)
    C[r.random((K, D)) < 0.05] = 0.0                      # sgn(0) = +1 cases
    if K > 2:
        C[2] = C[1]                                        # exact tie between classes 1 and 2
    kn = hd.knobs(D_eff, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    S_or = O.similarity(hb, C, D_eff, O.SIM_HAMMING, 1)
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_HAMMING)
    Hd = dev_bits(hb)                                      # bits beyond D_eff are NOT zero: must be ignored
    S = h.hdc_similarity(Hd, dev(C), kn).cpu().numpy()
    assert np.array_equal(S, S_or)
    lab, best, sec = h.hdc_classify(Hd, dev(C), kn, want_scores=True)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))


def test_hamming_padded_leading_dimensions(hd, h):
    r = rng(2)
    N, K, D = 100, 7, 1000
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.standard_normal((K, D + 24)).astype(np.float32)
    Hd = dev_bits(hb, ld_words=40)
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Cd = dev(C)[:, :D]                                     # ldc = D + 24
    S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    assert np.array_equal(S, O.similarity(hb, C[:, :D], D, O.SIM_HAMMING, 1))


# ------------------------------------------------------------------------------------ level-ID
@pytest.mark.parametrize("N,F,Q,D,D_eff", [(5, 1, 2, 64, 64), (33, 3, 4, 100, 100), (70, 16, 16, 2048, 2048),
                                           (70, 17, 256, 1100, 1000), (129, 100, 7, 3000, 2049),
                                           (40, 784, 256, 10000, 10000), (35, 1030, 256, 200, 33),
                                           (64, 31, 5, 40, 1)])
def test_levelid_bit_exact(hd, h, N, F, Q, D, D_eff):
    r = rng(3, N, F, Q, D_eff)
    lv = r.integers(0, Q, size=(N, F), dtype=np.uint8)
    lv[r.random((N, F)) < 0.5] = 0
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D_eff)
    kn = hd.knobs(D_eff)
    H = h.hdc_encode_levelid(dev(lv), dev_bits(ID), dev_bits(LV), D, kn)
    assert np.array_equal(host_bits(H, D_eff), bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:                                          # tail bits of the last word are zero
        assert (host_words(H)[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("zeros", [0.8, 0.97, 1.0])
@pytest.mark.parametrize("N,F,Q,D,D_eff", [(200, 784, 256, 10000, 10000), (97, 100, 16, 3000, 2049), (50, 36, 256, 1100, 1000),
                                           (130, 1020, 256, 200, 33), (49, 4, 3, 64, 64),
                                           (150, 617, 128, 1024, 1024), (60, 1023, 256, 96, 96), (75, 7, 9, 500, 499)])
def test_levelid_sparse_path_bit_exact(hd, h, zeros, N, F, Q, D, D_eff):
    """Mostly-zero level rows take the sparse path of the fast kernel (per-warp decision, base counter +
    listed features); a few fully dense rows mixed in exercise the per-warp fallback and the list
    capacity guard.  Bit-exact against the oracle either way."""
    r = rng(13, N, F, Q, D_eff, int(zeros * 100))
    lv = r.integers(1, Q, size=(N, F), dtype=np.uint8)
    lv[r.random((N, F)) < zeros] = 0
    lv[5 % N] = r.integers(1, Q, size=F, dtype=np.uint8)      # one fully dense sample
    if N > 60:
        lv[48:52] = r.integers(0, Q, size=(4, F), dtype=np.uint8)   # a dense group of four
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D_eff)
    H = h.hdc_encode_levelid(dev(lv), dev_bits(ID), dev_bits(LV), D, hd.knobs(D_eff))
    assert np.array_equal(host_bits(H, D_eff), bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (host_words(H)[:, W - 1] >> (D_eff % 32) == 0).all()


# ------------------------------------------------------------------------------------ RP encode
def _encode(hd, h, X, P, D_eff, prec, flags=0, bf16_inputs=False):
    kn = hd.knobs(D_eff, precision=prec, flags=flags)
    Xd, Pd = dev(X), dev(P)
    if bf16_inputs:
        Xd, Pd = Xd.to(torch.bfloat16), Pd.to(torch.bfloat16)
    H, raw = h.hdc_encode_rp(Xd, Pd, kn, want_raw=True)
    torch.cuda.synchronize()
    return host_bits(H, D_eff), raw.cpu().numpy(), host_words(H)


@pytest.mark.parametrize("prec", ["F32", "BF16", "F16", "I8", "B1"])
@pytest.mark.parametrize("flags", [0, 1, 2, 4])
@pytest.mark.parametrize("N,F,D,D_eff", [(200, 64, 2048, 2048), (131, 617, 1000, 999), (300, 100, 700, 33),
                                         (3, 7, 40, 40), (520, 784, 520, 515)])
def test_encode_rp_exact_arithmetic(hd, h, prec, flags, N, F, D, D_eff):
    """Integer features (0..255) and +-1 projections: every product and partial sum is an integer
    < 2^24, exact in bf16 operands and fp32 accumulation in any order, so fp32 / bf16 kernels
    (CUDA-core and tensor-core) must match the oracle bit for bit, sgn(0) cases included."""
    r = rng(4, N, F, D_eff)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    X[0] = 0                                                # all-zero row: every acc is 0 -> bit 0
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    if F % 2 == 0:
        P[1, ::2], P[1, 1::2] = 1.0, -1.0
        X[1] = 7.0                                          # acc[1,1] == 0 exactly
    p = getattr(O, prec)
    if prec == "I8":
        X[:, 0] = np.where(X.max(axis=1) > 0, 254.0, 0.0)   # row max 254 -> scale 0.5, ties to even
    bits_or, acc_or, _ = O.encode_rp(X, P, D_eff, p)
    bits, raw, words = _encode(hd, h, X, P, D_eff, getattr(hd, "HDC_" + prec), flags)
    assert np.array_equal(raw.astype(np.float64), acc_or)
    assert np.array_equal(bits, bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (words[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("prec", ["F32", "BF16", "I8"])
@pytest.mark.parametrize("flags", [0, 2, 4])
@pytest.mark.parametrize("D_eff,pad,off", [(10000, 0, 0), (10000, 3, 0), (10000, 7, 0), (10000, 3, 1), (4100, 0, 0),
                                           (4100, 3, 4), (8192, 0, 0), (8192, 4, 2), (240, 0, 0), (240, 4, 0)])
def test_encode_rp_row_stride_and_alignment_of_hbits(hd, h, prec, flags, D_eff, pad, off):
    """The sign+pack epilogue writes one 16-byte store per thread when the rows of Hbits are 16-byte aligned
    (ldh_words % 4 == 0 and an aligned base) and single words otherwise: every (ld, base offset) must give
    the oracle's bits, exactly W words per row, nothing else in the buffer touched (include/hdc.h)."""
    N, F = 300, 72
    r = rng(41, D_eff, pad, off)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D_eff, F))).astype(np.float32)
    bits_or, _, _ = O.encode_rp(X, P, D_eff, getattr(O, prec))
    W = (D_eff + 31) // 32
    ld = W + pad
    SENT = 0x5A5A5A5A
    buf = torch.full((N * ld + off + 8,), SENT, dtype=torch.int32, device="cuda")
    H = buf[off:off + N * ld].view(N, ld)[:, :W]
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), flags=flags)
    h.hdc_encode_rp(dev(X), dev(P), kn, Hbits=H)
    torch.cuda.synchronize()
    assert np.array_equal(host_bits(H, D_eff), bits_or)
    full = buf.cpu().numpy()
    assert (full[:off] == SENT).all() and (full[off + N * ld:] == SENT).all()
    if pad:
        assert (full[off:off + N * ld].reshape(N, ld)[:, W:] == SENT).all()
    if D_eff % 32:
        assert (host_words(H)[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("prec", ["F32", "BF16", "F16", "I8"])
@pytest.mark.parametrize("flags", [0, 1, 2, 4])
def test_encode_rp_float_c2_shape(hd, h, prec, flags):
    """Gaussian features / projection at the C2 shape (F=617, D=10000 sliced): raw accumulators
    within 1e-3 relative of the float64 oracle; sign mismatches only inside the rounding band."""
    w = gen.c2_isolet_shaped(D=1500, n_tr=8, n_te=300)
    X, P, D_eff = w["Xte"], w["P"], 1500
    p = getattr(O, prec)
    bits_or, acc_or, absum = O.encode_rp(X, P, D_eff, p, want_absum=True)
    bits, raw, _ = _encode(hd, h, X, P, D_eff, getattr(hd, "HDC_" + prec), flags)
    if prec == "I8":
        assert np.array_equal(raw.astype(np.float64), acc_or)
        assert np.array_equal(bits, bits_or)
    else:
        assert (np.abs(raw - acc_or) <= 1e-3 * np.abs(acc_or) + 1e-6 * absum).all()
        n = check_sign_band(bits, bits_or, acc_or, absum, X.shape[1])
        assert n <= 1e-4 * bits.size


def test_encode_rp_bf16_inputs_in_place(hd, h):
    """bf16 X and P handed over as bf16 (C5 style): used in place, identical to rounding fp32."""
    w = gen.c5_large_batch(n=200, D=768, K=10, F=1024, per_class=1)
    X, P = w["X"], w["P"]
    bits_or, acc_or, absum = O.encode_rp(X, P, 768, O.BF16, want_absum=True)
    bits, raw, _ = _encode(hd, h, X, P, 768, hd.HDC_BF16, 0, bf16_inputs=True)
    assert (np.abs(raw - acc_or) <= 1e-3 * np.abs(acc_or) + 1e-6 * absum).all()
    check_sign_band(bits, bits_or, acc_or, absum, 1024)


# ------------------------------------------------------------------------------------ dot / cos
@pytest.mark.parametrize("sim", ["DOT", "COS"])
@pytest.mark.parametrize("hv_bits", [32, 16, 17, 18, 8, 1])   # 17 = HDC_HV_F16 (IEEE half), 18 = HDC_HV_I16 (int16 codes)
@pytest.mark.parametrize("N,K,D,D_eff", [(150, 26, 2100, 2100), (64, 6, 10000, 4099), (33, 1, 500, 500),
                                         (140, 70, 1300, 1000), (140, 600, 1300, 1000), (300, 200, 700, 640),
                                         (130, 1000, 520, 520)])
@pytest.mark.parametrize("pad", [False, True])
def test_dot_cos_similarity_and_classify(hd, h, sim, hv_bits, N, K, D, D_eff, pad):
    """pad: query rows of W words rounded up to 4 (16-byte aligned rows, what Handle.alloc_hbits gives: class tiles of
    <= 128 rows then take sim_ts_kernel, fed by TMA) or exactly W words (any alignment: the cp.async rings)."""
    r = rng(5, N, K, D_eff, hv_bits)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 30).astype(np.float32)
    C[r.random((K, D)) < 0.03] = 0.0
    if K > 3:
        C[3] = 0.0                                          # zero-norm class: cosine 0
    simc = getattr(O, "SIM_" + sim)
    S_or = O.similarity(hb, C, D_eff, simc, hv_bits)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4 if pad else None), dev(C)
    S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
    lab = lab.cpu().numpy()
    lab_or, best_or, sec_or = O.classify(S_or, simc)
    if hv_bits in (18, 8, 1):                               # integer contraction: exact
        if sim == "DOT":
            # fp32 scores: the exact int32 sum, rounded once where it exceeds 24 bits (int16 codes only)
            assert np.array_equal(S, S_or.astype(np.float32))
            assert hv_bits == 18 or np.array_equal(S.astype(np.float64), S_or)
            Si = h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int32).cpu().numpy()
            assert np.array_equal(Si.astype(np.float64), S_or)
        else:
            assert np.allclose(S, S_or, rtol=1e-6, atol=1e-9)
        assert np.array_equal(lab, lab_or)
    else:
        cop = O.class_operand(C, D_eff, hv_bits)
        floor = 1e-6 * np.sqrt(D_eff) * np.sqrt((cop * cop).sum(axis=1))[None, :] if sim == "DOT" else 1e-6
        check_scores(S, S_or, floor)
        check_labels_float(lab, S_or, simc)
    same = lab == lab_or
    assert np.allclose(best.cpu().numpy()[same], best_or[same], rtol=1e-3, atol=1e-5)
    assert np.allclose(sec.cpu().numpy()[same], sec_or[same], rtol=1e-3, atol=1e-5)


@pytest.mark.parametrize("sim,hv_bits", [("COS", 32), ("DOT", 16), ("COS", 17), ("COS", 8), ("DOT", 8), ("DOT", 1), ("HAMMING", 1),
                                         ("COS", 18), ("DOT", 18)])
@pytest.mark.parametrize("N,K,D,D_eff,perf", [(300, 26, 2100, 2100, (0, 1)), (129, 1000, 520, 520, (0, 1)), (513, 200, 1300, 1000, (0, 1)),
                                              (1, 70, 700, 33, (0, 1)), (257, 600, 1300, 1000, (3, 8)), (640, 6, 10000, 4099, (0, 1))])
def test_similarity_on_cta_pairs(hd, h, sim, hv_bits, N, K, D, D_eff, perf):
    """sim_tc_kernel on CTA pairs (cta_group::2, HDC_FLAG_TC_2CTA forces it at any size): odd numbers of 256-query
    tiles, a pair whose peer has no valid row, class tiles of every width, perforation; scores and labels by the same
    rules as the one-CTA kernel, which must also give the same labels."""
    r = rng(55, N, K, D_eff, hv_bits)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 30).astype(np.float32)
    C[r.random((K, D)) < 0.03] = 0.0
    if K > 3:
        C[3] = 0.0
        C[2] = C[1]                                         # exact tie -> lowest index
    simc = getattr(O, "SIM_" + sim)
    S_or = O.similarity(hb, C, D_eff, simc, hv_bits, perf[0], perf[1])
    lab_or, best_or, sec_or = O.classify(S_or, simc)
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4 if N % 2 else None), dev(C)
    out = {}
    for flags in (hd.HDC_FLAG_TC_2CTA, hd.HDC_FLAG_TC_1CTA):
        kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), flags=flags, perf_begin=perf[0],
                      perf_stride=perf[1])
        S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
        lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
        lab = lab.cpu().numpy()
        if hv_bits in (18, 8, 1):
            if sim == "COS":
                assert np.allclose(S, S_or, rtol=1e-6, atol=1e-9)
            else:
                assert np.array_equal(S, S_or.astype(np.float32))
            assert np.array_equal(lab, lab_or)
            assert np.allclose(best.cpu().numpy(), best_or, rtol=1e-6, atol=1e-9)
            assert np.allclose(sec.cpu().numpy(), sec_or, rtol=1e-6, atol=1e-9)
        else:
            cop = O.class_operand(C[:, perf[0]:D_eff:perf[1]], len(range(perf[0], D_eff, perf[1])), hv_bits)
            floor = 1e-6 * np.sqrt(cop.shape[1]) * np.sqrt((cop * cop).sum(axis=1))[None, :] if sim == "DOT" else 1e-6
            check_scores(S, S_or, floor)
            check_labels_float(lab, S_or, simc)
        out[flags] = (S, lab)
    if hv_bits in (18, 8, 1):
        if sim == "COS":   # (the split-reduction path of the one-CTA kernel scales in double, the others in fp32)
            assert np.allclose(out[hd.HDC_FLAG_TC_2CTA][0], out[hd.HDC_FLAG_TC_1CTA][0], rtol=1e-6, atol=1e-9)
        else:
            assert np.array_equal(out[hd.HDC_FLAG_TC_2CTA][0], out[hd.HDC_FLAG_TC_1CTA][0])
        assert np.array_equal(out[hd.HDC_FLAG_TC_2CTA][1], out[hd.HDC_FLAG_TC_1CTA][1])


@pytest.mark.parametrize("hv_bits,K", [(16, 112), (16, 128), (16, 129), (8, 128), (8, 129), (1, 128), (1, 130), (32, 32),
                                       (32, 33), (18, 32), (18, 33), (17, 127), (32, 16), (8, 17)])
@pytest.mark.parametrize("N,D_eff", [(300, 4099), (2100, 1000), (129, 10000)])
def test_similarity_class_tile_width_boundaries(hd, h, hv_bits, K, N, D_eff):
    """Class tiles of exactly / just over 128 staged rows (96 / 144 for the three-part operands): the two sides of the
    switch between the kernel with the query tile in tensor memory and the one through shared memory, with few
    queries (split reduction axis) and many, rows 16-byte aligned; COS scores, labels, best / runner-up."""
    r = rng(77, hv_bits, K, N, D_eff)
    D = D_eff + 13
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 30).astype(np.float32)
    C[r.random((K, D)) < 0.03] = 0.0
    C[K - 1] = C[K - 2]                                     # exact tie between the last two classes of the tile
    S_or = O.similarity(hb, C, D_eff, O.SIM_COS, hv_bits)
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_COS)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=hd.HDC_SIM_COS)
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4), dev(C)
    S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
    lab = lab.cpu().numpy()
    if hv_bits in (18, 8, 1):
        assert np.allclose(S, S_or, rtol=1e-6, atol=1e-9)
        assert np.array_equal(lab, lab_or)
        assert np.allclose(best.cpu().numpy(), best_or, rtol=1e-6, atol=1e-9)
        assert np.allclose(sec.cpu().numpy(), sec_or, rtol=1e-6, atol=1e-9)
    else:
        check_scores(S, S_or, 1e-6)
        check_labels_float(lab, S_or, O.SIM_COS)


def test_classify_ties_go_to_lowest_index(hd, h):
    r = rng(6)
    N, K, D = 90, 9, 640
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-5, 6, size=(K, D)).astype(np.float32)
    C[5] = C[2]
    C[7] = C[2]
    for hv_bits, sim in [(32, "DOT"), (32, "COS"), (8, "COS"), (1, "HAMMING"), (1, "DOT")]:
        simc = getattr(O, "SIM_" + sim)
        lab_or, _, _ = O.classify(O.similarity(hb, C, D, simc, hv_bits), simc)
        kn = hd.knobs(D, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
        lab = h.hdc_classify(dev_bits(hb), dev(C), kn).cpu().numpy()
        assert np.array_equal(lab, lab_or), (hv_bits, sim)
        assert not np.isin(lab, [5, 7]).any()


# ------------------------------------------------------------------------------------ training
@pytest.mark.parametrize("N,K,D,D_eff", [(256, 4, 2048, 2048), (1000, 26, 1100, 1000), (70, 3, 64, 33)])
def test_bundle_exact(hd, h, N, K, D, D_eff):
    r = rng(7, N, K, D_eff)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    y = r.integers(0, K, size=N).astype(np.int32)
    C0 = r.integers(-3, 4, size=(K, D)).astype(np.float32)
    C_or = O.bundle(hb, y, K, D_eff, C0)
    Cd = dev(C0.copy())
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, dev_bits(hb), dev(y), Cd, hd.knobs(D_eff))
    out = Cd.cpu().numpy()
    assert np.array_equal(out[:, :D_eff], C_or)
    assert np.array_equal(out[:, D_eff:], C0[:, D_eff:])    # columns >= D_eff untouched


@pytest.mark.parametrize("B", [0, 1, 7, 64])
@pytest.mark.parametrize("hv_bits,sim", [(1, "HAMMING"), (8, "COS"), (18, "COS"), (18, "DOT"),
                                         (19, "COS"), (19, "DOT"), (20, "DOT")])   # 19 / 20 = HDC_HV_I32 / HDC_HV_I64
def test_perceptron_epoch_integer_paths_exact(hd, h, B, hv_bits, sim):
    """Integer similarity => identical predictions => identical Delta => identical fp32 update."""
    w = gen.c1_tiny(D=512)
    hb, _, _ = O.encode_rp(w["Xtr"], w["P"], 512, O.F32)
    y = w["ytr"].copy()
    y[::5] = (y[::5] + 1) % w["K"]                          # label noise so mispredictions persist
    D_eff = 500
    simc = getattr(O, "SIM_" + sim)
    C = O.bundle(hb, y, w["K"], 512)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
    Cd = dev(C.copy())
    Hd, yd = dev_bits(hb), dev(y)
    C_or = C[:, :D_eff].copy()
    for _ in range(3):
        C_or, wrong_or, pred_or = O.train_epoch(hb, y, C_or, D_eff, hv_bits, simc, 0.05, B)
        pred = torch.empty(len(y), dtype=torch.int32, device="cuda")
        nw = torch.zeros(1, dtype=torch.int64, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, Cd, kn, lr=0.05, batch=B, pred=pred, n_wrong=nw)
        assert np.array_equal(pred.cpu().numpy(), pred_or)
        assert int(nw.item()) == wrong_or
        assert np.array_equal(Cd.cpu().numpy()[:, :D_eff], C_or)
    assert np.array_equal(Cd.cpu().numpy()[:, D_eff:], C[:, D_eff:])


@pytest.mark.parametrize("hv_bits", [32, 16])
def test_perceptron_epoch_float_teacher_forced(hd, h, hv_bits):
    """fp32 / bf16 cosine: each epoch starts from the oracle's accumulators; predictions equal
    except near-ties; C_acc equal on every class row not touched by a near-tie sample."""
    w = gen.c2_isolet_shaped(D=2000, n_tr=1200, n_te=8)
    hb, _, _ = O.encode_rp(w["Xtr"], w["P"], 2000, O.F32)
    y, K, D_eff = w["ytr"], w["K"], 2000
    C_or = O.bundle(hb, y, K, D_eff)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=hd.HDC_SIM_COS)
    Hd, yd = dev_bits(hb), dev(y)
    for _ in range(3):
        S_or = O.similarity(hb, C_or, D_eff, O.SIM_COS, hv_bits)
        C_next, wrong_or, pred_or = O.train_epoch(hb, y, C_or, D_eff, hv_bits, O.SIM_COS, 0.05, 0)
        Cd = dev(C_or.copy())
        pred = torch.empty(len(y), dtype=torch.int32, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, Cd, kn, lr=0.05, batch=0, pred=pred)
        pred = pred.cpu().numpy()
        check_labels_float(pred, S_or, O.SIM_COS)
        near = np.nonzero(pred != pred_or)[0]
        touched = set(y[near]) | set(pred[near]) | set(pred_or[near])
        rows = [k for k in range(K) if k not in touched]
        assert np.array_equal(Cd.cpu().numpy()[rows], C_next[rows])
        assert wrong_or > 0
        C_or = C_next


# ------------------------------------------------------------------------------------ D_eff
@pytest.mark.parametrize("D_eff", [10000, 8192, 4096, 2048, 1024, 1000])
def test_d_eff_equals_physical_slice_on_gpu(hd, h, D_eff):
    """S3: results at D_eff equal those on arrays physically sliced to D_eff columns (bit-exact,
    GPU vs GPU and GPU vs oracle on the integer paths)."""
    w = gen.c4_har_shaped(D=10000, n_tr=8, n_te=96)
    X, P = w["Xte"], w["P"]
    kn_full = hd.knobs(D_eff, precision=hd.HDC_I8)
    H1 = h.hdc_encode_rp(dev(X), dev(P), kn_full)
    H2 = h.hdc_encode_rp(dev(X), dev(P[:D_eff].copy()), kn_full)
    assert torch.equal(H1, H2)
    bits_or, _, _ = O.encode_rp(X, P, D_eff, O.I8)
    assert np.array_equal(host_bits(H1, D_eff), bits_or)
    r = rng(8, D_eff)
    C = r.standard_normal((6, 10000)).astype(np.float32)
    kn = hd.knobs(D_eff, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Hfull = h.hdc_encode_rp(dev(X), dev(P), hd.knobs(10000, precision=hd.HDC_I8))
    S1 = h.hdc_similarity(Hfull, dev(C), kn)
    S2 = h.hdc_similarity(H1, dev(C[:, :D_eff].copy()), kn)
    assert torch.equal(S1, S2)


# ------------------------------------------------------------------------------------ HD-Clustering
@pytest.mark.parametrize("hv_bits,sim", [(1, "HAMMING"), (8, "COS"), (32, "COS"), (16, "COS")])
@pytest.mark.parametrize("N,K,D,D_eff", [(300, 5, 2048, 2048), (1000, 26, 3000, 2500), (40, 1, 96, 96)])
def test_kmeans_epochs_match_oracle(hd, h, hv_bits, sim, N, K, D, D_eff):
    """HD-Clustering epochs (PAPER.md L197 / L221, reading A16) from seeds taken among the samples,
    on noisy copies of K prototypes (clusters separated well enough that no cosine is a near-tie):
    assignments, moved-sample counts and re-bundled accumulators equal the oracle's exactly (the
    accumulators are small integers; empty clusters keep theirs)."""
    r = rng(9, N, K, D_eff, hv_bits)
    proto = r.integers(0, 2, size=(K, D), dtype=np.uint8)
    yt = r.integers(0, K, size=N)
    hb = proto[yt] ^ (r.random((N, D)) < 0.2).astype(np.uint8)
    seeds = r.choice(N, K, replace=False)
    C = np.zeros((K, D), dtype=np.float32)
    C[:, :] = 1.0 - 2.0 * hb[seeds]
    simc = getattr(O, "SIM_" + sim)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
    Cd, Hd = dev(C.copy()), dev_bits(hb)
    C_or, prev_or = C[:, :D_eff].copy(), None
    prev_d = None
    for _ in range(4):
        C_or, a_or, ch_or = O.kmeans_epoch(hb, C_or, D_eff, hv_bits, simc, prev_or)
        a_d = torch.empty(N, dtype=torch.int32, device="cuda")
        nch = torch.zeros(1, dtype=torch.int64, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_KMEANS, Hd, prev_d, Cd, kn, pred=a_d, n_wrong=nch)
        assert np.array_equal(a_d.cpu().numpy(), a_or)
        assert int(nch.item()) == ch_or
        assert np.array_equal(Cd.cpu().numpy()[:, :D_eff], C_or)
        prev_or, prev_d = a_or, a_d
    assert np.array_equal(Cd.cpu().numpy()[:, D_eff:], C[:, D_eff:])      # columns >= D_eff untouched


def test_kmeans_empty_cluster_keeps_accumulator(hd, h):
    r = rng(10)
    D = 512
    hb = r.integers(0, 2, size=(64, D), dtype=np.uint8)
    hb[:, :256] = hb[0, :256]                                # all samples close to sample 0
    c0 = 1.0 - 2.0 * hb[0].astype(np.float32)
    C = np.stack([c0, -c0, c0 * 0.5])                         # cluster 1 = antipode: never chosen; 2 ties with 0
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Cd = dev(C.copy())
    a_d = torch.empty(64, dtype=torch.int32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_KMEANS, dev_bits(hb), None, Cd, kn, pred=a_d)
    C_or, a_or, _ = O.kmeans_epoch(hb, C, D, 1, O.SIM_HAMMING)
    assert np.array_equal(a_d.cpu().numpy(), a_or) and (a_or == 0).all()   # ties -> lowest index
    got = Cd.cpu().numpy()
    assert np.array_equal(got, C_or)
    assert np.array_equal(got[1], C[1]) and np.array_equal(got[2], C[2])


# ------------------------------------------------------------------------------------ perforation
@pytest.mark.parametrize("begin,stride", [(0, 8), (3, 8), (5, 2), (1, 3), (17, 1), (0, 64)])
@pytest.mark.parametrize("sim,hv_bits", [("HAMMING", 1), ("DOT", 1), ("DOT", 8), ("COS", 8), ("COS", 32), ("COS", 16),
                                         ("DOT", 32), ("DOT", 18), ("COS", 18)])
@pytest.mark.parametrize("N,K,D,D_eff", [(150, 10, 2100, 2100), (70, 70, 1300, 1000), (33, 3, 10000, 8400)])
def test_perforated_similarity_and_classify(hd, h, begin, stride, sim, hv_bits, N, K, D, D_eff):
    """General reduction perforation of the similarity (reading A17): the kernels
    visit d = begin + j*stride < D_eff only and agree with the oracle's gather of those dimensions --
    exactly on the integer paths (popcount kernel for K < 64, +-1 / int8 tensor path), within the
    float rules otherwise."""
    r = rng(12, N, K, D_eff, hv_bits, begin, stride)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 30).astype(np.float32)
    C[r.random((K, D)) < 0.03] = 0.0
    simc = getattr(O, "SIM_" + sim)
    S_or = O.similarity(hb, C, D_eff, simc, hv_bits, begin, stride)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), perf_begin=begin, perf_stride=stride)
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4 if (begin + stride + N) % 2 else None), dev(C)
    S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    lab = h.hdc_classify(Hd, Cd, kn).cpu().numpy()
    lab_or, _, _ = O.classify(S_or, simc)
    if hv_bits in (18, 8, 1):
        if sim == "COS":
            assert np.allclose(S, S_or, rtol=1e-6, atol=1e-9)
        else:
            assert np.array_equal(S, S_or.astype(np.float32))
        assert np.array_equal(lab, lab_or)
    else:
        idx = O.perforated_index(D_eff, begin, stride)
        cop = O.class_operand(C[:, idx], len(idx), hv_bits)
        floor = 1e-6 * np.sqrt(len(idx)) * np.sqrt((cop * cop).sum(axis=1))[None, :] if sim == "DOT" else 1e-6
        check_scores(S, S_or, floor)
        check_labels_float(lab, S_or, simc)


@pytest.mark.parametrize("hv_bits,sim", [(1, "HAMMING"), (8, "COS")])
def test_perforated_training_epoch_exact(hd, h, hv_bits, sim):
    """Predictions use the perforated similarity, the update still touches every d < D_eff."""
    w = gen.c1_tiny(D=512)
    hb, _, _ = O.encode_rp(w["Xtr"], w["P"], 512, O.F32)
    y = w["ytr"].copy()
    y[::5] = (y[::5] + 1) % w["K"]
    simc = getattr(O, "SIM_" + sim)
    C = O.bundle(hb, y, w["K"], 512)
    kn = hd.knobs(500, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), perf_begin=2, perf_stride=4)
    Cd, Hd, yd = dev(C.copy()), dev_bits(hb), dev(y)
    C_or = C[:, :500].copy()
    for _ in range(2):
        C_or, wrong_or, pred_or = O.train_epoch(hb, y, C_or, 500, hv_bits, simc, 0.05, 64, begin=2, stride=4)
        pred = torch.empty(len(y), dtype=torch.int32, device="cuda")
        nw = torch.zeros(1, dtype=torch.int64, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, Cd, kn, lr=0.05, batch=64, pred=pred, n_wrong=nw)
        assert np.array_equal(pred.cpu().numpy(), pred_or)
        assert int(nw.item()) == wrong_or
        assert np.array_equal(Cd.cpu().numpy()[:, :500], C_or)


def test_perforation_argument_errors(hd, h):
    Hd = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    Cd = torch.ones((2, 128), dtype=torch.float32, device="cuda")
    for bad in (dict(perf_begin=128), dict(perf_begin=-1), dict(perf_stride=-2)):
        with pytest.raises(hd.HdcError) as ei:
            h.hdc_classify(Hd, Cd, hd.knobs(128, hv_bits=1, sim=hd.HDC_SIM_HAMMING, **bad))
        assert ei.value.code == hd.HDC_ERR_INVALID_ARG
    with pytest.raises(hd.HdcError) as ei:                  # CUDA-core DOT / COS kernels are not perforated
        h.hdc_classify(Hd, Cd, hd.knobs(128, hv_bits=32, sim=hd.HDC_SIM_COS, flags=hd.HDC_FLAG_SIMT, perf_stride=2))
    assert ei.value.code == hd.HDC_ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------ data-parallel training
@pytest.mark.parametrize("hv_bits,sim", [(1, "HAMMING"), (8, "COS"), (32, "COS"), (16, "COS")])
@pytest.mark.parametrize("B", [0, 100])
def test_train_delta_plus_apply_equals_train_epoch(hd, h, hv_bits, sim, B):
    """hdc_train_epoch(PERCEPTRON) = per mini-batch hdc_train_delta + hdc_train_apply; and the delta of
    a mini-batch is the integer sum of the deltas of its shards (two "ranks" emulated one after the
    other on this GPU -- predictions depend only on the current C_acc), so data-parallel replicas
    that all-reduce the int32 delta stay bit-identical to the single-GPU epoch."""
    w = gen.c1_tiny(D=512)
    hb, _, _ = O.encode_rp(w["Xtr"], w["P"], 512, O.F32)
    y = w["ytr"].copy()
    y[::4] = (y[::4] + 1) % w["K"]
    N, K, D_eff = len(y), w["K"], 500
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
    C0 = O.bundle(hb, y, K, 512)
    Hd, yd = dev_bits(hb), dev(y)
    C_ref, C_split, C_shard = dev(C0.copy()), dev(C0.copy()), dev(C0.copy())
    nw_ref = torch.zeros(1, dtype=torch.int64, device="cuda")
    nw_shard = torch.zeros(1, dtype=torch.int64, device="cuda")
    for _ in range(2):
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, C_ref, kn, lr=0.05, batch=B, n_wrong=nw_ref)
        Bb = N if B == 0 else B
        for b0 in range(0, N, Bb):
            b1 = min(N, b0 + Bb)
            d = h.hdc_train_delta(Hd[b0:b1], yd[b0:b1], C_split, kn)
            h.hdc_train_apply(C_split, kn, d, 0.05)
            mid = b0 + (b1 - b0 + 1) // 2                          # shard_bounds of two ranks
            d0 = h.hdc_train_delta(Hd[b0:mid], yd[b0:mid], C_shard, kn, n_wrong=nw_shard).clone()
            d1 = h.hdc_train_delta(Hd[mid:b1], yd[mid:b1], C_shard, kn, n_wrong=nw_shard)
            h.hdc_train_apply(C_shard, kn, d0 + d1, 0.05)          # what the all-reduce hands every rank
        assert torch.equal(C_split, C_ref)
        assert torch.equal(C_shard, C_ref)
    assert int(nw_shard.item()) == int(nw_ref.item())
    # and the oracle agrees on the integer paths
    if hv_bits in (1, 8):
        C_or = C0[:, :D_eff].copy()
        for _ in range(2):
            C_or, _, _ = O.train_epoch(hb, y, C_or, D_eff, hv_bits, getattr(O, "SIM_" + sim), 0.05, B)
        assert np.array_equal(C_ref.cpu().numpy()[:, :D_eff], C_or)


def test_train_delta_of_an_empty_shard_is_zero(hd, h):
    kn = hd.knobs(128, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Cc = torch.ones((3, 128), dtype=torch.float32, device="cuda")
    H0 = torch.zeros((0, 4), dtype=torch.int32, device="cuda")
    y0 = torch.zeros(0, dtype=torch.int32, device="cuda")
    d = torch.full((3, 128), 7, dtype=torch.int32, device="cuda")
    h.hdc_train_delta(H0, y0, Cc, kn, delta=d)
    assert int(d.abs().sum().item()) == 0


# ------------------------------------------------------------------------------------ 16-bit level indices
@pytest.mark.parametrize("N,F,Q,D,D_eff", [(70, 617, 814, 1024, 1024), (33, 617, 814, 1024, 512), (40, 64, 1000, 2048, 1999),
                                           (20, 1100, 300, 256, 256), (9, 5, 65535, 96, 96)])
def test_levelid_u16_indices_bit_exact(hd, h, N, F, Q, D, D_eff):
    """hdc_encode_levelid_u16: more than 256 levels (the Micro-HD comparison runs with up
    to 814 levels at D = 1024 / 512 on F = 617 features).  Bit-exact against the oracle."""
    r = rng(14, N, F, Q, D_eff)
    lv = r.integers(0, Q, size=(N, F)).astype(np.uint16)
    lv[0] = Q - 1
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D_eff)
    lvd = torch.from_numpy(lv.view(np.int16)).cuda()
    H = h.hdc_encode_levelid(lvd, dev_bits(ID), dev_bits(LV), D, hd.knobs(D_eff))
    assert np.array_equal(host_bits(H, D_eff), bits_or)


@pytest.mark.parametrize("N,F,Q,ld,col0,D,D_eff", [(333, 617, 814, 617, 0, 1024, 1024), (129, 617, 814, 620, 1, 1100, 1055),
                                                   (65, 640, 1024, 643, 3, 1024, 1000), (100, 63, 257, 63, 0, 4100, 4100),
                                                   (37, 1, 300, 4, 2, 64, 33), (50, 1020, 300, 1020, 0, 96, 96),
                                                   (40, 700, 1024, 700, 0, 512, 512)])
def test_levelid_u16_fast_kernel_shapes_bit_exact(hd, h, N, F, Q, ld, col0, D, D_eff):
    """16-bit level indices on the slice-resident fast kernel (Q <= 1024, tables + rows in shared memory): ragged
    batches (N not a multiple of 32), odd F, rows that start at odd element offsets of a wider matrix, several
    slices, partial last word; the last case exceeds the shared-memory budget and takes the general kernel."""
    r = rng(16, N, F, Q, D_eff)
    big = r.integers(0, Q, size=(N, ld)).astype(np.uint16)
    big[0, col0:col0 + F] = Q - 1
    big[r.random((N, ld)) < 0.2] = 0
    lv = big[:, col0:col0 + F]
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D_eff)
    lvd = torch.from_numpy(big.view(np.int16)).cuda()[:, col0:col0 + F]
    H = h.hdc_encode_levelid(lvd, dev_bits(ID), dev_bits(LV), D, hd.knobs(D_eff))
    assert np.array_equal(host_bits(H, D_eff), bits_or)


@pytest.mark.parametrize("F,ld,col0", [(617, 617, 0), (617, 620, 0), (616, 621, 1), (100, 107, 3), (1020, 1023, 3), (5, 9, 2)])
def test_levelid_unaligned_rows_bit_exact(hd, h, F, ld, col0):
    """Level rows that start at any byte offset (a column slice of a wider uint8 matrix; F not a
    multiple of 4): the fast kernel reads aligned words and re-aligns them with shuffles."""
    r = rng(15, F, ld, col0)
    N, Q, D = 101, 64, 1056
    big = r.integers(0, Q, size=(N, ld), dtype=np.uint8)
    big[r.random((N, ld)) < 0.6] = 0
    lv = big[:, col0:col0 + F]
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D)
    lvd = dev(big)[:, col0:col0 + F]
    H = h.hdc_encode_levelid(lvd, dev_bits(ID), dev_bits(LV), D, hd.knobs(D))
    assert np.array_equal(host_bits(H, D), bits_or)


# ------------------------------------------------------------------------------------ seeded fuzz
@pytest.mark.parametrize("case", range(48))
def test_similarity_classify_fuzz(hd, h, case):
    """Seeded random shapes / knobs through hdc_similarity + hdc_classify (every kernel choice the
    dispatcher can make: popcount, tensor path, split reduction axis, several n-tiles, perforation)."""
    r = rng(16, case)
    N = int(r.choice([1, 2, 31, 127, 128, 129, 300, 700, 2100]))
    K = int(r.choice([1, 2, 5, 16, 17, 63, 64, 65, 100, 257, 300]))
    D = int(r.choice([32, 33, 100, 512, 1000, 2048, 4099, 9000]))
    D_eff = int(r.integers(1, D + 1)) if r.random() < 0.5 else D
    sim, hv_bits = [("HAMMING", 1), ("DOT", 1), ("DOT", 8), ("COS", 8), ("COS", 32), ("COS", 16), ("DOT", 32),
                    ("DOT", 16)][int(r.integers(0, 8))]
    if hv_bits == 16 and case % 2:
        hv_bits = 17                                           # HDC_HV_F16
    if hv_bits == 8 and case % 3 == 0:
        hv_bits = 18                                           # HDC_HV_I16
    begin, stride = 0, 1
    if r.random() < 0.35:
        stride = int(r.choice([2, 3, 8, 32]))
        begin = int(r.integers(0, min(stride, D_eff)))
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 20).astype(np.float32)
    C[r.random((K, D)) < 0.02] = 0.0
    simc = getattr(O, "SIM_" + sim)
    S_or = O.similarity(hb, C, D_eff, simc, hv_bits, begin, stride)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), perf_begin=begin, perf_stride=stride)
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4 if case % 2 else None), dev(C)
    S = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    lab = h.hdc_classify(Hd, Cd, kn).cpu().numpy()
    lab_or, _, _ = O.classify(S_or, simc)
    if hv_bits in (18, 8, 1):
        if sim == "COS":
            assert np.allclose(S, S_or, rtol=1e-6, atol=1e-9)
        else:
            assert np.array_equal(S, S_or.astype(np.float32))
        assert np.array_equal(lab, lab_or)
    else:
        idx = O.perforated_index(D_eff, begin, stride)
        cop = O.class_operand(C[:, idx], len(idx), hv_bits)
        floor = 1e-6 * np.sqrt(len(idx)) * np.sqrt((cop * cop).sum(axis=1))[None, :] if sim == "DOT" else 1e-6
        check_scores(S, S_or, floor)
        check_labels_float(lab, S_or, simc)


@pytest.mark.parametrize("case", range(32))
def test_encode_rp_fuzz_exact(hd, h, case):
    """Seeded random shapes / precisions / kernel flags with integer-exact operands (see
    test_encode_rp_exact_arithmetic): accumulators and bits equal the oracle bit for bit."""
    r = rng(17, case)
    N = int(r.choice([1, 2, 127, 128, 129, 255, 257, 600, 1300]))
    F = int(r.choice([1, 2, 8, 31, 64, 65, 100, 617, 784, 1024, 1500]))
    D = int(r.choice([32, 33, 100, 255, 256, 257, 1000, 2048, 3001]))
    D_eff = int(r.integers(1, D + 1)) if r.random() < 0.5 else D
    prec = ["F32", "BF16", "I8", "B1"][int(r.integers(0, 4))]
    if prec == "BF16" and case % 2:
        prec = "F16"
    flags = int(r.choice([0, 1, 2, 4]))
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    if prec == "I8":
        X[:, 0] = np.where(X.max(axis=1) > 0, 254.0, 0.0)
    bits_or, acc_or, _ = O.encode_rp(X, P, D_eff, getattr(O, prec))
    bits, raw, words = _encode(hd, h, X, P, D_eff, getattr(hd, "HDC_" + prec), flags)
    assert np.array_equal(raw.astype(np.float64), acc_or)
    assert np.array_equal(bits, bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (words[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("case", range(32))
def test_levelid_fuzz_bit_exact(hd, h, case):
    """Seeded random (N, F, Q, D, D_eff, zero fraction, level dtype): general, fast dense and fast
    sparse kernels, aligned and unaligned rows."""
    r = rng(18, case)
    N = int(r.choice([1, 3, 4, 5, 47, 48, 49, 200]))
    F = int(r.choice([1, 2, 15, 16, 17, 63, 64, 65, 100, 617, 784, 1019, 1020, 1021, 1400]))
    wide = r.random() < 0.25
    Q = int(r.choice([2, 3, 16, 256])) if not wide else int(r.choice([257, 1000]))
    D = int(r.choice([32, 40, 100, 1024, 2049, 10000]))
    D_eff = int(r.integers(1, D + 1)) if r.random() < 0.5 else D
    zeros = float(r.choice([0.0, 0.5, 0.9, 0.99]))
    lv = r.integers(0, Q, size=(N, F)).astype(np.uint16 if wide else np.uint8)
    lv[r.random((N, F)) < zeros] = 0
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = gen.level_table(9, Q, D)
    bits_or = O.encode_levelid(lv, ID, LV, D_eff)
    lvd = torch.from_numpy(lv.astype(np.int16)).cuda() if wide else dev(lv)
    H = h.hdc_encode_levelid(lvd, dev_bits(ID), dev_bits(LV), D, hd.knobs(D_eff))
    assert np.array_equal(host_bits(H, D_eff), bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (host_words(H)[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("case", range(16))
def test_perceptron_epoch_fuzz_integer_paths(hd, h, case):
    """Seeded random (N, K, D, D_eff, batch, lr, perforation) on the integer-similarity paths: two
    epochs, predictions, wrong counts and accumulators bit-identical to the oracle."""
    r = rng(19, case)
    N = int(r.choice([1, 50, 257, 1100]))
    K = int(r.choice([1, 2, 7, 26, 70]))
    D = int(r.choice([64, 100, 1000, 2100]))
    D_eff = int(r.integers(1, D + 1)) if r.random() < 0.5 else D
    B = int(r.choice([0, 1, 13, 64, 4096]))
    hv_bits, sim = [(1, "HAMMING"), (8, "COS"), (8, "DOT"), (1, "DOT")][int(r.integers(0, 4))]
    begin, stride = 0, 1
    if r.random() < 0.3:
        stride = int(r.choice([2, 5, 8]))
        begin = int(r.integers(0, min(stride, D_eff)))
    lr = float(r.choice([1.0, 0.5, 0.03125]))
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    y = r.integers(0, K, size=N).astype(np.int32)
    C = r.integers(-5, 6, size=(K, D)).astype(np.float32)
    simc = getattr(O, "SIM_" + sim)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), perf_begin=begin, perf_stride=stride)
    Cd, Hd, yd = dev(C.copy()), dev_bits(hb), dev(y)
    C_or = C[:, :D_eff].copy()
    for _ in range(2):
        C_or, wrong_or, pred_or = O.train_epoch(hb, y, C_or, D_eff, hv_bits, simc, lr, B, begin, stride)
        pred = torch.empty(N, dtype=torch.int32, device="cuda")
        nw = torch.zeros(1, dtype=torch.int64, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, Cd, kn, lr=lr, batch=B, pred=pred, n_wrong=nw)
        assert np.array_equal(pred.cpu().numpy(), pred_or)
        assert int(nw.item()) == wrong_or
        assert np.array_equal(Cd.cpu().numpy()[:, :D_eff], C_or)
    assert np.array_equal(Cd.cpu().numpy()[:, D_eff:], C[:, D_eff:])


# ------------------------------------------------------------------------------------ A18 perforated encode
def _encode_perf(hd, h, X, P, D_eff, prec, begin, stride, flags=0, bf16_inputs=False):
    kn = hd.knobs(D_eff, precision=prec, flags=flags, enc_perf_begin=begin, enc_perf_stride=stride)
    Xd, Pd = dev(X), dev(P)
    if bf16_inputs:
        Xd, Pd = Xd.to(torch.bfloat16), Pd.to(torch.bfloat16)
    H, raw = h.hdc_encode_rp(Xd, Pd, kn, want_raw=True)
    torch.cuda.synchronize()
    assert raw.dtype == torch.float32
    return host_bits(H, D_eff), raw.cpu().numpy(), host_words(H)


@pytest.mark.parametrize("prec", ["F32", "BF16", "F16", "I8", "B1"])
@pytest.mark.parametrize("flags", [0, 1])
@pytest.mark.parametrize("N,F,D,D_eff,begin,stride", [(200, 64, 2048, 2048, 0, 2), (131, 617, 1000, 999, 5, 8),
                                                      (300, 100, 700, 33, 99, 3), (70, 784, 520, 515, 1, 2),
                                                      (129, 1024, 300, 300, 0, 4), (5, 7, 40, 40, 6, 1)])
def test_encode_rp_perforated_exact_arithmetic(hd, h, prec, flags, N, F, D, D_eff, begin, stride):
    """Perforated F reduction (reading A18) on integer-exact operands: bits equal the
    oracle bit for bit; the scaled accumulators agree to fp32 rounding of the scale (exactly when
    F / F_visited is a power of two)."""
    r = rng(20, N, F, D_eff, begin, stride)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    if prec == "I8":
        vis = O.perforated_index(F, begin, stride)
        X[:, vis[0]] = np.where(X[:, vis].max(axis=1) > 0, 254.0, 0.0)   # row max 254 over the visited columns
        X[:, np.setdiff1d(np.arange(F), vis)] *= 3.0                     # skipped columns must not set the scale
    bits_or, acc_or, _ = O.encode_rp(X, P, D_eff, getattr(O, prec), f_begin=begin, f_stride=stride)
    bits, raw, words = _encode_perf(hd, h, X, P, D_eff, getattr(hd, "HDC_" + prec), begin, stride, flags)
    assert np.array_equal(bits, bits_or)
    n_vis = len(O.perforated_index(F, begin, stride))
    if (F / n_vis) == 2.0 ** round(np.log2(F / n_vis)):
        assert np.array_equal(raw.astype(np.float64), acc_or)
    else:
        assert np.allclose(raw, acc_or, rtol=3e-7, atol=0)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (words[:, W - 1] >> (D_eff % 32) == 0).all()


@pytest.mark.parametrize("prec", ["F32", "BF16"])
def test_encode_rp_perforated_float_c2_shape(hd, h, prec):
    w = gen.c2_isolet_shaped(D=1500, n_tr=8, n_te=300)
    X, P, D_eff = w["Xte"], w["P"], 1500
    for begin, stride, bf in [(0, 2, False), (3, 8, False), (1, 2, True)]:
        Xo, Po = X, P
        if bf:   # bf16 inputs handed over as bf16: the compacted copies stay bf16
            Xo = np.asarray(torch.from_numpy(X).to(torch.bfloat16).float())
            Po = np.asarray(torch.from_numpy(P).to(torch.bfloat16).float())
        bits_or, acc_or, absum = O.encode_rp(Xo, Po, D_eff, getattr(O, prec), want_absum=True, f_begin=begin,
                                             f_stride=stride)
        bits, raw, _ = _encode_perf(hd, h, Xo, Po, D_eff, getattr(hd, "HDC_" + prec), begin, stride, 0, bf)
        assert (np.abs(raw - acc_or) <= 1e-3 * np.abs(acc_or) + 1e-6 * absum).all()
        n = check_sign_band(bits, bits_or, acc_or, absum, X.shape[1])
        assert n <= 1e-4 * bits.size


def test_encode_rp_perforation_argument_errors_and_workspace(hd, h):
    X = torch.zeros((8, 16), dtype=torch.float32, device="cuda")
    P = torch.zeros((128, 16), dtype=torch.float32, device="cuda")
    before = h.launch_count()
    for kw in ({"enc_perf_begin": 16}, {"enc_perf_begin": -1}, {"enc_perf_stride": -2}):
        with pytest.raises(hd.HdcError) as ei:
            h.hdc_encode_rp(X, P, hd.knobs(128, **kw))
        assert ei.value.code == hd.HDC_ERR_INVALID_ARG
    assert h.launch_count() == before
    kn0, kn1 = hd.knobs(128), hd.knobs(128, enc_perf_stride=2)
    assert h.workspace_bytes(hd.HDC_OP_ENCODE_RP, 8, 16, 128, 0, kn1) > 0
    # a perforated similarity knob does not touch the encoder and vice versa
    H0 = h.hdc_encode_rp(X + 1.0, P + 1.0, kn0)
    H1 = h.hdc_encode_rp(X + 1.0, P + 1.0, hd.knobs(128, perf_begin=3, perf_stride=8))
    assert torch.equal(H0, H1)


def test_infer_rp_host_with_perforated_encode_equals_device_calls(hd, h):
    """hdc_infer_rp_host reads the same knobs: a perforated encode (enc_perf_*) and a perforated
    similarity (perf_*) in one call give the labels of the two device calls; integer paths, exact."""
    r = rng(21)
    N, F, D, K = 40000, 100, 1100, 7                       # > 2 chunks of the host pipeline
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = r.integers(-9, 10, size=(K, D)).astype(np.float32)
    kn = hd.knobs(1000, precision=hd.HDC_BF16, hv_bits=1, sim=hd.HDC_SIM_HAMMING, perf_begin=1, perf_stride=2,
                  enc_perf_begin=2, enc_perf_stride=3)
    Pd, Cd = dev(P), dev(C)
    lab_dev = h.hdc_classify(h.hdc_encode_rp(dev(X), Pd, kn), Cd, kn).cpu().numpy()
    lab_host = h.hdc_infer_rp_host(torch.from_numpy(X).pin_memory(), Pd, Cd, kn).numpy()
    assert np.array_equal(lab_host, lab_dev)
    sub = slice(0, 300)
    bits_or, _, _ = O.encode_rp(X[sub], P, 1000, O.BF16, f_begin=2, f_stride=3)
    lab_or, _, _ = O.classify(O.similarity(bits_or, C, 1000, O.SIM_HAMMING, 1, 1, 2), O.SIM_HAMMING)
    assert np.array_equal(lab_dev[sub], lab_or)


# ------------------------------------------------------------------------------------ S12 / A19 ADC-quantised chunked dot
@pytest.mark.parametrize("res,step,fl,ce", [(8, 1, -127, 128), (8, 2, -3, 128), (6, 9, -3, 128), (3, 7, -40, 90),
                                            (16, 1, -128, 128), (1, 50, 0, 128)])
@pytest.mark.parametrize("N,K,D,D_eff", [(300, 26, 10000, 10000), (77, 6, 1100, 1024), (50, 70, 2100, 2047),
                                         (33, 1, 256, 129), (9, 40, 128, 1), (130, 33, 4500, 4099),
                                         (64, 100, 16384, 16384)])
def test_adc_similarity_bit_exact(hd, h, res, step, fl, ce, N, K, D, D_eff):
    """hdc_similarity_adc (reading A19): integer scores and labels equal the oracle."""
    r = rng(22, N, K, D_eff, res, step)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.standard_normal((K, D)).astype(np.float32)
    C[r.random((K, D)) < 0.05] = 0.0
    if K > 2:
        C[2] = C[1]                                            # exact tie between classes 1 and 2
        hb[0] = (C[1] < 0)                                      # query 0 == class 1 == class 2
    S_or = O.similarity_adc(hb, C, D_eff, res, step, fl, ce)
    lab_or, _, _ = O.classify(S_or, O.SIM_DOT)
    S, lab = h.hdc_similarity_adc(dev_bits(hb), dev(C), hd.knobs(D_eff), res, step, fl, ce)
    assert np.array_equal(S.cpu().numpy().astype(np.int64), S_or)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    _, lab2 = h.hdc_similarity_adc(dev_bits(hb), dev(C), hd.knobs(D_eff), res, step, fl, ce, want_scores=False)
    assert np.array_equal(lab2.cpu().numpy(), lab_or)


def test_adc_similarity_transparent_window_equals_hamming_path(hd, h):
    """The paper's baseline window is transparent: scores = D_eff - 2 * hdc_similarity(HAMMING)."""
    r = rng(23)
    N, K, D, D_eff = 500, 26, 10000, 8400
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.standard_normal((K, D)).astype(np.float32)
    Hd, Cd = dev_bits(hb), dev(C)
    S, _ = h.hdc_similarity_adc(Hd, Cd, hd.knobs(D_eff), 8, 1, -127, 128)
    ham = h.hdc_similarity(Hd, Cd, hd.knobs(D_eff, hv_bits=1, sim=hd.HDC_SIM_HAMMING))
    assert torch.equal(S, D_eff - 2 * ham)


def test_adc_similarity_argument_errors(hd, h):
    H = torch.zeros((8, 4), dtype=torch.int32, device="cuda")
    Cc = torch.ones((3, 128), dtype=torch.float32, device="cuda")
    before = h.launch_count()
    for bad in [(0, 1, -3, 128), (17, 1, -3, 128), (8, 0, -3, 128), (8, 1, 5, 4), (8, 1, -40000, 128),
                (8, 65537, -3, 128)]:
        with pytest.raises(hd.HdcError) as ei:
            h.hdc_similarity_adc(H, Cc, hd.knobs(128), *bad)
        assert ei.value.code == hd.HDC_ERR_INVALID_ARG
    with pytest.raises(hd.HdcError):
        h.hdc_similarity_adc(H, Cc, hd.knobs(128), 8, 1, -127, 128, want_scores=False, want_labels=False)
    assert h.launch_count() == before
    S, lab = h.hdc_similarity_adc(H[:0], Cc, hd.knobs(128), 8, 1, -127, 128)
    assert S.shape == (0, 3) and lab.shape == (0,)
    assert h.launch_count() == before


# ------------------------------------------------------------------------------------ fp16 class operand (L165)
@pytest.mark.parametrize("flags", [0, 1])
def test_fp16_class_operand_exact_on_small_integer_accumulators(hd, h, flags):
    """Accumulators that are integers of magnitude <= 2048 are exact in IEEE half (not in bf16), so the
    HDC_HV_F16 contraction (tcgen05 kind::f16 with half operands, or the CUDA-core kernel) must give
    the exact integer dot products -- and differ from the bf16 operand's."""
    r = rng(24, flags)
    N, K, D, D_eff = 300, 26, 2100, 2047
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-2048, 2049, size=(K, D)).astype(np.float32)
    S_or = O.similarity(hb, C, D_eff, O.SIM_DOT, O.HV_F16)
    assert np.array_equal(S_or, O.similarity(hb, C, D_eff, O.SIM_DOT, 32))
    kn = hd.knobs(D_eff, hv_bits=hd.HDC_HV_F16, sim=hd.HDC_SIM_DOT, flags=flags)
    S = h.hdc_similarity(dev_bits(hb), dev(C), kn).cpu().numpy()
    assert np.array_equal(S.astype(np.float64), S_or)          # |s| < 2^24: exact in the fp32 accumulator
    lab = h.hdc_classify(dev_bits(hb), dev(C), kn).cpu().numpy()
    assert np.array_equal(lab, O.classify(S_or, O.SIM_DOT)[0])
    S16 = h.hdc_similarity(dev_bits(hb), dev(C), hd.knobs(D_eff, hv_bits=16, sim=hd.HDC_SIM_DOT, flags=flags))
    assert not np.array_equal(S16.cpu().numpy(), S)


def test_fp16_perceptron_epoch_teacher_forced(hd, h):
    w = gen.c2_isolet_shaped(D=2000, n_tr=1200, n_te=8)
    hb, _, _ = O.encode_rp(w["Xtr"], w["P"], 2000, O.F32)
    y, K, D_eff = w["ytr"], w["K"], 2000
    C_or = O.bundle(hb, y, K, D_eff)
    kn = hd.knobs(D_eff, hv_bits=hd.HDC_HV_F16, sim=hd.HDC_SIM_COS)
    Hd, yd = dev_bits(hb), dev(y)
    for _ in range(2):
        S_or = O.similarity(hb, C_or, D_eff, O.SIM_COS, O.HV_F16)
        C_next, wrong_or, pred_or = O.train_epoch(hb, y, C_or, D_eff, O.HV_F16, O.SIM_COS, 0.05, 0)
        Cd = dev(C_or.copy())
        pred = torch.empty(len(y), dtype=torch.int32, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Hd, yd, Cd, kn, lr=0.05, batch=0, pred=pred)
        pred = pred.cpu().numpy()
        check_labels_float(pred, S_or, O.SIM_COS)
        near = np.nonzero(pred != pred_or)[0]
        touched = set(y[near]) | set(pred[near]) | set(pred_or[near])
        rows = [k for k in range(K) if k not in touched]
        assert np.array_equal(Cd.cpu().numpy()[rows], C_next[rows])
        C_or = C_next


def test_encode_rp_fp16_precision_on_bf16_inputs(hd, h):
    """precision HDC_F16 with bf16 inputs: widened exactly, then rounded to half (both kernels)."""
    w = gen.c5_large_batch(n=200, D=768, K=10, F=1024, per_class=1)
    Xb = np.asarray(torch.from_numpy(w["X"]).to(torch.bfloat16).float())
    Pb = np.asarray(torch.from_numpy(w["P"]).to(torch.bfloat16).float())
    bits_or, acc_or, absum = O.encode_rp(Xb, Pb, 768, O.F16, want_absum=True)
    for flags in (0, 1):
        bits, raw, _ = _encode(hd, h, Xb, Pb, 768, hd.HDC_F16, flags, bf16_inputs=True)
        assert (np.abs(raw - acc_or) <= 1e-3 * np.abs(acc_or) + 1e-6 * absum).all()
        check_sign_band(bits, bits_or, acc_or, absum, 1024)


@pytest.mark.parametrize("prec,hv_bits,sim,K,perf", [("F32", 32, "COS", 26, False), ("I8", 8, "COS", 6, False),
                                                     ("BF16", 1, "HAMMING", 10, True), ("F16", 17, "DOT", 7, False),
                                                     ("B1", 1, "HAMMING", 100, False), ("BF16", 16, "COS", 3, True)])
def test_infer_rp_host_chunks_reuse_staged_operands(hd, h, prec, hv_bits, sim, K, perf):
    """hdc_infer_rp_host stages P and prepares the class operand once and reuses them for the following
    chunks of equal size (the last, shorter chunk prepares again): labels equal the two device calls on
    the whole batch, for every precision / class-operand kind; exact-integer operands."""
    r = rng(25, K, hv_bits)
    N, F, D, D_eff = 16384 * 2 + 5000, 64, 1100, 1000
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = r.integers(-20, 21, size=(K, D)).astype(np.float32)
    kw = dict(perf_begin=3, perf_stride=4) if perf else {}
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), **kw)
    Pd, Cd = dev(P), dev(C)
    lab_dev = h.hdc_classify(h.hdc_encode_rp(dev(X), Pd, kn), Cd, kn).cpu().numpy()
    lab_host = h.hdc_infer_rp_host(torch.from_numpy(X).pin_memory(), Pd, Cd, kn).numpy()
    assert np.array_equal(lab_host, lab_dev)
    # a second call with another class model through the same workspace must not see stale operands
    C2 = -C
    lab_dev2 = h.hdc_classify(h.hdc_encode_rp(dev(X), Pd, kn), dev(C2), kn).cpu().numpy()
    lab_host2 = h.hdc_infer_rp_host(torch.from_numpy(X).pin_memory(), Pd, dev(C2), kn).numpy()
    assert np.array_equal(lab_host2, lab_dev2)
    assert not np.array_equal(lab_host2, lab_host)


# ------------------------------------------------------------------------------------ HDC_FLAG_F32_FAST (2 x fp16 split)
@pytest.mark.parametrize("flags", [8, 8 | 2, 8 | 4])
@pytest.mark.parametrize("N,F,D,D_eff", [(200, 64, 2048, 2048), (131, 617, 1000, 999), (300, 100, 700, 33),
                                         (3, 7, 40, 40), (520, 784, 520, 515)])
def test_encode_rp_f32_fast_exact_arithmetic(hd, h, flags, N, F, D, D_eff):
    """Integer features and +-1 projections are exact in the row-scaled half split, so the 3-product
    contraction must match the oracle bit for bit, raw accumulators (scales undone exactly) included."""
    r = rng(26, N, F, D_eff)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    X[0] = 0
    X[1 % N] *= 2.0 ** -20                                   # a tiny row: its own scale
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    P[2 % D] *= 2.0 ** 9
    bits_or, acc_or, _ = O.encode_rp(X, P, D_eff, O.F32)
    bits, raw, words = _encode(hd, h, X, P, D_eff, hd.HDC_F32, flags)
    assert np.array_equal(raw.astype(np.float64), acc_or)
    assert np.array_equal(bits, bits_or)
    W = (D_eff + 31) // 32
    if D_eff % 32:
        assert (words[:, W - 1] >> (D_eff % 32) == 0).all()


def test_encode_rp_f32_fast_error_bound_and_sign_band(hd, h):
    """Gaussian operands with a wide dynamic range inside each row (magnitudes over 2^-24 .. 1): the
    accumulators are as close to the float64 oracle as the CUDA-core fp32 FFMA kernel's, sign mismatches
    only inside the fp32 rounding band, and the result passes the same checks as the 6-product path."""
    r = rng(27)
    N, F, D = 300, 617, 1500
    X = (r.standard_normal((N, F)) * np.exp2(-24.0 * r.random((N, F)))).astype(np.float32)
    P = (r.standard_normal((D, F)) * np.exp2(-10.0 * r.random((D, F)))).astype(np.float32)
    X[:, 0] = 3.0                                            # one dominant element per row
    bits_or, acc_or, absum = O.encode_rp(X, P, D, O.F32, want_absum=True)
    bits, raw, _ = _encode(hd, h, X, P, D, hd.HDC_F32, hd.HDC_FLAG_F32_FAST)
    err = np.abs(raw - acc_or)
    # operand truncation is bounded by 3 * 2^-22 * sum|x p|; on top sits the fp32 accumulation error every
    # fp32 kernel has (here, with one dominant term per row, the larger of the two): hold the fast path to
    # the CUDA-core FFMA kernel's measured error on the same data
    _, raw_ffma, _ = _encode(hd, h, X, P, D, hd.HDC_F32, hd.HDC_FLAG_SIMT)
    ref = (np.abs(raw_ffma - acc_or) / absum).max()
    assert (err / absum).max() <= 1.5 * ref + 3 * 2.0 ** -22
    assert (err <= 4 * F * 2.0 ** -24 * absum).all()
    n = check_sign_band(bits, bits_or, acc_or, absum, F)
    assert n <= 1e-4 * bits.size
    # C2-shaped data: same tolerances as test_encode_rp_float_c2_shape
    w = gen.c2_isolet_shaped(D=1500, n_tr=8, n_te=300)
    bits_or, acc_or, absum = O.encode_rp(w["Xte"], w["P"], 1500, O.F32, want_absum=True)
    bits, raw, _ = _encode(hd, h, w["Xte"], w["P"], 1500, hd.HDC_F32, hd.HDC_FLAG_F32_FAST)
    assert (np.abs(raw - acc_or) <= 1e-3 * np.abs(acc_or) + 1e-6 * absum).all()
    n = check_sign_band(bits, bits_or, acc_or, absum, 617)
    assert n <= 1e-4 * bits.size
    print("f32_fast: max err / absum =", float((np.abs(raw - acc_or) / absum).max()), "sign mismatches", n)


def test_infer_rp_host_with_f32_fast_flag(hd, h):
    r = rng(28)
    N, F, D, K = 40000, 100, 1100, 7
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = r.integers(-9, 10, size=(K, D)).astype(np.float32)
    kn = hd.knobs(1000, precision=hd.HDC_F32, hv_bits=8, sim=hd.HDC_SIM_COS, flags=hd.HDC_FLAG_F32_FAST)
    Pd, Cd = dev(P), dev(C)
    lab_dev = h.hdc_classify(h.hdc_encode_rp(dev(X), Pd, kn), Cd, kn).cpu().numpy()
    lab_host = h.hdc_infer_rp_host(torch.from_numpy(X).pin_memory(), Pd, Cd, kn).numpy()
    assert np.array_equal(lab_host, lab_dev)
    bits_or, _, _ = O.encode_rp(X[:300], P, 1000, O.F32)
    lab_or, _, _ = O.classify(O.similarity(bits_or, C, 1000, O.SIM_COS, 8), O.SIM_COS)
    assert np.array_equal(lab_dev[:300], lab_or)
