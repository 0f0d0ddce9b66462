"""32- and 64-bit integer class operands ("integer data types (8, 16, 32, or 64-bit)"; hv codes
HDC_HV_I32 / HDC_HV_I64, reading A22: q = rint(C_acc), no scale, symmetric saturation) through the C ABI:
the tensor-core route contracts the balanced 16-bit pieces of the codes on tcgen05 kind::i8 (sim_tc_kernel) and recombines
the pieces' int32 scores in 64 bits; widedot.cu's dp4a kernel over the byte planes of the codes is the CUDA-core route
(HDC_FLAG_SIMT).  On both the 64-bit integer sums must equal the oracle's python / int64 integers bit for bit at every shape (ragged query tiles, class
counts around the register tile, D_eff not a multiple of 4 / 32 / 512), saturating 32-bit codes, sums beyond 2^53,
perforation, ties, a zero class, padded query rows with dirty bits beyond D_eff."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O

from gpu_util import dev, dev_bits

pytestmark = pytest.mark.gpu

HV = {"I32": (19, O.HV_I32, 1.2e9), "I64": (20, O.HV_I64, 2.0 ** 52)}   # hv code, oracle code, accumulator magnitude


@pytest.fixture(scope="module")
def hd():
    import paper_2606_26547_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def h(hd):
    hh = hd.Handle(0)
    yield hh
    hh.close()


def test_codes_match_header(hd):
    assert (hd.HDC_HV_I32, hd.HDC_HV_I64, hd.HDC_I64) == (19, 20, 7)


@pytest.mark.parametrize("width", ["I32", "I64"])
@pytest.mark.parametrize("N,K,D,D_eff,perf", [(1, 1, 33, 33, (0, 1)), (5, 3, 100, 77, (0, 1)), (130, 9, 1000, 999, (0, 1)),
                                              (300, 26, 10000, 10000, (0, 1)), (257, 70, 2100, 2047, (0, 1)),
                                              (129, 8, 513, 513, (0, 1)), (128, 4, 512, 512, (0, 1)),
                                              (200, 13, 1300, 1000, (3, 4)), (64, 5, 700, 640, (1, 7))])
@pytest.mark.parametrize("pad", [False, True])
@pytest.mark.parametrize("flags_name", ["", "HDC_FLAG_SIMT", "HDC_FLAG_TC_2CTA"])
def test_wide_integer_similarity_and_classify(hd, h, width, N, K, D, D_eff, perf, pad, flags_name):
    """flags: default = the tensor-core route (16-bit pieces of the codes on sim_tc_kernel, recombined in 64 bits),
    HDC_FLAG_SIMT = the dp4a kernel over byte planes, HDC_FLAG_TC_2CTA = the pieces on CTA pairs."""
    flags = getattr(hd, flags_name) if flags_name else 0
    code, ocode, mag = HV[width]
    r = np.random.default_rng([71, code, N, K, D_eff])
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)       # bits beyond D_eff are random: they must not count
    C = (r.standard_normal((K, D)) * mag).astype(np.float32)
    C[r.random((K, D)) < 0.05] = 0.5                         # ties to even (-> 0) among the codes
    C[r.random((K, D)) < 0.05] = -2.5                        # -> -2
    if K > 4:
        C[3] = 0.0                                           # zero class: cosine 0
        C[4] = C[1]                                          # exact tie -> lowest index
    S_or = O.similarity(hb, C, D_eff, O.SIM_DOT, ocode, perf[0], perf[1])
    assert S_or.dtype == np.int64
    if width == "I64" and D_eff >= 1000 and perf[1] == 1:
        assert np.abs(S_or).max() > 2 ** 53                  # a float64 contraction would round here
    Hd, Cd = dev_bits(hb, (D + 127) // 128 * 4 if pad else None), dev(C)
    kn = hd.knobs(D_eff, hv_bits=code, sim=hd.HDC_SIM_DOT, flags=flags, perf_begin=perf[0], perf_stride=perf[1])
    Si = h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int64).cpu().numpy()
    assert np.array_equal(Si, S_or)
    Sf = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    assert np.array_equal(Sf, S_or.astype(np.float32))       # the exact sum rounded once
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_DOT)
    lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert K <= 4 or not (lab_or == 4).any()
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
    # cosine over the integer codes
    knc = hd.knobs(D_eff, hv_bits=code, sim=hd.HDC_SIM_COS, flags=flags, perf_begin=perf[0], perf_stride=perf[1])
    Sc_or = O.similarity(hb, C, D_eff, O.SIM_COS, ocode, perf[0], perf[1])
    Sc = h.hdc_similarity(Hd, Cd, knc).cpu().numpy()
    assert np.allclose(Sc, Sc_or, rtol=1e-6, atol=1e-12)
    assert K <= 4 or (Sc[:, 3] == 0.0).all()
    labc_or, bestc_or, secc_or = O.classify(Sc_or, O.SIM_COS)
    labc, bestc, secc = h.hdc_classify(Hd, Cd, knc, want_scores=True)
    assert np.array_equal(labc.cpu().numpy(), labc_or)
    assert np.allclose(bestc.cpu().numpy(), bestc_or, rtol=1e-6, atol=1e-12)
    assert np.allclose(secc.cpu().numpy(), secc_or, rtol=1e-6, atol=1e-12)


@pytest.mark.parametrize("width", ["I32", "I64"])
@pytest.mark.parametrize("flags_name", ["", "HDC_FLAG_SIMT"])
def test_wide_integer_operand_is_the_trained_accumulator(hd, h, width, flags_name):
    """Integer accumulators as bundling leaves them (L53 / L181): the 32- / 64-bit operand IS the accumulator -- DOT scores
    equal those of hv_bits = 32 computed by the oracle in float64, winners decided by 2 units at sums ~ 1e9 (far beyond
    what an fp32 accumulate holds); K = 1000 covers 125 / 250 class passes per CTA."""
    code, ocode, _ = HV[width]
    N, K, D = 200, 1000, 4100
    r = np.random.default_rng([72, code])
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-(2 ** 19), 2 ** 19, size=(K, D)).astype(np.float32)
    C[2] = C[1]
    C[2, 17] = C[1, 17] - 2.0 if C[1, 17] > 0 else C[1, 17] + 2.0
    hb[:8] = (C[1] < 0).astype(np.uint8)[None, :]
    hb[:8, 17] = np.arange(8) % 2
    S_or = O.similarity(hb, C, D, O.SIM_DOT, ocode)
    assert np.array_equal(S_or.astype(np.float64), O.similarity(hb, C, D, O.SIM_DOT, 32))
    assert np.abs(S_or).max() > 2 ** 29
    Hd, Cd = dev_bits(hb), dev(C)
    kn = hd.knobs(D, hv_bits=code, sim=hd.HDC_SIM_DOT, flags=getattr(hd, flags_name) if flags_name else 0)
    assert np.array_equal(h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int64).cpu().numpy(), S_or)
    lab_or = O.classify(S_or, O.SIM_DOT)[0]
    assert set(lab_or[:8].tolist()) == {1, 2}
    assert np.array_equal(h.hdc_classify(Hd, Cd, kn).cpu().numpy(), lab_or)


@pytest.mark.parametrize("width", ["I32", "I64"])
def test_wide_integer_row_passes_of_the_tensor_core_route(hd, h, width):
    """More queries than one pass of the tensor-core route holds (18944 rows at this K): two passes, the second one
    ragged; scores, labels and best / runner-up land in the right rows."""
    code, ocode, mag = HV[width]
    N, K, D = 19100, 450, 96
    r = np.random.default_rng([73, code])
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * mag).astype(np.float32)
    S_or = O.similarity(hb, C, D, O.SIM_DOT, ocode)
    Hd, Cd = dev_bits(hb), dev(C)
    kn = hd.knobs(D, hv_bits=code, sim=hd.HDC_SIM_DOT)
    assert np.array_equal(h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int64).cpu().numpy(), S_or)
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_DOT)
    lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
    knc = hd.knobs(D, hv_bits=code, sim=hd.HDC_SIM_COS)
    Sc_or = O.similarity(hb, C, D, O.SIM_COS, ocode)
    assert np.allclose(h.hdc_similarity(Hd, Cd, knc).cpu().numpy(), Sc_or, rtol=1e-6, atol=1e-12)
    assert np.array_equal(h.hdc_classify(Hd, Cd, knc).cpu().numpy(), O.classify(Sc_or, O.SIM_COS)[0])


@pytest.mark.parametrize("width", ["I32", "I64"])
def test_wide_integer_all_zero_pieces_are_skipped_exactly(hd, h, width):
    """The tensor-core route does not contract a 16-bit piece of the codes that is zero everywhere (small accumulators:
    the upper pieces) and the recombination skips its never-written scores: alternating models with and without live
    upper pieces on one handle (same workspace, stale piece scores in it) must each give the oracle's integers."""
    code, ocode, mag = HV[width]
    N, K, D = 700, 26, 1500
    r = np.random.default_rng([74, code])
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    Hd = dev_bits(hb)
    models = [(r.standard_normal((K, D)) * mag).astype(np.float32),                    # every piece live
              r.integers(-40, 41, size=(K, D)).astype(np.float32),                     # piece 0 only
              np.zeros((K, D), dtype=np.float32),                                      # no piece at all
              (r.integers(-3, 4, size=(K, D)) * 65536.0).astype(np.float32),           # piece 1 only
              (r.standard_normal((K, D)) * mag).astype(np.float32)]
    kn = hd.knobs(D, hv_bits=code, sim=hd.HDC_SIM_DOT)
    knc = hd.knobs(D, hv_bits=code, sim=hd.HDC_SIM_COS)
    for C in models:
        Cd = dev(C)
        S_or = O.similarity(hb, C, D, O.SIM_DOT, ocode)
        assert np.array_equal(h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int64).cpu().numpy(), S_or)
        lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
        lab_or, best_or, sec_or = O.classify(S_or, O.SIM_DOT)
        assert np.array_equal(lab.cpu().numpy(), lab_or)
        assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
        assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
        Sc_or = O.similarity(hb, C, D, O.SIM_COS, ocode)
        assert np.allclose(h.hdc_similarity(Hd, Cd, knc).cpu().numpy(), Sc_or, rtol=1e-6, atol=1e-12)


@pytest.mark.parametrize("width", ["I32", "I64"])
def test_wide_integer_classes_through_the_host_pipeline(hd, h, width):
    """hdc_infer_rp_host (chunks of 2048, 3072, ... rows; the first one prepares the class pieces, the later ones reuse
    them) and hdc_infer_rp on the same inputs: labels identical, and equal to the oracle's on exact-arithmetic inputs."""
    code, ocode, mag = HV[width]
    N, F, D, K = 30000, 48, 640, 11
    r = np.random.default_rng([75, code])
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = (r.standard_normal((K, D)) * mag).astype(np.float32)
    kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=code, sim=hd.HDC_SIM_DOT)
    Pd, Cd = dev(P), dev(C)
    lab = h.hdc_infer_rp(dev(X), Pd, Cd, kn).cpu().numpy()
    lab_host = h.hdc_infer_rp_host(torch.from_numpy(X).pin_memory(), Pd, Cd, kn).numpy()
    assert np.array_equal(lab_host, lab)
    bits = O.encode_rp(X, P, D, O.BF16)[0]
    assert np.array_equal(lab, O.classify(O.similarity(bits, C, D, O.SIM_DOT, ocode), O.SIM_DOT)[0])


def test_wide_integer_argument_errors(hd, h):
    hb = np.zeros((4, 64), dtype=np.uint8)
    C = np.ones((2, 64), dtype=np.float32)
    Hd, Cd = dev_bits(hb), dev(C)
    for code in (19, 20):
        with pytest.raises(Exception):                       # int32 scores cannot hold the sums
            h.hdc_similarity(Hd, Cd, hd.knobs(64, hv_bits=code, sim=hd.HDC_SIM_DOT), s_dtype=torch.int32)
        with pytest.raises(Exception):                       # the cosine is fp32
            h.hdc_similarity(Hd, Cd, hd.knobs(64, hv_bits=code, sim=hd.HDC_SIM_COS), s_dtype=torch.int64)
        with pytest.raises(Exception):                       # Hamming needs sign bits
            h.hdc_classify(Hd, Cd, hd.knobs(64, hv_bits=code, sim=hd.HDC_SIM_HAMMING))
    with pytest.raises(Exception):                           # int64 scores are for the wide integer operands
        h.hdc_similarity(Hd, Cd, hd.knobs(64, hv_bits=8, sim=hd.HDC_SIM_DOT), s_dtype=torch.int64)
