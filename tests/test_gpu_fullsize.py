"""Full-size launches of BASELINE.json configs[2..4]: the CUDA path runs the whole batch in
the launch configuration bench.py / bench_rows.py time; the oracle checks rows sampled at the start, the middle
and the end of the batch one by one, and a property that holds at any size covers the rest.  Plus: repeated
launches of the CTA-pair kernels at awkward tile counts (every run must reproduce the first: cheap race / hang
evidence while compute-sanitizer is closed on this pool), and the exactness of the fp32 class operand on large
integer accumulators (16 / 32 / 64-bit integer element types)."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O
from workloads import gen

from gpu_util import check_labels_float, check_sign_band, dev, dev_bits, host_bits

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


def _spread(n, per):
    """`per` row indices at the start, the middle and the end of n rows (tile / batch / tail positions)."""
    mid = n // 2 - per // 2
    return np.concatenate([np.arange(0, per), np.arange(mid, mid + per), np.arange(n - per, n)])


# ------------------------------------------------------------------------------------ C3, full size
def test_c3_full_size_levelid_bundle_hamming(hd, h):
    """configs[2] at 60000 / 10000 samples: level-ID encode (bit-exact on 3 x 256 sampled rows of each split),
    bundle of all 60000 hypervectors (exact against the oracle's bundle of the hypervectors the kernel
    returned), Hamming classify of all 10000 test hypervectors (every label and distance exact)."""
    w = gen.c3_mnist_shaped()
    D, K, F = w["D"], w["K"], w["F"]
    assert w["Ltr"].shape == (60000, 784) and w["Lte"].shape == (10000, 784)
    IDd, LVd = dev_bits(w["ID"]), dev_bits(w["LV"])
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Htr = h.hdc_encode_levelid(dev(w["Ltr"]), IDd, LVd, D, kn)
    Hte = h.hdc_encode_levelid(dev(w["Lte"]), IDd, LVd, D, kn)
    for H, L in ((Htr, w["Ltr"]), (Hte, w["Lte"])):
        pos = _spread(L.shape[0], 256)
        got = host_bits(H[torch.from_numpy(pos).cuda()], D)
        assert np.array_equal(got, O.encode_levelid(L[pos], w["ID"], w["LV"], D))
    # identical images must give identical hypervectors wherever they sit (the rest of the batch)
    _, first, inv = np.unique(w["Lte"], axis=0, return_index=True, return_inverse=True)
    Hte_h = Hte.cpu().numpy()
    assert np.array_equal(Hte_h, Hte_h[first[inv.ravel()]])
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, dev(w["ytr"]), C, kn)
    btr = host_bits(Htr, D)
    C_or = None
    for n0 in range(0, btr.shape[0], 6000):                   # the oracle's bundle, accumulated in chunks
        C_or = O.bundle(btr[n0:n0 + 6000], w["ytr"][n0:n0 + 6000], K, D, C_acc=C_or)
    assert np.array_equal(C.cpu().numpy(), C_or)
    del btr
    lab, best, sec = h.hdc_classify(Hte, C, kn, want_scores=True)
    S_or = O.similarity(host_bits(Hte, D), C_or, D, O.SIM_HAMMING, 1)
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_HAMMING)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
    assert (lab_or == w["yte"]).mean() > 0.9


# ------------------------------------------------------------------------------------ C4, E = 20, full size
@pytest.mark.parametrize("prec,hv_bits,sim,D_eff", [("I8", 8, "COS", 10000), ("B1", 1, "HAMMING", 4096)])
def test_c4_full_size_twenty_epochs_integer_paths(hd, h, prec, hv_bits, sim, D_eff):
    """configs[3] at 7352 / 2947 samples, E = 20 retraining epochs (lr 0.05, B = N) on the integer paths: the
    class accumulators after every epoch count, the mispredictions per epoch and the test labels are the
    oracle's, bit for bit."""
    w = gen.c4_har_shaped()
    D, K = w["D"], w["K"]
    p, simc = getattr(O, prec), getattr(O, "SIM_" + sim)
    btr_or, acc_tr, ab_tr = O.encode_rp(w["Xtr"], w["P"], D_eff, p, want_absum=True)
    bte_or, _, _ = O.encode_rp(w["Xte"], w["P"], D_eff, p)
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim))
    Htr = h.hdc_encode_rp(dev(w["Xtr"]), dev(w["P"]), kn)
    if prec == "I8":
        assert np.array_equal(host_bits(Htr, D_eff), btr_or)
    else:
        check_sign_band(host_bits(Htr, D_eff), btr_or, acc_tr, ab_tr, w["F"])
    del acc_tr, ab_tr
    Htr_or, Hte_or, ytr = dev_bits(btr_or), dev_bits(bte_or), dev(w["ytr"])
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr_or, ytr, C, kn)
    C_or = O.bundle(btr_or, w["ytr"], K, D_eff)
    nw = torch.zeros(1, dtype=torch.int64, device="cuda")
    for e in range(20):
        C_or, wrong_or, _ = O.train_epoch(btr_or, w["ytr"], C_or, D_eff, hv_bits, simc, w["lr"], 0)
        nw.zero_()
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr_or, ytr, C, kn, lr=w["lr"], batch=0, n_wrong=nw)
        assert int(nw.item()) == wrong_or, e
        if e in (0, 4, 19):
            assert np.array_equal(C.cpu().numpy()[:, :D_eff], C_or), e
    lab = h.hdc_classify(Hte_or, C, kn).cpu().numpy()
    lab_or, _, _ = O.classify(O.similarity(bte_or, C_or, D_eff, simc, hv_bits), simc)
    assert np.array_equal(lab, lab_or)
    assert (lab_or == w["yte"]).mean() > 0.6


# ------------------------------------------------------------------------------------ C5, a whole batch
@pytest.mark.parametrize("variant", ["bf16", "1bit"])
def test_c5_whole_batch_encode_classify(hd, h, variant):
    """configs[4]: one whole 65536-query batch of the seeded C5 stream (F = 1024 bf16, D = 16384, K = 1000) through
    hdc_encode_rp + hdc_classify; the oracle checks 3 x 384 rows (start, middle, end of the batch) -- hypervectors in
    the sign band, labels by the class-operand rule on the oracle's similarity of the returned hypervectors --
    and every row of the batch must come back with the class it was drawn around (the set is cleanly separable)."""
    nb, D, K, F = 65536, 16384, 1000, 1024
    w = gen.c5_large_batch(nb, batch=0)
    Xd, Pd = dev(w["X"]).to(torch.bfloat16), dev(w["P"]).to(torch.bfloat16)
    H = h.hdc_encode_rp(Xd, Pd, hd.knobs(D, precision=hd.HDC_BF16))
    pos = _spread(nb, 384)
    bits_or, acc_or, absum = O.encode_rp(w["X"][pos], w["P"], D, O.BF16, want_absum=True)
    bits = host_bits(H[torch.from_numpy(pos).cuda()], D)
    check_sign_band(bits, bits_or, acc_or, absum, F)
    btr, _, _ = O.encode_rp(w["Xtr"], w["P"], D, O.BF16)
    C_or = O.bundle(btr, w["ytr"], K, D)
    Cd = dev(C_or)
    if variant == "bf16":
        kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=16, sim=hd.HDC_SIM_COS)
        lab = h.hdc_classify(H, Cd, kn).cpu().numpy()
        check_labels_float(lab[pos], O.similarity(bits, C_or, D, O.SIM_COS, 16), O.SIM_COS)
    else:
        kn = hd.knobs(D, precision=hd.HDC_B1, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
        lab, best, _ = h.hdc_classify(H, Cd, kn, want_scores=True)
        lab = lab.cpu().numpy()
        lab_or, best_or, _ = O.classify(O.similarity(bits, C_or, D, O.SIM_HAMMING, 1), O.SIM_HAMMING)
        assert np.array_equal(lab[pos], lab_or)
        assert np.array_equal(best.cpu().numpy()[pos], best_or.astype(np.float32))
    assert (lab == w["y"]).mean() > 0.999


# ------------------------------------------------------------------------------------ repeated launches
@pytest.mark.parametrize("prec", ["F32", "BF16", "I8"])
@pytest.mark.parametrize("N,D_eff,flags", [(257, 10000, 4), (256 * 37 + 1, 272, 4), (5000, 16, 4), (12345, 1000, 4),
                                           (74 * 256 + 255, 520, 0), (130, 10000, 2)])
def test_contraction_repeats_bit_for_bit(hd, h, prec, N, D_eff, flags):
    """The tcgen05 contraction (CTA pairs: odd pair counts, a pair with an empty peer, one-column tail tiles;
    single CTAs) launched 200 times back to back on the same inputs: every run must equal the first and the
    first must equal the oracle.  A lost mbarrier phase, a TMEM hand-back too early or a stale shared-memory
    slot shows up as a differing bit or a trapped wait."""
    F = 200
    r = np.random.default_rng([31, N, D_eff])
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D_eff, F))).astype(np.float32)
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), flags=flags)
    Xd, Pd = dev(X), dev(P)
    m = h.hdc_model_prepare(Pd, None, kn)
    H0 = h.hdc_encode_rp_m(Xd, m)
    assert np.array_equal(host_bits(H0, D_eff), O.encode_rp(X, P, D_eff, getattr(O, prec))[0])
    Hs = [h.alloc_hbits(N, D_eff) for _ in range(4)]
    bad = torch.zeros((), dtype=torch.int64, device="cuda")
    for i in range(200):
        Hi = Hs[i & 3]
        Hi.fill_(-1)
        h.hdc_encode_rp_m(Xd, m, Hbits=Hi)
        bad += (Hi != H0).any()
    torch.cuda.synchronize()
    assert int(bad.item()) == 0


@pytest.mark.parametrize("flags", [0, 4])
@pytest.mark.parametrize("hv_bits,sim,N,K,D_eff", [(32, "COS", 300, 26, 10000), (16, "COS", 129, 1000, 4100),
                                                   (1, "HAMMING", 777, 100, 10000), (8, "COS", 6238, 26, 10000),
                                                   (16, "COS", 74 * 256 + 130, 300, 1100)])
def test_similarity_repeats_bit_for_bit(hd, h, hv_bits, sim, N, K, D_eff, flags):
    """sim_tc_kernel (bit expanders + TMA + tcgen05; one CTA with and without the split reduction axis, CTA pairs
    with flags = HDC_FLAG_TC_2CTA or by size) 200 times."""
    r = np.random.default_rng([37, N, K])
    bits = r.integers(0, 2, size=(N, D_eff), dtype=np.uint8)
    C = (9 - 2 * r.binomial(9, 0.5, size=(K, D_eff))).astype(np.float32)
    kn = hd.knobs(D_eff, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim), flags=flags)
    Hd, Cd = dev_bits(bits), dev(C)
    m = h.hdc_model_prepare(None, Cd, kn)
    lab0, b0, s0 = h.hdc_classify_m(Hd, m, want_scores=True)
    S_or = O.similarity(bits, C, D_eff, getattr(O, "SIM_" + sim), hv_bits)
    if hv_bits in (8, 1):
        assert np.array_equal(lab0.cpu().numpy(), O.classify(S_or, getattr(O, "SIM_" + sim))[0])
    else:
        check_labels_float(lab0.cpu().numpy(), S_or, getattr(O, "SIM_" + sim))
    bad = torch.zeros((), dtype=torch.int64, device="cuda")
    for i in range(200):
        lab, b, s = h.hdc_classify_m(Hd, m, want_scores=True)
        bad += (lab != lab0).any() | (b != b0).any() | (s != s0).any()
    torch.cuda.synchronize()
    assert int(bad.item()) == 0


def test_fused_inference_repeats_bit_for_bit(hd, h):
    N, F, D, K = 74 * 256 + 131, 96, 1000, 26
    r = np.random.default_rng(41)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = (9 - 2 * r.binomial(9, 0.5, size=(K, D))).astype(np.float32)
    kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=8, sim=hd.HDC_SIM_COS, flags=hd.HDC_FLAG_FUSED_INFER)
    Xd = dev(X)
    m = h.hdc_model_prepare(dev(P), dev(C), kn)
    lab0, b0, s0 = h.hdc_infer_rp_m(Xd, m, want_scores=True)
    bad = torch.zeros((), dtype=torch.int64, device="cuda")
    for i in range(100):
        lab, b, s = h.hdc_infer_rp_m(Xd, m, want_scores=True)
        bad += (lab != lab0).any() | (b != b0).any() | (s != s0).any()
    torch.cuda.synchronize()
    assert int(bad.item()) == 0


# ------------------------------------------------------------------------------------ wide integer accumulators
@pytest.mark.parametrize("K", [26, 1000])
def test_fp32_class_operand_carries_24_bit_integers_exactly(hd, h, K):
    """PAPER.md L165 lists 16 / 32 / 64-bit integer element types.  Class accumulators are fp32 (A10) and hv_bits = 32
    contracts them as three bf16 parts: every integer |c| < 2^24 is carried EXACTLY (no operand rounding), and the
    contraction accumulates in fp32.  (i) accumulators with one entry near 2^24 and small ones elsewhere, every
    partial sum below 2^24: DOT scores equal the oracle's integers exactly; (ii) dense 24-bit accumulators, sums far
    beyond 2^24: scores within fp32 accumulation of the exact sum (2^-22 relative to sum|c|), labels by the 1e-3
    rule.  Wider integer storage types would differ from this only in how sums beyond 2^24 are rounded."""
    N, D = 384, 10000
    r = np.random.default_rng([43, K])
    bits = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = np.zeros((K, D), dtype=np.float64)
    C[:, :] = r.integers(-3, 4, size=(K, D)) * (r.random((K, D)) < 0.2)
    big = r.integers(0, D, size=K)
    C[np.arange(K), big] = (2 ** 24 - 1 - 40000 - r.integers(0, 1000, size=K)) * (1 - 2 * r.integers(0, 2, size=K))
    C[0, big[0]] = 2 ** 24 - 1 - 40000                                         # the largest operand used
    C32 = C.astype(np.float32)
    assert np.array_equal(C32.astype(np.float64), C)
    Hd = dev_bits(bits)
    kn = hd.knobs(D, hv_bits=32, sim=hd.HDC_SIM_DOT)
    S = h.hdc_similarity(Hd, dev(C32), kn).cpu().numpy().astype(np.float64)
    S_or = O.similarity(bits, C32, D, O.SIM_DOT, 32)
    assert np.abs(S_or).max() < 2 ** 24 and np.abs(S_or).max() > 2 ** 23
    assert np.array_equal(S, S_or)                                             # exact integers
    lab = h.hdc_classify(Hd, dev(C32), kn).cpu().numpy()
    assert np.array_equal(lab, O.classify(S_or, O.SIM_DOT)[0])
    # (ii) dense
    Cd = r.integers(-(2 ** 24 - 1), 2 ** 24, size=(K, D)).astype(np.float32)
    S = h.hdc_similarity(Hd, dev(Cd), kn).cpu().numpy().astype(np.float64)
    S_or = O.similarity(bits, Cd, D, O.SIM_DOT, 32)
    absum = np.abs(Cd.astype(np.float64)).sum(axis=1)
    assert (np.abs(S - S_or) <= 2.0 ** -22 * absum[None, :]).all()
    check_labels_float(h.hdc_classify(Hd, dev(Cd), kn).cpu().numpy(), S_or, O.SIM_DOT)


@pytest.mark.parametrize("K", [26, 1000])
@pytest.mark.parametrize("flags_name", ["", "HDC_FLAG_TC_1CTA", "HDC_FLAG_SIMT"])
def test_int16_class_operand_is_exact_in_int32(hd, h, K, flags_name):
    """PAPER.md L165 "integer data types (8, 16, ...": hv code HDC_HV_I16 (reading A21).  Dense 16-bit accumulators with
    max|c| = 32767 (scale exactly 1: the codes ARE the accumulators), D_eff = 10000, sums up to 3e8 -- far beyond what
    fp32 holds exactly: the int32 DOT scores equal the oracle's integers, the fp32 scores are those integers rounded
    once, labels (decided on the integers: adjacent integers above 2^24 collide as floats) and cosines agree; the
    tensor path (three base-128 digits on kind::i8, CTA pairs and one CTA) and the CUDA-core path alike."""
    N, D = 300, 10000
    flags = getattr(hd, flags_name) if flags_name else 0
    r = np.random.default_rng([44, K])
    bits = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-32767, 32768, size=(K, D)).astype(np.float32)
    C[0, 0] = 32767.0
    # class 2 = class 1 except one +-2 change in one dimension: their scores differ by 2 or 4 around 1e6..3e8
    C[2] = C[1]
    C[2, 17] = C[1, 17] - 2.0 if C[1, 17] > 0 else C[1, 17] + 2.0
    # queries 0..7 are (nearly) class 1's sign pattern: scores ~ sum|c| ~ 1.6e8 >> 2^24, winner decided by 2 units
    bits[:8] = (C[1] < 0).astype(np.uint8)[None, :]
    bits[:8, 17] = np.arange(8) % 2
    Hd, Cd = dev_bits(bits), dev(C)
    S_or = O.similarity(bits, C, D, O.SIM_DOT, O.HV_I16)
    assert np.array_equal(S_or, O.similarity(bits, C, D, O.SIM_DOT, 32))        # scale 1: codes = accumulators
    assert np.abs(S_or).max() > 2 ** 27
    kn = hd.knobs(D, hv_bits=hd.HDC_HV_I16, sim=hd.HDC_SIM_DOT, flags=flags)
    Si = h.hdc_similarity(Hd, Cd, kn, s_dtype=torch.int32).cpu().numpy()
    assert np.array_equal(Si.astype(np.float64), S_or)
    Sf = h.hdc_similarity(Hd, Cd, kn).cpu().numpy()
    assert np.array_equal(Sf, S_or.astype(np.float32))
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_DOT)
    assert set(lab_or[:8].tolist()) <= {1, 2} and len(set(lab_or[:8].tolist())) == 2
    lab, best, sec = h.hdc_classify(Hd, Cd, kn, want_scores=True)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
    # cosine: codes' norms in double, labels exact
    knc = hd.knobs(D, hv_bits=hd.HDC_HV_I16, sim=hd.HDC_SIM_COS, flags=flags)
    Sc_or = O.similarity(bits, C, D, O.SIM_COS, O.HV_I16)
    assert np.allclose(h.hdc_similarity(Hd, Cd, knc).cpu().numpy(), Sc_or, rtol=1e-6, atol=1e-9)
    assert np.array_equal(h.hdc_classify(Hd, Cd, knc).cpu().numpy(), O.classify(Sc_or, O.SIM_COS)[0])
    # a non-unit scale (max|c| not 32767) and a D_eff prefix
    C2 = (r.standard_normal((K, D)) * 30).astype(np.float32)
    kn2 = hd.knobs(4099, hv_bits=hd.HDC_HV_I16, sim=hd.HDC_SIM_DOT, flags=flags)
    S2_or = O.similarity(bits, C2, 4099, O.SIM_DOT, O.HV_I16)
    assert np.array_equal(h.hdc_similarity(Hd, dev(C2), kn2, s_dtype=torch.int32).cpu().numpy().astype(np.float64), S2_or)
    assert np.array_equal(h.hdc_classify(Hd, dev(C2), kn2).cpu().numpy(), O.classify(S2_or, O.SIM_DOT)[0])
