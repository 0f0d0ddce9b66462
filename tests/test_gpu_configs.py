"""End-to-end parity per BASELINE.json config (C1..C5) -- `-m gpu`.  The CUDA path runs the whole
pipeline through the C ABI; the oracle runs the same pipeline on the same seeded inputs.  Stage-wise
checks feed the GPU stage with the ORACLE's upstream output where a float stage would otherwise
make downstream integers incomparable."""
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


def _labels_ok_given_bitflips(lab, S_or, sim, flips_per_query):
    """Downstream of a float encode: labels equal except where the oracle's top-2 Hamming margin
    is <= 2 * (#mismatched bits of that query)."""
    lab_or, best, second = O.classify(S_or, sim)
    d = np.nonzero(lab != lab_or)[0]
    assert (np.abs(best - second)[d] <= 2 * flips_per_query[d]).all()
    return lab_or


def test_c1_tiny_end_to_end(hd, h):
    w = gen.c1_tiny()
    D, K = w["D"], w["K"]
    btr_or, acc_tr, ab_tr = O.encode_rp(w["Xtr"], w["P"], D, O.F32, want_absum=True)
    bte_or, acc_te, ab_te = O.encode_rp(w["Xte"], w["P"], D, O.F32, want_absum=True)
    kn_e = hd.knobs(D, precision=hd.HDC_F32)
    Htr = h.hdc_encode_rp(dev(w["Xtr"]), dev(w["P"]), kn_e)
    Hte = h.hdc_encode_rp(dev(w["Xte"]), dev(w["P"]), kn_e)
    check_sign_band(host_bits(Htr, D), btr_or, acc_tr, ab_tr, w["F"])
    check_sign_band(host_bits(Hte, D), bte_or, acc_te, ab_te, w["F"])
    flips = (host_bits(Hte, D) != bte_or).sum(axis=1)
    # free-running GPU pipeline
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, dev(w["ytr"]), C, hd.knobs(D))
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    lab = h.hdc_classify(Hte, C, kn).cpu().numpy()
    # oracle pipeline
    C_or = O.bundle(btr_or, w["ytr"], K, D)
    if np.array_equal(host_bits(Htr, D), btr_or):
        assert np.array_equal(C.cpu().numpy(), C_or)
    S_or = O.similarity(bte_or, C_or, D, O.SIM_HAMMING, 1)
    lab_or = _labels_ok_given_bitflips(lab, S_or, O.SIM_HAMMING, flips + 2 * int((host_bits(Htr, D) != btr_or).sum()))
    acc_gpu = (lab == w["yte"]).mean()
    acc_or = (lab_or == w["yte"]).mean()
    assert acc_or > 0.9 and abs(acc_gpu - acc_or) <= 0.01


def test_c2_isolet_shaped_full_size(hd, h):
    """configs[1] at full size: fp32 RP encode D=10000, bundle, 20 retraining epochs lr=0.05 (B=N),
    cosine classify.  Encode: sign band.  Inference from the oracle's hypervectors and class
    accumulators: score / label rules.  Free-running training: accuracy within 0.5 % and per-class
    cosine(C_gpu, C_oracle) >= 0.999."""
    w = gen.c2_isolet_shaped()
    D, K, F = w["D"], w["K"], w["F"]
    Pd = dev(w["P"])
    kn_e = hd.knobs(D, precision=hd.HDC_F32)
    btr_or, acc_tr, ab_tr = O.encode_rp(w["Xtr"], w["P"], D, O.F32, want_absum=True)
    Htr = h.hdc_encode_rp(dev(w["Xtr"]), Pd, kn_e)
    n_tr = check_sign_band(host_bits(Htr, D), btr_or, acc_tr, ab_tr, F)
    del acc_tr, ab_tr
    bte_or, acc_te, ab_te = O.encode_rp(w["Xte"], w["P"], D, O.F32, want_absum=True)
    Hte = h.hdc_encode_rp(dev(w["Xte"]), Pd, kn_e)
    n_te = check_sign_band(host_bits(Hte, D), bte_or, acc_te, ab_te, F)
    assert n_tr + n_te <= 1e-5 * (btr_or.size + bte_or.size) + 5
    # oracle training
    C_or, hist_or = O.train(btr_or, w["ytr"], K, D, 32, O.SIM_COS, w["epochs"], w["lr"])
    S_or = O.similarity(bte_or, C_or, D, O.SIM_COS, 32)
    # stage-wise inference: oracle H and oracle C through the GPU similarity / classify
    kn = hd.knobs(D, hv_bits=32, sim=hd.HDC_SIM_COS)
    Hte_or = dev_bits(bte_or)
    S = h.hdc_similarity(Hte_or, dev(C_or), kn).cpu().numpy()
    assert (np.abs(S - S_or) <= 1e-3 * np.abs(S_or) + 1e-6).all()
    lab = h.hdc_classify(Hte_or, dev(C_or), kn).cpu().numpy()
    check_labels_float(lab, S_or, O.SIM_COS)
    # free-running GPU training on the GPU's own hypervectors
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    ytr = dev(w["ytr"])
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, ytr, C, hd.knobs(D))
    nw = torch.zeros(1, dtype=torch.int64, device="cuda")
    hist = []
    for _ in range(w["epochs"]):
        nw.zero_()
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, C, kn, lr=w["lr"], batch=0, n_wrong=nw)
        hist.append(int(nw.item()))
    lab_free = h.hdc_classify(Hte, C, kn).cpu().numpy()
    lab_or, _, _ = O.classify(S_or, O.SIM_COS)
    acc_gpu, acc_or = (lab_free == w["yte"]).mean(), (lab_or == w["yte"]).mean()
    assert abs(acc_gpu - acc_or) <= 0.005
    Cg = C.cpu().numpy().astype(np.float64)
    cosk = (Cg * C_or).sum(1) / (np.linalg.norm(Cg, axis=1) * np.linalg.norm(C_or.astype(np.float64), axis=1))
    assert cosk.min() >= 0.999
    assert abs(hist[0] - hist_or[0]) <= 3 and hist[-1] <= hist[0]
    assert acc_or > 3.0 / K


def test_c3_mnist_shaped_levelid_pipeline(hd, h):
    """configs[2] (sample counts reduced so the oracle finishes in seconds; F, Q, D, K as stated):
    level-ID encode, bundle -> sign, packed Hamming classify.  Integer path: bit-exact throughout."""
    w = gen.c3_mnist_shaped(n_tr=1500, n_te=400)
    D, K, F, Q = w["D"], w["K"], w["F"], w["Q"]
    assert 0.7 < (w["Ltr"] == 0).mean() < 0.9
    IDd, LVd = dev_bits(w["ID"]), dev_bits(w["LV"])
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Htr = h.hdc_encode_levelid(dev(w["Ltr"]), IDd, LVd, D, kn)
    Hte = h.hdc_encode_levelid(dev(w["Lte"]), IDd, LVd, D, kn)
    btr_or = O.encode_levelid(w["Ltr"], w["ID"], w["LV"], D)
    bte_or = O.encode_levelid(w["Lte"], w["ID"], w["LV"], D)
    assert np.array_equal(host_bits(Htr, D), btr_or)
    assert np.array_equal(host_bits(Hte, D), bte_or)
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, dev(w["ytr"]), C, kn)
    C_or = O.bundle(btr_or, w["ytr"], K, D)
    assert np.array_equal(C.cpu().numpy(), C_or)
    lab, best, sec = h.hdc_classify(Hte, C, kn, want_scores=True)
    S_or = O.similarity(bte_or, C_or, D, O.SIM_HAMMING, 1)
    lab_or, best_or, sec_or = O.classify(S_or, O.SIM_HAMMING)
    assert np.array_equal(lab.cpu().numpy(), lab_or)
    assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32))
    assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32))
    assert (lab_or == w["yte"]).mean() > 0.8
    # one perceptron epoch on the packed path is exact too
    C2, wrong_or, pred_or = O.train_epoch(btr_or, w["ytr"], C_or, D, 1, O.SIM_HAMMING, 1.0, 256)
    nw = torch.zeros(1, dtype=torch.int64, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, dev(w["ytr"]), C, kn, lr=1.0, batch=256, n_wrong=nw)
    assert int(nw.item()) == wrong_or
    assert np.array_equal(C.cpu().numpy(), C2)


PRECS = [("fp32", "F32", 32, "COS"), ("bf16", "BF16", 16, "COS"), ("int8", "I8", 8, "COS"),
         ("1bit", "B1", 1, "HAMMING")]


@pytest.mark.parametrize("name,prec,hv_bits,sim", PRECS)
def test_c4_sweep_points(hd, h, name, prec, hv_bits, sim):
    """configs[3] (sample counts reduced): D_eff x precision x epochs.  Encode once at D=10000 per
    precision (prefix-stable, S3); per point the GPU trains on the ORACLE's hypervectors
    teacher-free and must reproduce the oracle's accuracy (integer paths: identical labels)."""
    w = gen.c4_har_shaped(n_tr=1500, n_te=600)
    D, K, F = w["D"], w["K"], w["F"]
    p, simc = getattr(O, prec), getattr(O, "SIM_" + sim)
    btr_or, acc_tr, ab_tr = O.encode_rp(w["Xtr"], w["P"], D, p, want_absum=True)
    bte_or, acc_te, ab_te = O.encode_rp(w["Xte"], w["P"], D, p, want_absum=True)
    kn_e = hd.knobs(D, precision=getattr(hd, "HDC_" + prec))
    Htr = h.hdc_encode_rp(dev(w["Xtr"]), dev(w["P"]), kn_e)
    Hte = h.hdc_encode_rp(dev(w["Xte"]), dev(w["P"]), kn_e)
    if prec == "I8":
        assert np.array_equal(host_bits(Htr, D), btr_or) and np.array_equal(host_bits(Hte, D), bte_or)
    else:
        check_sign_band(host_bits(Htr, D), btr_or, acc_tr, ab_tr, F)
        check_sign_band(host_bits(Hte, D), bte_or, acc_te, ab_te, F)
    Htr_or, Hte_or, ytr = dev_bits(btr_or), dev_bits(bte_or), dev(w["ytr"])
    for D_eff in w["d_eff"]:
        for E in (0, 5):
            C_or, _ = O.train(btr_or, w["ytr"], K, D_eff, hv_bits, simc, E, w["lr"])
            S_or = O.similarity(bte_or, C_or, D_eff, simc, hv_bits)
            lab_or, _, _ = O.classify(S_or, simc)
            kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits,
                          sim=getattr(hd, "HDC_SIM_" + sim))
            C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
            h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr_or, ytr, C, kn)
            for _ in range(E):
                h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr_or, ytr, C, kn, lr=w["lr"], batch=0)
            lab = h.hdc_classify(Hte_or, C, kn).cpu().numpy()
            if hv_bits in (8, 1):
                assert np.array_equal(C.cpu().numpy()[:, :D_eff], C_or), (name, D_eff, E)
                assert np.array_equal(lab, lab_or), (name, D_eff, E)
            else:
                acc_g, acc_o = (lab == w["yte"]).mean(), (lab_or == w["yte"]).mean()
                assert abs(acc_g - acc_o) <= 0.01, (name, D_eff, E, acc_g, acc_o)
            # inference from the oracle's model: score / label rules
            lab2 = h.hdc_classify(Hte_or, dev(np.pad(C_or, ((0, 0), (0, D - D_eff)))), kn).cpu().numpy()
            if hv_bits in (8, 1):
                assert np.array_equal(lab2, lab_or)
            else:
                check_labels_float(lab2, S_or, simc)


@pytest.mark.parametrize("variant", ["bf16", "1bit"])
def test_c5_large_batch_launch_config_sampled(hd, h, variant):
    """configs[4] in the launch configuration bench.py times (one 65536-query batch, F=1024 bf16,
    D=16384, K=1000), checked on sampled rows the oracle computes one by one (256 structured + 256
    unstructured near-tie queries placed at the start, middle and end of the batch)."""
    nb, ns, D, K, F = 65536, 256, 16384, 1000, 1024
    w = gen.c5_large_batch(n=ns, n_unstructured=ns, per_class=4)
    Xs, P = w["X"], w["P"]
    r = np.random.default_rng(5)
    filler = gen.from_bf16_bits(gen.to_bf16_bits(r.standard_normal((1024, F))))
    X = gen.tile_rows(filler, nb)
    pos = np.concatenate([np.arange(0, 128), np.arange(30000, 30000 + 256), np.arange(nb - 128, nb)])
    X[pos] = Xs
    Xd = dev(X).to(torch.bfloat16)
    Pd = dev(P).to(torch.bfloat16)
    kn_e = hd.knobs(D, precision=hd.HDC_BF16)
    H = h.hdc_encode_rp(Xd, Pd, kn_e)
    bits_or, acc_or, absum = O.encode_rp(Xs, P, D, O.BF16, want_absum=True)
    Hs = host_bits(H[torch.from_numpy(pos).cuda()], D)
    check_sign_band(Hs, bits_or, acc_or, absum, F)
    # class model from the oracle's encode of the training samples (even count per class)
    btr, _, _ = O.encode_rp(w["Xtr"], P, D, O.BF16)
    C_or = O.bundle(btr, w["ytr"], K, D)
    assert 0.01 < (C_or == 0).mean()
    Cd = dev(C_or)
    # classification of the whole batch with the oracle's sampled hypervectors spliced in
    Hin = H.clone()
    Hin[torch.from_numpy(pos).cuda()] = dev_bits(bits_or)
    if variant == "bf16":
        kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=16, sim=hd.HDC_SIM_COS)
        S_or = O.similarity(bits_or, C_or, D, O.SIM_COS, 16)
        lab = h.hdc_classify(Hin, Cd, kn).cpu().numpy()[pos]
        check_labels_float(lab, S_or, O.SIM_COS)
        lab_or, _, _ = O.classify(S_or, O.SIM_COS)
    else:
        kn = hd.knobs(D, precision=hd.HDC_B1, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
        S_or = O.similarity(bits_or, C_or, D, O.SIM_HAMMING, 1)
        lab_or, _, _ = O.classify(S_or, O.SIM_HAMMING)
        lab = h.hdc_classify(Hin, Cd, kn).cpu().numpy()[pos]
        assert np.array_equal(lab, lab_or)
    assert (lab_or[:ns] == w["y"][:ns]).mean() > 0.95


def test_c2_bench_launch_configuration_sampled(hd, h):
    """The step bench.py times: 131072 tiled C2 queries, fp32 encode on CTA pairs (886 waves of 256x256
    tiles) + cosine classify, and the host entry point.  The oracle checks the first 1559 rows (the
    test set once) bit by bit / label by label; a property that holds at any size covers the rest:
    row i is a copy of row i mod 1559, so every hypervector and label must repeat with that period
    wherever the row sits in a tile, a CTA pair or a chunk of the host pipeline."""
    w = gen.c2_isolet_shaped()
    D, K, F = w["D"], w["K"], w["F"]
    NQ, n_te = 131072, w["Xte"].shape[0]
    Xq = gen.tile_rows(w["Xte"], NQ)
    Pd = dev(w["P"])
    kn_e = hd.knobs(D, precision=hd.HDC_F32)
    kn = hd.knobs(D, precision=hd.HDC_F32, hv_bits=32, sim=hd.HDC_SIM_COS)
    Hq = h.hdc_encode_rp(dev(Xq), Pd, kn_e)
    bte_or, acc_te, ab_te = O.encode_rp(w["Xte"], w["P"], D, O.F32, want_absum=True)
    check_sign_band(host_bits(Hq[:n_te], D), bte_or, acc_te, ab_te, F)
    Hw = Hq.cpu().numpy()
    idx = np.arange(NQ)
    assert np.array_equal(Hw, Hw[idx % n_te]), "a tiled row encoded differently from its first copy"
    btr_or, _, _ = O.encode_rp(w["Xtr"][:2048], w["P"], D, O.F32)
    C_or = O.bundle(btr_or, w["ytr"][:2048], K, D)
    Cd = dev(C_or)
    lab = h.hdc_classify(Hq, Cd, kn).cpu().numpy()
    S_or = O.similarity(bte_or, C_or, D, O.SIM_COS, 32)
    check_labels_float(lab[:n_te], S_or, O.SIM_COS)
    assert np.array_equal(lab, lab[idx % n_te])
    Xh = torch.from_numpy(Xq).pin_memory()
    lab_host = h.hdc_infer_rp_host(Xh, Pd, Cd, kn).numpy()
    # the host pipeline runs the fused kernel per chunk: same hypervectors, scores summed in another order, so
    # it answers to the oracle by the same rule rather than to the two-kernel path bit for bit
    check_labels_float(lab_host[:n_te], S_or, O.SIM_COS)
    assert np.array_equal(lab_host, lab_host[idx % n_te])
