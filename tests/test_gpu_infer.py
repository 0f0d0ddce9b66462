"""Parity of hdc_infer_rp -- encode + similarity + arg-max in one call; with HDC_FLAG_FUSED_INFER ONE tcgen05
kernel for small class models (include/hdc.h; Listing 1 L63-L81, L161) -- against the CPU oracle,
through the C ABI.

The encode stage is checked as in test_gpu_kernels.py (bit-exact on exact-arithmetic inputs, sign band on float
inputs); the similarity + arg-max stage is checked against the oracle's similarity of the hypervectors the call
itself returned (stage-wise: a legitimately flipped bit of a float encode must not be charged to the classifier),
bit-exact for the integer class operands (hv_bits 8 and 1), by the 1e-3 rules for the float ones."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O
from workloads import gen

from gpu_util import check_labels_float, check_sign_band, dev, host_bits

pytestmark = pytest.mark.gpu

SIMS = {"DOT": O.SIM_DOT, "COS": O.SIM_COS, "HAMMING": O.SIM_HAMMING}


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
    return np.random.default_rng([977, *[int(k) for k in key]])


def _int_inputs(N, F, D, K, key):
    """Exact-arithmetic encode inputs (integer features, +-1 projection) and integer class accumulators shaped
    like a bundle of 21 hypervectors per class, with exact zeros and tied classes."""
    r = rng(*key)
    X = r.integers(0, 256, size=(N, F)).astype(np.float32)
    X[r.random((N, F)) < 0.3] = 0
    X[0] = 0
    P = (1.0 - 2.0 * r.integers(0, 2, size=(D, F))).astype(np.float32)
    C = (21 - 2 * r.binomial(21, 0.5, size=(K, D))).astype(np.float32)
    C[:, ::7] = 0.0                                       # sgn(0) in the class operand
    if K >= 3:
        C[2] = C[1]                                       # a tie between classes 1 and 2 -> lowest index
    return X, P, C


def _check_stage2(hd, lab, best, second, bits, C, D_eff, sim_name, hv_bits, begin=0, stride=1):
    sim = SIMS[sim_name]
    S_or = O.similarity(bits, C, D_eff, sim, hv_bits, begin, stride)
    lab_or, b_or, s_or = O.classify(S_or, sim)
    if hv_bits in (20, 19, 18, 8, 1):
        assert np.array_equal(lab, lab_or)
        assert np.allclose(best, b_or, rtol=1e-6, atol=1e-6) and np.allclose(second, s_or, rtol=1e-6, atol=1e-6)
    else:
        check_labels_float(lab, S_or, sim)
        n = np.arange(lab.size)
        floor = 1e-6 if sim == O.SIM_COS else 1e-6 * np.sqrt(D_eff) * np.linalg.norm(C[:, :D_eff], axis=1).max()
        assert (np.abs(best - S_or[n, lab]) <= 1e-3 * np.abs(S_or[n, lab]) + floor).all()


@pytest.mark.parametrize("prec", ["F32", "BF16", "I8"])
@pytest.mark.parametrize("sim_name,hv_bits", [("COS", 32), ("DOT", 32), ("COS", 16), ("COS", 17), ("COS", 8), ("DOT", 8),
                                              ("DOT", 1), ("HAMMING", 1)])
@pytest.mark.parametrize("N,F,D,D_eff,K", [(12288 + 37, 64, 1000, 1000, 26), (12500, 72, 4100, 4100, 6),
                                           (12288, 64, 300, 257, 32), (13000, 40, 256, 256, 1),
                                           (12800, 64, 700, 33, 9), (12345, 96, 520, 515, 16), (12300, 64, 640, 640, 8)])
def test_infer_rp_fused_exact_arithmetic(hd, h, prec, sim_name, hv_bits, N, F, D, D_eff, K):
    X, P, C = _int_inputs(N, F, D, K, (1, N, F, D_eff, K))
    if prec == "I8":
        X[:, 0] = np.where(X.max(axis=1) > 0, 254.0, 0.0)
    bits_or, _, _ = O.encode_rp(X, P, D_eff, getattr(O, prec))
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim_name),
                  flags=hd.HDC_FLAG_FUSED_INFER)
    H = h.alloc_hbits(N, D_eff)
    f0 = h.stat(hd.HDC_STAT_INFER_FUSED)
    lab, best, second = h.hdc_infer_rp(dev(X), dev(P), dev(C), kn, want_scores=True, Hbits=H)
    torch.cuda.synchronize()
    assert h.stat(hd.HDC_STAT_INFER_FUSED) == f0 + 1, "the fused kernel was not taken"
    bits = host_bits(H, D_eff)
    assert np.array_equal(bits, bits_or)                       # exact arithmetic: bit for bit, sgn(0) included
    _check_stage2(hd, lab.cpu().numpy(), best.cpu().numpy(), second.cpu().numpy(), bits, C, D_eff, sim_name, hv_bits)
    # without the hypervector output: same labels and scores
    lab2, best2, second2 = h.hdc_infer_rp(dev(X), dev(P), dev(C), kn, want_scores=True)
    assert torch.equal(lab2, lab) and torch.equal(best2, best) and torch.equal(second2, second)


@pytest.mark.parametrize("prec", ["F32", "BF16", "F16", "I8", "B1"])
@pytest.mark.parametrize("sim_name,hv_bits", [("COS", 32), ("COS", 8), ("HAMMING", 1)])
def test_infer_rp_fused_float_c2_shape(hd, h, prec, sim_name, hv_bits):
    """Gaussian mixture features / Gaussian projection at the C2 shape (F = 617, K = 26), D sliced to 1500."""
    w = gen.c2_isolet_shaped(D=1500, n_tr=600, n_te=1559)
    D_eff, K, F = 1500, w["K"], w["F"]
    N = 12288 + 131
    X = gen.tile_rows(w["Xte"], N)
    p = getattr(O, prec)
    btr, _, _ = O.encode_rp(w["Xtr"], w["P"], D_eff, p)
    C = O.bundle(btr, w["ytr"], K, D_eff)
    C, _, _ = O.train_epoch(btr, w["ytr"], C, D_eff, 32, O.SIM_COS, 0.05, 0)     # non-integer accumulators
    n_te = w["Xte"].shape[0]
    bits_or, acc_or, absum = O.encode_rp(w["Xte"], w["P"], D_eff, p, want_absum=True)
    kn = hd.knobs(D_eff, precision=getattr(hd, "HDC_" + prec), hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim_name),
                  flags=hd.HDC_FLAG_FUSED_INFER)
    H = h.alloc_hbits(N, D_eff)
    f0 = h.stat(hd.HDC_STAT_INFER_FUSED)
    lab, best, second = h.hdc_infer_rp(dev(X), dev(w["P"]), dev(C), kn, want_scores=True, Hbits=H)
    torch.cuda.synchronize()
    assert h.stat(hd.HDC_STAT_INFER_FUSED) == f0 + 1
    bits = host_bits(H, D_eff)
    if prec == "I8":
        assert np.array_equal(bits[:n_te], bits_or)
    else:
        check_sign_band(bits[:n_te], bits_or, acc_or, absum, F)
    assert np.array_equal(bits, bits[np.arange(N) % n_te])       # tiled rows: same hypervector wherever the row sits
    _check_stage2(hd, lab.cpu().numpy(), best.cpu().numpy(), second.cpu().numpy(), bits, C, D_eff, sim_name, hv_bits)
    # end to end against the oracle's own pipeline (its hypervectors, its labels): same accuracy
    lab_or, _, _ = O.classify(O.similarity(bits_or, C, D_eff, SIMS[sim_name], hv_bits), SIMS[sim_name])
    acc, acc_or = (lab.cpu().numpy()[:n_te] == w["yte"]).mean(), (lab_or == w["yte"]).mean()
    assert abs(acc - acc_or) <= 0.01 and acc_or > 2.0 / K


@pytest.mark.parametrize("sim_name,hv_bits,begin,stride", [("COS", 32, 0, 8), ("COS", 8, 3, 8), ("HAMMING", 1, 5, 2),
                                                           ("DOT", 16, 100, 1)])
def test_infer_rp_fused_perforated_similarity(hd, h, sim_name, hv_bits, begin, stride):
    N, F, D, K = 12300, 64, 1000, 26
    X, P, C = _int_inputs(N, F, D, K, (3, begin, stride))
    kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=hv_bits, sim=getattr(hd, "HDC_SIM_" + sim_name), perf_begin=begin,
                  perf_stride=stride, flags=hd.HDC_FLAG_FUSED_INFER)
    H = h.alloc_hbits(N, D)
    lab, best, second = h.hdc_infer_rp(dev(X), dev(P), dev(C), kn, want_scores=True, Hbits=H)
    bits = host_bits(H, D)
    assert np.array_equal(bits, O.encode_rp(X, P, D, O.BF16)[0])       # the encode is not perforated by these knobs
    _check_stage2(hd, lab.cpu().numpy(), best.cpu().numpy(), second.cpu().numpy(), bits, C, D, sim_name, hv_bits, begin,
                  stride)


@pytest.mark.parametrize("N,K,flags,hv_bits", [(12288, 26, 0, 8), (12288, 33, 16, 8), (500, 26, 16, 8),
                                               (12288, 26, 16 | 1, 8), (12288, 26, 16 | 2, 8), (0, 26, 16, 8),
                                               (12288, 26, 16, 18), (700, 26, 0, 18),
                                               (12288, 26, 16, 19), (700, 26, 0, 20)])   # 19 / 20 = HDC_HV_I32 / _I64
def test_infer_rp_two_kernel_path_and_stats(hd, h, N, K, flags, hv_bits):
    """The default (no HDC_FLAG_FUSED_INFER = 16), and with the flag: large K, small N, HDC_FLAG_SIMT,
    HDC_FLAG_TC_1CTA and int16 class codes (hv code 18: sums beyond what the fused fp32 search holds exactly),
    take hdc_encode_rp + hdc_classify; the result obeys the same rules and hdc_stat reports which path ran."""
    F, D = 64, 600
    X, P, C = _int_inputs(max(N, 1), F, D, K, (4, N, K, flags))
    X = X[:N]
    kn = hd.knobs(D, precision=hd.HDC_BF16, hv_bits=hv_bits, sim=hd.HDC_SIM_COS, flags=flags)
    u0, f0 = h.stat(hd.HDC_STAT_INFER_UNFUSED), h.stat(hd.HDC_STAT_INFER_FUSED)
    H = h.alloc_hbits(N, D)
    lab, best, second = h.hdc_infer_rp(dev(X) if N else torch.empty((0, F), device="cuda"), dev(P), dev(C), kn,
                                       want_scores=True, Hbits=H)
    torch.cuda.synchronize()
    assert h.stat(hd.HDC_STAT_INFER_FUSED) == f0
    assert h.stat(hd.HDC_STAT_INFER_UNFUSED) == u0 + (1 if N else 0)
    if N:
        bits = host_bits(H, D)
        assert np.array_equal(bits, O.encode_rp(X, P, D, O.BF16)[0])
        _check_stage2(hd, lab.cpu().numpy(), best.cpu().numpy(), second.cpu().numpy(), bits, C, D, "COS", hv_bits)


def test_infer_rp_argument_errors(hd, h):
    X, P, C = (torch.zeros((4, 8), device="cuda"), torch.zeros((64, 8), device="cuda"), torch.zeros((3, 64), device="cuda"))
    with pytest.raises(hd.HdcError) as e:
        h.hdc_infer_rp(X, P, C, hd.knobs(65))
    assert e.value.code == hd.HDC_ERR_INVALID_ARG
    with pytest.raises(hd.HdcError) as e:
        h.hdc_infer_rp(X, P, C, hd.knobs(64, hv_bits=8, sim=hd.HDC_SIM_HAMMING))
    assert e.value.code == hd.HDC_ERR_INVALID_ARG
    assert h.stat(99) == -1


def test_infer_rp_bench_launch_configuration_sampled(hd, h):
    """The headline shape through the fused kernel: ONE hdc_infer_rp over 131072 tiled C2 queries (fp32-precision
    encode on CTA pairs, K = 26 fp32 classes searched in the epilogue, cosine), with and without the hypervector
    output, and the host entry point in its chunks.  The oracle checks the first 1559 rows; the rest must repeat with that period
    (row i is a copy of row i mod 1559) wherever the row sits in a tile, a CTA pair or a chunk."""
    w = gen.c2_isolet_shaped()
    D, K, F = w["D"], w["K"], w["F"]
    NQ, n_te = 131072, w["Xte"].shape[0]
    Xq = gen.tile_rows(w["Xte"], NQ)
    Pd = dev(w["P"])
    kn = hd.knobs(D, precision=hd.HDC_F32, hv_bits=32, sim=hd.HDC_SIM_COS, flags=hd.HDC_FLAG_FUSED_INFER)
    btr_or, _, _ = O.encode_rp(w["Xtr"][:2048], w["P"], D, O.F32)
    C_or = O.bundle(btr_or, w["ytr"][:2048], K, D)
    C_or, _, _ = O.train_epoch(btr_or, w["ytr"][:2048], C_or, D, 32, O.SIM_COS, 0.05, 0)
    Cd = dev(C_or)
    H = h.alloc_hbits(NQ, D)
    f0 = h.stat(hd.HDC_STAT_INFER_FUSED)
    lab, best, second = h.hdc_infer_rp(dev(Xq), Pd, Cd, kn, want_scores=True, Hbits=H)
    torch.cuda.synchronize()
    assert h.stat(hd.HDC_STAT_INFER_FUSED) == f0 + 1
    bte_or, acc_te, ab_te = O.encode_rp(w["Xte"], w["P"], D, O.F32, want_absum=True)
    bits = host_bits(H[:n_te], D)
    check_sign_band(bits, bte_or, acc_te, ab_te, F)
    Hw = H.cpu().numpy()
    idx = np.arange(NQ)
    assert np.array_equal(Hw, Hw[idx % n_te])
    lab_h, best_h, second_h = lab.cpu().numpy(), best.cpu().numpy(), second.cpu().numpy()
    _check_stage2(hd, lab_h[:n_te], best_h[:n_te], second_h[:n_te], bits, C_or, D, "COS", 32)
    assert np.array_equal(lab_h, lab_h[idx % n_te]) and np.array_equal(best_h, best_h[idx % n_te])
    lab2 = h.hdc_infer_rp(dev(Xq), Pd, Cd, kn)                               # no hypervector output
    assert torch.equal(lab2, lab)
    Xh = torch.from_numpy(Xq).pin_memory()
    # the host pipeline: its small ramp-up chunks take the two-kernel path, the later ones the fused kernel, so
    # it answers to the oracle by the same rule (scores summed in another order), and repeats with the period
    lab_host = h.hdc_infer_rp_host(Xh, Pd, Cd, kn).numpy()
    check_labels_float(lab_host[:n_te], O.similarity(bits, C_or, D, O.SIM_COS, 32), O.SIM_COS)
    assert np.array_equal(lab_host, lab_host[idx % n_te]) or (lab_host != lab_h).mean() < 1e-3
    assert (lab_host != lab_h).mean() < 1e-3
