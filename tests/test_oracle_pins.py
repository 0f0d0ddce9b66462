"""Pins for the CPU oracle (`oracle/hdc_oracle.py`) against things other than itself:
brute-force python loops on tiny inputs, closed forms, invariants, library routines
(ml_dtypes bfloat16), and the one value the paper prints (tests/golden/).  CPU only."""
import math
import os

import ml_dtypes
import numpy as np
import pytest

import workloads as wl
from oracle import hdc_oracle as o

HERE = os.path.dirname(os.path.abspath(__file__))
rng = lambda s: np.random.default_rng(s)      # noqa: E731


# ------------------------------------------------------------------ S0 layout
def test_pack_layout_by_hand():
    bits = np.zeros((1, 70), dtype=np.uint8)
    bits[0, [0, 5, 31, 33, 69]] = 1
    w = o.pack_bits(bits)
    assert w.shape == (1, 3)
    assert int(w[0, 0]) == (1 << 0) | (1 << 5) | (1 << 31)
    assert int(w[0, 1]) == (1 << 1)
    assert int(w[0, 2]) == (1 << 5)           # bit 69 = word 2, bit 5; bits 70..95 zero
    assert np.array_equal(o.unpack_bits(w, 70), bits)
    # the generator's packer (a separate implementation) uses the same layout
    assert np.array_equal(wl.pack_bits_lsb(bits), w)


@pytest.mark.parametrize("D", [1, 31, 32, 33, 64, 100, 313 * 32 - 16])
def test_pack_roundtrip(D):
    b = rng(D).integers(0, 2, size=(5, D), dtype=np.uint8)
    w = o.pack_bits(b)
    assert w.shape[1] == (D + 31) // 32
    assert np.array_equal(o.unpack_bits(w, D), b)
    if D % 32:
        assert (w[:, -1] >> (D % 32) == 0).all()          # tail bits zero


# ------------------------------------------------------------------ S1 precision conversions
def test_bf16_rne_against_ml_dtypes():
    r = rng(1)
    x = np.concatenate([r.standard_normal(20000) * 10.0 ** r.integers(-20, 20, 20000),
                        [0.0, -0.0, 1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0 + 2.0 ** -7,
                         -(1.0 + 2.0 ** -8), 3.3895314e38 * 0.5, 1e-40]]).astype(np.float32)
    want = x.astype(ml_dtypes.bfloat16).astype(np.float32)
    got = o.round_bf16(x)
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
    # ties to even, by hand: 1+2^-8 is halfway between 1 and 1+2^-7 -> 1 (even mantissa)
    assert o.round_bf16(np.float32(1.0 + 2.0 ** -8)) == np.float32(1.0)
    assert o.round_bf16(np.float32(1.0 + 3 * 2.0 ** -8)) == np.float32(1.0 + 2.0 ** -6)


def test_int8_rows_fixed_points():
    q = np.array([[127, -127, 0, 5, -64], [0, 0, 0, 0, 0], [1, 2, 127, -3, 4]], dtype=np.float32)
    assert np.array_equal(o.quantize_int8_rows(q), q.astype(np.int32))   # max 127 -> identity
    x = np.array([[0.5, -1.0, 0.25, 1.0 / 127]], dtype=np.float32)
    assert np.array_equal(o.quantize_int8_rows(x), [[64, -127, 32, 1]])  # 63.5 -> 64 (RNE), 31.75 -> 32
    assert np.abs(o.quantize_int8_rows(rng(2).standard_normal((7, 33)).astype(np.float32))).max() == 127
    # per-tensor variant: the single max maps to 127
    c = rng(3).standard_normal((4, 9)).astype(np.float32)
    qt = o.quantize_int8_tensor(c)
    assert np.abs(qt).max() == 127 and (np.abs(qt) == 127).sum() == 1
    assert np.array_equal(o.quantize_int8_tensor(np.zeros((2, 3), np.float32)), np.zeros((2, 3)))


# ------------------------------------------------------------------ S1 random projection
def _brute_encode(X, P, D_eff):
    N, F = X.shape
    out = np.zeros((N, D_eff), dtype=np.uint8)
    for n in range(N):
        for d in range(D_eff):
            s = 0.0
            for f in range(F):
                s += float(X[n, f]) * float(P[d, f])
            out[n, d] = 1 if s < 0 else 0
    return out


@pytest.mark.parametrize("N,F,D,D_eff", [(3, 5, 40, 40), (8, 16, 64, 33), (2, 1, 7, 7), (4, 17, 130, 31)])
def test_encode_rp_brute_force(N, F, D, D_eff):
    r = rng(N * 1000 + F)
    X = r.standard_normal((N, F)).astype(np.float32)
    P = r.standard_normal((D, F)).astype(np.float32)
    bits, acc, absum = o.encode_rp(X, P, D_eff, o.F32, want_absum=True)
    assert bits.shape == (N, D_eff)
    assert np.array_equal(bits, _brute_encode(X, P, D_eff))
    assert (absum >= np.abs(acc) - 1e-12).all()


def test_encode_rp_transposed_operand_would_fail():
    # P is [D][F] (Listing 1: hypermatrix<2048,617>): row d is projection d.
    X = np.array([[1.0, 0.0]], dtype=np.float32)
    P = np.array([[1.0, -5.0], [-1.0, 5.0], [-2.0, 1.0]], dtype=np.float32)     # D=3, F=2
    bits, acc, _ = o.encode_rp(X, P, 3)
    assert np.array_equal(acc, [[1.0, -1.0, -2.0]])
    assert np.array_equal(bits, [[0, 1, 1]])


def test_encode_rp_f1_scale_invariance_and_sign_zero():
    r = rng(7)
    X = r.standard_normal((6, 1)).astype(np.float32)
    P = r.standard_normal((50, 1)).astype(np.float32)
    bits, _, _ = o.encode_rp(X, P, 50)
    assert np.array_equal(bits, ((X * P.T) < 0).astype(np.uint8))               # F=1: sgn(x*p)
    X = r.standard_normal((5, 9)).astype(np.float32)
    P = r.standard_normal((64, 9)).astype(np.float32)
    b1, _, _ = o.encode_rp(X, P, 64)
    b2, _, _ = o.encode_rp(np.float32(8.0) * X, P, 64)                          # alpha > 0 (exact *8)
    assert np.array_equal(b1, b2)
    # sgn(0) = +1 -> bit 0 (A1); sgn(-0.0) too
    Xz = np.array([[1.0, 1.0], [0.0, -0.0]], dtype=np.float32)
    Pz = np.array([[1.0, -1.0], [1.0, 1.0], [-1.0, -1.0]], dtype=np.float32)
    bz, az, _ = o.encode_rp(Xz, Pz, 3)
    assert np.array_equal(az[0], [0.0, 2.0, -2.0]) and np.array_equal(bz, [[0, 0, 1], [0, 0, 0]])


def test_encode_rp_integer_inputs_exact_all_precisions():
    r = rng(11)
    X = r.integers(0, 128, size=(9, 23)).astype(np.float32)
    X[:, 0] = 127                                           # row max 127 -> int8 quantisation is identity
    P = (1 - 2 * r.integers(0, 2, size=(77, 23))).astype(np.float32) * 127
    want = (X.astype(np.int64) @ P.astype(np.int64).T)
    for prec in (o.F32, o.I8):
        bits, acc, _ = o.encode_rp(X, P, 77, prec)
        assert np.array_equal(acc, want) and np.array_equal(bits, (want < 0))
    Xs = r.integers(0, 256, size=(9, 23)).astype(np.float32)        # 8-bit ints are exact in bf16
    Ps = (1 - 2 * r.integers(0, 2, size=(77, 23))).astype(np.float32)
    wants = Xs.astype(np.int64) @ Ps.astype(np.int64).T
    for prec in (o.F32, o.BF16, o.B1):
        bits, acc, _ = o.encode_rp(Xs, Ps, 77, prec)
        assert np.array_equal(acc, wants) and np.array_equal(bits, (wants < 0))


def test_encode_rp_angle_closed_form():
    """Gaussian P: P(sign bit differs) = theta(x,y)/pi per dimension (random hyperplane)."""
    D, F = 20000, 24
    r = rng(13)
    P = r.standard_normal((D, F)).astype(np.float32)
    x = r.standard_normal(F)
    for theta in (0.2, 1.0, math.pi / 2, 2.5):
        u = r.standard_normal(F)
        u -= (u @ x) / (x @ x) * x
        yv = math.cos(theta) * x / np.linalg.norm(x) + math.sin(theta) * u / np.linalg.norm(u)
        bits, _, _ = o.encode_rp(np.stack([x, 3.0 * yv]).astype(np.float32), P, D)
        frac = (bits[0] != bits[1]).mean()
        p = theta / math.pi
        assert abs(frac - p) <= 4.0 * math.sqrt(p * (1 - p) / D), (theta, frac, p)


def test_near_orthogonality_of_random_hypervectors():
    D = 10000
    bits = rng(17).integers(0, 2, size=(40, D), dtype=np.uint8)
    S = o.cosine(bits, o.bipolar(bits), D)
    off = S[~np.eye(40, dtype=bool)]
    assert np.allclose(np.diag(S), 1.0) and np.abs(off).max() < 4.5 / math.sqrt(D)
    assert np.sqrt((off ** 2).mean()) < 1.3 / math.sqrt(D)      # sd of cos is 1/sqrt(D)
    # encoded independent inputs are near-orthogonal too (north_star: |cos| <~ 3/sqrt(D))
    r = rng(18)
    hb, _, _ = o.encode_rp(r.standard_normal((12, 300)).astype(np.float32),
                           r.standard_normal((D, 300)).astype(np.float32), D)
    Sx = o.cosine(hb, o.bipolar(hb), D)
    assert np.abs(Sx[~np.eye(12, dtype=bool)]).max() < 0.25    # inputs in R^300 are ~1/sqrt(300) apart


# ------------------------------------------------------------------ S6 similarity
@pytest.mark.parametrize("D_eff", [1, 31, 32, 33, 64, 100, 257])
def test_bipolar_identity_dot_equals_D_minus_2_hamming(D_eff):
    r = rng(D_eff)
    h = r.integers(0, 2, size=(6, 257), dtype=np.uint8)
    c = r.integers(0, 2, size=(5, 257), dtype=np.uint8)
    ham = o.hamming(h, c, D_eff)
    dt = o.dot(h, o.bipolar(c), D_eff)
    assert np.array_equal(dt, D_eff - 2 * ham)
    # brute force Hamming
    for n in range(6):
        for k in range(5):
            assert ham[n, k] == sum(int(h[n, d] != c[k, d]) for d in range(D_eff))


def test_cosine_against_textbook_formula_and_zero_norm():
    r = rng(23)
    h = r.integers(0, 2, size=(7, 90), dtype=np.uint8)
    C = r.standard_normal((4, 90)).astype(np.float32)
    C[2] = 0.0
    S = o.cosine(h, C, 64)
    v = 1.0 - 2.0 * h[:, :64].astype(np.float64)
    for n in range(7):
        for k in range(4):
            c = C[k, :64].astype(np.float64)
            want = 0.0 if k == 2 else float(v[n] @ c) / (np.linalg.norm(v[n]) * np.linalg.norm(c))
            assert abs(S[n, k] - want) < 1e-14
    assert np.allclose(o.cosine(h, o.bipolar(h), 90).diagonal(), 1.0)
    assert np.allclose(o.cosine(h, -o.bipolar(h), 90).diagonal(), -1.0)


def test_similarity_precisions_of_class_operand():
    r = rng(29)
    h = r.integers(0, 2, size=(5, 70), dtype=np.uint8)
    C = (r.standard_normal((3, 70)) * 7).astype(np.float32)
    v = o.bipolar(h)
    assert np.allclose(o.similarity(h, C, 70, o.SIM_DOT, 32), v @ C.astype(np.float64).T)
    cb = C.astype(ml_dtypes.bfloat16).astype(np.float64)
    assert np.array_equal(o.similarity(h, C, 70, o.SIM_DOT, 16), v @ cb.T)
    q = o.similarity(h, C, 70, o.SIM_DOT, 8)
    assert np.array_equal(q, np.rint(q)) and np.abs(q).max() <= 127 * 70
    # per-tensor scale over the D_eff prefix only (S5): the max inside the prefix maps to 127
    C2 = C.copy(); C2[0, 69] = 1e6
    assert np.abs(o.class_operand(C2, 64, 8)).max() == 127
    # hv_bits=1: sign bits; Hamming and bipolar dot agree through the identity
    ham = o.similarity(h, C, 70, o.SIM_HAMMING, 1)
    assert np.array_equal(o.similarity(h, C, 70, o.SIM_DOT, 1), 70 - 2 * ham)
    Cz = C.copy(); Cz[1, 3] = 0.0
    assert o.class_operand(Cz, 70, 1)[1, 3] == 0                 # sgn(0)=+1 -> bit 0


# ------------------------------------------------------------------ S7 classify
def test_classify_ties_and_runner_up():
    S = np.array([[1.0, 3.0, 3.0, 2.0], [5.0, 1.0, 0.0, 5.0], [-1.0, -2.0, -3.0, -4.0]])
    lab, best, second = o.classify(S, o.SIM_COS)
    assert lab.tolist() == [1, 0, 0] and best.tolist() == [3.0, 5.0, -1.0]
    assert second.tolist() == [3.0, 5.0, -2.0]
    Hd = np.array([[7, 2, 2, 9], [4, 4, 4, 4]])
    lab, best, second = o.classify(Hd, o.SIM_HAMMING)
    assert lab.tolist() == [1, 0] and best.tolist() == [2, 4] and second.tolist() == [2, 4]
    lab, best, second = o.classify(np.array([[0.25], [-3.0]]), o.SIM_DOT)          # K = 1
    assert lab.tolist() == [0, 0] and second.tolist() == best.tolist()


# ------------------------------------------------------------------ S2 level-ID
def _brute_levelid(levels, ID, LV, D_eff):
    N, F = levels.shape
    out = np.zeros((N, D_eff), dtype=np.uint8)
    for n in range(N):
        for d in range(D_eff):
            cnt = 0
            for f in range(F):
                cnt += int(ID[f, d]) ^ int(LV[levels[n, f], d])
            out[n, d] = 1 if 2 * cnt > F else 0
    return out


@pytest.mark.parametrize("N,F,Q,D,D_eff", [(3, 7, 5, 40, 40), (4, 8, 4, 70, 33), (2, 1, 3, 35, 35), (5, 3, 2, 64, 64)])
def test_levelid_brute_force(N, F, Q, D, D_eff):
    r = rng(N + 10 * F + 100 * Q)
    lv = r.integers(0, Q, size=(N, F)).astype(np.uint8)
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = r.integers(0, 2, size=(Q, D), dtype=np.uint8)
    got = o.encode_levelid(lv, ID, LV, D_eff)
    assert np.array_equal(got, _brute_levelid(lv, ID, LV, D_eff))
    if F == 1:
        assert np.array_equal(got, (ID[0] ^ LV[lv[:, 0]])[:, :D_eff])
    if F == 3:
        a, b, c = (ID[f] ^ LV[lv[:, f]] for f in range(3))
        assert np.array_equal(got, ((a & b) | (a & c) | (b & c))[:, :D_eff])      # bitwise majority


def test_levelid_even_F_tie_gives_bit0():
    ID = np.array([[0, 1], [1, 1]], dtype=np.uint8)         # F=2, D=2
    LV = np.array([[0, 0]], dtype=np.uint8)
    got = o.encode_levelid(np.zeros((1, 2), np.uint8), ID, LV, 2)
    assert got.tolist() == [[0, 1]]                          # d=0: cnt 1 of 2 -> tie -> 0; d=1: 2 of 2 -> 1


@pytest.mark.parametrize("F", [9, 101])
def test_majority_bundling_recovers_components_above_chance(F):
    """For odd F and iid bound vectors, P(maj_d == component_f,d) = 1/2 + C(F-1,(F-1)/2)/2^F."""
    D = 20000
    r = rng(F)
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = r.integers(0, 2, size=(8, D), dtype=np.uint8)
    lv = r.integers(0, 8, size=(6, F)).astype(np.uint8)
    hb = o.encode_levelid(lv, ID, LV, D)
    p = 0.5 + math.comb(F - 1, (F - 1) // 2) / 2.0 ** F
    agree = np.mean([(hb[n] == (ID[f] ^ LV[lv[n, f]])).mean() for n in range(6) for f in range(F)])
    sd = math.sqrt(p * (1 - p) / (D * 6 * F))
    assert abs(agree - p) < 6 * sd + 1e-4, (agree, p)
    assert {9: 0.6367, 101: 0.5398}[F] == round(p, 4)


def test_level_table_hamming_closed_form():
    Q, D = 17, 1000
    LV = wl.level_table(99, Q, D)
    m = [(q * (D // 2)) // (Q - 1) for q in range(Q)]
    for a in range(Q):
        for b in range(Q):
            assert int((LV[a] != LV[b]).sum()) == abs(m[a] - m[b])
    assert int((LV[0] != LV[Q - 1]).sum()) == D // 2


# ------------------------------------------------------------------ S3 D_eff
def test_listing1_first_1024_of_2048_golden():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "listing1_redperf.txt"))
            if l.strip() and not l.startswith("#")]
    D, start, end, stride, D_eff, first, last = rows[0]
    D, D_eff = int(D), int(D_eff)
    assert int(math.floor(float(end) * D)) == D_eff and float(start) == 0.0 and int(stride) == 1
    # Listing 1 shapes: F=617, D=2048, K=26
    r = rng(2048)
    h = r.integers(0, 2, size=(3, D), dtype=np.uint8)
    c = r.integers(0, 2, size=(26, D), dtype=np.uint8)
    want = (h[:, None, int(first):int(last) + 1] != c[None, :, int(first):int(last) + 1]).sum(axis=2)
    assert np.array_equal(o.hamming(h, c, D_eff), want)


@pytest.mark.parametrize("D_eff", [1, 31, 32, 33, 100, 200])
def test_d_eff_slice_equivalence(D_eff):
    r = rng(300 + D_eff)
    D, F, K, N = 200, 11, 4, 24
    X = r.standard_normal((N, F)).astype(np.float32)
    P = r.standard_normal((D, F)).astype(np.float32)
    y = r.integers(0, K, size=N)
    for prec, hvb, sim in ((o.F32, 32, o.SIM_COS), (o.BF16, 16, o.SIM_DOT), (o.I8, 8, o.SIM_COS), (o.B1, 1, o.SIM_HAMMING)):
        hb_full, _, _ = o.encode_rp(X, P, D, prec)
        hb, _, _ = o.encode_rp(X, P, D_eff, prec)
        hb_sl, _, _ = o.encode_rp(X, P[:D_eff], D_eff, prec)
        assert np.array_equal(hb, hb_sl) and np.array_equal(hb, hb_full[:, :D_eff])
        C_full = o.bundle(hb_full, y, K, D)
        C = o.bundle(hb_full, y, K, D_eff)
        assert np.array_equal(C, C_full[:, :D_eff])
        S = o.similarity(hb_full, C_full, D_eff, sim, hvb)
        S_sl = o.similarity(hb_full[:, :D_eff].copy(), C_full[:, :D_eff].copy(), D_eff, sim, hvb)
        assert np.array_equal(S, S_sl)
        C1, w1, p1 = o.train_epoch(hb_full, y, C_full, D_eff, hvb, sim, 0.25, 5)
        C2, w2, p2 = o.train_epoch(hb_sl, y, C_full[:, :D_eff].copy(), D_eff, hvb, sim, 0.25, 5)
        assert np.array_equal(C1, C2) and w1 == w2 and np.array_equal(p1, p2)


# ------------------------------------------------------------------ S8 bundle
def test_bundle_sums_and_counts():
    r = rng(41)
    hb = r.integers(0, 2, size=(50, 77), dtype=np.uint8)
    y = r.integers(0, 5, size=50)
    C = o.bundle(hb, y, 5, 77)
    assert C.dtype == np.float32
    v = 1 - 2 * hb.astype(np.int64)
    assert np.array_equal(C.sum(axis=0), v.sum(axis=0))
    for k in range(5):
        want = np.zeros(77, dtype=np.int64)
        for n in range(50):
            if y[n] == k:
                want += v[n]
        assert np.array_equal(C[k], want)
        assert np.abs(C[k]).max() <= (y == k).sum()
    C2 = o.bundle(hb, y, 5, 77, C_acc=C)
    assert np.array_equal(C2, 2 * C)


# ------------------------------------------------------------------ S9 retraining
def _textbook_online_perceptron(hb, y, C, lr):
    """Separate 10-line statement of the B=1 rule: on a mistake add lr*h to the true class and
    subtract it from the predicted one (dot similarity, fp32 class vectors)."""
    C = C.astype(np.float32).copy()
    wrong = 0
    for n in range(hb.shape[0]):
        h = (1.0 - 2.0 * hb[n]).astype(np.float32)
        scores = [float(np.dot(h.astype(np.float64), C[k].astype(np.float64))) for k in range(C.shape[0])]
        yh = int(np.argmax(scores))
        if yh != y[n]:
            wrong += 1
            C[y[n]] = C[y[n]] + np.float32(lr) * h
            C[yh] = C[yh] - np.float32(lr) * h
    return C, wrong


def test_train_epoch_b1_is_online_perceptron():
    r = rng(43)
    hb = r.integers(0, 2, size=(60, 96), dtype=np.uint8)
    y = r.integers(0, 4, size=60)
    C0 = o.bundle(hb[:8], y[:8], 4, 96)
    for lr in (1.0, 0.05):
        C1, w1, _ = o.train_epoch(hb, y, C0, 96, 32, o.SIM_DOT, lr, batch=1)
        C2, w2 = _textbook_online_perceptron(hb, y, C0, lr)
        assert w1 == w2 and w1 > 0 and np.array_equal(C1, C2)


@pytest.mark.parametrize("B", [0, 1, 7, 64])
def test_train_epoch_invariants(B):
    r = rng(47 + B)
    hb = r.integers(0, 2, size=(90, 130), dtype=np.uint8)
    y = r.integers(0, 5, size=90)
    C = o.bundle(hb, y, 5, 130)
    col = C.astype(np.float64).sum(axis=0)
    for _ in range(3):                                   # sum_k Delta[k,d] = 0: column sums conserved (lr = 2^-2 exact)
        C, wrong, pred = o.train_epoch(hb, y, C, 130, 32, o.SIM_COS, 0.25, B)
        assert np.array_equal(C.astype(np.float64).sum(axis=0), col)
        assert 0 <= wrong <= 90 and pred.shape == (90,)
    if B == 0:                                           # epoch-synchronous: mistakes counted against the epoch-start model
        assert wrong == int((pred != y).sum())


def test_train_separable_converges_and_fixed_point():
    r = rng(53)
    K, D, per = 3, 512, 20
    protos = r.integers(0, 2, size=(K, D), dtype=np.uint8)
    y = np.repeat(np.arange(K), per)
    hb = protos[y] ^ (r.random((K * per, D)) < 0.15).astype(np.uint8)
    C = o.bundle(hb[::7], y[::7], K, D)
    hist = []
    for _ in range(6):
        C, wrong, _ = o.train_epoch(hb, y, C, D, 32, o.SIM_COS, 1.0, 0)
        hist.append(wrong)
    assert hist[-1] == 0 and hist[-2] == 0
    C2, wrong, _ = o.train_epoch(hb, y, C, D, 32, o.SIM_COS, 1.0, 0)
    assert wrong == 0 and np.array_equal(C2, C)           # zero mispredicts => unchanged


def test_train_update_two_rounded_fp32_ops():
    # one sample, one mistake: C_acc' = fl32(C + fl32(lr*delta)); check against python floats
    hb = np.array([[0, 1, 0]], dtype=np.uint8)
    C = np.array([[0.1, 0.2, 0.3], [5.0, -5.0, 5.0]], dtype=np.float32)   # class 1 wins: h=(+1,-1,+1)
    Cn, wrong, pred = o.train_epoch(hb, np.array([0]), C, 3, 32, o.SIM_DOT, 0.05, 0)
    assert wrong == 1 and pred.tolist() == [1]
    lr = np.float32(0.05)
    for d, v in enumerate([1.0, -1.0, 1.0]):
        assert Cn[0, d] == np.float32(C[0, d] + np.float32(lr * np.float32(v)))
        assert Cn[1, d] == np.float32(C[1, d] + np.float32(lr * np.float32(-v)))


# ------------------------------------------------------------------ S5 per-tensor int8, by hand
def test_int8_tensor_rounding_mode_and_scale_by_hand():
    """quantize_int8_tensor (S5 / A7; "projecting ... onto lower-precision integer
    types"): ONE scale for the whole array, s = fl32(127 / max|c|), q = rint-to-nearest-EVEN of
    fl32(c*s).  Worked by hand, non-unit scales, with halves of both parities so that truncation,
    round-half-up, round-half-away and a per-row scale each fail."""
    # max|c| = 2  ->  s = 63.5 (exact in fp32)
    #   2.0*63.5 = 127        -> 127
    #   1.0*63.5 = 63.5       -> 64   (tie, 64 is even; trunc gives 63)
    #   0.5*63.5 = 31.75      -> 32   (trunc gives 31)
    #  -0.75*63.5 = -47.625   -> -48  (trunc gives -47)
    #   0.0123*63.5 = 0.78..  -> 1    (trunc gives 0)
    c = np.array([[2.0, 1.0, 0.5, -0.75, 0.0123]], dtype=np.float32)
    assert o.quantize_int8_tensor(c).tolist() == [[127, 64, 32, -48, 1]]
    # max|c| = 254 -> s = 0.5 (exact): products are exact halves
    #   125*0.5 = 62.5 -> 62 (tie to EVEN; half-up and half-away give 63)
    #   127*0.5 = 63.5 -> 64 (tie to even; trunc gives 63)
    #  -125*0.5 = -62.5 -> -62 (half-away gives -63);  -127*0.5 = -63.5 -> -64
    #   -254*0.5 = -127 -> -127 (the negative extreme is -127, never -128);  1*0.5 = 0.5 -> 0;  3*0.5 = 1.5 -> 2
    c = np.array([[125.0, 127.0, -125.0, -127.0], [-254.0, 1.0, 3.0, 0.0]], dtype=np.float32)
    assert o.quantize_int8_tensor(c).tolist() == [[62, 64, -62, -64], [-127, 0, 2, 0]]
    # the scale is per TENSOR: the second row is quantised with the first row's maximum
    # (a per-row scheme would give [[127, 64], [127, 64]])
    c = np.array([[2.0, 1.0], [0.5, 0.25]], dtype=np.float32)
    assert o.quantize_int8_tensor(c).tolist() == [[127, 64], [32, 16]]         # 0.25*63.5 = 15.875 -> 16
    # the class operand at hv_bits = 8 takes the scale over d < D_eff only (S5): the large entry in the
    # truncated column must not change it
    C = np.array([[2.0, 1.0, 1000.0], [0.5, 0.25, -1000.0]], dtype=np.float32)
    assert o.class_operand(C, 2, 8).tolist() == [[127.0, 64.0], [32.0, 16.0]]
    # all-zero tensor: scale 1, codes 0
    assert o.quantize_int8_tensor(np.zeros((2, 3), dtype=np.float32)).tolist() == [[0, 0, 0], [0, 0, 0]]


# ------------------------------------------------------------------ S9 mini-batches 1 < B < N, brute force
def _py_round_half_even(x: float) -> int:
    return int(round(x))          # python's round() is round-half-to-even on floats


def _brute_minibatch_epoch(hb, y, C0, lr, B, hv_bits, sim, epoch_start_model=False, drop_partial=False):
    """S9 written out with python loops only, sharing nothing with the oracle: for every mini-batch
    [b0, b0+B) in index order -- including the shorter last one -- (i) re-derive the class operand from
    the CURRENT accumulators, (ii) predict each sample of the batch against it, (iii) integer Delta over the
    batch's mispredictions, (iv) C = fl32(C + fl32(lr*Delta)).  The two keyword switches build the MUTANTS
    the pin has to reject (every batch predicted from the epoch-start model; last partial batch dropped)."""
    N, D = hb.shape
    K = C0.shape[0]
    C = [[np.float32(C0[k, d]) for d in range(D)] for k in range(K)]
    Cstart = [row[:] for row in C]
    pred, wrong = [-1] * N, 0

    def operand(Cm):
        if hv_bits == 32:
            return [[float(v) for v in row] for row in Cm]
        amax = max(abs(float(v)) for row in Cm for v in row)
        s = np.float32(127.0) / np.float32(amax) if amax > 0 else np.float32(1.0)
        return [[float(max(-127, min(127, _py_round_half_even(float(np.float32(v * s)))))) for v in row] for row in Cm]

    for b0 in range(0, N, B):
        b1 = min(N, b0 + B)
        if drop_partial and b1 - b0 < B:
            break
        op = operand(Cstart if epoch_start_model else C)
        nrm = [math.sqrt(sum(c * c for c in op[k])) for k in range(K)]
        delta = [[0] * D for _ in range(K)]
        for n in range(b0, b1):
            v = [1 - 2 * int(hb[n, d]) for d in range(D)]
            sc = []
            for k in range(K):
                t = float(sum(v[d] * op[k][d] for d in range(D)))
                if sim == o.SIM_COS:
                    t = t / (math.sqrt(D) * nrm[k]) if nrm[k] > 0 else 0.0
                sc.append(t)
            yh = max(range(K), key=lambda k: (sc[k], -k))          # arg-max, ties -> lowest index
            pred[n] = yh
            if yh != int(y[n]):
                wrong += 1
                for d in range(D):
                    delta[int(y[n])][d] += v[d]
                    delta[yh][d] -= v[d]
        for k in range(K):
            for d in range(D):
                C[k][d] = np.float32(C[k][d] + np.float32(np.float32(lr) * np.float32(delta[k][d])))
    return np.array(C, dtype=np.float32), wrong, pred


@pytest.mark.parametrize("hv_bits,sim", [(32, o.SIM_DOT), (32, o.SIM_COS), (8, o.SIM_DOT)])
def test_train_epoch_minibatches_brute_force(hv_bits, sim):
    """1 < B < N with B not dividing N (N = 23, B = 5: batches of 5,5,5,5,3), K = 3, D = 40, two epochs,
    lr = 0.25 (a power of two: no score is decided by a rounding).  Pins S9 step (i) -- the operand is
    re-derived and the batch re-predicted from the CURRENT accumulators -- and the ragged last batch."""
    r = rng(61)
    N, B, K, D = 23, 5, 3, 40
    protos = r.integers(0, 2, size=(K, D), dtype=np.uint8)
    y = r.integers(0, K, size=N)
    hb = protos[y] ^ (r.random((N, D)) < 0.35).astype(np.uint8)
    C = o.bundle(hb[:6], y[:6], K, D)                    # a weak start so that several batches hold mistakes
    Cm, Cd = C.copy(), C.copy()
    differs_start = differs_drop = False
    for _ in range(2):
        want_C, want_wrong, want_pred = _brute_minibatch_epoch(hb, y, C, 0.25, B, hv_bits, sim)
        got_C, got_wrong, got_pred = o.train_epoch(hb, y, C, D, hv_bits, sim, 0.25, B)
        assert np.array_equal(got_C, want_C) and got_wrong == want_wrong and got_pred.tolist() == want_pred
        assert want_wrong > 0
        # the two mutants, built from the same brute force, must be distinguishable on this data --
        # otherwise the equality above would not pin what it says it pins
        m_C, m_wrong, m_pred = _brute_minibatch_epoch(hb, y, C, 0.25, B, hv_bits, sim, epoch_start_model=True)
        differs_start |= (not np.array_equal(m_C, want_C)) or m_pred != want_pred
        d_C, d_wrong, d_pred = _brute_minibatch_epoch(hb, y, C, 0.25, B, hv_bits, sim, drop_partial=True)
        differs_drop |= (not np.array_equal(d_C, want_C)) or d_pred != want_pred
        C = got_C
    assert differs_start, "data does not separate per-batch re-prediction from the epoch-start model"
    assert differs_drop, "data does not exercise the ragged last mini-batch"


# ------------------------------------------------------------------ end-to-end sanity (not parity)
def test_pipeline_sanity_c1():
    c = wl.c1_tiny()
    hb, _, _ = o.encode_rp(c["Xtr"], c["P"], c["D"], o.F32)
    C = o.bundle(hb, c["ytr"], c["K"], c["D"])
    ht, _, _ = o.encode_rp(c["Xte"], c["P"], c["D"], o.F32)
    lab, best, second, S = o.infer(ht, C, c["D"], o.SIM_HAMMING, 1)
    assert (lab == c["yte"]).mean() > 0.9                   # far above 1/K = 0.25
    lab512, _, _, _ = o.infer(ht, C, 512, o.SIM_HAMMING, 1)
    assert (lab512 == c["yte"]).mean() > 0.8


def test_generators_are_seeded_and_shaped():
    a, b = wl.c2_isolet_shaped(D=64, n_tr=50, n_te=20), wl.c2_isolet_shaped(D=64, n_tr=50, n_te=20)
    assert a["Xtr"].shape == (50, 617) and a["P"].shape == (64, 617) and a["K"] == 26
    assert np.array_equal(a["Xtr"], b["Xtr"]) and np.array_equal(a["P"], b["P"])
    full = wl.c2_isolet_shaped(D=128, n_tr=50, n_te=20)
    assert np.array_equal(full["P"][:64], a["P"])            # prefix-stable in D (S3)
    c3 = wl.c3_mnist_shaped(D=256, n_tr=400, n_te=50)
    assert c3["Ltr"].dtype == np.uint8 and c3["Ltr"].shape == (400, 784)
    assert 0.70 < (c3["Ltr"] == 0).mean() < 0.90             # ~80 % zeros
    c5 = wl.c5_large_batch(64, D=128, K=10, n_unstructured=16, per_class=2)
    assert c5["X"].shape == (80, 1024) and c5["P"].shape == (128, 1024)
    assert np.array_equal(o.round_bf16(c5["X"]), c5["X"])     # bf16-representable
    assert abs(float(c5["X"][:64].std()) - 1.0) < 0.05


# ------------------------------------------------------------------------------------- S11 k-means
def _kmeans_brute(hb, C, D_eff, sim):
    """Plain python loops: assign by cosine (double) or Hamming to sign bits, re-bundle members."""
    N, K = hb.shape[0], C.shape[0]
    a = []
    for n in range(N):
        best, bi = None, 0
        for k in range(K):
            if sim == o.SIM_HAMMING:
                s = -sum(int(hb[n, d]) != int(C[k, d] < 0) for d in range(D_eff))
            else:
                dotv = sum((1 - 2 * int(hb[n, d])) * float(C[k, d]) for d in range(D_eff))
                nrm = sum(float(C[k, d]) ** 2 for d in range(D_eff)) ** 0.5
                s = dotv / (D_eff ** 0.5 * nrm) if nrm > 0 else 0.0
            if best is None or s > best:
                best, bi = s, k
        a.append(bi)
    Cn = np.array(C[:, :D_eff], dtype=np.float32)
    for k in range(K):
        mem = [n for n in range(N) if a[n] == k]
        if mem:
            Cn[k] = [sum(1 - 2 * int(hb[n, d]) for n in mem) for d in range(D_eff)]
    return Cn, np.array(a, dtype=np.int32)


@pytest.mark.parametrize("sim,hv_bits", [(o.SIM_COS, 32), (o.SIM_HAMMING, 1)])
@pytest.mark.parametrize("N,K,D,D_eff", [(9, 3, 40, 40), (12, 4, 70, 33), (5, 1, 16, 16)])
def test_kmeans_epoch_brute_force(sim, hv_bits, N, K, D, D_eff):
    r = np.random.default_rng(N * 100 + K)
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-5, 6, size=(K, D)).astype(np.float32)
    C[C == 0] = 1.0
    Cn, a, ch = o.kmeans_epoch(hb, C, D_eff, hv_bits, sim, prev=np.zeros(N, dtype=np.int32))
    Cb, ab = _kmeans_brute(hb, C, D_eff, sim)
    assert np.array_equal(a, ab)
    assert np.array_equal(Cn, Cb)
    assert ch == int((ab != 0).sum())


def test_kmeans_empty_cluster_keeps_its_accumulator_and_k1_is_the_bundle():
    r = np.random.default_rng(7)
    hb = r.integers(0, 2, size=(20, 64), dtype=np.uint8)
    c0 = 1.0 - 2.0 * hb[0].astype(np.float32)
    C = np.stack([c0, -c0])               # cluster 1 = the antipode of sample 0
    far = (hb ^ hb[0]).sum(axis=1) > 32  # samples closer to the antipode
    hb = hb[~far]
    Cn, a, _ = o.kmeans_epoch(hb, C, 64, 32, o.SIM_COS)
    assert (a == 0).all()
    assert np.array_equal(Cn[1], C[1])                                   # empty: unchanged
    assert np.array_equal(Cn[0], o.bundle(hb, np.zeros(len(hb), dtype=np.int64), 1, 64)[0])
    C1, a1, _ = o.kmeans_epoch(hb, C[:1], 64, 32, o.SIM_COS)           # K = 1 -> the bundle of everything
    assert (a1 == 0).all() and np.array_equal(C1[0], Cn[0])


def test_kmeans_spherical_objective_never_decreases_and_reaches_a_fixed_point():
    """With cosine similarity, (assign to the most similar centre, centre = sum of members) is
    spherical k-means: J = sum_n <v_n, c_hat_a(n)> is non-decreasing from one epoch to the next and
    the iteration stops at a fixed point (textbook property, independent of the oracle's code)."""
    r = np.random.default_rng(11)
    D, K, N = 512, 5, 300
    proto = r.integers(0, 2, size=(K, D), dtype=np.uint8)
    yt = r.integers(0, K, size=N)
    hb = proto[yt] ^ (r.random((N, D)) < 0.3).astype(np.uint8)
    C = (1.0 - 2.0 * hb[r.choice(N, K, replace=False)]).astype(np.float32)   # random samples as seeds
    v = 1.0 - 2.0 * hb.astype(np.float64)

    def J(Cc, a):
        ch = Cc.astype(np.float64)
        ch = ch / np.maximum(np.linalg.norm(ch, axis=1, keepdims=True), 1e-300)
        return float((v * ch[a]).sum())

    prev, hist = None, []
    for _ in range(30):
        C2, a, ch = o.kmeans_epoch(hb, C, D, 32, o.SIM_COS, prev)
        hist.append(J(C2, a))
        if prev is not None and ch == 0:
            assert np.array_equal(C2, C)                                 # fixed point
            break
        C, prev = C2, a
    else:
        raise AssertionError("k-means did not converge in 30 epochs")
    assert all(b >= a_ - 1e-9 for a_, b in zip(hist, hist[1:]))


def test_kmeans_recovers_well_separated_clusters():
    r = np.random.default_rng(12)
    D, K, N = 2048, 4, 200
    proto = r.integers(0, 2, size=(K, D), dtype=np.uint8)
    yt = np.arange(N) % K
    hb = proto[yt] ^ (r.random((N, D)) < 0.1).astype(np.uint8)
    for sim, bits in ((o.SIM_COS, 32), (o.SIM_HAMMING, 1)):
        C = (1.0 - 2.0 * hb[:K]).astype(np.float32)                      # one seed per true cluster
        C, a, _ = o.kmeans_epoch(hb, C, D, bits, sim)
        assert np.array_equal(a, yt)
        C2, a2, ch = o.kmeans_epoch(hb, C, D, bits, sim, prev=a)
        assert ch == 0 and np.array_equal(C2, C)


# ------------------------------------------------------------------------------------- A17 perforation
@pytest.mark.parametrize("begin,stride,D_eff", [(0, 1, 40), (0, 8, 40), (3, 8, 37), (5, 2, 33), (39, 7, 40), (1, 3, 32)])
def test_perforated_similarity_brute_force(begin, stride, D_eff):
    """Reduction perforation: loops over the visited dimensions written out by hand;
    dot = n_visited - 2 * Hamming on them; (0, 1) is the unperforated similarity."""
    r = np.random.default_rng(begin * 100 + stride)
    N, K, D = 6, 4, 40
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.integers(-9, 10, size=(K, D)).astype(np.float32)
    C[C == 0] = 2.0
    vis = [d for d in range(D_eff) if d >= begin and (d - begin) % stride == 0]
    assert list(o.perforated_index(D_eff, begin, stride)) == vis
    H = o.similarity(hb, C, D_eff, o.SIM_HAMMING, 1, begin, stride)
    Dt = o.similarity(hb, C, D_eff, o.SIM_DOT, 1, begin, stride)
    Dd = o.similarity(hb, C, D_eff, o.SIM_DOT, 32, begin, stride)
    Cs = o.similarity(hb, C, D_eff, o.SIM_COS, 32, begin, stride)
    for n in range(N):
        for k in range(K):
            ham = sum(int(hb[n, d]) != int(C[k, d] < 0) for d in vis)
            dt = sum((1 - 2 * int(hb[n, d])) * float(C[k, d]) for d in vis)
            nrm = math.sqrt(sum(float(C[k, d]) ** 2 for d in vis))
            assert H[n, k] == ham
            assert Dt[n, k] == len(vis) - 2 * ham
            assert Dd[n, k] == dt
            assert abs(Cs[n, k] - dt / (math.sqrt(len(vis)) * nrm)) < 1e-12
    if (begin, stride) == (0, 1):
        assert np.array_equal(H, o.similarity(hb, C, D_eff, o.SIM_HAMMING, 1))


def test_perforated_int8_scale_is_taken_over_the_visited_dimensions():
    hb = np.zeros((1, 8), dtype=np.uint8)
    C = np.array([[1000.0, 2.0, 3.0, 127.0, 5.0, 6.0, 7.0, 8.0]], dtype=np.float32)
    # visiting 1, 3, 5, 7: max |c| = 127 -> scale 1 -> the integers themselves
    S = o.similarity(hb, C, 8, o.SIM_DOT, 8, begin=1, stride=2)
    assert S[0, 0] == 2 + 127 + 6 + 8
    # unperforated: 1000 sets the scale and the small entries collapse
    assert o.similarity(hb, C, 8, o.SIM_DOT, 8)[0, 0] != S[0, 0]


def test_perforated_training_updates_every_dimension():
    """Only the similarity reduction is perforated (L155); the class update still touches d < D_eff."""
    w = wl.c1_tiny(D=256)
    hb, _, _ = o.encode_rp(w["Xtr"], w["P"], 256, o.F32)
    y = w["ytr"].copy()
    y[::3] = (y[::3] + 1) % w["K"]
    C0 = o.bundle(hb, y, w["K"], 256)
    C1, wrong, pred = o.train_epoch(hb, y, C0, 256, 1, o.SIM_HAMMING, 1.0, 0, begin=2, stride=4)
    lab, _, _ = o.classify(o.similarity(hb, C0, 256, o.SIM_HAMMING, 1, 2, 4), o.SIM_HAMMING)
    assert np.array_equal(pred, lab) and wrong == int((lab != y).sum()) and wrong > 0
    touched = np.nonzero((C1 != C0).any(axis=0))[0]
    assert (touched % 4 != 2).any()                      # columns outside the visited set changed too


# ------------------------------------------------------------------------------------- random shapes
from hypothesis import given, settings, strategies as st  # noqa: E402


@settings(max_examples=40, deadline=None)
@given(st.integers(1, 8), st.integers(1, 17), st.integers(1, 130), st.integers(0, 2 ** 31 - 1), st.data())
def test_encode_and_similarity_random_shapes_against_loops(N, F, D, seed, data):
    """Random small shapes (incl. D_eff = 1, 31, 32, 33 and tails): RP encode bits, Hamming, dot and the
    arg-extremum against plain python loops."""
    D_eff = data.draw(st.sampled_from(sorted({1, min(D, 31), min(D, 32), min(D, 33), D})))
    K = data.draw(st.integers(1, 5))
    r = np.random.default_rng(seed)
    X = r.integers(-3, 4, size=(N, F)).astype(np.float32)
    P = r.integers(-2, 3, size=(D, F)).astype(np.float32)
    bits, acc, _ = o.encode_rp(X, P, D_eff, o.F32)
    for n in range(N):
        for d in range(D_eff):
            a = sum(float(X[n, f]) * float(P[d, f]) for f in range(F))
            assert acc[n, d] == a and bits[n, d] == (1 if a < 0 else 0)
    C = r.integers(-4, 5, size=(K, D)).astype(np.float32)
    H = o.similarity(bits, C, D_eff, o.SIM_HAMMING, 1)
    Dt = o.similarity(bits, C, D_eff, o.SIM_DOT, 32)
    for n in range(N):
        for k in range(K):
            assert H[n, k] == sum(int(bits[n, d]) != int(C[k, d] < 0) for d in range(D_eff))
            assert Dt[n, k] == sum((1 - 2 * int(bits[n, d])) * float(C[k, d]) for d in range(D_eff))
    lab, best, _ = o.classify(H, o.SIM_HAMMING)
    for n in range(N):
        assert lab[n] == min(range(K), key=lambda k: (H[n, k], k)) and best[n] == H[n, lab[n]]
    lab2, _, _ = o.classify(Dt, o.SIM_DOT)
    for n in range(N):
        assert lab2[n] == min(range(K), key=lambda k: (-Dt[n, k], k))


@settings(max_examples=40, deadline=None)
@given(st.integers(1, 6), st.integers(1, 12), st.integers(1, 9), st.integers(1, 70), st.integers(0, 2 ** 31 - 1))
def test_levelid_random_shapes_against_loops(N, F, Q, D, seed):
    r = np.random.default_rng(seed)
    lv = r.integers(0, Q, size=(N, F)).astype(np.uint16)
    ID = r.integers(0, 2, size=(F, D), dtype=np.uint8)
    LV = r.integers(0, 2, size=(Q, D), dtype=np.uint8)
    D_eff = int(r.integers(1, D + 1))
    bits = o.encode_levelid(lv, ID, LV, D_eff)
    assert bits.shape == (N, D_eff)
    for n in range(N):
        for d in range(D_eff):
            cnt = sum(int(ID[f, d]) ^ int(LV[lv[n, f], d]) for f in range(F))
            assert bits[n, d] == (1 if 2 * cnt > F else 0)


# ------------------------------------------------------------------------------------- A18 encode perforation
@pytest.mark.parametrize("begin,stride,F", [(0, 2, 16), (1, 3, 17), (5, 4, 9), (0, 1, 7), (3, 8, 12)])
def test_perforated_encode_brute_force(begin, stride, F):
    """the reduction loop skips iterations at a stride and, for matrix-vector dot
    products, "the results are scaled appropriately to compensate for the skipped iterations"
    (reading A18: by F / F_visited).  Loops written out by hand, fp32 operands."""
    r = rng(181)
    N, D = 5, 11
    X = r.standard_normal((N, F)).astype(np.float32)
    P = r.standard_normal((D, F)).astype(np.float32)
    vis = [f for f in range(F) if f >= begin and (f - begin) % stride == 0]
    want = np.zeros((N, D))
    for n in range(N):
        for d in range(D):
            t = 0.0
            for f in vis:
                t += float(X[n, f]) * float(P[d, f])
            want[n, d] = t * F / len(vis)
    bits, acc, absum = o.encode_rp(X, P, D, o.F32, want_absum=True, f_begin=begin, f_stride=stride)
    assert np.allclose(acc, want, rtol=1e-12, atol=1e-12)
    assert np.array_equal(bits, (want < 0).astype(np.uint8))
    assert (absum >= np.abs(acc) - 1e-9).all()


def test_perforated_encode_of_a_constant_summand_is_exact():
    """The compensation is exact when every term of the reduction is the same: x = p = 1 gives
    acc = F at every stride and offset, also when the stride does not divide F."""
    F = 617
    X, P = np.ones((2, F), dtype=np.float32), np.ones((3, F), dtype=np.float32)
    for begin, stride in [(0, 2), (0, 8), (5, 7), (616, 3), (0, 617)]:
        _, acc, _ = o.encode_rp(X, P, 3, o.F32, f_begin=begin, f_stride=stride)
        assert np.allclose(acc, F, rtol=1e-14)
    # and an alternating summand +1, -1, ... at stride 2 sees only one sign: acc = +F or -F
    X[:, 1::2] = -1.0
    _, acc0, _ = o.encode_rp(X, P, 3, o.F32, f_begin=0, f_stride=2)
    _, acc1, _ = o.encode_rp(X, P, 3, o.F32, f_begin=1, f_stride=2)
    assert np.allclose(acc0, F) and np.allclose(acc1, -F)


def test_perforated_encode_int8_scales_come_from_the_visited_features():
    """Per-row int8 quantisation of a perforated contraction sees only the gathered columns: a large
    value in a skipped column must not change the codes of the visited ones."""
    X = np.array([[1.0, 1000.0, -2.0, 1000.0, 4.0, 1000.0]], dtype=np.float32)
    P = np.array([[1.0, 9.0, 1.0, 9.0, 1.0, 9.0], [1.0, 9.0, -1.0, 9.0, -1.0, 9.0]], dtype=np.float32)
    bits, acc, _ = o.encode_rp(X, P, 2, o.I8, f_begin=0, f_stride=2)
    # visited x = (1, -2, 4): scale 127/4 -> codes (32, -64, 127) (31.75 -> 32, -63.5 -> -64 ties to even);
    # p rows (1,1,1) and (1,-1,-1) -> (127,127,127) and (127,-127,-127)
    assert np.array_equal(acc, np.array([[(32 - 64 + 127) * 127 * 2.0, (32 + 64 - 127) * 127 * 2.0]]))
    assert bits.tolist() == [[0, 1]]
    # without perforation the 1000s set the scale: x codes (0, 127, 0, 127, 1, 127) (4 * 0.127 = 0.508 -> 1),
    # p row 0 codes (14, 127, 14, 127, 14, 127) (127/9 = 14.1)
    _, acc_full, _ = o.encode_rp(X, P, 2, o.I8)
    assert acc_full[0, 0] == 3 * 127 * 127 + 14


def test_unperforated_encode_arguments_change_nothing():
    r = rng(182)
    X = r.standard_normal((6, 13)).astype(np.float32)
    P = r.standard_normal((9, 13)).astype(np.float32)
    for prec in (o.F32, o.BF16, o.I8):
        a = o.encode_rp(X, P, 9, prec, want_absum=True)
        b = o.encode_rp(X, P, 9, prec, want_absum=True, f_begin=0, f_stride=1)
        assert all(np.array_equal(u, v) for u, v in zip(a, b))


# ------------------------------------------------------------------------------------- S12 / A19 ADC-quantised chunked dot
def test_adc_transfer_function_by_hand():
    """Reading A19 written out on small windows.  Baseline window (L273: floor -127, ceil 128, RES 8,
    step 1): 256 codes, transparent on [-127, 128], -128 clips to -127."""
    p = np.arange(-128, 129)
    q = o.adc_quantize(p, 8, 1, -127, 128)
    assert np.array_equal(q[1:], p[1:]) and q[0] == -127
    # the paper's best window: floor -3, ceil 128, RES 8, step 2 -> levels -3, -1, 1, 3, ...
    q = o.adc_quantize(np.array([-128, -4, -3, -2, -1, 0, 1, 2, 127, 128]), 8, 2, -3, 128)
    #  clip -> -3,-3,-3,-2,-1,0,1,2,127,128 ; (p+3+1)//2 -> 0,0,0,1,1,2,2,3,65,66 ; -3 + 2*code
    assert q.tolist() == [-3, -3, -3, -1, -1, 1, 1, 3, 127, 129]
    # RES limits the code: RES 2, step 9, floor -3 -> levels -3, 6, 15, 24 and nothing above
    q = o.adc_quantize(np.array([-10, 1, 2, 10, 11, 19, 20, 128]), 2, 9, -3, 128)
    assert q.tolist() == [-3, -3, 6, 6, 15, 15, 24, 24]
    # idempotent and monotone
    for res, step, fl, ce in [(8, 2, -3, 128), (6, 9, -3, 128), (4, 5, -20, 60), (8, 1, -127, 128)]:
        q = o.adc_quantize(p, res, step, fl, ce)
        assert (np.diff(q) >= 0).all()
        assert np.array_equal(o.adc_quantize(q, res, step, fl, max(ce, int(q.max()))), q)


@pytest.mark.parametrize("D_eff", [128, 256, 300, 127, 1, 129, 1000])
def test_adc_similarity_with_a_transparent_window_is_the_bipolar_dot(D_eff):
    """PAPER.md L273 baseline window is transparent unless a whole chunk is anti-aligned, so the chunked
    sum is the plain dot = D_eff - 2 * Hamming (S0/S6 identity) -- also with a ragged last chunk."""
    r = rng(190 + D_eff)
    hb = r.integers(0, 2, size=(9, 1024), dtype=np.uint8)
    C = r.standard_normal((5, 1024)).astype(np.float32)
    C[0, :40] = 0.0
    S = o.similarity_adc(hb, C, D_eff, 8, 1, -127, 128)
    ham = o.similarity(hb, C, D_eff, o.SIM_HAMMING, 1)
    assert np.array_equal(S, D_eff - 2 * ham.astype(np.int64))
    # an anti-aligned full chunk reads -127, not -128
    hb2 = np.zeros((1, 256), dtype=np.uint8)
    C2 = -np.ones((1, 256), dtype=np.float32)
    assert o.similarity_adc(hb2, C2, 256, 8, 1, -127, 128)[0, 0] == -254


@pytest.mark.parametrize("res,step,fl,ce", [(8, 2, -3, 128), (6, 9, -3, 128), (3, 7, -40, 90), (8, 1, -127, 128)])
def test_adc_similarity_brute_force(res, step, fl, ce):
    r = rng(195)
    N, K, D, D_eff, chunk = 4, 3, 400, 300, 128
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = r.standard_normal((K, D)).astype(np.float32)
    S = o.similarity_adc(hb, C, D_eff, res, step, fl, ce)
    for n in range(N):
        for k in range(K):
            total = 0
            for j0 in range(0, D_eff, chunk):
                part = 0
                for d in range(j0, min(j0 + chunk, D_eff)):
                    v = -1 if hb[n, d] else 1
                    c = -1 if C[k, d] < 0 else 1
                    part += v * c
                x = min(max(part, fl), ce)
                code = min((x - fl + step // 2) // step, 2 ** res - 1)
                total += fl + code * step
            assert S[n, k] == total


def test_adc_floor_clipping_keeps_the_label_of_a_separable_query():
    """L273: "Clipping below -3 therefore preserves the classification outcome": a query equal to one
    class hypervector keeps its label under the paper's tuned window."""
    r = rng(196)
    K, D = 6, 2048
    C = np.where(r.integers(0, 2, size=(K, D)) == 1, -1.0, 1.0).astype(np.float32)
    hb = (C < 0).astype(np.uint8)                      # query n == class n
    flip = r.random((K, D)) < 0.2
    hb ^= flip.astype(np.uint8)                         # 20 % noise
    for res, step in [(8, 2), (6, 9)]:
        lab, _, _ = o.classify(o.similarity_adc(hb, C, D, res, step, -3, 128), o.SIM_DOT)
        assert lab.tolist() == list(range(K))


# ------------------------------------------------------------------------------------- S5 fp16 class operand
def _half_rne_by_hand(x: float) -> float:
    """binary16 round-to-nearest-even from the definition (normal and subnormal range, no overflow)."""
    if x == 0.0:
        return 0.0
    s = -1.0 if x < 0 else 1.0
    a = abs(x)
    e = max(math.floor(math.log2(a)), -14)           # exponent of the binade; subnormals share 2^-14
    ulp = 2.0 ** (e - 10)
    q = a / ulp                                       # exact: power-of-two scaling
    f = math.floor(q)
    r = q - f
    if r > 0.5 or (r == 0.5 and f % 2 == 1):
        f += 1
    return s * f * ulp


def test_fp16_class_operand_rounding_by_hand():
    """hv code HV_F16 (PAPER.md L165 FP16): IEEE half RNE, checked against the definition on ties
    (2049 -> 2048, 2051 -> 2052), the largest finite value, subnormals and random values."""
    r = rng(200)
    vals = np.concatenate([np.array([0.0, 1.0, -1.0, 2049.0, 2051.0, -2049.0, 65504.0, 65519.0, 1.0 + 2.0 ** -11,
                                     1.0 + 3 * 2.0 ** -11, 6e-8, 3e-8, 2.0 ** -25, 1e-5, 0.1, 32.0, -33.3],
                                    dtype=np.float32),
                           (r.standard_normal(500) * r.choice([1e-3, 1.0, 40.0, 3000.0], size=500)).astype(np.float32)])
    got = o.class_operand(vals[None, :], len(vals), o.HV_F16)[0]
    want = np.array([_half_rne_by_hand(float(v)) for v in vals])
    assert np.array_equal(got, want)
    assert got[3] == 2048.0 and got[4] == 2052.0 and got[6] == 65504.0 and got[7] == 65504.0
    # exact integers up to 2048 are representable: a bundle of <= 2048 hypervectors is held exactly
    ints = np.arange(-2048, 2049, dtype=np.float32)
    assert np.array_equal(o.class_operand(ints[None, :], len(ints), o.HV_F16)[0], ints.astype(np.float64))


def test_fp16_similarity_equals_fp32_on_small_integer_accumulators():
    r = rng(201)
    hb = r.integers(0, 2, size=(7, 300), dtype=np.uint8)
    C = r.integers(-2048, 2049, size=(4, 300)).astype(np.float32)
    for sim in (o.SIM_DOT, o.SIM_COS):
        assert np.array_equal(o.similarity(hb, C, 300, sim, o.HV_F16), o.similarity(hb, C, 300, sim, 32))


def test_fp16_encode_operands_by_hand():
    """precision F16: both operands rounded to binary16 (definition written out in
    _half_rne_by_hand), then the plain contraction."""
    r = rng(202)
    X = (r.standard_normal((5, 9)) * 3).astype(np.float32)
    P = r.standard_normal((7, 9)).astype(np.float32)
    Xh = np.array([[_half_rne_by_hand(float(v)) for v in row] for row in X])
    Ph = np.array([[_half_rne_by_hand(float(v)) for v in row] for row in P])
    want = np.zeros((5, 7))
    for n in range(5):
        for d in range(7):
            want[n, d] = sum(Xh[n, f] * Ph[d, f] for f in range(9))
    bits, acc, _ = o.encode_rp(X, P, 7, o.F16)
    assert np.allclose(acc, want, rtol=1e-14, atol=1e-14)
    assert np.array_equal(bits, (want < 0).astype(np.uint8))
    # operands already representable in half: identical to fp32
    Xi = r.integers(0, 256, size=(4, 9)).astype(np.float32)
    Pi = (1.0 - 2.0 * r.integers(0, 2, size=(6, 9))).astype(np.float32)
    assert np.array_equal(o.encode_rp(Xi, Pi, 6, o.F16)[1], o.encode_rp(Xi, Pi, 6, o.F32)[1])


# ------------------------------------------------------------------ S5 per-tensor int16 (A21), by hand
def test_int16_tensor_rounding_mode_and_scale_by_hand():
    """quantize_int16_tensor ("integer data types (8, 16, 32, or 64-bit)"; reading A21 = A7 at
    16 bits): ONE scale s = fl32(32767 / max|c|) for the array, q = rint-to-nearest-EVEN of fl32(c*s), codes in
    [-32767, 32767].  Worked by hand so that truncation, half-up, half-away, a per-row scale and a 32768 full
    scale each fail."""
    # max|c| = 16383.5 -> s = 2 (exact): products are exact
    #   16383.5*2 = 32767; 0.25*2 = 0.5 -> 0 (tie to even; half-up gives 1); 0.75*2 = 1.5 -> 2 (trunc gives 1)
    #   1.25*2 = 2.5 -> 2 (tie to even; half-up / half-away give 3; a 32768 full scale gives 2.50004 -> 3)
    #   -1.25*2 = -2.5 -> -2; 100.3*2 = 200.6 -> 201; -16383.5 -> -32767 (never -32768)
    c = np.array([[16383.5, 0.25, 0.75, 1.25], [-1.25, 100.3, -16383.5, 0.0]], dtype=np.float32)
    assert o.quantize_int16_tensor(c).tolist() == [[32767, 0, 2, 2], [-2, 201, -32767, 0]]
    # max|c| = 2 -> s = 16383.5 (exact in fp32)
    #   1.0*s = 16383.5 -> 16384 (tie, even); 0.5*s = 8191.75 -> 8192; -0.75*s = -12287.625 -> -12288
    #   second row uses the SAME scale (per tensor): 0.25*s = 4095.875 -> 4096; a per-row scale would give 32767
    c = np.array([[2.0, 1.0, 0.5, -0.75], [0.25, 0.0, 0.0, 0.0]], dtype=np.float32)
    assert o.quantize_int16_tensor(c).tolist() == [[32767, 16384, 8192, -12288], [4096, 0, 0, 0]]
    # the class operand takes the scale over d < D_eff only (S5)
    C = np.array([[2.0, 1.0, 1000.0], [0.5, 0.25, -1000.0]], dtype=np.float32)
    assert o.class_operand(C, 2, o.HV_I16).tolist() == [[32767.0, 16384.0], [8192.0, 4096.0]]
    assert o.quantize_int16_tensor(np.zeros((2, 3), dtype=np.float32)).tolist() == [[0, 0, 0], [0, 0, 0]]


def test_int16_similarity_brute_force_and_small_integer_identity():
    """hv code HV_I16 through similarity(): DOT = python-integer sum of v*q over d < D_eff, COS = DOT /
    (sqrt(D_eff) * |q|) with the norm of the CODES; integer accumulators whose max is 32767/2^j are held
    exactly up to the power-of-two scale (labels and cosines of hv_bits = 32 are reproduced)."""
    r = rng(210)
    N, K, D, D_eff = 6, 4, 90, 77
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 50).astype(np.float32)
    amax = max(abs(float(C[k, d])) for k in range(K) for d in range(D_eff))
    s = np.float32(32767.0) / np.float32(amax)
    q = [[int(round(float(np.float32(C[k, d]) * s))) for d in range(D_eff)] for k in range(K)]   # python round: half-even
    dot = o.similarity(hb, C, D_eff, o.SIM_DOT, o.HV_I16)
    cos = o.similarity(hb, C, D_eff, o.SIM_COS, o.HV_I16)
    for n in range(N):
        for k in range(K):
            acc = sum((1 - 2 * int(hb[n, d])) * q[k][d] for d in range(D_eff))
            assert dot[n, k] == acc
            nrm = sum(v * v for v in q[k]) ** 0.5
            assert abs(cos[n, k] - acc / (D_eff ** 0.5 * nrm)) < 1e-12
    # integer accumulators with max|c| = 32767: scale exactly 1 -> the int16 operand IS the accumulator
    Ci = r.integers(-32767, 32768, size=(K, D)).astype(np.float32)
    Ci[0, 0] = 32767.0
    assert np.array_equal(o.similarity(hb, Ci, D, o.SIM_DOT, o.HV_I16), o.similarity(hb, Ci, D, o.SIM_DOT, 32))
    assert np.allclose(o.similarity(hb, Ci, D, o.SIM_COS, o.HV_I16), o.similarity(hb, Ci, D, o.SIM_COS, 32),
                       rtol=1e-14, atol=0)


# ------------------------------------------------------------------ S5 32- / 64-bit integer class operand (A22)
def test_int32_int64_codes_by_hand():
    """round_int_tensor ("integer data types (8, 16, 32, or 64-bit)"; reading A22): the codes
    ARE the accumulators, q = rint-to-nearest-EVEN(c), no scale, symmetric saturation at 2^(w-1) - 1.  By hand,
    so that truncation (1.5 -> 1), half-up (0.5 -> 1, -1.5 -> -1), half-away (2.5 -> 3), any A7-style scale
    (7 -> 7 * s), a clamp at -2^31 and a wrap of out-of-range values each fail."""
    c = np.array([[0.5, 1.5, 2.5, 3.49, 7.0, 16777216.0],
                  [-0.5, -1.5, -2.5, -3.51, 1e10, -3e9]], dtype=np.float32)
    # 1e10 = 2^10 * 9765625 and 3e9 = 2^9 * 5859375 are fp32 values (odd parts < 2^24)
    assert o.round_int_tensor(c, 32).tolist() == [[0, 2, 2, 3, 7, 16777216],
                                                  [0, -2, -2, -4, 2147483647, -2147483647]]
    assert o.round_int_tensor(c, 64).tolist() == [[0, 2, 2, 3, 7, 16777216],
                                                  [0, -2, -2, -4, 10000000000, -3000000000]]
    # the edges: 2^31 itself saturates to 2^31 - 1 (and -2^31 to -(2^31 - 1)); the largest fp32 below 2^31 does not
    e = np.array([[2147483648.0, -2147483648.0, 2147483520.0, -2147483520.0]], dtype=np.float32)
    assert o.round_int_tensor(e, 32).tolist() == [[2147483647, -2147483647, 2147483520, -2147483520]]
    assert o.round_int_tensor(e, 64).tolist() == [[2147483648, -2147483648, 2147483520, -2147483520]]
    e = np.array([[2.0 ** 63, -2.0 ** 63, 1e30, -1e30, 2.0 ** 62]], dtype=np.float32)
    assert o.round_int_tensor(e, 64).tolist() == [[2 ** 63 - 1, -(2 ** 63 - 1), 2 ** 63 - 1, -(2 ** 63 - 1), 2 ** 62]]
    # the class operand is the prefix d < D_eff, as int64
    C = np.array([[2.5, -7.0, 1000.0], [0.5, 3.5, -1000.0]], dtype=np.float32)
    for hv in (o.HV_I32, o.HV_I64):
        got = o.class_operand(C, 2, hv)
        assert got.dtype == np.int64 and got.tolist() == [[2, -7], [0, 4]]


def test_int32_int64_similarity_brute_force_and_identities():
    """hv codes HV_I32 / HV_I64 through similarity(): DOT = the python-integer sum of v*q over d < D_eff
    (beyond 2^53 for the 64-bit codes: a float64 contraction would round there), COS = DOT / (sqrt(D_eff) |q|);
    for integer accumulators the scores of hv_bits = 32 are reproduced exactly, and the two widths agree
    wherever the 32-bit codes do not saturate."""
    r = rng(220)
    N, K, D, D_eff = 6, 4, 90, 77
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    for hv, mag in ((o.HV_I32, 1.2e9), (o.HV_I64, 2.0 ** 52)):
        C = (r.standard_normal((K, D)) * mag).astype(np.float32)
        C[1, 3] = 0.5                                    # a tie (-> 0) and a non-integer (-> rint) among them
        C[2, 5] = -1234.5
        w = 32 if hv == o.HV_I32 else 64
        lim = 2 ** (w - 1) - 1
        q = [[max(-lim, min(lim, int(round(float(C[k, d]))))) for d in range(D_eff)] for k in range(K)]  # python round: half-even, exact ints
        assert hv == o.HV_I64 or any(abs(v) == lim for row in q for v in row)   # the 32-bit case does saturate
        dot = o.similarity(hb, C, D_eff, o.SIM_DOT, hv)
        cos = o.similarity(hb, C, D_eff, o.SIM_COS, hv)
        assert dot.dtype == np.int64
        big = 0
        for n in range(N):
            for k in range(K):
                acc = sum((1 - 2 * int(hb[n, d])) * q[k][d] for d in range(D_eff))
                assert int(dot[n, k]) == acc
                big = max(big, abs(acc))
                nrm = float(sum(v * v for v in q[k])) ** 0.5
                assert abs(cos[n, k] - acc / (D_eff ** 0.5 * nrm)) <= 1e-12 * abs(cos[n, k]) + 1e-300
        assert hv == o.HV_I32 or big > 2 ** 53
    # integer accumulators as training leaves them: the integer operand IS the accumulator
    Ci = r.integers(-5000, 5001, size=(K, D)).astype(np.float32)
    want = o.similarity(hb, Ci, D_eff, o.SIM_DOT, 32)
    for hv in (o.HV_I32, o.HV_I64):
        assert np.array_equal(o.similarity(hb, Ci, D_eff, o.SIM_DOT, hv).astype(np.float64), want)
        assert np.allclose(o.similarity(hb, Ci, D_eff, o.SIM_COS, hv), o.similarity(hb, Ci, D_eff, o.SIM_COS, 32),
                           rtol=1e-14, atol=0)
        lab, best, second = o.classify(o.similarity(hb, Ci, D_eff, o.SIM_DOT, hv), o.SIM_DOT)
        lab32, best32, second32 = o.classify(want, o.SIM_DOT)
        assert np.array_equal(lab, lab32) and np.array_equal(best, best32) and np.array_equal(second, second32)
    # a zero class row has cosine 0 (A8), perforation gathers the visited dimensions (A17)
    Cz = Ci.copy()
    Cz[2] = 0.0
    assert np.all(o.similarity(hb, Cz, D_eff, o.SIM_COS, o.HV_I32)[:, 2] == 0.0)
    idx = np.arange(3, D_eff, 4)
    assert np.array_equal(o.similarity(hb, Ci, D_eff, o.SIM_DOT, o.HV_I64, 3, 4),
                          o.similarity(hb[:, idx], Ci[:, idx], len(idx), o.SIM_DOT, o.HV_I64))
