"""CPU ORACLE for the HDC hot path of arxiv/paper_2606_26547 (ApproxHDC) -- TEST INFRASTRUCTURE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module.  It shares no code with `paper_2606_26547_b200/` (the CUDA path)
and imports nothing from it.  It is a plain, slow restatement, in numpy float64 / exact
integers, of what the paper defines; every function cites the PAPER.md passage (Lnn) it
follows and, where the paper is silent, the DESIGN.md reading (A1..A15, S0..S10) it adopts.
There is no blocking, fusion or reordering: each function is the definition written out, with
a library routine (float64 matmul, sum, argmax, packbits) as a step.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): brute-force python loops on tiny inputs, the
bipolar identity dot = D_eff - 2*Hamming, near-orthogonality |cos| <~ 3/sqrt(D), the
angle/Hamming closed form for Gaussian projections, majority-bundling recovery probability
1/2 + C(F-1,(F-1)/2)/2^F, D_eff slice-equivalence and Listing 1's "first 1024 of 2048",
bf16 RNE against ml_dtypes, per-row and per-tensor int8 / int16 codes worked by hand (non-unit scales, ties of
both parities), the 32- / 64-bit integer class codes (A22) by hand and against python-integer sums beyond 2^53, perceptron invariants (sum_k Delta = 0; B=1 == textbook online perceptron; 1 < B < N with
a ragged last batch == a python-loop restatement that re-derives the operand per mini-batch); the ADC-quantised chunked dot (S12) against hand loops, the transparent-window case
(= D_eff - 2*Hamming) and a hand-worked clipped example -- its transfer function itself is a
reading (A19), the paper prints no formula: "parity unpinned" for the ADC formula.  Unpinned: accuracy parity with the paper's ISOLET numbers (datasets absent) --
"parity unpinned" for that one item only.

Conventions (S0; paper silent, readings A1-A3): bipolar v in {+1,-1}; bit b = [v == -1], so
XOR of bits == product of bipolars; sgn(a) = -1 iff a < 0 (0 -> +1, bit 0); packed element d
sits in uint32 word d>>5 at bit d&31 (LSB first), tail bits zero; arg-extremum ties -> lowest
index.
"""
from __future__ import annotations

import numpy as np

# precision / hv_bits / sim codes mirror include/hdc.h numerically but are typed here by hand
F32, BF16, I8, B1 = 0, 1, 2, 3
F16 = 6         # encode operands as IEEE half ("floating-point types (FP16 or FP32)")
SIM_DOT, SIM_COS, SIM_HAMMING = 0, 1, 2
HV_F16 = 17      # hv_bits code (not a width): class operand as 16-bit IEEE half ("FP16")
HV_I16 = 18      # hv_bits code (not a width): class operand as 16-bit integers ("integer data types (8, 16, ...")
HV_I32 = 19      # hv_bits codes: class operand as 32- / 64-bit integers ("... 32, or 64-bit)"; reading A22)
HV_I64 = 20


# ------------------------------------------------------------------------------------- S0
def unpack_bits(words: np.ndarray, D: int) -> np.ndarray:
    """[R][>=ceil(D/32)] uint32 -> [R][D] uint8 bits, LSB-first (S0 / A2)."""
    w = np.ascontiguousarray(words, dtype="<u4")
    by = w.view(np.uint8).reshape(w.shape[0], -1)
    return np.unpackbits(by, axis=1, bitorder="little")[:, :D].copy()


def pack_bits(bits: np.ndarray) -> np.ndarray:
    """[R][D] bits -> [R][ceil(D/32)] uint32, LSB-first, tail bits zero (S0 / A2)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint8)
    R, D = bits.shape
    W = (D + 31) // 32
    pad = np.zeros((R, W * 32), dtype=np.uint8)
    pad[:, :D] = bits
    return np.packbits(pad, axis=1, bitorder="little").view("<u4").reshape(R, W).copy()


def bipolar(bits: np.ndarray) -> np.ndarray:
    """bit -> +1/-1 as float64 (bit 1 <=> -1, A2)."""
    return 1.0 - 2.0 * bits.astype(np.float64)


# ------------------------------------------------------------------------------------- S1
def round_bf16(x: np.ndarray) -> np.ndarray:
    """fp32 -> nearest bfloat16 (ties to even), returned as float32 holding that value.
    PAPER.md L165 ("element type representation"); RNE is reading A7.  Finite inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return r.astype(np.uint32).view(np.float32).reshape(np.shape(x))


def quantize_int8_rows(x: np.ndarray) -> np.ndarray:
    """Per-row symmetric int8 (reading A7; "projecting ... onto lower-precision
    integer types"): a = max_f |x|, s = fl32(127/a) (s = 1 if a == 0),
    q = clamp(rint(fl32(x*s)), -127, 127).  Every step is one correctly rounded fp32 op."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    a = np.max(np.abs(x), axis=1, keepdims=True).astype(np.float32)
    s = np.where(a > 0, np.float32(127.0) / np.where(a > 0, a, np.float32(1)), np.float32(1.0))
    s = s.astype(np.float32)
    q = np.rint((x * s).astype(np.float32))
    return np.clip(q, -127, 127).astype(np.int32)


def quantize_int8_tensor(c: np.ndarray) -> np.ndarray:
    """Per-tensor symmetric int8 over the given array (S5 / A7): s = fl32(127/max|c|)."""
    c = np.ascontiguousarray(c, dtype=np.float32)
    a = np.float32(np.max(np.abs(c))) if c.size else np.float32(0)
    s = np.float32(127.0) / a if a > 0 else np.float32(1.0)
    q = np.rint((c * np.float32(s)).astype(np.float32))
    return np.clip(q, -127, 127).astype(np.int32)


def quantize_int16_tensor(c: np.ndarray) -> np.ndarray:
    """Per-tensor symmetric int16 over the given array (hypervectors "represented using
    integer data types (8, 16, 32, or 64-bit)", inference "projecting class ... hypervectors onto
    lower-precision integer types"; reading A7 carried to 16 bits, A21): s = fl32(32767/max|c|) (1 if the
    array is all zero), q = clamp(rint(fl32(c*s)), -32767, 32767), rint = round half to even."""
    c = np.ascontiguousarray(c, dtype=np.float32)
    a = np.float32(np.max(np.abs(c))) if c.size else np.float32(0)
    s = np.float32(32767.0) / a if a > 0 else np.float32(1.0)
    q = np.rint((c * np.float32(s)).astype(np.float32))
    return np.clip(q, -32767, 32767).astype(np.int32)


def round_int_tensor(c: np.ndarray, width: int) -> np.ndarray:
    """Class operand as 32- or 64-bit integers (hypervectors "represented using integer data
    types (8, 16, 32, or 64-bit)"; L53 / L181: class hypervectors are sums of +-1 hypervectors, i.e. integers;
    reading A22): the accumulators themselves, q = rint(c), round half to even, NO scale (an fp32 value has 24
    significant bits: stretching it to 2^31 adds rounding and no information; for the integer accumulators
    that training produces q = c), saturating symmetrically at +-(2^(width-1) - 1).  Returns int64."""
    if width not in (32, 64):
        raise ValueError("width")
    c = np.ascontiguousarray(c, dtype=np.float32).astype(np.float64)     # every fp32 is a float64
    q = np.rint(c)                                                        # half to even; integers in float64
    lim = (1 << (width - 1)) - 1
    edge = float(1 << (width - 1))                                        # 2^(width-1): first value out of range
    inside = np.abs(q) < edge                                             # these convert exactly (fp32-valued)
    out = np.where(inside, q, 0.0).astype(np.int64)
    out[~inside & (q > 0)] = lim
    out[~inside & (q < 0)] = -lim
    return out


def rp_operands(X: np.ndarray, P: np.ndarray, precision: int):
    """Operands of the random-projection contraction at `precision` (S1): FP32 identity;
    BF16 RNE of both; F16 IEEE-half RNE of both; INT8 per-row of X and per-row (per projection d) of P.  B1 means packed
    hypervectors with the real-valued contraction done in bf16 (reading A6)."""
    if precision == F32:
        return X.astype(np.float64), P.astype(np.float64)
    if precision in (BF16, B1):
        return round_bf16(X).astype(np.float64), round_bf16(P).astype(np.float64)
    if precision == F16:
        # IEEE binary16 RNE of both operands, products and sums exact / float64 (fp32 accumulate on the GPU)
        return (np.asarray(X, dtype=np.float32).astype(np.float16).astype(np.float64),
                np.asarray(P, dtype=np.float32).astype(np.float16).astype(np.float64))
    if precision == I8:
        return quantize_int8_rows(X).astype(np.float64), quantize_int8_rows(P).astype(np.float64)
    raise ValueError("precision")


def encode_rp(X: np.ndarray, P: np.ndarray, D_eff: int, precision: int = F32,
              want_absum: bool = False, f_begin: int = 0, f_stride: int = 1):
    """Random-projection encode + sign (Listing 1 L68-L70 `__hetero_hdc_matmul`,
    L155 "matrix-vector dot-product", L161 "{+1,-1} representation"; always binarised: A5).

        acc[n,d] = sum_{f<F} x~[n,f] * p~[d,f]      (P is [D][F]: `hypermatrix<2048,617>`, L65)
        bit[n,d] = [acc[n,d] < 0]  for d < D_eff     (sgn(0) = +1, A1)

    float64 accumulation; for INT8 the operands are integers <= 127 so every product and sum is
    exact in float64.  Returns bits [N][D_eff] uint8, acc [N][D_eff] float64 and optionally
    absum[n,d] = sum_f |x~ p~| (used by the sign-agreement band, S4).

    Reduction perforation of the F axis (off by default: L157 / L187 keep it out of the encoders
    because it "often degrades the quality-of-service"; L155 defines it: "for operations such as
    matrix-vector dot products, the results are scaled appropriately to compensate for the skipped
    iterations"; reading A18): the loop visits f = f_begin, f_begin + f_stride, ... < F, the operands
    at `precision` are those of the gathered columns (per-row int8 scales over the visited features),
    and acc (and absum) are multiplied by F / F_visited."""
    X, P = np.asarray(X), np.asarray(P)[:D_eff]
    scale = 1.0
    if f_begin != 0 or f_stride != 1:
        F = X.shape[1]
        idx = perforated_index(F, f_begin, f_stride)
        X, P = X[:, idx], P[:, idx]
        scale = F / len(idx)
    Xo, Po = rp_operands(X, P, precision)
    acc = (Xo @ Po.T) * scale
    bits = (acc < 0).astype(np.uint8)
    absum = (np.abs(Xo) @ np.abs(Po).T) * scale if want_absum else None
    return bits, acc, absum


# ------------------------------------------------------------------------------------- S2
def encode_levelid(levels: np.ndarray, ID: np.ndarray, LV: np.ndarray, D_eff: int) -> np.ndarray:
    """Level-ID ("ID-based", record) encoding ("ID-based encoding [12]", L183
    N_LEVELS, L239 "Level-ID encoding"; bind = XOR, bundle = majority: BASELINE north_star).

        cnt[n,d] = sum_{f<F} ( ID[f,d] XOR LV[levels[n,f], d] )
        bit[n,d] = [ 2*cnt[n,d] > F ]          (tie, F even -> bit 0 <=> bipolar sum 0 -> +1: A3)

    levels [N][F] integer level indices < Q; ID [F][D], LV [Q][D] are 0/1 arrays."""
    levels = np.asarray(levels)
    ID = np.asarray(ID, dtype=np.uint8)[:, :D_eff]
    LV = np.asarray(LV, dtype=np.uint8)[:, :D_eff]
    N, F = levels.shape
    out = np.empty((N, D_eff), dtype=np.uint8)
    for n in range(N):
        bound = ID ^ LV[levels[n].astype(np.int64)]           # [F][D_eff]
        cnt = bound.sum(axis=0, dtype=np.int64)
        out[n] = (2 * cnt > F)
    return out


# ------------------------------------------------------------------------------------- S5
def class_operand(C_acc: np.ndarray, D_eff: int, hv_bits: int) -> np.ndarray:
    """Class operand derived from the fp32 accumulators at the hypervector element width
    (training in high precision, inference "projecting class ... hypervectors
    onto lower-precision integer types"; S5): 32 -> C_acc; 16 -> bf16 RNE; 8 -> per-tensor
    symmetric int8 over k<K, d<D_eff; 1 -> bit [C_acc < 0]; HV_F16 -> IEEE half RNE; HV_I16 -> per-tensor
    symmetric int16 over k<K, d<D_eff; HV_I32 / HV_I64 -> rint(C_acc) as 32- / 64-bit integers (A22).
    Returned as float64 values (bits as uint8, the 32- / 64-bit integer codes as int64)."""
    c = np.asarray(C_acc, dtype=np.float32)[:, :D_eff]
    if hv_bits == 32:
        return c.astype(np.float64)
    if hv_bits == 16:
        return round_bf16(c).astype(np.float64)
    if hv_bits == HV_F16:
        # IEEE binary16, round-to-nearest-even (L165 "floating-point types (FP16 or FP32)");
        # |c| > 65504 overflows to +-inf: outside the contract (S0: finite operands)
        return c.astype(np.float16).astype(np.float64)
    if hv_bits == 8:
        return quantize_int8_tensor(c).astype(np.float64)
    if hv_bits == HV_I16:
        return quantize_int16_tensor(c).astype(np.float64)
    if hv_bits in (HV_I32, HV_I64):
        return round_int_tensor(c, 32 if hv_bits == HV_I32 else 64)
    if hv_bits == 1:
        return (c < 0).astype(np.uint8)
    raise ValueError("hv_bits")


# ------------------------------------------------------------------------------------- S6
def hamming(hbits: np.ndarray, cbits: np.ndarray, D_eff: int) -> np.ndarray:
    """dist[n,k] = sum_{d<D_eff} [h[n,d] != c[k,d]]  (Listing 1 L72-L74
    `__hetero_hdc_hamming_distance`, L161 xor+popcount; prefix reduction-perforation L61,
    L76-L77, result used as-is L155)."""
    h = np.asarray(hbits, dtype=np.uint8)[:, :D_eff]
    c = np.asarray(cbits, dtype=np.uint8)[:, :D_eff]
    out = np.empty((h.shape[0], c.shape[0]), dtype=np.int64)
    for k in range(c.shape[0]):
        out[:, k] = (h ^ c[k][None, :]).sum(axis=1, dtype=np.int64)
    return out


def dot(hbits: np.ndarray, cop: np.ndarray, D_eff: int) -> np.ndarray:
    """s[n,k] = sum_{d<D_eff} v[n,d]*c[k,d], v bipolar (PAPER.md L197/L229 dot-product
    similarity; L155 perforated similarity "used as-is": no rescale, A11).  float64; exact
    for integer operands."""
    v = bipolar(np.asarray(hbits)[:, :D_eff])
    return v @ np.asarray(cop, dtype=np.float64)[:, :D_eff].T


def cosine(hbits: np.ndarray, cop: np.ndarray, D_eff: int) -> np.ndarray:
    """s[n,k] = dot[n,k] / ( sqrt(D_eff) * sqrt(sum_{d<D_eff} c[k,d]^2) ), 0 where the class
    norm is 0 ("cosine similarity", L110 `__hetero_hdc_cos_sim`; A8).  The query
    norm of a bipolar vector restricted to D_eff dims is sqrt(D_eff)."""
    c = np.asarray(cop, dtype=np.float64)[:, :D_eff]
    s = dot(hbits, c, D_eff)
    nrm = np.sqrt((c * c).sum(axis=1))
    out = np.zeros_like(s)
    nz = nrm > 0
    out[:, nz] = s[:, nz] / (np.sqrt(float(D_eff)) * nrm[nz])[None, :]
    return out


def dot_int(hbits: np.ndarray, q: np.ndarray, D_eff: int) -> np.ndarray:
    """s[n,k] = sum_{d<D_eff} v[n,d]*q[k,d] for integer codes q, in 64-bit integer arithmetic (exact while
    sum_d |q[k,d]| < 2^63: the contract of the 32- / 64-bit integer class operands, A22).  int64 [N][K]."""
    v = (1 - 2 * np.asarray(hbits, dtype=np.int64)[:, :D_eff])
    q = np.asarray(q, dtype=np.int64)[:, :D_eff]
    out = np.empty((v.shape[0], q.shape[0]), dtype=np.int64)
    for k in range(q.shape[0]):
        out[:, k] = (v * q[k][None, :]).sum(axis=1, dtype=np.int64)
    return out


def cosine_int(hbits: np.ndarray, q: np.ndarray, D_eff: int) -> np.ndarray:
    """Cosine for integer codes: dot_int / (sqrt(D_eff) * |q[k]|), 0 where the class norm is 0 (A8); the
    squared norm is summed in python integers (exact), the division done in float64."""
    s = dot_int(hbits, q, D_eff)
    out = np.zeros(s.shape, dtype=np.float64)
    for k in range(s.shape[1]):
        n2 = sum(int(x) * int(x) for x in np.asarray(q)[k, :D_eff])
        if n2 > 0:
            out[:, k] = s[:, k].astype(np.float64) / (np.sqrt(float(D_eff)) * np.sqrt(float(n2)))
    return out


def perforated_index(D_eff: int, begin: int = 0, stride: int = 1) -> np.ndarray:
    """Reduction perforation (the reduction-axis loop "skip[s] iterations at regular
    intervals, defined by a specified stride", annotation parameters "starting offset, ending offset,
    and stride"; L76-L77 red_perf(v, 0, 0.5, 1); L130 {"stride": 8, "extent": 0.84}): the dimensions
    a similarity reduction visits are d = begin, begin + stride, ... < D_eff (end offset = D_eff)."""
    if stride < 1 or not 0 <= begin < D_eff:
        raise ValueError("bad perforation")
    return np.arange(begin, D_eff, stride)


def similarity(hbits: np.ndarray, C_acc: np.ndarray, D_eff: int, sim: int, hv_bits: int,
               begin: int = 0, stride: int = 1):
    """Scores of every query against every class at the given knobs (S5 + S6).
    Perforation (reading A17): the result equals that of physically gathering the visited
    dimensions of both operands and running with D = their number -- nothing is rescaled
    (L155: "for similarity and dissimilarity computations, the resultant values are used as-is"),
    the cosine is the cosine of the sub-vectors, the per-tensor int8 scale is taken over them."""
    if begin != 0 or stride != 1:
        idx = perforated_index(D_eff, begin, stride)
        hb = np.asarray(hbits, dtype=np.uint8)[:, idx]
        Cg = np.asarray(C_acc, dtype=np.float32)[:, idx]
        return similarity(hb, Cg, len(idx), sim, hv_bits)
    cop = class_operand(C_acc, D_eff, hv_bits)
    if sim == SIM_HAMMING:
        if hv_bits != 1:
            raise ValueError("Hamming needs hv_bits=1")
        return hamming(hbits, cop, D_eff)
    if hv_bits in (HV_I32, HV_I64):
        if sim == SIM_DOT:
            return dot_int(hbits, cop, D_eff)
        if sim == SIM_COS:
            return cosine_int(hbits, cop, D_eff)
        raise ValueError("sim")
    if hv_bits == 1:
        cop = bipolar(cop)
    if sim == SIM_DOT:
        return dot(hbits, cop, D_eff)
    if sim == SIM_COS:
        return cosine(hbits, cop, D_eff)
    raise ValueError("sim")


# ------------------------------------------------------------------------------------- S12
def adc_quantize(p: np.ndarray, res: int, step: int, floor: int, ceil: int) -> np.ndarray:
    """Transfer function of the analogue-to-digital converter that reads one array chunk's partial
    dot product in the SpecPCM simulator (knobs ADC_RES, ADC_STEP, ADC_FLOOR, ADC_CEIL;
    "each partial dot product quantized by the ADC before accumulation"; "Clipping below -3 ...
    narrowing the ADC input range ... allows fewer quantization levels (lower ADC_RES)").  The paper
    gives no formula; reading A19: the input is clipped to [floor, ceil], converted to the nearest of
    2^res codes spaced `step` apart starting at `floor` (halves round up, codes saturate at
    2^res - 1), and read back as floor + code*step.  The paper's baseline window (floor -127, ceil 128,
    res 8, step 1) is then exactly 256 codes and transparent on [-127, 128].  Integers in, out."""
    if res < 1 or res > 16 or step < 1 or floor > ceil:
        raise ValueError("bad ADC parameters")
    p = np.clip(np.asarray(p, dtype=np.int64), floor, ceil)
    code = (p - floor + step // 2) // step
    code = np.minimum(code, (1 << res) - 1)
    return floor + code * step


def similarity_adc(hbits: np.ndarray, C_acc: np.ndarray, D_eff: int, res: int, step: int, floor: int,
                   ceil: int, chunk: int = 128) -> np.ndarray:
    """Chunked, ADC-quantised dot-product similarity ("The SpecPCM simulator computes
    dot-product similarity over 128-element array chunks, with each partial dot product quantized by
    the ADC before accumulation"; MLC=1, "+-1 encoded hypervectors": query and class operand bipolar,
    class operand = sign of the accumulators, S5 at hv_bits = 1):

        s[n,k] = sum_j  adc( sum_{d in chunk j, d < D_eff} v[n,d] * c[k,d] )

    chunks are [j*chunk, (j+1)*chunk); the last one may hold fewer than `chunk` dimensions.
    Returns int64 [N][K]; the label is the arg-max (ties -> lowest index, S7)."""
    v = bipolar(np.asarray(hbits, dtype=np.uint8)[:, :D_eff]).astype(np.int64)
    c = bipolar(class_operand(C_acc, D_eff, 1)).astype(np.int64)
    S = np.zeros((v.shape[0], c.shape[0]), dtype=np.int64)
    for j0 in range(0, D_eff, chunk):
        part = v[:, j0:j0 + chunk] @ c[:, j0:j0 + chunk].T
        S += adc_quantize(part, res, step, floor, ceil)
    return S


# ------------------------------------------------------------------------------------- S7
def classify(S: np.ndarray, sim: int):
    """Label = arg-max of DOT/COS scores, arg-min of Hamming distances (Listing 1
    L79-L80 `__hetero_hdc_arg_min` "select nearest cluster"); ties -> lowest index (A14).
    Also returns best and runner-up values (runner-up = best of the rest; = best on a tie;
    = best when K == 1)."""
    S = np.asarray(S)
    key = -S if sim == SIM_HAMMING else S
    lab = np.argmax(key, axis=1).astype(np.int32)            # first occurrence = lowest index
    n = np.arange(S.shape[0])
    best = S[n, lab]
    if S.shape[1] == 1:
        return lab, best, best.copy()
    rest = np.array(key, dtype=np.float64, copy=True)
    rest[n, lab] = -np.inf
    second = S[n, np.argmax(rest, axis=1)]
    return lab, best, second


# ------------------------------------------------------------------------------------- S8
def bundle(hbits: np.ndarray, y: np.ndarray, K: int, D_eff: int, C_acc: np.ndarray | None = None):
    """One-pass training: C_acc[k,d] += sum_{n: y_n = k} v[n,d]  ("hypervectors
    corresponding to inputs from the same class are combined ... vector addition").  fp32
    accumulators (A10) hold these integers exactly (|.| < 2^24)."""
    v = bipolar(np.asarray(hbits)[:, :D_eff])
    out = np.zeros((K, D_eff), dtype=np.float64) if C_acc is None else \
        np.array(C_acc, dtype=np.float64)[:, :D_eff].copy()
    for k in range(K):
        out[k] += v[np.asarray(y) == k].sum(axis=0)
    return out.astype(np.float32)


# ------------------------------------------------------------------------------------- S9
def train_epoch(hbits: np.ndarray, y: np.ndarray, C_acc: np.ndarray, D_eff: int, hv_bits: int,
                sim: int, lr: float, batch: int = 0, begin: int = 0, stride: int = 1):
    """One retraining epoch (PAPER.md L181 TRAIN_ITERATIONS "number of retraining epochs";
    the per-sample rule is not in the paper -- reading A9 / S9, "perceptron-style" per
    BASELINE north_star).  Samples in index order, no shuffle; per mini-batch of B samples:
      (i)   class operands from the current C_acc (S5);
      (ii)  yhat_n = classify(h_n) with the inference similarity;
      (iii) Delta[k,d] = sum_{n in batch, yhat_n != y_n} ([k=y_n] - [k=yhat_n]) * v[n,d]  (integer);
      (iv)  C_acc[k,d] = fl32( C_acc[k,d] + fl32( lr * (float)Delta[k,d] ) )   two rounded ops.
    Returns (C_acc' fp32 [K][D_eff], number of mispredictions, predictions int32 [N])."""
    hb = np.asarray(hbits, dtype=np.uint8)[:, :D_eff]
    y = np.asarray(y)
    C = np.array(C_acc, dtype=np.float32)[:, :D_eff].copy()
    K = C.shape[0]
    N = hb.shape[0]
    B = N if batch in (0, None) or batch > N else int(batch)
    lr32 = np.float32(lr)
    pred = np.empty(N, dtype=np.int32)
    wrong = 0
    for b0 in range(0, N, B):
        sl = slice(b0, min(N, b0 + B))
        S = similarity(hb[sl], C, D_eff, sim, hv_bits, begin, stride)   # only the similarity is perforated
        yh, _, _ = classify(S, sim)
        pred[sl] = yh
        v = bipolar(hb[sl])
        delta = np.zeros((K, D_eff), dtype=np.int64)
        for i in np.nonzero(yh != y[sl])[0]:
            vi = v[i].astype(np.int64)
            delta[y[sl][i]] += vi
            delta[yh[i]] -= vi
            wrong += 1
        step = (lr32 * delta.astype(np.float32)).astype(np.float32)
        C = (C + step).astype(np.float32)
    return C, wrong, pred


# ------------------------------------------------------------------------------------- S10
def train(hbits, y, K, D_eff, hv_bits, sim, epochs, lr, batch=0):
    """Bundle then `epochs` retraining epochs (S10); "skipped retraining iterations" = fewer
    epochs (10 -> 3)."""
    C = bundle(hbits, y, K, D_eff)
    hist = []
    for _ in range(int(epochs)):
        C, wrong, _ = train_epoch(hbits, y, C, D_eff, hv_bits, sim, lr, batch)
        hist.append(wrong)
    return C, hist


# ------------------------------------------------------------------------------------- S11
def kmeans_epoch(hbits: np.ndarray, C_acc: np.ndarray, D_eff: int, hv_bits: int, sim: int, prev=None,
                 begin: int = 0, stride: int = 1):
    """One iteration of HD-Clustering ("HD-Clustering implements K-Means clustering
    using HDC", L221: cosine or Hamming similarity, TRAIN_ITERATIONS epochs).  The paper gives no
    pseudo-code; reading A16 is Lloyd's iteration with the path's own primitives:
      (i)   a_n = classify(h_n) against the current cluster accumulators (S5-S7: the similarity and
            element precision of the knobs, ties to the lowest cluster index);
      (ii)  every cluster that received at least one sample is re-bundled from its members,
            C_acc[k,d] = sum_{n: a_n = k} v[n,d]   (S8);  a cluster with no member keeps its
            accumulator unchanged.
    Returns (C_acc' fp32 [K][D_eff], assignments int32 [N], number of n with a_n != prev[n]
    (0 if prev is None))."""
    hb = np.asarray(hbits, dtype=np.uint8)[:, :D_eff]
    C = np.array(C_acc, dtype=np.float32)[:, :D_eff].copy()
    K = C.shape[0]
    S = similarity(hb, C, D_eff, sim, hv_bits, begin, stride)
    a, _, _ = classify(S, sim)
    a = a.astype(np.int32)
    v = bipolar(hb).astype(np.int64)
    for k in range(K):
        members = np.nonzero(a == k)[0]
        if members.size:
            C[k] = v[members].sum(axis=0).astype(np.float32)
    changed = 0 if prev is None else int((a != np.asarray(prev)).sum())
    return C, a, changed


def infer(hbits, C_acc, D_eff, sim, hv_bits):
    """similarity + arg-extremum (Listing 1 L72-L80)."""
    S = similarity(hbits, C_acc, D_eff, sim, hv_bits)
    return classify(S, sim) + (S,)
