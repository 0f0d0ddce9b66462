"""Per-row measurements of the hot path beyond bench.py's headline step:
each row times one entry point of the C ABI on device-resident, seeded synthetic inputs of the
shapes of BASELINE.json's configs, with CUDA events around the calls and the library's own per-kernel
events (hdc_kernel_time) for the dominant kernel, and states the roofline it is held against.

    python -m paper_2606_26547_b200.bench_rows [--row NAME] [--reps R]

Used by `bench.py --rows` and as the (committed) command of the ncu captures under profiles/.
No arithmetic of the method lives here.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_2606_26547_b200 as hd  # noqa: E402

SEED = 26547


def _gen(seed):
    g = torch.Generator(device="cuda")
    g.manual_seed(SEED + seed)
    return g


def _time(fn, reps, warm=3):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def _kernel(h, kid, fn, reps):
    h.kernel_timing(True)
    for _ in range(reps):
        fn()
    torch.cuda.synchronize()
    ms, n = h.kernel_time(kid)
    h.kernel_timing(False)
    return ms / max(1, n), n // max(1, reps)


def _rand_bits(n, w, seed):
    return torch.randint(-2 ** 31, 2 ** 31 - 1, (n, w), dtype=torch.int32, device="cuda", generator=_gen(seed))


def _class_acc(K, D, seed, per_class=32):
    """Accumulators shaped like a bundle of `per_class` bipolar hypervectors per class (exact ints)."""
    u = torch.randint(0, 2, (per_class, K, D), dtype=torch.int8, device="cuda", generator=_gen(seed))
    return (per_class - 2 * u.sum(0, dtype=torch.int32)).to(torch.float32).contiguous()


# ------------------------------------------------------------------------------------ encode rows
def row_encode(h, peaks, reps, N, F, D, prec_name, x_bf16=False):
    flags = 0
    if prec_name == "f32_fast":   # HDC_FLAG_F32_FAST: 2-way half splits, three products
        flags = hd.HDC_FLAG_F32_FAST
    prec = {"f32": hd.HDC_F32, "f32_fast": hd.HDC_F32, "bf16": hd.HDC_BF16, "f16": hd.HDC_F16,
            "i8": hd.HDC_I8}[prec_name]
    X = torch.randn((N, F), device="cuda", generator=_gen(1))
    P = torch.randn((D, F), device="cuda", generator=_gen(2))
    if x_bf16:
        X, P = X.to(torch.bfloat16), P.to(torch.bfloat16)
    kn = hd.knobs(D, precision=prec, flags=flags)
    H = torch.empty((N, (D + 31) // 32), dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_encode_rp(X, P, kn, Hbits=H)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_ENCODE_GEMM, fn, reps)
    flops = 2.0 * N * F * D
    mult = {"f32": 1.0 / 6.0, "f32_fast": 1.0 / 3.0, "bf16": 1.0, "f16": 1.0, "i8": 2.0}[prec_name]
    peak = peaks["bf16_tflops"] * mult
    ach = flops / (k_ms * 1e-3) / 1e12
    return {"what": f"hdc_encode_rp N={N} F={F} D={D} precision={prec_name}" + (" (bf16 inputs in place)" if x_bf16 else ""),
            "call_ms": call_ms, "kernel_ms": k_ms, "queries_per_s": N / (call_ms * 1e-3),
            "roofline": {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "peak_source": f"bf16_tflops (burst, measured) x {mult:.4g}"}}


# ------------------------------------------------------------------------------------ similarity rows
def row_classify(h, peaks, reps, N, K, D, hv_bits, sim_name):
    sim = {"cos": hd.HDC_SIM_COS, "dot": hd.HDC_SIM_DOT, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    W = (D + 31) // 32
    H = _rand_bits(N, W, 3)
    C = _class_acc(K, D, 4)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_classify(H, C, kn, labels=lab)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, reps)
    out = {"what": f"hdc_classify N={N} K={K} D={D} hv_bits={hv_bits} sim={sim_name}", "call_ms": call_ms,
           "kernel_ms": k_ms, "queries_per_s": N / (call_ms * 1e-3)}
    hbm = N * W * 4 / (k_ms * 1e-3) / 1e9
    out["hbm_GBps_query_bits"] = hbm
    if sim_name == "hamming" and K < 64:
        popc = float(N) * K * W / (k_ms * 1e-3) / 1e12
        peak = 148 * 16 * peaks["sm_max_mhz"] * 1e6 / 1e12
        out["roofline"] = {"bound": "alu", "achieved": popc, "peak": peak, "unit": "Tpopc/s", "frac": popc / peak,
                           "peak_source": "148 SM x 16 POPC lanes x sm_max_mhz"}
    else:
        parts = 3 if hv_bits == 32 else 1
        mult = 2.0 if hv_bits in (8, 1) else 1.0
        kp = ((K + 15) // 16) * 16
        flops = 2.0 * N * D * kp * parts
        ach = flops / (k_ms * 1e-3) / 1e12
        peak = peaks["bf16_tflops"] * mult
        out["roofline"] = {"bound": "tensor" if K >= 128 else "hbm",
                           "achieved": ach if K >= 128 else hbm,
                           "peak": peak if K >= 128 else peaks["hbm_gbs"],
                           "unit": "TFLOP/s" if K >= 128 else "GB/s",
                           "frac": (ach / peak) if K >= 128 else hbm / peaks["hbm_gbs"],
                           "executed_tflops": ach}
    return out


def row_adc(h, peaks, reps, N=131072, K=26, D=1024):
    """SpecPCM-simulator similarity (PAPER.md L273 best configuration: D = 1024, ADC_RES 8, ADC_STEP 2,
    ADC_FLOOR -3, ADC_CEIL 128; ISOLET-shaped K = 26): chunked ADC-quantised dot + arg-max."""
    W = (D + 31) // 32
    H = _rand_bits(N, W, 3)
    C = _class_acc(K, D, 4)
    kn = hd.knobs(D)
    fn = lambda: h.hdc_similarity_adc(H, C, kn, 8, 2, -3, 128, want_scores=False)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, reps)
    popc = float(N) * K * W / (k_ms * 1e-3) / 1e12
    peak = 148 * 16 * peaks["sm_max_mhz"] * 1e6 / 1e12
    return {"what": f"hdc_similarity_adc N={N} K={K} D={D} window (8, 2, -3, 128), labels only", "call_ms": call_ms,
            "kernel_ms": k_ms, "queries_per_s": N / (call_ms * 1e-3),
            "hbm_GBps_query_bits": N * W * 4 / (k_ms * 1e-3) / 1e9,
            "roofline": {"bound": "alu", "achieved": popc, "peak": peak, "unit": "Tpopc/s", "frac": popc / peak,
                         "peak_source": "148 SM x 16 POPC lanes x sm_max_mhz"}}


# ------------------------------------------------------------------------------------ level-ID row
def row_levelid(h, peaks, reps, N=65536, F=784, Q=256, D=10000, dense_input=False):
    from workloads import gen
    import numpy as np
    w = gen.c3_mnist_shaped(D=D, n_tr=16, n_te=4096, Q=Q)
    lv = torch.from_numpy(gen.tile_rows(w["Lte"], N)).cuda()
    if dense_input:  # uniformly random levels: no zeros to skip, every warp takes the dense path
        lv = torch.randint(0, Q, (N, F), dtype=torch.uint8, device="cuda", generator=_gen(30))
    ID = torch.from_numpy(gen.pack_bits_lsb(w["ID"]).view(np.int32)).cuda()
    LV = torch.from_numpy(gen.pack_bits_lsb(w["LV"]).view(np.int32)).cuda()
    Wd = (D + 31) // 32
    H = torch.empty((N, Wd), dtype=torch.int32, device="cuda")
    kn = hd.knobs(D)
    fn = lambda: h.hdc_encode_levelid(lv, ID, LV, D, kn, Hbits=H)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_LEVELID, fn, reps)
    # algorithmic logic ops per sample: one bind XOR plus one full
    # adder (2 LOP3) per (feature, word) = 3*F*W; the kernel executes 3.69 (address + ripple extra)
    ops = 3.0 * F * Wd * N
    ach = ops / (k_ms * 1e-3) / 1e12
    peak = 148 * 64 * peaks["sm_max_mhz"] * 1e6 / 1e12
    what = (f"hdc_encode_levelid N={N} F={F} Q={Q} D={D} (uniform random levels: dense path)" if dense_input else
            f"hdc_encode_levelid N={N} F={F} Q={Q} D={D} (C3-shaped, ~80% zero pixels: sparse path, exact; the "
            "fraction is against the DENSE definition's 3*F*W ops, fewer are executed)")
    return {"what": what, "call_ms": call_ms,
            "kernel_ms": k_ms, "samples_per_s": N / (call_ms * 1e-3),
            "hbm_GBps": N * (F + 4 * Wd) / (k_ms * 1e-3) / 1e9,
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "Tlop/s (32-bit logic ops)",
                         "frac": ach / peak, "peak_source": "148 SM x 64 INT lanes x sm_max_mhz"}}


# ------------------------------------------------------------------------------------ training row
def row_train(h, peaks, reps, N=6238, K=26, D=10000, hv_bits=32, sim_name="cos"):
    sim = {"cos": hd.HDC_SIM_COS, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    W = (D + 31) // 32
    H = _rand_bits(N, W, 5)
    y = torch.randint(0, K, (N,), dtype=torch.int32, device="cuda", generator=_gen(6))
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, H, y, C, kn)
    fn = lambda: h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, H, y, C, kn, lr=0.05, batch=0)  # noqa: E731
    call_ms = _time(fn, reps)
    out = {"what": f"hdc_train_epoch (perceptron, B=N) N={N} K={K} D={D} hv_bits={hv_bits} sim={sim_name} "
                   "on random hypervectors (every sample mispredicted: worst case for the class update)",
           "call_ms": call_ms, "samples_per_s": N / (call_ms * 1e-3)}
    # The C ABI neither allocates nor synchronises, so an epoch loop can be captured in a CUDA graph
    # (the 8 launches of an epoch are launch-latency bound at this size): 20 epochs per replay.
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                for _ in range(20):
                    fn()
        torch.cuda.current_stream().wait_stream(side)
        gm = _time(g.replay, max(2, reps // 2)) / 20.0
        out["graph_epoch_ms"] = gm
        out["graph_samples_per_s"] = N / (gm * 1e-3)
    except Exception as e:  # noqa: BLE001
        out["graph_error"] = repr(e)[:200]
    return out


def row_c5_stream(h, peaks, reps, hv_bits, sim_name, N=1 << 20, B=65536, F=1024, D=16384, K=1000):
    """BASELINE.json configs[4]: N = 2^20 bf16 queries streamed in 64K-query device-resident batches
    through hdc_encode_rp (bf16) + hdc_classify against K = 1000 classes (bf16 cosine or packed 1-bit
    Hamming).  Four distinct input batches (537 MB > L2) are cycled."""
    sim = {"cos": hd.HDC_SIM_COS, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    nb = N // B
    Xs = [torch.randn((B, F), device="cuda", generator=_gen(20 + i)).to(torch.bfloat16) for i in range(4)]
    P = torch.randn((D, F), device="cuda", generator=_gen(2)).to(torch.bfloat16)
    C = _class_acc(K, D, 4)
    kn_e = hd.knobs(D, precision=hd.HDC_BF16)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    H = torch.empty((B, (D + 31) // 32), dtype=torch.int32, device="cuda")
    lab = torch.empty(N, dtype=torch.int32, device="cuda")

    def fn():
        for i in range(nb):
            h.hdc_encode_rp(Xs[i & 3], P, kn_e, Hbits=H)
            h.hdc_classify(H, C, kn, labels=lab[i * B:(i + 1) * B])

    call_ms = _time(fn, max(1, reps // 5), warm=1)
    flops = 2.0 * N * D * (F + (K if hv_bits != 1 else 0))
    out = {"what": f"C5 stream: N={N} in {nb} batches of {B}, F={F} bf16, D={D}, K={K}, classes hv_bits={hv_bits} "
                   f"sim={sim_name}: hdc_encode_rp + hdc_classify per batch",
           "call_ms": call_ms, "queries_per_s": N / (call_ms * 1e-3)}
    if hv_bits != 1:
        ach = flops / (call_ms * 1e-3) / 1e12
        out["roofline"] = {"bound": "tensor", "achieved": ach, "peak": peaks["bf16_tflops_sustained"],
                           "unit": "TFLOP/s", "frac": ach / peaks["bf16_tflops_sustained"],
                           "peak_source": "bf16_tflops_sustained (measured); 2*D*(F+K) flop per query"}
    else:
        t_ideal = (2.0 * N * D * F / (peaks["bf16_tflops_sustained"] * 1e12)
                   + 2.0 * N * D * 1008 / (2.0 * peaks["bf16_tflops_sustained"] * 1e12))
        out["roofline"] = {"bound": "tensor", "achieved": N / (call_ms * 1e-3), "peak": N / t_ideal,
                           "unit": "queries/s", "frac": t_ideal / (call_ms * 1e-3),
                           "peak_source": "bf16 encode at bf16_tflops_sustained + +-1 int8 similarity at 2x that"}
    return out


def row_levelid_microhd(h, peaks, reps, N=131072, F=617, Q=128, D=1024):
    """The paper's Micro-HD-Classification reference shape (ISOLET F = 617, D = 1024,
    L = 128 levels): dense uniform levels, rows of 617 bytes (not word-aligned)."""
    if Q <= 256:
        lv = torch.randint(0, Q, (N, F), dtype=torch.uint8, device="cuda", generator=_gen(31))
    else:   # 16-bit level indices (hdc_encode_levelid_u16): L255 tunes the level count up to 814
        lv = torch.randint(0, Q, (N, F), dtype=torch.int16, device="cuda", generator=_gen(31))
    Wd = (D + 31) // 32
    ID = _rand_bits(F, Wd, 32)
    LV = _rand_bits(Q, Wd, 33)
    H = torch.empty((N, Wd), dtype=torch.int32, device="cuda")
    kn = hd.knobs(D)
    fn = lambda: h.hdc_encode_levelid(lv, ID, LV, D, kn, Hbits=H)  # noqa: E731
    call_ms = _time(fn, reps)
    ops = 3.0 * F * Wd * N
    ach = ops / (call_ms * 1e-3) / 1e12
    peak = 148 * 64 * peaks["sm_max_mhz"] * 1e6 / 1e12
    return {"what": f"hdc_encode_levelid N={N} F={F} Q={Q} D={D} (Micro-HD reference shape, dense levels)",
            "call_ms": call_ms, "samples_per_s": N / (call_ms * 1e-3),
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "Tlop/s (32-bit logic ops)",
                         "frac": ach / peak, "peak_source": "148 SM x 64 INT lanes x sm_max_mhz"}}


def row_c3_pipeline(h, peaks, reps, N=65536, F=784, Q=256, D=10000, K=10):
    """configs[2] inference: level-ID encode + packed Hamming classify against K = 10 classes."""
    from workloads import gen
    import numpy as np
    w = gen.c3_mnist_shaped(D=D, n_tr=16, n_te=4096, Q=Q)
    lv = torch.from_numpy(gen.tile_rows(w["Lte"], N)).cuda()
    ID = torch.from_numpy(gen.pack_bits_lsb(w["ID"]).view(np.int32)).cuda()
    LV = torch.from_numpy(gen.pack_bits_lsb(w["LV"]).view(np.int32)).cuda()
    H = torch.empty((N, (D + 31) // 32), dtype=torch.int32, device="cuda")
    C = _class_acc(K, D, 4)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")
    kn_e, kn = hd.knobs(D), hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)

    def fn():
        h.hdc_encode_levelid(lv, ID, LV, D, kn_e, Hbits=H)
        h.hdc_classify(H, C, kn, labels=lab)

    call_ms = _time(fn, reps)
    ops = 3.0 * F * ((D + 31) // 32) * N
    ach = ops / (call_ms * 1e-3) / 1e12
    peak = 148 * 64 * peaks["sm_max_mhz"] * 1e6 / 1e12
    return {"what": f"C3 inference: hdc_encode_levelid + hdc_classify (Hamming) N={N} F={F} Q={Q} D={D} K={K}",
            "call_ms": call_ms, "queries_per_s": N / (call_ms * 1e-3),
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "Tlop/s (32-bit logic ops)",
                         "frac": ach / peak, "peak_source": "148 SM x 64 INT lanes x sm_max_mhz; 3*F*W ops per query"}}


def c4_sweep(h, peaks, reps=5, NQ=131072):
    """configs[3]: D_eff x precision x retraining epochs on the HAR-shaped Gaussian mixture.  Per
    point: inference queries/s (encode at D_eff + classify, test set tiled to NQ), training
    samples/s of one retraining epoch, and the test accuracy after E = 0 / 5 / 20 epochs (accuracy
    parity with the oracle is the job of tests/test_gpu_configs.py)."""
    from workloads import gen
    import numpy as np
    w = gen.c4_har_shaped()
    D, K = w["D"], w["K"]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    Xtr, Xte, ytr, P = dev(w["Xtr"]), dev(w["Xte"]), dev(w["ytr"]), dev(w["P"])
    Xq = dev(gen.tile_rows(w["Xte"], NQ))
    yte = w["yte"]
    points = []
    precs = [("fp32", hd.HDC_F32, 32, hd.HDC_SIM_COS), ("bf16", hd.HDC_BF16, 16, hd.HDC_SIM_COS),
             ("int8", hd.HDC_I8, 8, hd.HDC_SIM_COS), ("1bit", hd.HDC_B1, 1, hd.HDC_SIM_HAMMING)]
    for name, prec, hv_bits, sim in precs:
        for D_eff in w["d_eff"]:
            kn_e = hd.knobs(D_eff, precision=prec)
            kn = hd.knobs(D_eff, precision=prec, hv_bits=hv_bits, sim=sim)
            Htr = h.hdc_encode_rp(Xtr, P, kn_e)
            Hte = h.hdc_encode_rp(Xte, P, kn_e)
            C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
            h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, ytr, C, kn)
            acc = {}
            done = 0
            for E in w["epochs"]:
                for _ in range(E - done):
                    h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, C, kn, lr=w["lr"], batch=0)
                done = E
                lab = h.hdc_classify(Hte, C, kn).cpu().numpy()
                acc[f"E{E}"] = float((lab == yte).mean())
            Ct = C.clone()
            ep_ms = _time(lambda: h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, Ct, kn, lr=w["lr"], batch=0),
                          reps)
            Hq = torch.empty((NQ, (D_eff + 31) // 32), dtype=torch.int32, device="cuda")
            lab_q = torch.empty(NQ, dtype=torch.int32, device="cuda")

            def infer():
                h.hdc_encode_rp(Xq, P, kn_e, Hbits=Hq)
                h.hdc_classify(Hq, C, kn, labels=lab_q)

            time.sleep(0.3)
            inf_ms = _time(infer, reps)
            points.append({"precision": name, "D_eff": D_eff, "queries_per_s": NQ / (inf_ms * 1e-3),
                           "train_samples_per_s": Xtr.shape[0] / (ep_ms * 1e-3), "accuracy": acc})
            del Hq, lab_q
            torch.cuda.empty_cache()
    return points


def adc_sweep(h, peaks, reps=5, NQ=131072):
    """SpecPCM-simulator knobs on the ISOLET-shaped mixture (D = 1024, TRAINING_ITER = 2, MLC = 1):
    test accuracy and queries/s of hdc_similarity_adc for the paper's ADC windows, beside the exact
    Hamming classify at the same D.  Accuracy parity with the oracle: tests/test_gpu_kernels.py."""
    from workloads import gen
    import numpy as np
    w = gen.c2_isolet_shaped()
    K, D = w["K"], w["D"]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    Xtr, Xte, ytr, P = dev(w["Xtr"]), dev(w["Xte"]), dev(w["ytr"]), dev(w["P"])
    yte = w["yte"]
    out = []
    for D_eff in (1024, 2048, 10000):
        kn_e = hd.knobs(D_eff, precision=hd.HDC_F32)
        kn = hd.knobs(D_eff, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
        Htr, Hte = h.hdc_encode_rp(Xtr, P, kn_e), h.hdc_encode_rp(Xte, P, kn_e)
        C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, ytr, C, kn)
        for _ in range(2):
            h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, C, kn, lr=w["lr"], batch=0)
        Hq = dev(gen.tile_rows(Hte.cpu().numpy(), NQ))
        lab = h.hdc_classify(Hte, C, kn).cpu().numpy()
        ms = _time(lambda: h.hdc_classify(Hq, C, kn), reps)
        out.append({"D_eff": D_eff, "similarity": "hamming (exact)", "accuracy": float((lab == yte).mean()),
                    "queries_per_s": NQ / (ms * 1e-3)})
        for res, step, fl, ce in [(8, 1, -127, 128), (8, 2, -3, 128), (6, 9, -3, 128), (4, 9, -3, 128), (2, 32, -3, 128)]:
            _, lab = h.hdc_similarity_adc(Hte, C, kn, res, step, fl, ce, want_scores=False)
            ms = _time(lambda: h.hdc_similarity_adc(Hq, C, kn, res, step, fl, ce, want_scores=False), reps)
            out.append({"D_eff": D_eff, "similarity": f"adc res={res} step={step} floor={fl} ceil={ce}",
                        "accuracy": float((lab.cpu().numpy() == yte).mean()), "queries_per_s": NQ / (ms * 1e-3)})
    return out


def row_kmeans(h, peaks, reps, N=7797, K=26, D=10000, hv_bits=32, sim_name="cos"):
    """HD-Clustering epoch (assign + re-bundle) on noisy copies of K prototypes, ISOLET-sized."""
    sim = {"cos": hd.HDC_SIM_COS, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    W = (D + 31) // 32
    proto = _rand_bits(K, W, 7)
    yt = torch.randint(0, K, (N,), device="cuda", generator=_gen(8))
    noise = _rand_bits(N, W, 9) & _rand_bits(N, W, 10) & _rand_bits(N, W, 11)      # ~12.5 % flipped bits
    H = (proto[yt] ^ noise).contiguous()
    C = _class_acc(K, D, 12, per_class=1)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    a = torch.empty(N, dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_train_epoch(hd.HDC_TRAIN_KMEANS, H, None, C, kn, pred=a)  # noqa: E731
    call_ms = _time(fn, reps)
    return {"what": f"hdc_train_epoch (k-means epoch) N={N} K={K} D={D} hv_bits={hv_bits} sim={sim_name}",
            "call_ms": call_ms, "samples_per_s": N / (call_ms * 1e-3)}


ROWS = {
    "c2_encode_f32": lambda h, p, r: row_encode(h, p, r, 131072, 617, 10000, "f32"),
    "c2_encode_f32_fast": lambda h, p, r: row_encode(h, p, r, 131072, 617, 10000, "f32_fast"),
    "c2_encode_bf16": lambda h, p, r: row_encode(h, p, r, 131072, 617, 10000, "bf16"),
    "c2_encode_f16": lambda h, p, r: row_encode(h, p, r, 131072, 617, 10000, "f16"),
    "c2_encode_i8": lambda h, p, r: row_encode(h, p, r, 131072, 617, 10000, "i8"),
    "c2_classify_cos32": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, 32, "cos"),
    "c4_classify_cos8": lambda h, p, r: row_classify(h, p, r, 131072, 6, 10000, 8, "cos"),
    "c3_levelid": lambda h, p, r: row_levelid(h, p, r),
    "c3_levelid_dense_input": lambda h, p, r: row_levelid(h, p, r, dense_input=True),
    "microhd_levelid": lambda h, p, r: row_levelid_microhd(h, p, r),
    "microhd_levelid_q814": lambda h, p, r: row_levelid_microhd(h, p, r, Q=814),
    "c3_hamming_k10": lambda h, p, r: row_classify(h, p, r, 131072, 10, 10000, 1, "hamming"),
    "c5_encode_bf16": lambda h, p, r: row_encode(h, p, r, 65536, 1024, 16384, "bf16", x_bf16=True),
    "c5_classify_bf16": lambda h, p, r: row_classify(h, p, r, 65536, 1000, 16384, 16, "cos"),
    "c5_classify_1bit": lambda h, p, r: row_classify(h, p, r, 65536, 1000, 16384, 1, "hamming"),
    "c3_pipeline": lambda h, p, r: row_c3_pipeline(h, p, r),
    "c5_stream_bf16": lambda h, p, r: row_c5_stream(h, p, r, 16, "cos"),
    "c5_stream_1bit": lambda h, p, r: row_c5_stream(h, p, r, 1, "hamming"),
    "specpcm_adc_d1024": lambda h, p, r: row_adc(h, p, r, 131072, 26, 1024),
    "specpcm_adc_d10000": lambda h, p, r: row_adc(h, p, r, 131072, 26, 10000),
    "c2_train_epoch": lambda h, p, r: row_train(h, p, r),
    "c2_kmeans_epoch": lambda h, p, r: row_kmeans(h, p, r),
}


def run(h, peaks, reps=5, only=None):
    out = {}
    for name, fn in ROWS.items():
        if only and name != only:
            continue
        time.sleep(1.0)   # let the part cool between rows: each row is a burst measurement of its own
        out[name] = fn(h, peaks, reps)
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--row", default=None, choices=sorted(ROWS))
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--c4-sweep", action="store_true", help="configs[3]: D_eff x precision x epochs table")
    ap.add_argument("--adc-sweep", action="store_true", help="SpecPCM ADC windows (PAPER.md L273): accuracy, queries/s")
    a = ap.parse_args()
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        with open(pk) as f:
            peaks = json.load(f)
    else:  # the profiling guide's fallback figures
        peaks = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}
    torch.cuda.set_device(0)
    h = hd.Handle(0)
    if a.c4_sweep:
        for pt in c4_sweep(h, peaks, a.reps):
            print(json.dumps({"c4_sweep": pt}), flush=True)
        h.close()
        return
    if a.adc_sweep:
        for pt in adc_sweep(h, peaks, a.reps):
            print(json.dumps({"adc_sweep": pt}), flush=True)
        h.close()
        return
    res = run(h, peaks, a.reps, a.row)
    for k, v in res.items():
        print(json.dumps({k: v}), flush=True)
    h.close()


if __name__ == "__main__":
    main()
