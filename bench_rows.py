"""Per-row measurements of the hot path beyond bench.py's headline step:
each row times one entry point of the C ABI on device-resident, SEEDED synthetic inputs drawn by
workloads/gen.py with the shapes of BASELINE.json's configs, with CUDA events around the calls and the
library's own per-kernel events (hdc_kernel_time) for the dominant kernel, samples the SM clock during
its timed region (ClockSampler), and states the roofline it is held against.

    python bench_rows.py [--row NAME] [--reps R]      (also the command of the ncu captures under profiles/)

`bench.py` folds DEFAULT_ROWS into its JSON line on every run (so the driver's record carries them) and
all of ROWS with `--rows`.  No arithmetic of the method lives here and nothing under oracle/ is imported:
the oracle-timed baselines beside these rows are bench.py's cpu_baseline leg.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_2606_26547_b200 as hd  # noqa: E402
from workloads import gen  # noqa: E402

SM_COUNT = 148


def load_peaks():
    """MEASURED_PEAKS.json (driver-written, this pool's B200s) or the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "sm_max_mhz": 1965.0, "_source": "fallback"}


def sustained_clock_mhz(peaks):
    """SM clock at which the driver measured bf16_tflops_sustained (1300 MHz: the guide's figure)."""
    return float((peaks.get("clocks_under_load") or {}).get("sm_mhz_median") or 1300.0)


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while a timed region runs."""

    def __init__(self, index: int = 0):
        self.ok = False
        self.samples, self.reasons = [], set()
        self._stop = threading.Event()
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.max_mhz = None

    def _run(self):
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev))
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop.wait(0.004)

    def __enter__(self):
        if self.ok:
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *a):
        if self.ok:
            self._stop.set()
            self.t.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


_CLOCKS = {}          # clocks of the last _time() call, picked up by run()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _bits(b):
    return _dev(gen.pack_bits_lsb(b).view(np.int32))


def _time(fn, reps, warm=3):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(torch.cuda.current_device()) as cs:
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
    _CLOCKS["last"] = cs.summary()
    return a.elapsed_time(b) / reps


def _kernel(h, kid, fn, reps):
    h.kernel_timing(True)
    for _ in range(reps):
        fn()
    torch.cuda.synchronize()
    ms, n = h.kernel_time(kid)
    h.kernel_timing(False)
    return ms / max(1, n), n // max(1, reps)


def _rand_bits(n, w, name):
    """[n][w] packed words of iid uniform bits from the seeded stream (0, name), in rows of w rounded up to 4 words
    (16-byte aligned rows: the layout Handle.alloc_hbits gives the hypervectors hdc_encode_* write)."""
    ld = (w + 3) // 4 * 4
    host = np.zeros((n, ld), dtype=np.uint32)
    host[:, :w] = gen.rng_for(0, name).integers(0, 2 ** 32, size=(n, w), dtype=np.uint32)
    return _dev(host.view(np.int32))[:, :w]


def _class_acc(K, D, name, per_class=32):
    """Accumulators shaped like a bundle of `per_class` bipolar hypervectors per class (exact ints)."""
    ones = gen.rng_for(0, name).binomial(per_class, 0.5, size=(K, D))
    return _dev((per_class - 2 * ones).astype(np.float32))


def _c2():
    if "c2" not in _CACHE:
        _CACHE["c2"] = gen.c2_isolet_shaped()
    return _CACHE["c2"]


def _c4():
    if "c4" not in _CACHE:
        _CACHE["c4"] = gen.c4_har_shaped()
    return _CACHE["c4"]


_CACHE = {}


# ------------------------------------------------------------------------------------ encode rows
def row_encode(h, peaks, reps, cfg, N, prec_name):
    """hdc_encode_rp on the C2 / C4 test set tiled to N rows (fp32 inputs) or one C5 batch (bf16 inputs)."""
    flags = 0
    if prec_name == "f32_fast":   # HDC_FLAG_F32_FAST: 2-way half splits, three products
        flags = hd.HDC_FLAG_F32_FAST
    prec = {"f32": hd.HDC_F32, "f32_fast": hd.HDC_F32, "bf16": hd.HDC_BF16, "f16": hd.HDC_F16,
            "i8": hd.HDC_I8}[prec_name]
    if cfg == "c5":
        w = gen.c5_large_batch(N, batch=0, per_class=1)
        X, P = _dev(w["X"]).to(torch.bfloat16), _dev(w["P"]).to(torch.bfloat16)
    else:
        w = _c2() if cfg == "c2" else _c4()
        X, P = _dev(gen.tile_rows(w["Xte"], N)), _dev(w["P"])
    F, D = X.shape[1], P.shape[0]
    kn = hd.knobs(D, precision=prec, flags=flags)
    H = h.alloc_hbits(N, D)
    fn = lambda: h.hdc_encode_rp(X, P, kn, Hbits=H)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_ENCODE_GEMM, fn, reps)
    flops = 2.0 * N * F * D
    mult = {"f32": 1.0 / 6.0, "f32_fast": 1.0 / 3.0, "bf16": 1.0, "f16": 1.0, "i8": 2.0}[prec_name]
    peak = peaks["bf16_tflops"] * mult
    ach = flops / (k_ms * 1e-3) / 1e12
    return {"what": f"hdc_encode_rp {cfg.upper()}-shaped N={N} F={F} D={D} precision={prec_name}"
                    + (" (bf16 inputs in place)" if cfg == "c5" else " (fp32 inputs, staging pass inside call_ms)"),
            "call_ms": call_ms, "kernel_ms": k_ms, "queries_per_s": N / (call_ms * 1e-3),
            "roofline": {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "peak_source": f"bf16_tflops (burst, {peaks.get('_source', 'measured')}) x {mult:.4g}; contraction kernel"}}


def row_point(h, peaks, reps, cfg, N, prec_name):
    """One precision point end to end (encode + classify, SURVEY.md 8(d) rows 'C2 bf16', 'C4 bf16 / int8' at
    D_eff = 10000): queries/s against 2*D*(F+K) flop per query at the tensor peak of the precision."""
    w = _c2() if cfg == "c2" else _c4()
    prec, hv, mult = {"bf16": (hd.HDC_BF16, 16, 1.0), "i8": (hd.HDC_I8, 8, 2.0)}[prec_name]
    D, K, F = w["D"], w["K"], w["F"]
    X, P = _dev(gen.tile_rows(w["Xte"], N)), _dev(w["P"])
    kn_e = hd.knobs(D, precision=prec)
    kn = hd.knobs(D, precision=prec, hv_bits=hv, sim=hd.HDC_SIM_COS)
    Htr = h.hdc_encode_rp(_dev(w["Xtr"]), P, kn_e)
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, _dev(w["ytr"]), C, kn)
    H = h.alloc_hbits(N, D)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")

    def fn():
        h.hdc_encode_rp(X, P, kn_e, Hbits=H)
        h.hdc_classify(H, C, kn, labels=lab)

    call_ms = _time(fn, reps)
    enc_ms, _ = _kernel(h, hd.HDC_K_ENCODE_GEMM, fn, reps)
    sim_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, reps)
    qps = N / (call_ms * 1e-3)
    peak_qps = peaks["bf16_tflops_sustained"] * mult * 1e12 / (2.0 * D * (F + K))
    n_te = w["Xte"].shape[0]
    return {"what": f"{cfg.upper()} precision point {prec_name}: hdc_encode_rp + hdc_classify (cosine, hv_bits={hv}) "
                    f"N={N} F={F} D_eff={D} K={K}",
            "call_ms": call_ms, "encode_kernel_ms": enc_ms, "classify_kernel_ms": sim_ms, "queries_per_s": qps,
            "test_accuracy": float((lab[:n_te].cpu().numpy() == w["yte"]).mean()),
            "roofline": {"bound": "tensor", "achieved": qps, "peak": peak_qps, "unit": "queries/s",
                         "frac": qps / peak_qps,
                         "peak_source": f"bf16_tflops_sustained x {mult:.3g} / (2*D*(F+K) flop per query) "
                                        "(SURVEY.md 8(d); whole call incl. staging)"}}


# ------------------------------------------------------------------------------------ similarity rows
def row_classify(h, peaks, reps, N, K, D, hv_bits, sim_name, flags=0, acc_scale=None):
    """acc_scale: multiplies the bundle-shaped accumulators (|c| <= 32) -- 32- / 64-bit integer classes whose every
    16-bit piece holds nonzero codes (without it only the lowest piece does and the others are skipped)."""
    sim = {"cos": hd.HDC_SIM_COS, "dot": hd.HDC_SIM_DOT, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    W = (D + 31) // 32
    H = _rand_bits(N, W, "rows_query_bits")
    C = _class_acc(K, D, "rows_class_acc")
    if isinstance(acc_scale, (list, tuple)):   # one scale per class, cycling (an fp32 value spans at most 24 bits)
        sc = torch.tensor([float(acc_scale[k % len(acc_scale)]) for k in range(K)], device=C.device)
        C = C * sc[:, None]
    elif acc_scale is not None:
        C = C * float(acc_scale)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim, flags=flags)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_classify(H, C, kn, labels=lab)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, reps)
    out = {"what": f"hdc_classify N={N} K={K} D={D} hv_bits={hv_bits} sim={sim_name}"
                   + (f" accumulators x {acc_scale} (every 16-bit piece live)" if acc_scale is not None else ""),
           "call_ms": call_ms,
           "kernel_ms": k_ms, "queries_per_s": N / (call_ms * 1e-3)}
    hbm = N * W * 4 / (k_ms * 1e-3) / 1e9
    out["hbm_GBps_query_bits"] = hbm
    if sim_name == "hamming" and K < 64:
        popc = float(N) * K * W / (k_ms * 1e-3) / 1e12
        peak = 148 * 16 * peaks["sm_max_mhz"] * 1e6 / 1e12
        out["roofline"] = {"bound": "alu", "achieved": popc, "peak": peak, "unit": "Tpopc/s", "frac": popc / peak,
                           "peak_source": "148 SM x 16 POPC lanes x sm_max_mhz"}
    elif hv_bits in (hd.HDC_HV_I32, hd.HDC_HV_I64) and (flags & hd.HDC_FLAG_SIMT):
        # widedot.cu: one dp4a per (query, class, 4 dimensions, byte plane of the codes); the integer dot-product
        # instruction issues at 64 lanes per clock and SM (measured: DESIGN.md section 6)
        planes = 4 if hv_bits == hd.HDC_HV_I32 else 8
        dp4a = float(N) * K * ((D + 3) // 4) * planes / (k_ms * 1e-3) / 1e12
        peak = 148 * 64 * peaks["sm_max_mhz"] * 1e6 / 1e12
        out["roofline"] = {"bound": "alu", "achieved": dp4a, "peak": peak, "unit": "Tdp4a/s", "frac": dp4a / peak,
                           "peak_source": "148 SM x 64 dp4a lanes x sm_max_mhz"}
    else:
        # (32- / 64-bit integer codes: two / four 16-bit pieces, each three base-128 digits on kind::i8; kernel_ms
        # spans the pieces' contractions and the 64-bit recombination)
        parts = {32: 3, hd.HDC_HV_I16: 3, hd.HDC_HV_I32: 6, hd.HDC_HV_I64: 12}.get(hv_bits, 1)
        mult = 2.0 if hv_bits in (hd.HDC_HV_I16, hd.HDC_HV_I32, hd.HDC_HV_I64, 8, 1) else 1.0
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
    H = _rand_bits(N, W, "rows_query_bits")
    C = _class_acc(K, D, "rows_class_acc")
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
    w = gen.c3_mnist_shaped(D=D, n_tr=16, n_te=4096, Q=Q)
    lv = _dev(gen.tile_rows(w["Lte"], N))
    if dense_input:  # uniformly random levels: no zeros to skip, every warp takes the dense path
        lv = _dev(gen.rng_for(3, "rows_dense_levels").integers(0, Q, size=(N, F), dtype=np.uint8))
    ID, LV = _bits(w["ID"]), _bits(w["LV"])
    Wd = (D + 31) // 32
    H = h.alloc_hbits(N, D)
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
    H = _rand_bits(N, W, "rows_train_bits")
    y = _dev(gen.rng_for(0, "rows_train_y").integers(0, K, size=N).astype(np.int32))
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


def _c5_setup(h, nbatches, B, D, K, F):
    """C5 inputs (workloads/gen.py recipe): `nbatches` device-resident bf16 query batches, bf16 P, and class
    accumulators = bundle of 32 encoded noisy samples per class (through the library)."""
    key = ("c5", nbatches, B, D, K, F)
    if key not in _CACHE:
        w0 = gen.c5_large_batch(B, batch=0, D=D, K=K, F=F)
        Xs = [_dev(w0["X"]).to(torch.bfloat16)]
        for i in range(1, nbatches):
            Xs.append(_dev(gen.c5_large_batch(B, batch=i, D=D, K=K, F=F, per_class=1)["X"]).to(torch.bfloat16))
        P = _dev(w0["P"]).to(torch.bfloat16)
        kn_e = hd.knobs(D, precision=hd.HDC_BF16)
        Htr = h.hdc_encode_rp(_dev(w0["Xtr"]).to(torch.bfloat16), P, kn_e)
        C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
        h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, _dev(w0["ytr"]), C, hd.knobs(D))
        _CACHE.clear()          # one large set resident at a time
        _CACHE[key] = (Xs, P, C, w0["y"])
    return _CACHE[key]


def row_c5_stream(h, peaks, reps, hv_bits, sim_name, N=1 << 20, B=65536, F=1024, D=16384, K=1000):
    """BASELINE.json configs[4]: N = 2^20 bf16 queries streamed in 64K-query device-resident batches
    through hdc_encode_rp (bf16) + hdc_classify against K = 1000 classes (bf16 cosine or packed 1-bit
    Hamming).  Four distinct seeded input batches (537 MB > L2) are cycled over the 16 batches."""
    sim = {"cos": hd.HDC_SIM_COS, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    nb = N // B
    Xs, P, C, y0 = _c5_setup(h, 4, B, D, K, F)
    kn_e = hd.knobs(D, precision=hd.HDC_BF16)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    H = h.alloc_hbits(B, D)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")

    def fn():
        for i in range(nb):
            h.hdc_encode_rp(Xs[i & 3], P, kn_e, Hbits=H)
            h.hdc_classify(H, C, kn, labels=lab[i * B:(i + 1) * B])

    call_ms = _time(fn, max(1, reps // 5), warm=1)
    enc_ms, _ = _kernel(h, hd.HDC_K_ENCODE_GEMM, fn, 1)
    sim_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, 1)
    flops = 2.0 * N * D * (F + (K if hv_bits != 1 else 0))
    out = {"what": f"C5 stream: N={N} in {nb} batches of {B}, F={F} bf16, D={D}, K={K}, classes hv_bits={hv_bits} "
                   f"sim={sim_name}: hdc_encode_rp + hdc_classify per batch",
           "call_ms": call_ms, "queries_per_s": N / (call_ms * 1e-3),
           "encode_kernel_ms_per_batch": enc_ms, "classify_kernel_ms_per_batch": sim_ms,
           "accuracy_batch0": float((lab[:B].cpu().numpy() == y0).mean())}
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


def row_c5_classify(h, peaks, reps, hv_bits, sim_name, B=65536, F=1024, D=16384, K=1000):
    """hdc_classify of one ENCODED C5 batch (the hypervectors of seeded batch 0) against the K = 1000 classes."""
    sim = {"cos": hd.HDC_SIM_COS, "hamming": hd.HDC_SIM_HAMMING}[sim_name]
    Xs, P, C, y0 = _c5_setup(h, 4, B, D, K, F)
    H = h.hdc_encode_rp(Xs[0], P, hd.knobs(D, precision=hd.HDC_BF16))
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    lab = torch.empty(B, dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_classify(H, C, kn, labels=lab)  # noqa: E731
    call_ms = _time(fn, reps)
    k_ms, _ = _kernel(h, hd.HDC_K_SIM, fn, reps)
    # int16 class codes (hv code 18): algorithmic flops 2*B*D*K against the int8 tensor peak; the kernel executes
    # three int8 digit columns per class, so a third of that peak is its ceiling
    # (32-bit integer codes, hv code 19: two 16-bit pieces = six digit columns per class, a sixth of that peak)
    mult = 2.0 if hv_bits in (hd.HDC_HV_I16, hd.HDC_HV_I32, hd.HDC_HV_I64, 8, 1) else 1.0
    flops = 2.0 * B * D * (((K + 15) // 16) * 16)
    ach = flops / (k_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops"] * mult
    return {"what": f"hdc_classify of one encoded C5 batch N={B} K={K} D={D} hv_bits={hv_bits} sim={sim_name}",
            "call_ms": call_ms, "kernel_ms": k_ms, "queries_per_s": B / (call_ms * 1e-3),
            "accuracy": float((lab.cpu().numpy() == y0).mean()),
            "roofline": {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "peak_source": f"bf16_tflops (burst, measured) x {mult:.3g}"}}


def row_levelid_microhd(h, peaks, reps, N=131072, F=617, Q=128, D=1024):
    """The paper's Micro-HD-Classification reference shape (ISOLET F = 617, D = 1024,
    L = 128 levels): dense uniform levels, rows of 617 bytes (not word-aligned)."""
    lv = gen.rng_for(0, "rows_microhd_levels").integers(0, Q, size=(N, F), dtype=np.uint8 if Q <= 256 else np.int16)
    lv = _dev(lv)    # Q > 256: 16-bit level indices (hdc_encode_levelid_u16): L255 tunes the level count up to 814
    Wd = (D + 31) // 32
    ID, LV = _bits(gen.id_table(0, F, D)), _bits(gen.level_table(0, Q, D))
    H = h.alloc_hbits(N, D)
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
    w = gen.c3_mnist_shaped(D=D, n_tr=16, n_te=4096, Q=Q)
    lv = _dev(gen.tile_rows(w["Lte"], N))
    ID, LV = _bits(w["ID"]), _bits(w["LV"])
    H = h.alloc_hbits(N, D)
    C = _class_acc(K, D, "rows_class_acc")
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
            Hq = h.alloc_hbits(NQ, D_eff)
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
    proto = _rand_bits(K, W, "rows_km_proto")
    yt = _dev(gen.rng_for(0, "rows_km_y").integers(0, K, size=N))
    noise = _rand_bits(N, W, "rows_km_n1") & _rand_bits(N, W, "rows_km_n2") & _rand_bits(N, W, "rows_km_n3")  # ~12.5 % flipped bits
    H = (proto[yt] ^ noise).contiguous()
    C = _class_acc(K, D, "rows_km_seed", per_class=1)
    kn = hd.knobs(D, hv_bits=hv_bits, sim=sim)
    a = torch.empty(N, dtype=torch.int32, device="cuda")
    fn = lambda: h.hdc_train_epoch(hd.HDC_TRAIN_KMEANS, H, None, C, kn, pred=a)  # noqa: E731
    call_ms = _time(fn, reps)
    return {"what": f"hdc_train_epoch (k-means epoch) N={N} K={K} D={D} hv_bits={hv_bits} sim={sim_name}",
            "call_ms": call_ms, "samples_per_s": N / (call_ms * 1e-3)}


ROWS = {
    "c2_encode_f32": lambda h, p, r: row_encode(h, p, r, "c2", 131072, "f32"),
    "c2_encode_f32_fast": lambda h, p, r: row_encode(h, p, r, "c2", 131072, "f32_fast"),
    "c2_encode_bf16": lambda h, p, r: row_encode(h, p, r, "c2", 131072, "bf16"),
    "c2_encode_f16": lambda h, p, r: row_encode(h, p, r, "c2", 131072, "f16"),
    "c2_encode_i8": lambda h, p, r: row_encode(h, p, r, "c2", 131072, "i8"),
    "c2_point_bf16": lambda h, p, r: row_point(h, p, r, "c2", 131072, "bf16"),
    "c4_point_bf16": lambda h, p, r: row_point(h, p, r, "c4", 131072, "bf16"),
    "c4_point_i8": lambda h, p, r: row_point(h, p, r, "c4", 131072, "i8"),
    "c2_classify_cos32": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, 32, "cos"),
    "c4_classify_cos8": lambda h, p, r: row_classify(h, p, r, 131072, 6, 10000, 8, "cos"),
    "c3_levelid": lambda h, p, r: row_levelid(h, p, r),
    "c3_levelid_dense_input": lambda h, p, r: row_levelid(h, p, r, dense_input=True),
    "microhd_levelid": lambda h, p, r: row_levelid_microhd(h, p, r),
    "microhd_levelid_q814": lambda h, p, r: row_levelid_microhd(h, p, r, Q=814),
    "c3_hamming_k10": lambda h, p, r: row_classify(h, p, r, 131072, 10, 10000, 1, "hamming"),
    "c3_pipeline": lambda h, p, r: row_c3_pipeline(h, p, r),
    "c5_encode_bf16": lambda h, p, r: row_encode(h, p, r, "c5", 65536, "bf16"),
    "c5_classify_bf16": lambda h, p, r: row_c5_classify(h, p, r, 16, "cos"),
    "c5_classify_1bit": lambda h, p, r: row_c5_classify(h, p, r, 1, "hamming"),
    "c5_classify_i8": lambda h, p, r: row_c5_classify(h, p, r, 8, "cos"),
    "c5_classify_i16": lambda h, p, r: row_c5_classify(h, p, r, hd.HDC_HV_I16, "cos"),
    "c2_classify_cos_i16": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I16, "cos"),
    "c2_classify_cos_i32": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I32, "cos"),
    "c2_classify_dot_i64": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I64, "dot"),
    "c2_classify_cos_i32_full": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I32, "cos", acc_scale=6.0e7),
    "c2_classify_dot_i64_full": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I64, "dot",
                                                                 acc_scale=(1.0, 2.0 ** 16, 2.0 ** 32, 2.0 ** 44)),
    "c2_classify_cos_i32_dp4a": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I32, "cos", hd.HDC_FLAG_SIMT),
    "c2_classify_dot_i64_dp4a": lambda h, p, r: row_classify(h, p, r, 131072, 26, 10000, hd.HDC_HV_I64, "dot", hd.HDC_FLAG_SIMT),
    "c5_classify_i32": lambda h, p, r: row_c5_classify(h, p, r, hd.HDC_HV_I32, "cos"),
    "c5_stream_bf16": lambda h, p, r: row_c5_stream(h, p, r, 16, "cos"),
    "c5_stream_1bit": lambda h, p, r: row_c5_stream(h, p, r, 1, "hamming"),
    "specpcm_adc_d1024": lambda h, p, r: row_adc(h, p, r, 131072, 26, 1024),
    "specpcm_adc_d10000": lambda h, p, r: row_adc(h, p, r, 131072, 26, 10000),
    "c2_train_epoch": lambda h, p, r: row_train(h, p, r),
    "c2_kmeans_epoch": lambda h, p, r: row_kmeans(h, p, r),
}

# the rows bench.py folds into its default JSON line (every run; about a minute on one B200)
DEFAULT_ROWS = ("c2_encode_bf16", "c2_encode_i8", "c4_point_bf16", "c4_point_i8", "c2_classify_cos32",
                "c3_levelid", "c3_levelid_dense_input", "microhd_levelid_q814", "c3_hamming_k10", "c3_pipeline",
                "c5_classify_bf16", "c5_classify_1bit", "c5_stream_bf16", "c5_stream_1bit", "c2_train_epoch",
                "c2_classify_cos_i32")


def run(h, peaks, reps=5, only=None, cool_s=0.5):
    """only: None = every row, a name, or a collection of names.  Every row carries the SM clock sampled
    during its (last) timed region."""
    if isinstance(only, str):
        only = (only,)
    out = {}
    for name, fn in ROWS.items():
        if only is not None and name not in only:
            continue
        time.sleep(cool_s)   # let the part cool between rows: each row is a burst measurement of its own
        t0 = time.perf_counter()
        _CLOCKS.pop("last", None)
        row = fn(h, peaks, reps)
        row["clocks"] = _CLOCKS.get("last")
        row["wall_s"] = round(time.perf_counter() - t0, 2)
        out[name] = row
        torch.cuda.empty_cache()
    _CACHE.clear()
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--row", default=None, choices=sorted(ROWS))
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--c4-sweep", action="store_true", help="configs[3]: D_eff x precision x epochs table")
    ap.add_argument("--adc-sweep", action="store_true", help="SpecPCM ADC windows (PAPER.md L273): accuracy, queries/s")
    a = ap.parse_args()
    peaks = load_peaks()
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
