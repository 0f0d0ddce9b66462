"""bench.py -- HDC inference queries/s (encode + similarity + argmax) at D=10000 on B200.

Headline workload = BASELINE.json configs[1] ("C2", ISOLET-shaped): F=617 fp32 features, K=26,
D=10000 fp32 Gaussian random projection, cosine similarity against class hypervectors trained by
bundling + 20 retraining epochs (lr 0.05); the 1559-query test set is tiled to 131072 queries per
step so that the timed inputs (323 MB) exceed L2.  One step = hdc_encode_rp + hdc_classify over
that batch, through the C ABI.  Synthetic seeded data (workloads/gen.py) stands in for ISOLET.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--rows]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/hdc_oracle.py, as
it stands) on the host cores for the same metric / config.  `--rows` adds per-row measurements of
the other hot-path steps (level-ID encode, Hamming, training, bf16 / int8 precisions).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hdc_inference_queries_per_sec_D10000"
UNIT = "queries/s"
NQ = 131072            # queries per step (test set tiled)
NCU_TRAFFIC_BYTES = 804.4e6
NCU_TRAFFIC_SOURCE = "profiles/r1_final_kernels.md (gemm_tc_kernel, fp32-precision encode, 131072 x 617 x 10000)"
SM_COUNT = 148
FP32_LANES = 128       # FFMA lanes per SM per clock


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "sm_max_mhz": 1965.0, "_source": "fallback"}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
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


def c2_workload(world: int = 1, rank: int = 0):
    """C2 model inputs + this rank's shard of the query stream: the test set tiled to world*NQ rows,
    split by shard.shard_bounds (contiguous blocks, NQ rows per rank: weak scaling)."""
    from workloads import gen
    from paper_2606_26547_b200 import shard
    w = gen.c2_isolet_shaped()
    lo, hi = shard.shard_bounds(world * NQ, world, rank)
    n_te = w["Xte"].shape[0]
    idx = np.arange(lo, hi) % n_te
    Xq = np.ascontiguousarray(w["Xte"][idx])
    return w, Xq


# ------------------------------------------------------------------------------------ reference arm
def oracle_infer(O, X, P, C_acc, D):
    bits, _, _ = O.encode_rp(X, P, D, O.F32)
    lab, _, _, _ = O.infer(bits, C_acc, D, O.SIM_COS, 32)
    return lab


def oracle_model(O, w, n_train=1024):
    """Class accumulators for the timing legs of the oracle (bundle of a training subset; the
    timed work -- encode + cosine + argmax -- does not depend on how well the model is trained)."""
    btr, _, _ = O.encode_rp(w["Xtr"][:n_train], w["P"], w["D"], O.F32)
    return O.bundle(btr, w["ytr"][:n_train], w["K"], w["D"])


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import hdc_oracle as O
    w, Xq = c2_workload()
    C = oracle_model(O, w)
    sample = 16384
    X = Xq[:sample]
    for _ in range(max(1, args.warmup) if args.warmup else 0):
        oracle_infer(O, X[:256], w["P"], C, w["D"])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_infer(O, X, w["P"], C, w["D"])
    dt = time.perf_counter() - t0
    val = sample * args.steps / dt
    cores = os.cpu_count()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "C2 ISOLET-shaped: F=617 fp32, K=26, D=10000 RP encode + cosine + argmax",
                       "queries_per_step": sample, "timing": "host wall clock"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{sample} queries of the tiled C2 test set per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ own arm
def run_gpu(args):
    import torch
    import torch.distributed as dist

    import paper_2606_26547_b200 as hd
    from paper_2606_26547_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = load_peaks()
    h = hd.Handle(local)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731

    w, Xq = c2_workload(world, rank)
    D, K, F = w["D"], w["K"], w["F"]
    Pd = dev(w["P"])
    kn_e = hd.knobs(D, precision=hd.HDC_F32)
    kn = hd.knobs(D, precision=hd.HDC_F32, hv_bits=32, sim=hd.HDC_SIM_COS)

    # ---- model: encode train, bundle, 20 retraining epochs (setup; also timed as training rows)
    Xtr, ytr = dev(w["Xtr"]), dev(w["ytr"])
    Htr = h.hdc_encode_rp(Xtr, Pd, kn_e)
    C = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, ytr, C, kn)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    torch.cuda.synchronize()
    ev[0].record()
    for _ in range(w["epochs"]):
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, C, kn, lr=w["lr"], batch=0)
    ev[1].record()
    torch.cuda.synchronize()
    train_ms = ev[0].elapsed_time(ev[1])
    train_sps = w["epochs"] * Xtr.shape[0] / (train_ms * 1e-3)

    # ---- timed inference steps (device-resident inputs)
    Xd = dev(Xq)
    W = (D + 31) // 32
    Hq = torch.empty((NQ, W), dtype=torch.int32, device="cuda")
    labels = torch.empty(NQ, dtype=torch.int32, device="cuda")

    def step():
        h.hdc_encode_rp(Xd, Pd, kn_e, Hbits=Hq)
        h.hdc_classify(Hq, C, kn, labels=labels)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    l0 = h.launch_count()
    with ClockSampler(local) as cs:
        ev[0].record()
        for _ in range(args.steps):
            step()
        ev[1].record()
        torch.cuda.synchronize()
    launches = h.launch_count() - l0
    ms = ev[0].elapsed_time(ev[1])
    if world > 1:
        dist.barrier()
    ms = shard.max_over_ranks(ms, torch.device("cuda", local))
    value = world * NQ * args.steps / (ms * 1e-3)
    n_te = w["Xte"].shape[0]
    acc = float((labels[:n_te].cpu().numpy() == w["yte"][np.arange(rank * NQ, rank * NQ + n_te) % n_te]).mean())

    # ---- dominant kernel: the encode contraction.  Its launches are bracketed by CUDA events
    # inside the library (hdc_kernel_timing) on the stream they are launched on; measured (a) over a
    # re-run of the timed steps (sustained regime) and (b) alone, back to back (burst regime).
    h.kernel_timing(True)
    torch.cuda.synchronize()
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    enc_ms_tot, enc_n = h.kernel_time(hd.HDC_K_ENCODE_GEMM)
    sim_ms_tot, sim_n = h.kernel_time(hd.HDC_K_SIM)
    enc_ms = enc_ms_tot / max(1, enc_n)
    cls_ms = sim_ms_tot / max(1, sim_n)
    reps = max(3, args.steps)
    ev[0].record()
    for _ in range(reps):
        h.hdc_encode_rp(Xd, Pd, kn_e, Hbits=Hq)
    ev[1].record()
    torch.cuda.synchronize()
    enc_call_ms = ev[0].elapsed_time(ev[1]) / reps
    enc_alone_tot, enc_alone_n = h.kernel_time(hd.HDC_K_ENCODE_GEMM)
    enc_alone_ms = enc_alone_tot / max(1, enc_alone_n)
    h.kernel_timing(False)
    # fp32-precision contraction on tensor cores = six bf16 products per fp32 MAC:
    # algorithmic flops are the fp32 ones, the peak is the measured bf16 peak / 6.
    flops = 2.0 * NQ * F * D
    achieved = flops / (enc_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops_sustained"] / 6.0
    clocks = cs.summary()
    roofline = {"bound": "tensor",
                "kernel": "gemm_tc_kernel<bf16,EPI_SIGN,cta_group::2> (tcgen05 fp32-precision encode on CTA pairs: 6 "
                          "bf16 segment products per MAC over 3-way split operands, sign+pack epilogue)",
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": f"bf16_tflops_sustained / 6 ({peaks['_source']} MEASURED_PEAKS.json; kernel timed "
                               "inside the step loop)",
                "algorithmic_flops_per_launch": flops, "ms_per_launch": enc_ms,
                "executed_bf16_tflops": 6.0 * 2.0 * NQ * 640 * D / (enc_ms * 1e-3) / 1e12,
                "alone": {"ms_per_launch": enc_alone_ms, "achieved": flops / (enc_alone_ms * 1e-3) / 1e12,
                          "peak": peaks["bf16_tflops"] / 6.0,
                          "frac": flops / (enc_alone_ms * 1e-3) / 1e12 / (peaks["bf16_tflops"] / 6.0),
                          "peak_source": "bf16_tflops (burst) / 6"},
                "encode_call_ms": enc_call_ms, "classify_kernel_ms": cls_ms,
                "share_of_step": enc_ms / (ms / args.steps),
                "fp32_alu_peak_tflops": SM_COUNT * FP32_LANES * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12,
                # dram__bytes_read.sum + dram__bytes_write.sum of this kernel at this shape, one launch, from
                # the ncu --set full capture summarised in profiles/ (bytes)
                "traffic": NCU_TRAFFIC_BYTES, "traffic_source": NCU_TRAFFIC_SOURCE,
                "algorithmic_bytes_per_launch": float(NQ) * 3 * 640 * 2 + float(D) * 3 * 640 * 2 + float(NQ) * W * 4}

    # ---- NOT the headline: the same step with the opt-in HDC_FLAG_F32_FAST encode (fp32 operands as 2-way
    # IEEE-half splits, 22 mantissa bits, three tensor-core products instead of six).  Reported beside the
    # headline so that the cost of the last two operand bits is on record; `value` above never uses it.
    kn_fast = hd.knobs(D, precision=hd.HDC_F32, flags=hd.HDC_FLAG_F32_FAST)
    labels_fast = torch.empty(NQ, dtype=torch.int32, device="cuda")

    def step_fast():
        h.hdc_encode_rp(Xd, Pd, kn_fast, Hbits=Hq)
        h.hdc_classify(Hq, C, kn, labels=labels_fast)

    for _ in range(3):
        step_fast()
    torch.cuda.synchronize()
    ev[0].record()
    for _ in range(args.steps):
        step_fast()
    ev[1].record()
    torch.cuda.synchronize()
    fast_ms = ev[0].elapsed_time(ev[1]) / args.steps
    f32_fast = {"queries_per_s_per_gpu": NQ / (fast_ms * 1e-3), "ms_per_step": fast_ms,
                "labels_differing_from_headline_path": int((labels_fast != labels).sum().item()),
                "what": "same step with knobs.flags = HDC_FLAG_F32_FAST (opt-in; 22-bit operands, 3 products); "
                        "not the headline value"}
    h.hdc_encode_rp(Xd, Pd, kn_e, Hbits=Hq)                  # leave Hq / labels as the headline path wrote them
    h.hdc_classify(Hq, C, kn, labels=labels)

    # ---- fingerprint of the seeded inputs (a run is reproducible even if the RNG library changes)
    import hashlib
    hsh = hashlib.sha256()
    for a in (w["Xte"], w["yte"], w["Xtr"], w["ytr"], w["P"]):
        hsh.update(np.ascontiguousarray(a).tobytes())
    inputs_sha = hsh.hexdigest()[:16]

    # ---- single-pass latency at the true test-set size: one encode + classify of the
    # 1559 C2 test queries, device-resident, median of 20 passes
    Xt = dev(w["Xte"])
    Ht = torch.empty((n_te, W), dtype=torch.int32, device="cuda")
    lt = torch.empty(n_te, dtype=torch.int32, device="cuda")
    lat = []
    for i in range(23):
        ev[0].record()
        h.hdc_encode_rp(Xt, Pd, kn_e, Hbits=Ht)
        h.hdc_classify(Ht, C, kn, labels=lt)
        ev[1].record()
        torch.cuda.synchronize()
        if i >= 3:
            lat.append(ev[0].elapsed_time(ev[1]))
    latency = {"queries": int(n_te), "ms_median": float(np.median(lat)), "ms_best": float(min(lat))}

    # ---- end to end through the host entry point (pinned host buffers, H2D + D2H inside)
    e2e = None
    if rank == 0 or world > 1:
        Xh = torch.from_numpy(Xq).pin_memory()
        Lh = torch.empty(NQ, dtype=torch.int32).pin_memory()
        h.hdc_infer_rp_host(Xh, Pd, C, kn, labels_host=Lh)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            h.hdc_infer_rp_host(Xh, Pd, C, kn, labels_host=Lh)      # synchronises before returning
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, torch.device("cuda", local))
        assert np.array_equal(Lh.numpy(), labels.cpu().numpy()), "e2e labels differ from the device path"
        e2e = {"value": world * NQ * args.steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(Xh.numel() * 4),
               "d2h_bytes_per_step": int(NQ * 4), "api": "hdc_infer_rp_host"}

    line = None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "C2 ISOLET-shaped: F=617 fp32, K=26, D=10000 fp32 RP encode + cosine + argmax",
                           "queries_per_step_per_gpu": NQ, "l2": "inputs (323 MB/step) larger than L2",
                           "sharding": "queries split across ranks, P and C replicated, no collective",
                           "test_accuracy": acc, "inputs_sha256": inputs_sha},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "f32_fast_variant": f32_fast, "latency_true_size": latency,
                "train": {"samples_per_s": train_sps, "what": "C2 retraining epochs (classify + class update), B=N",
                          "epochs": w["epochs"], "ms": train_ms}}
        if world == 1:
            line["cpu_baseline"] = cpu_baseline(w, Xq)
        if args.rows and world == 1:
            from paper_2606_26547_b200 import bench_rows
            line["rows"] = bench_rows.run(h, peaks)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    h.close()


def cpu_baseline(w, Xq):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    from oracle import hdc_oracle as O
    C = oracle_model(O, w)
    sample = 131072
    X = Xq[:sample]
    oracle_infer(O, X[:128], w["P"], C, w["D"])
    t0 = time.perf_counter()
    oracle_infer(O, X, w["P"], C, w["D"])
    dt = time.perf_counter() - t0
    return {"value": sample / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
            "sample": f"{sample} queries of the tiled C2 test set (encode + cosine + argmax), {dt:.1f} s"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--rows", action="store_true", help="also measure the other hot-path rows")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
