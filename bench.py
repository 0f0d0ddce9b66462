"""bench.py -- HDC inference queries/s (encode + similarity + argmax) at D=10000 on B200.

Headline workload = BASELINE.json configs[1] ("C2", ISOLET-shaped): F=617 fp32 features, K=26,
D=10000 fp32 Gaussian random projection, cosine similarity against class hypervectors trained by
bundling + 20 retraining epochs (lr 0.05); the 1559-query test set is tiled to 131072 queries per
step so that the timed inputs (323 MB) exceed L2.  One step = hdc_encode_rp + hdc_classify over
that batch, through the C ABI.  Synthetic seeded data (workloads/gen.py) stands in for ISOLET.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--rows] [--no-rows]

`--gpus N` with N > 1 and no torchrun environment re-executes itself as N ranks (one per GPU) under
`python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1`; launched by
torchrun it checks WORLD_SIZE == N.  Queries are sharded over the ranks (weak scaling, no collective
on the inference path); the `train_sharded` block times data-parallel retraining (one int32 all-reduce
of the class update per mini-batch: paper_2606_26547_b200/shard.py) and checks it against a single-rank
epoch bit for bit.

Prints ONE JSON line (rank 0).  Besides the headline it carries `rows`: the other hot-path rows
(bench_rows.DEFAULT_ROWS: bf16 / int8 encode, the C4 precision points, level-ID, Hamming, C5, retraining),
each with its own SM-clock sample, and -- at N = 1 -- the oracle timed beside them (`rows_cpu_baseline`).
`--rows` measures every row of bench_rows.ROWS, `--no-rows` none.  `--impl reference` times the CPU oracle
(oracle/hdc_oracle.py, as it stands) on the host cores for the same metric / config.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hdc_inference_queries_per_sec_D10000"
UNIT = "queries/s"
NQ = 131072            # queries per step and rank (test set tiled)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the headline contraction kernel, from the
# `ncu --set full` capture named beside it (a static figure: ncu cannot run inside the timed bench)
NCU_TRAFFIC_BYTES = 812.8e6
NCU_TRAFFIC_SOURCE = ("profiles/r2_final_kernels.md (static: ncu --set full capture of gemm_tc_kernel, fp32-precision "
                      "encode, 131072 x 617 x 10000, round 2 build; command in that file)")
SM_COUNT = 148
FP32_LANES = 128       # FFMA lanes per SM per clock
NOMINAL_BF16_TFLOPS = 2250.0   # dense, at sm_max_mhz (guide)


# ------------------------------------------------------------------------------------ launcher
def launcher_command(gpus: int, argv: list, port: int) -> list:
    """Command line that runs this file as `gpus` ranks, one per GPU, over NCCL (the form the driver uses)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(gpus)}",
            "--master-addr", "127.0.0.1", "--master-port", str(int(port)), os.path.abspath(__file__)] + list(argv)


def free_port() -> int:
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def resolve_world(gpus: int, env=os.environ):
    """(world, rank, local_rank, must_spawn).  Under torchrun WORLD_SIZE must equal --gpus; without it
    --gpus > 1 asks for a re-exec under the launcher.  Never falls back to fewer ranks than asked."""
    if gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if "WORLD_SIZE" in env:
        world = int(env["WORLD_SIZE"])
        if world != gpus:
            raise SystemExit(f"bench.py: --gpus {gpus} but the launcher started WORLD_SIZE={world} ranks")
        return world, int(env.get("RANK", "0")), int(env.get("LOCAL_RANK", "0")), False
    return gpus, 0, 0, gpus > 1


def spawn_ranks(args):
    """Re-exec as args.gpus ranks.  Fails loudly when the box has fewer GPUs (no silent 1-rank run)."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this box has {have} "
                         "(there is no CPU or fewer-rank fallback)")
    cmd = launcher_command(args.gpus, sys.argv[1:], free_port())
    sys.stdout.flush()
    os.execv(cmd[0], cmd)


from bench_rows import ClockSampler, load_peaks, sustained_clock_mhz  # noqa: E402  (imports torch)


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
    world, rank, _, _ = resolve_world(args.gpus) if "WORLD_SIZE" in os.environ else (1, 0, 0, False)
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
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "C2 ISOLET-shaped: F=617 fp32, K=26, D=10000 RP encode + cosine + argmax",
                       "queries_per_step": sample, "timing": "host wall clock; rank 0 only, no GPU is used"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{sample} queries of the tiled C2 test set per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ own arm
def train_sharded_block(h, hd, shard, dist, world, rank, local, w, Htr, ytr, kn, epochs):
    """Data-parallel retraining: every mini-batch (B = N here) is split over the ranks,
    each rank computes the int32 class update of its shard (hdc_train_delta), ONE all-reduce(sum) per
    mini-batch (NCCL when world > 1) hands every rank the same integers, hdc_train_apply performs the
    identical fp32 update.  Checked bit for bit against hdc_train_epoch run by this rank alone."""
    import torch
    K, D = w["K"], w["D"]
    N = Htr.shape[0]
    C0 = torch.zeros((K, D), dtype=torch.float32, device="cuda")
    h.hdc_train_epoch(hd.HDC_TRAIN_BUNDLE, Htr, ytr, C0, kn)
    C_single = C0.clone()
    for _ in range(epochs):
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, C_single, kn, lr=w["lr"], batch=0)
    C = C0.clone()
    delta = torch.empty((K, ((D + 31) // 32) * 32), dtype=torch.int32, device="cuda")
    delta_fn = lambda lo, hi: h.hdc_train_delta(Htr[lo:hi], ytr[lo:hi], C, kn, delta=delta)   # noqa: E731
    apply_fn = lambda d: h.hdc_train_apply(C, kn, d, w["lr"])                                    # noqa: E731
    shard.train_epoch_sharded(delta_fn, apply_fn, N, 0)            # warm-up epoch (NCCL communicator, workspaces)
    C.copy_(C0)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ev[0].record()
    for _ in range(epochs):
        shard.train_epoch_sharded(delta_fn, apply_fn, N, 0)
    ev[1].record()
    torch.cuda.synchronize()
    ms = shard.max_over_ranks(ev[0].elapsed_time(ev[1]), torch.device("cuda", local))
    same = bool(torch.equal(C, C_single))
    if world > 1:
        flag = torch.tensor([1 if same else 0], device="cuda")
        dist.all_reduce(flag, op=dist.ReduceOp.MIN)
        same = bool(flag.item())
    if not same:
        raise RuntimeError("sharded retraining differs from the single-rank epochs (replicas must be bit-identical)")
    return {"samples_per_s": epochs * N / (ms * 1e-3), "ms": ms, "epochs": epochs, "ranks": world,
            "scaling": "strong (the 6238 C2 training samples are split over the ranks)",
            "collective": "none (1 rank)" if world == 1 else "all_reduce(sum) of int32 Delta[K x D] per mini-batch, NCCL",
            "bit_identical_to_single_rank": same,
            "what": "C2 retraining epochs as hdc_train_delta -> all-reduce -> hdc_train_apply, B = N"}


def run_gpu(args):
    world, rank, local, must_spawn = resolve_world(args.gpus)
    if must_spawn:
        spawn_ranks(args)          # does not return
    import torch
    import torch.distributed as dist

    import paper_2606_26547_b200 as hd
    from paper_2606_26547_b200 import shard

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
    Fp = -(-F // 64) * 64            # reduction axis as staged (k-blocks of 64 bf16)
    Pd = dev(w["P"])
    kn_e = hd.knobs(D, precision=hd.HDC_F32)
    kn = hd.knobs(D, precision=hd.HDC_F32, hv_bits=32, sim=hd.HDC_SIM_COS)

    # ---- model: encode train, bundle, 20 retraining epochs (setup; warm epochs are timed afterwards)
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
    train_cold_ms = ev[0].elapsed_time(ev[1])
    Cw = C.clone()                                       # the same epochs again, warm (model already converged)
    ev[0].record()
    for _ in range(w["epochs"]):
        h.hdc_train_epoch(hd.HDC_TRAIN_PERCEPTRON, Htr, ytr, Cw, kn, lr=w["lr"], batch=0)
    ev[1].record()
    torch.cuda.synchronize()
    train_ms = ev[0].elapsed_time(ev[1])
    train_sps = w["epochs"] * Xtr.shape[0] / (train_ms * 1e-3)
    del Cw

    # ---- timed inference steps (device-resident inputs)
    Xd = dev(Xq)
    W = (D + 31) // 32
    Hq = h.alloc_hbits(NQ, D)
    labels = torch.empty(NQ, dtype=torch.int32, device="cuda")

    # the query-independent operands (3 x bf16 split of P, class operand and cosine scales) are converted once
    # ("the one-time conversion of P and of the class model is not per-query work"); a step is
    # one hdc_infer_rp_m: staging of the step's X, the encode contraction, the classify kernel
    model = h.hdc_model_prepare(Pd, C, kn)

    def step():
        h.hdc_infer_rp_m(Xd, model, labels=labels, Hbits=Hq)

    def step_plain():   # the same through the plain entry points (operands re-derived inside every call)
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
    labels_model = labels.clone()
    ev[0].record()
    for _ in range(args.steps):
        step_plain()
    ev[1].record()
    torch.cuda.synchronize()
    plain_ms = ev[0].elapsed_time(ev[1]) / args.steps
    assert torch.equal(labels, labels_model), "prepared-model step and plain calls disagree"
    value = world * NQ * args.steps / (ms * 1e-3)
    n_te = w["Xte"].shape[0]
    acc = float((labels[:n_te].cpu().numpy() == w["yte"][np.arange(rank * NQ, rank * NQ + n_te) % n_te]).mean())

    # ---- dominant kernel: the encode contraction.  Its launches are bracketed by CUDA events
    # inside the library (hdc_kernel_timing) on the stream they are launched on; measured (a) over a
    # re-run of the timed steps (sustained regime) and (b) alone, back to back (burst regime).
    h.kernel_timing(True)
    torch.cuda.synchronize()
    with ClockSampler(local) as cs_k:
        ev[0].record()
        for _ in range(args.steps):
            step()
        ev[1].record()
        torch.cuda.synchronize()
    pass2_step_ms = ev[0].elapsed_time(ev[1]) / args.steps   # the step as timed in THIS pass (its own clocks)
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
    clk_k = cs_k.summary()
    # the same fraction against the peak RESCALED to the SM clock sampled while the kernel ran:
    # (a) the measured sustained cuBLAS rate per MHz of the clock it was measured at, (b) the nominal dense rate
    f_k = clk_k.get("sm_mhz") or clocks.get("sm_mhz")
    rescaled = None
    if f_k:
        pk_meas = peaks["bf16_tflops_sustained"] * f_k / sustained_clock_mhz(peaks) / 6.0
        pk_nom = NOMINAL_BF16_TFLOPS * f_k / peaks["sm_max_mhz"] / 6.0
        rescaled = {"sm_mhz_during_kernel_pass": f_k,
                    "peak_measured_rate_at_this_clock": pk_meas, "frac_of_measured_rate_at_this_clock": achieved / pk_meas,
                    "peak_nominal_at_this_clock": pk_nom, "frac_of_nominal_at_this_clock": achieved / pk_nom,
                    "how": "bf16_tflops_sustained x sm_mhz / (clock the driver measured it at) / 6; "
                           "2250 TFLOP/s nominal dense x sm_mhz / sm_max_mhz / 6"}
    roofline = {"bound": "tensor",
                "kernel": "gemm_tc_kernel<bf16,EPI_SIGN,cta_group::2> (tcgen05 fp32-precision encode on CTA pairs: 6 "
                          "bf16 segment products per MAC over 3-way split operands, sign+pack epilogue)",
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": f"bf16_tflops_sustained / 6 ({peaks['_source']} MEASURED_PEAKS.json; kernel timed "
                               "inside the step loop)",
                "frac_of_burst_peak": achieved / (peaks["bf16_tflops"] / 6.0),
                "clock_rescaled": rescaled,
                "algorithmic_flops_per_launch": flops, "ms_per_launch": enc_ms,
                "executed_bf16_tflops": 6.0 * 2.0 * NQ * Fp * D / (enc_ms * 1e-3) / 1e12,
                "alone": {"ms_per_launch": enc_alone_ms, "achieved": flops / (enc_alone_ms * 1e-3) / 1e12,
                          "peak": peaks["bf16_tflops"] / 6.0,
                          "frac": flops / (enc_alone_ms * 1e-3) / 1e12 / (peaks["bf16_tflops"] / 6.0),
                          "peak_source": "bf16_tflops (burst) / 6"},
                "encode_call_ms": enc_call_ms, "classify_kernel_ms": cls_ms,
                "later_passes": "ms_per_launch and classify_kernel_ms come from a second pass over the same steps with "
                                "the library's per-kernel events on, encode_call_ms and `alone` from a third pass of "
                                "encode calls only; each ran after the timed region, at the clocks the part had then, "
                                "so they need not add up to ms_per_step",
                "share_of_step": enc_ms / pass2_step_ms, "step_ms_in_kernel_pass": pass2_step_ms,
                "share_of_step_how": "contraction ms per launch / ms per step, both from the second pass (same clocks); "
                                     "compare with the ncu launch list profiles/r2_launches.md",
                "fp32_alu_peak_tflops": SM_COUNT * FP32_LANES * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12,
                "traffic": NCU_TRAFFIC_BYTES, "traffic_source": NCU_TRAFFIC_SOURCE,
                "algorithmic_bytes_per_launch": float(NQ) * 3 * Fp * 2 + float(D) * 3 * Fp * 2 + float(NQ) * W * 4}

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
    Ht = h.alloc_hbits(n_te, D)
    lt = torch.empty(n_te, dtype=torch.int32, device="cuda")
    lat, lat_plain = [], []
    for i in range(23):
        ev[0].record()
        h.hdc_infer_rp_m(Xt, model, labels=lt, Hbits=Ht)
        ev[1].record()
        torch.cuda.synchronize()
        if i >= 3:
            lat.append(ev[0].elapsed_time(ev[1]))
    for i in range(23):
        ev[0].record()
        h.hdc_encode_rp(Xt, Pd, kn_e, Hbits=Ht)
        h.hdc_classify(Ht, C, kn, labels=lt)
        ev[1].record()
        torch.cuda.synchronize()
        if i >= 3:
            lat_plain.append(ev[0].elapsed_time(ev[1]))
    latency = {"queries": int(n_te), "ms_median": float(np.median(lat)), "ms_best": float(min(lat)),
               "what": "hdc_infer_rp_m on the prepared model",
               "plain_calls_ms_median": float(np.median(lat_plain)),
               "plain_calls": "hdc_encode_rp + hdc_classify, P split and class operand re-derived in the calls"}

    # ---- end to end through the host entry point (pinned host buffers, H2D + D2H inside)
    Xh = torch.from_numpy(Xq).pin_memory()
    Lh = torch.empty(NQ, dtype=torch.int32).pin_memory()
    for _ in range(max(3, args.warmup)):      # the same number of warm-up steps as the device-resident loop
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
    e2e = {"value": world * NQ * args.steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(world * Xh.numel() * 4),
           "d2h_bytes_per_step": int(world * NQ * 4), "api": "hdc_infer_rp_host"}
    del Xh, Lh

    # ---- data-parallel retraining (every N; NCCL all-reduce when N > 1)
    train_sharded = train_sharded_block(h, hd, shard, dist, world, rank, local, w, Htr, ytr, kn, w["epochs"])

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
                "step": {"api": "hdc_infer_rp_m (prepared model): X staging + encode contraction + classify kernel",
                         "plain_calls_ms_per_step": plain_ms,
                         "plain_calls": "hdc_encode_rp + hdc_classify, labels identical"},
                "train": {"samples_per_s": train_sps, "what": "C2 retraining epochs (classify + class update), B=N, "
                          "warm (second run of the 20 epochs)", "epochs": w["epochs"], "ms": train_ms,
                          "first_run_ms": train_cold_ms},
                "train_sharded": train_sharded}
    # ---- the other hot-path rows, each with its own clock sample (rank 0's GPU; N = 1 only: they are 1-GPU rows)
    if rank == 0 and world == 1 and not args.no_rows:
        import bench_rows
        del Xd, Hq, Xt, Ht
        torch.cuda.empty_cache()
        t0 = time.perf_counter()
        line["rows"] = bench_rows.run(h, peaks, reps=5, only=None if args.rows else bench_rows.DEFAULT_ROWS)
        line["rows_wall_s"] = round(time.perf_counter() - t0, 1)
        line["cpu_baseline"] = cpu_baseline(w, Xq)
        line["rows_cpu_baseline"] = rows_cpu_baseline(w)
    elif rank == 0 and world == 1:
        line["cpu_baseline"] = cpu_baseline(w, Xq)
    if rank == 0:
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


def rows_cpu_baseline(w):
    """The oracle, as it stands, timed on the host cores beside the rows of `rows` (north_star: "absolute
    queries/sec and training samples/sec ... beside the oracle timed on the box's host cores in the same
    run"): bounded samples, wall clock, each labelled; a baseline, not a target."""
    from oracle import hdc_oracle as O
    from workloads import gen
    cores = os.cpu_count()
    out = {}

    def timed(fn):
        t0 = time.perf_counter()
        r = fn()
        return r, time.perf_counter() - t0

    # retraining epoch, C2 (train set encoded by the oracle first; one epoch B = N timed)
    n_tr = w["Xtr"].shape[0]
    btr, _, _ = O.encode_rp(w["Xtr"][:n_tr], w["P"], w["D"], O.F32)
    C = O.bundle(btr, w["ytr"][:n_tr], w["K"], w["D"])
    _, dt = timed(lambda: O.train_epoch(btr, w["ytr"][:n_tr], C, w["D"], 32, O.SIM_COS, w["lr"], 0))
    out["c2_train_epoch"] = {"value": n_tr / dt, "unit": "samples/s", "cores": cores, "kind": "oracle",
                             "sample": f"one retraining epoch (B=N) over the {n_tr} C2 training samples (pre-encoded), {dt:.2f} s"}
    # classify against the class accumulators held as 32-bit integers (exact 64-bit sums), C2 shape
    nq = 2048
    _, dt = timed(lambda: O.infer(btr[:nq], C, w["D"], O.SIM_COS, O.HV_I32))
    out["c2_classify_cos_i32"] = {"value": nq / dt, "unit": "queries/s", "cores": cores, "kind": "oracle",
                                  "sample": f"{nq} encoded C2 queries against K={w['K']} classes as 32-bit integers "
                                            f"(cosine + argmax), {dt:.2f} s; the integer sums are numpy loops over "
                                            "the classes: one core"}
    # level-ID encode, C3
    c3 = gen.c3_mnist_shaped(n_tr=16, n_te=256)
    hb3, dt = timed(lambda: O.encode_levelid(c3["Lte"], c3["ID"], c3["LV"], c3["D"]))
    out["c3_levelid"] = {"value": 256 / dt, "unit": "samples/s", "cores": cores, "kind": "oracle",
                         "sample": f"256 C3-shaped images (F=784, Q=256, D=10000), {dt:.2f} s; the oracle loops over "
                                   "samples in python: one core"}
    # Hamming similarity + arg-min, C3 shape (K = 10)
    C3 = O.bundle(hb3, c3["yte"], c3["K"], c3["D"])
    reps = 16
    q = np.concatenate([hb3] * reps, axis=0)
    _, dt = timed(lambda: O.infer(q, C3, c3["D"], O.SIM_HAMMING, 1))
    out["c3_hamming_k10"] = {"value": q.shape[0] / dt, "unit": "queries/s", "cores": cores, "kind": "oracle",
                             "sample": f"{q.shape[0]} encoded C3 queries (256 tiled x{reps}) against K=10, {dt:.2f} s"}
    out["c3_pipeline"] = {"value": 1.0 / (1.0 / out["c3_levelid"]["value"] + 1.0 / out["c3_hamming_k10"]["value"]),
                          "unit": "queries/s", "cores": cores, "kind": "oracle",
                          "sample": "harmonic combination of the two rows above (same samples)"}
    # C5: the SURVEY 8(d) subsample -- first 4096 queries of batch 0 + 64 of each remaining batch = 5056 queries
    c5 = gen.c5_large_batch(4096, batch=0)
    X5 = np.concatenate([c5["X"]] + [gen.c5_large_batch(64, batch=i, per_class=1)["X"] for i in range(1, 16)], axis=0)
    btr5, _, _ = O.encode_rp(c5["Xtr"], c5["P"], c5["D"], O.BF16)
    C5 = O.bundle(btr5, c5["ytr"], c5["K"], c5["D"])
    (hb5, _, _), dt_e = timed(lambda: O.encode_rp(X5, c5["P"], c5["D"], O.BF16))
    _, dt_c = timed(lambda: O.infer(hb5, C5, c5["D"], O.SIM_COS, 16))
    n5h = 512                        # the oracle's Hamming loops over the 1000 classes: a smaller sample
    _, dt_h = timed(lambda: O.infer(hb5[:n5h], C5, c5["D"], O.SIM_HAMMING, 1))
    dt_h *= X5.shape[0] / n5h
    n5 = X5.shape[0]
    out["c5_stream_bf16"] = {"value": n5 / (dt_e + dt_c), "unit": "queries/s", "cores": cores, "kind": "oracle",
                             "sample": f"{n5}-query subsample (4096 of batch 0 + 64 of each other batch): encode {dt_e:.1f} s "
                                       f"+ bf16 cosine classify {dt_c:.1f} s; extrapolated linearly to 2^20 queries: "
                                       f"{(dt_e + dt_c) * (1 << 20) / n5:.0f} s"}
    out["c5_stream_1bit"] = {"value": n5 / (dt_e + dt_h), "unit": "queries/s", "cores": cores, "kind": "oracle",
                             "sample": f"same subsample: encode {dt_e:.1f} s + Hamming classify {dt_h:.1f} s (timed on its first {n5h} queries, scaled); extrapolated "
                                       f"linearly to 2^20 queries: {(dt_e + dt_h) * (1 << 20) / n5:.0f} s"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--rows", action="store_true", help="measure every row of bench_rows.ROWS (default: DEFAULT_ROWS)")
    ap.add_argument("--no-rows", action="store_true", help="headline only")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
