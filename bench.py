#!/usr/bin/env python
"""bench.py -- the headline benchmark of the MosaicQuant / ZipperEngine hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

Workload (default): BASELINE.json configs[1], "LLaMA3-8B-shaped decode layers":
M in {1, 8, 32} tokens x {qkv 4096x6144, o 4096x4096, gate_up 4096x28672, down 14336x4096},
W ~ N(0, 0.02) + 0.5% block-clustered x20 outliers, 64x64 residual blocks at 5% density chosen by
the Delta-Hessian score (mq_pack_weights = Algorithm 1), fp16 activations, bf16 output.
One STEP = the whole hot path once over one batch for every (M, projection):
mq_quantize_act + mq_gemm, 12 pairs = 24 kernel launches, replayed from a CUDA graph.
Every call reads a weight copy that was last touched > 3x L2 ago (4 rotating copies, 460 MB).

Prints ONE JSON line (see the keys at the bottom).  `--impl reference` times the CPU oracle
(this tier's reference arm) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fused W4A4+residual GEMM TOPS & frac of INT8/HBM roofline; tokens/s vs W16A16"
RHO, BS = 0.05, 64
E2E_STREAMS = 4         # streams the end-to-end leg spreads a step's independent mq_linear_host calls over
N_COPIES = 4            # weight copies the STEP graphs rotate (458 MB of other layers' weights between two uses)
L2_BYTES = 126e6        # the per-shape loops rotate enough copies of ONE layer for 3 x L2 (SURVEY 8(d) cold-HBM rule)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_sustained=1400.0, source="fallback")


def workload_shapes(name: str):
    import synth
    cfg = synth.CONFIGS[name]
    return cfg, [(m, l) for m in cfg["Ms"] for l in cfg["layers"]]


def algo_bytes(M, K, N, nnz, bs):
    """SURVEY 8(d) algorithmic bytes of one mq_gemm launch: packed base + residual blocks + block
    metadata + scales + packed activations (+ their scales) in, 16-bit Y out."""
    return N * K // 2 + nnz * bs * bs // 2 + 8 * nnz + 8 * N + M * K // 2 + 4 * M + 2 * M * N


def algo_ops(M, K, N, nnz, bs):
    return 2 * M * N * K + 2 * M * nnz * bs * bs


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                pw.append(float(r[2]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                    samples=len(sm), reasons=sorted(reasons))


class Layer:
    """One projection: host tensors, N_COPIES packed device copies, per-M device buffers."""

    def __init__(self, mq, torch, synth, seed, shape, Ms, n_copies, rho=RHO, bs=BS, cold_rule=True):
        self.name, self.K, self.N = shape.name, shape.K, shape.N
        t0 = time.time()
        self.W = synth.gen_weight(seed, self.N, self.K)
        X = synth.gen_calib(seed, self.K, 256)
        self.h = (2.0 / X.shape[0] * (X.astype(np.float64) ** 2).sum(0)).astype(np.float32)   # calibration input
        self.budget = synth.budget_from_density(rho, self.N, self.K, bs)
        w0 = mq.mq_pack_weights(self.W, self.h, bs, self.budget)
        # cold-HBM rule: copies x packed bytes >= 3 x L2 for the loops that replay ONE layer back to back
        if cold_rule:
            n_copies = max(n_copies, int(np.ceil(3 * L2_BYTES / w0.info()["device_bytes"])) + 1)
        self.copies = [w0] + [w0.clone() for _ in range(n_copies - 1)]
        self.nnz = w0.info()["nnz"]
        # the same layer with budget 0 (dense-only W4A4): the zero-residual baseline of the same kernel
        z0 = mq.mq_pack_weights(self.W, self.h, bs, 0) if self.budget else w0
        self.dense = [z0] + [z0.clone() for _ in range(n_copies - 1)] if self.budget else self.copies
        self.pack_s = time.time() - t0
        self.W = None                                            # the fp32 weights are not needed any more
        self.A_host, self.A, self.qA, self.sA, self.Y, self.ws = {}, {}, {}, {}, {}, {}
        for m in Ms:
            a = synth.gen_act(seed + m, m, self.K)
            self.A_host[m] = torch.from_numpy(a).pin_memory()
            self.A[m] = self.A_host[m].cuda()
            self.qA[m] = torch.empty((m, self.K // 2), dtype=torch.uint8, device="cuda")
            self.sA[m] = torch.empty((m,), dtype=torch.float32, device="cuda")
            self.Y[m] = torch.empty((m, self.N), dtype=torch.bfloat16, device="cuda")
            self.ws[m] = mq.new_workspace(mq.mq_gemm_workspace_bytes(w0, m))


def measure(workload, steps, warmup, torch, mq, synth, world, dist, local, with_e2e=True, extras=True):
    """Times one workload (BASELINE.json config): the whole step, the GEMM kernels alone (roofline),
    the cuBLAS bf16 comparator and the end-to-end path through mq_linear with host buffers."""
    cfg, _ = workload_shapes(workload)
    Ms, layers_cfg = cfg["Ms"], cfg["layers"]
    layers = [Layer(mq, torch, synth, cfg["seed"] + i, l, Ms, N_COPIES) for i, l in enumerate(layers_cfg)]
    calls = [(m, L) for m in Ms for L in layers]           # one step, in order

    def step(si: int):
        for ci, (m, L) in enumerate(calls):
            w = L.copies[(si * len(Ms) + ci // len(layers)) % N_COPIES]
            mq.mq_quantize_act(L.A[m], L.qA[m], L.sA[m])
            mq.mq_gemm(w, L.qA[m], L.sA[m], m, Y=L.Y[m], workspace=L.ws[m])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        step(0)                                                  # first-call setup outside capture
        stream.synchronize()
        graphs = []
        for si in range(N_COPIES):                               # pattern of copies repeats every 4 steps
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                step(si)
            graphs.append(g)
        for i in range(warmup):
            graphs[i % N_COPIES].replay()
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        time.sleep(0.25)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            graphs[(warmup + i) % N_COPIES].replay()
        e1.record(stream)
        barrier()
        ms_step = e0.elapsed_time(e1) / steps
        clocks = sampler.stop()

        # ---- roofline of the dominant kernel, timed alone: graphs of GEMM launches only.
        # COLD: one launch per weight copy of the layer, copies x bytes >= 3 x L2, so every launch streams its
        # weights from HBM; WARM: the same number of launches on ONE copy (L2-resident when it fits), labelled.
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def time_graph(call, n, repeats=5):
            """us per launch of `call(r)` for r in range(n), replayed from a CUDA graph (best of `repeats`)."""
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for r in range(n):
                    call(r)
            for _ in range(2):
                g.replay()
            best = 1e30
            for _ in range(repeats):
                a0.record(stream)
                g.replay()
                a1.record(stream)
                stream.synchronize()
                best = min(best, a0.elapsed_time(a1) / n)
            del g
            return best * 1e3

        per_shape = []
        quant_shapes = {}
        for (m, L) in calls:
            nc = len(L.copies)
            reps = max(nc, 4) if m <= 512 else max(2, min(nc, 4))    # long launches need fewer repetitions
            gemm = lambda ws_, r: mq.mq_gemm(ws_[r % len(ws_)], L.qA[m], L.sA[m], m, Y=L.Y[m], workspace=L.ws[m])
            us = time_graph(lambda r: gemm(L.copies, r), reps)
            us_warm = time_graph(lambda r: gemm(L.copies[:1], r), reps)
            # the zero-residual baseline: same kernel, same protocol, the budget-0 packing of the same W
            us0 = time_graph(lambda r: gemm(L.dense, r), reps)
            row = dict(M=m, layer=L.name, K=L.K, N=L.N, us=us, us_warm=us_warm, us_dense=us0, copies=nc,
                       bytes=algo_bytes(m, L.K, L.N, L.nnz, BS), ops=algo_ops(m, L.K, L.N, L.nnz, BS))
            if extras:
                # the W4A8 variant of the same launch: int8 per-token activations, same packed weights
                q8, s8 = mq.mq_quantize_act8(L.A[m])
                row["us_a8"] = time_graph(lambda r: mq.mq_gemm_a8(L.copies[r % nc], q8, s8, m, Y=L.Y[m], workspace=L.ws[m]), reps, 3)
                del q8, s8
                # the paper's naive 3-kernel pipeline on the same launch (Fig.3)
                scr = torch.empty((m, L.N), dtype=torch.int32, device="cuda")
                row["us_naive"] = time_graph(lambda r: mq.mq_gemm_naive(L.copies[r % nc], L.qA[m], L.sA[m], m, Y=L.Y[m],
                                                                         workspace=L.ws[m], scratch=scr), reps, 3)
                del scr
                # per-group activation scales (the paper's W4A4 activation setting), group 128
                qg, sg = mq.mq_quantize_act_group(L.A[m], 128)
                wsg = torch.empty(max(mq.mq_gemm_group_workspace_bytes(L.copies[0], m), 16), dtype=torch.uint8, device="cuda")
                row["us_group"] = time_graph(lambda r: mq.mq_gemm_group(L.copies[r % nc], qg, sg, 128, m, Y=L.Y[m], workspace=wsg), reps, 3)
                del qg, sg, wsg
            per_shape.append(row)
            # the activation quantizer alone (kernel i): HBM, 2 B read + 0.5 B written per element
            if (m, L.K) not in quant_shapes:
                nq = 8 if m <= 512 else 3
                quant_shapes[(m, L.K)] = dict(M=m, K=L.K, us=time_graph(lambda r: mq.mq_quantize_act(L.A[m], L.qA[m], L.sA[m]), nq, 3),
                                              bytes=int(2.5 * m * L.K) + 4 * m)

        # ---- W16A16 comparator: cuBLAS bf16 on the same shapes, same rotation
        w16 = {L.name: [torch.randn((L.N, L.K), device="cuda", dtype=torch.bfloat16) * 0.02 for _ in range(2)]
               for L in layers}
        a16 = {(m, L.name): L.A[m].to(torch.bfloat16) for (m, L) in calls}

        def step16(si):
            for ci, (m, L) in enumerate(calls):
                torch.matmul(a16[(m, L.name)], w16[L.name][(si + ci // len(layers)) % 2].t())
        step16(0)
        stream.synchronize()
        g16 = []
        for si in range(2):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                step16(si)
            g16.append(g)
        for i in range(3):
            g16[i % 2].replay()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        for i in range(steps):
            g16[i % 2].replay()
        c1.record(stream)
        stream.synchronize()
        ms16 = c0.elapsed_time(c1) / steps
        del w16, g16, a16

        # ---- e2e: host buffers through the C ABI (mq_linear_host), H2D + D2H inside the timed region
        e2e_ms = None
        if with_e2e:
            Yh = {(m, L.name): torch.empty((m, L.N), dtype=torch.bfloat16).pin_memory() for (m, L) in calls}
            stg = {(m, L.name): torch.empty(mq.mq_linear_host_staging_bytes(L.copies[0], m), dtype=torch.uint8, device="cuda")
                   for (m, L) in calls}
            lws = {(m, L.name): mq.new_workspace(mq.mq_linear_workspace_bytes(L.copies[0], m)) for (m, L) in calls}

            # The 12 calls of a step are independent (each has its own host buffers, staging and workspace), so they
            # go round-robin onto E2E_STREAMS streams, largest copies first: one call's H2D and D2H copies overlap
            # another's kernels.  Every call still moves its own A in and its own Y out inside the timed region.
            e2e_streams = [torch.cuda.Stream() for _ in range(E2E_STREAMS)]
            e2e_order = sorted(range(len(calls)), key=lambda ci: -(calls[ci][0] * (calls[ci][1].K + calls[ci][1].N)))

            def step_e2e(si):
                # ONE C-ABI call per layer with host pointers: H2D copy of A, quantize + GEMM, D2H copy of Y
                for j, ci in enumerate(e2e_order):
                    m, L = calls[ci]
                    k = (m, L.name)
                    mq.mq_linear_host(L.copies[(si * len(Ms) + ci // len(layers)) % N_COPIES], L.A_host[m], Yh[k], stg[k], lws[k],
                                      e2e_streams[j % E2E_STREAMS])
                for s in e2e_streams:                                # the caller reads the results
                    s.synchronize()

            for i in range(3):
                step_e2e(i)
            barrier()
            t0 = time.perf_counter()
            for i in range(steps):
                step_e2e(i)
            torch.cuda.synchronize()
            e2e_ms = (time.perf_counter() - t0) * 1e3 / steps

    if world > 1:
        ms_step, e2 = max_over_ranks([ms_step, e2e_ms or 0.0], torch, dist, "cuda")
        e2e_ms = e2 if with_e2e else None
    return dict(cfg=cfg, Ms=Ms, layers_cfg=layers_cfg, layers=layers, calls=calls, ms_step=ms_step, clocks=clocks,
                per_shape=per_shape, quant=list(quant_shapes.values()), ms16=ms16, e2e_ms=e2e_ms,
                ops_step=sum(algo_ops(m, L.K, L.N, L.nnz, BS) for (m, L) in calls),
                bytes_step=sum(algo_bytes(m, L.K, L.N, L.nnz, BS) for (m, L) in calls),
                h2d=sum(L.A_host[m].numel() * 2 for (m, L) in calls), d2h=sum(m * L.N * 2 for (m, L) in calls),
                pack_s=sum(L.pack_s for L in layers))


def measure_sweep(workload, torch, mq, synth, layer_names=None):
    """BASELINE.json configs[3]: the residual density x block size sweep of the Qwen3-8B-shaped layers.  Per (layer,
    block, rho, M): the GEMM launch alone, cold weights (copies x bytes >= 3 x L2), same protocol as the roofline loop."""
    cfg, _ = workload_shapes(workload)
    stream = torch.cuda.Stream()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rows = []
    with torch.cuda.stream(stream):
        for i, l in enumerate(cfg["layers"]):
            if layer_names and l.name not in layer_names:
                continue
            for bs in cfg.get("block_sweep", [cfg["block"]]):
                for rho in cfg.get("rho_sweep", [cfg["rho"]]):
                    L = Layer(mq, torch, synth, cfg["seed"] + i, l, cfg["Ms"], N_COPIES, rho=rho, bs=bs)
                    for m in cfg["Ms"]:
                        mq.mq_quantize_act(L.A[m], L.qA[m], L.sA[m])
                        nc = len(L.copies)
                        reps = nc if m <= 512 else max(2, min(nc, 4))
                        g = torch.cuda.CUDAGraph()
                        mq.mq_gemm(L.copies[0], L.qA[m], L.sA[m], m, Y=L.Y[m], workspace=L.ws[m])
                        stream.synchronize()
                        with torch.cuda.graph(g, stream=stream):
                            for r in range(reps):
                                mq.mq_gemm(L.copies[r % nc], L.qA[m], L.sA[m], m, Y=L.Y[m], workspace=L.ws[m])
                        g.replay()
                        best = 1e30
                        for _ in range(3):
                            a0.record(stream)
                            g.replay()
                            a1.record(stream)
                            stream.synchronize()
                            best = min(best, a0.elapsed_time(a1) / reps)
                        del g
                        us = best * 1e3
                        by, ops = algo_bytes(m, l.K, l.N, L.nnz, bs), algo_ops(m, l.K, l.N, L.nnz, bs)
                        rows.append(dict(layer=l.name, K=l.K, N=l.N, block=bs, rho=rho, nnz=L.nnz, M=m, us=round(us, 3),
                                         gbs=round(by / (us * 1e-6) / 1e9, 1), tops=round(ops / (us * 1e-6) / 1e12, 2)))
                    del L
                    torch.cuda.empty_cache()
    # overhead of the residual against the rho = 0 run of the same (layer, block, M)
    base = {(r["layer"], r["block"], r["M"]): r["us"] for r in rows if r["rho"] == 0.0}
    for r in rows:
        b = base.get((r["layer"], r["block"], r["M"]))
        if b:
            r["over_rho0"] = round(r["us"] / b - 1.0, 4)
    return rows


def max_over_ranks(values, torch, dist, device):
    """Replicas only: the ranks share nothing on the data path; the job's time
    is the slowest rank's, so every timing is reduced with MAX over the ranks."""
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_value(ops_step, ms_step, world):
    """Whole-job throughput in TOPS: every rank processes the same step (weak scaling)."""
    return world * ops_step / (ms_step * 1e-3) / 1e12


def roofline_of(r, peaks, traffic):
    """Roofline object of the dominant kernel (the GEMM launches of one step timed alone, cold weights).
    Decode-shaped workloads are bound by HBM (algorithmic bytes), prefill-shaped ones by
    the INT8 tensor pipe; which one is decided by the slower of the two ideal times."""
    us = sum(s["us"] for s in r["per_shape"])
    by = sum(s["bytes"] for s in r["per_shape"])
    ops = sum(s["ops"] for s in r["per_shape"])
    int8_proxy = 2.0 * peaks["bf16_tflops"]          # kind::i8 runs at twice the bf16 rate (nominal 4.5 vs 2.25 PF)
    int8_peak = peaks.get("int8_probe_tops") or int8_proxy
    t_hbm, t_tensor = by / (peaks["hbm_gbs"] * 1e9), ops / (int8_peak * 1e12)
    has = lambda k: all(k in s for s in r["per_shape"])
    per_shape = []
    for s in r["per_shape"]:
        d = dict(M=s["M"], layer=s["layer"], us_cold=round(s["us"], 3), us_warm=round(s["us_warm"], 3),
                 us_dense_only=round(s["us_dense"], 3), copies=s["copies"],
                 gbs=round(s["bytes"] / (s["us"] * 1e-6) / 1e9, 1), tops=round(s["ops"] / (s["us"] * 1e-6) / 1e12, 2))
        for k, name in (("us_a8", "us_w4a8"), ("us_naive", "us_naive3"), ("us_group", "us_group128")):
            if k in s:
                d[name] = round(s[k], 3)
        per_shape.append(d)
    kern = ("mq_decode_kernel" if max(s["M"] for s in r["per_shape"]) <= 32 else "mq_gemm_kernel") + \
           f" ({len(r['per_shape'])} launches of the step, timed alone; cold = one launch per weight copy, copies x bytes >= 3 x L2)"
    us0 = sum(s["us_dense"] for s in r["per_shape"])
    extra = {"us_cold": us, "us_warm": sum(s["us_warm"] for s in r["per_shape"]),
             "residual_overhead": us / us0 - 1.0,
             "residual_overhead_note": f"time of the {len(r['per_shape'])} launches at rho={RHO} over the same launches on the "
                                       "budget-0 packing of the same weights (floor = rho: the residual adds rho x bytes and ops)"}
    if has("us_a8"):
        extra["w4a8_time_over_w4a4"] = sum(s["us_a8"] for s in r["per_shape"]) / us
    if has("us_group"):
        extra["group128_time_over_per_token"] = sum(s["us_group"] for s in r["per_shape"]) / us
        extra["group128_note"] = ("mq_gemm_group (per-group activation scales, group 128, P:441; tcgen05 kernel with a "
                                  "per-K-step accumulator drain for M >= 64, the decode kernel with a per-K-step "
                                  "conversion for M <= 32) over the per-token kernel, same launches")
    if has("us_naive"):
        extra["naive3_time_over_fused"] = sum(s["us_naive"] for s in r["per_shape"]) / us
        extra["naive3_note"] = ("the paper's naive pipeline (dense GEMM, separate sparse-block GEMM, reduce-add: mq_gemm_naive) "
                                "over the fused kernel, same launches; paper: 1.9x on RTX 4090 for Qwen3-8B V-proj (Fig.3)")
    # kernel (i) alone: HBM, 2.5 B per element; launch-bound for decode-sized M
    qus, qby = sum(q["us"] for q in r["quant"]), sum(q["bytes"] for q in r["quant"])
    extra["quantize_act"] = {"bound": "hbm", "achieved": qby / (qus * 1e-6) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": qby / (qus * 1e-6) / 1e9 / peaks["hbm_gbs"],
                             "kernel": "mq_quantize_act_kernel, timed alone (graph replay, inputs L2-resident for small M)",
                             "per_shape": [dict(M=q["M"], K=q["K"], us=round(q["us"], 3),
                                                gbs=round(q["bytes"] / (q["us"] * 1e-6) / 1e9, 1)) for q in r["quant"]]}
    if t_hbm >= t_tensor:
        a = by / (us * 1e-6) / 1e9
        return {"bound": "hbm", "achieved": a, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": a / peaks["hbm_gbs"],
                "traffic": traffic, "peak_source": peaks["source"], "kernel": kern, **extra, "per_shape": per_shape}
    a = ops / (us * 1e-6) / 1e12
    return {"bound": "tensor", "achieved": a, "peak": int8_peak, "unit": "TFLOP/s", "frac": a / int8_peak,
            "frac_of_proxy_2x_bf16_burst": a / int8_proxy, "proxy_peak": int8_proxy,
            "traffic": traffic,
            "peak_source": ("measured on this device: mq_probe_int8_peak, a pure tcgen05.mma kind::i8 issue loop (128 x 256 x 32)"
                            if peaks.get("int8_probe_tops") else peaks["source"] + " bf16 burst x 2 (int8 : bf16 nominal ratio; PROXY)"),
            "kernel": kern, **extra, "per_shape": per_shape}


def load_traffic(workload):
    """dram__bytes_read + dram__bytes_write of the dominant kernel per step, from the committed ncu
    summary (profiles/traffic.json, written by hand from an `ncu --set full` capture); None if absent."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        return json.load(open(p)).get(workload)
    return None


def run_ours(args, rank, world):
    import torch
    import synth
    import paper_2606_15652_b200 as mq

    mq.lib()  # no fallback: raises if libmq.so is missing
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    assert torch.cuda.get_device_capability() == (10, 0), "bench.py needs a B200 (sm_100a)"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = load_peaks()
    if "rho_sweep" in synth.CONFIGS[args.workload] and args.sweep_only:
        if rank == 0:
            print(json.dumps({"metric": METRIC, "workload": args.workload, "unit": "us per mq_gemm launch, cold weights",
                              "sweep": measure_sweep(args.workload, torch, mq, synth)}))
        return
    try:
        peaks["int8_probe_tops"] = max(mq.mq_probe_int8_peak(256, 4000), mq.mq_probe_int8_peak(128, 4000))
    except Exception:
        peaks["int8_probe_tops"] = None
    r = measure(args.workload, args.steps, args.warmup, torch, mq, synth, world, dist, local)
    Ms, layers_cfg, calls = r["Ms"], r["layers_cfg"], r["calls"]
    ms_step, e2e_ms = r["ms_step"], r["e2e_ms"]
    out = {
        "metric": METRIC, "value": aggregate_value(r["ops_step"], ms_step, world), "unit": "TOPS",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int4 storage / int8 MMA / int32 acc",
        "data": "synthetic",
        "config": {"workload": f"{args.workload}: M in {Ms} x {[l.name for l in layers_cfg]} (K,N)="
                               f"{[(l.K, l.N) for l in layers_cfg]}, rho={RHO}, block={BS}, fp16 in, bf16 out",
                   "step": f"mq_quantize_act + mq_gemm for each of the {len(calls)} (M, projection) pairs, CUDA-graph "
                           "replay, kernels chained by programmatic dependent launch",
                   "l2": f"step: {N_COPIES} rotating weight copies per layer ({N_COPIES * r['bytes_step'] / len(Ms) / 1e6:.0f} MB of other "
                         "weights between two uses of a copy > 3x L2); per-shape roofline loops: one launch per copy, copies x bytes >= 3x L2",
                   "parallelism": "replicas (no collective on the path)" if world > 1 else "single GPU"},
        "tokens_per_s": world * sum(Ms) / (ms_step * 1e-3),
        "hbm_gbs_step": r["bytes_step"] / (ms_step * 1e-3) / 1e9,
        "w16a16_cublas_bf16": {"ms_per_step": r["ms16"], "speedup_vs_w16a16": r["ms16"] / ms_step,
                               "paper_context": "up to 1.24x over W16A16 on RTX 4090 (P:43)"},
        "roofline": roofline_of(r, peaks, load_traffic(args.workload)),
        "e2e": {"value": world * r["ops_step"] / (e2e_ms * 1e-3) / 1e12, "unit": "TOPS", "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"],
                "api": "mq_linear_host (C ABI, pinned host buffers in and out)",
                "streams": E2E_STREAMS,
                "note": "the step's independent calls go round-robin onto the streams, largest copies first; "
                        "wall clock from the first call to the last stream's synchronize"},
        "gpu_launches": args.steps * 2 * len(calls),
        "int8_peak_tops": {"probe_tcgen05_kind_i8": peaks.get("int8_probe_tops"), "proxy_2x_bf16_burst": 2.0 * peaks["bf16_tflops"],
                           "nominal": 4500.0},
        "clocks": r["clocks"],
        "pack_seconds": round(r["pack_s"], 2),
    }
    del r
    if rank == 0 and world == 1 and args.also and args.also != args.workload:
        # the other regime of the north star (prefill: tensor-bound), same protocol, fewer steps
        torch.cuda.empty_cache()
        r2 = measure(args.also, max(3, args.steps // 4), 3, torch, mq, synth, world, dist, local, with_e2e=False, extras=False)
        rf = roofline_of(r2, peaks, load_traffic(args.also))
        out["also"] = {"workload": args.also, "ms_per_step": r2["ms_step"],
                       "value": r2["ops_step"] / (r2["ms_step"] * 1e-3) / 1e12, "unit": "TOPS",
                       "tokens_per_s": sum(r2["Ms"]) / (r2["ms_step"] * 1e-3),
                       "w16a16_cublas_bf16": {"ms_per_step": r2["ms16"], "speedup_vs_w16a16": r2["ms16"] / r2["ms_step"]},
                       "roofline": rf, "clocks": r2["clocks"]}
        del r2
    if rank == 0 and world == 1 and args.also2:
        # BASELINE.json configs[3] (Qwen3-8B-shaped): density x block sweep on one projection (the full sweep over the
        # four projections is `--workload qwen3_8b`, committed under profiles/)
        wl, _, ln = args.also2.partition(":")
        torch.cuda.empty_cache()
        out["also2"] = {"workload": wl, "layers": ln or "all", "unit": "us per mq_gemm launch, cold weights",
                        "sweep": measure_sweep(wl, torch, mq, synth, [ln] if ln else None)}
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(args.workload, budget_s=20.0)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()

# ------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
# ------------------------------------------------------------------------------------------
_ORACLE_GMACS = 1.0   # rough int64 MAC/ns of the plain oracle on ~8 cores; only sizes the sample


def _oracle_layers(workload):
    import oracle
    import synth
    cfg, _ = workload_shapes(workload)
    out = []
    for i, l in enumerate(cfg["layers"]):
        seed = cfg["seed"] + i
        W = synth.gen_weight(seed, l.N, l.K)
        X = synth.gen_calib(seed, l.K, 256)
        h = oracle.hessian_diag(X).astype(np.float32)
        out.append((seed, l, oracle.algorithm1(W, h, BS, synth.budget_from_density(RHO, l.N, l.K, BS))))
        del W
    return cfg, out


def _oracle_sample_rows(cfg, layers, seconds_per_step):
    """Largest token count m_s (<= max M of the workload) whose pass over all projections is
    estimated to fit in `seconds_per_step`."""
    macs_per_token = sum(l.N * l.K * (1 + RHO) for (_, l, _) in layers)
    m = max(cfg["Ms"])
    while m > 1 and m * macs_per_token / (_ORACLE_GMACS * 1e9) > seconds_per_step:
        m //= 2
    return m


def _oracle_step(layers, acts):
    import oracle
    for (_, l, L), A in zip(layers, acts):
        oracle.forward_timed(A, L)


def cpu_baseline(workload, budget_s=20.0, steps=2):
    import oracle
    import synth
    cfg, layers = _oracle_layers(workload)
    m = _oracle_sample_rows(cfg, layers, budget_s / steps)
    acts = [synth.gen_act(seed + m, m, l.K) for (seed, l, _) in layers]
    best, spent, passes = 1e30, 0.0, 0
    while passes < steps or (spent < budget_s / 2 and passes < 200):   # ~10 s of oracle work in total
        t0 = time.perf_counter()
        _oracle_step(layers, acts)
        dt = time.perf_counter() - t0
        best, spent, passes = min(best, dt), spent + dt, passes + 1
    ops = sum(algo_ops(m, l.K, l.N, L.nnz, BS) for (_, l, L) in layers)
    return {"value": ops / best / 1e12, "unit": "TOPS", "cores": min(oracle.num_threads(), m), "kind": "oracle",
            "threads_available": oracle.num_threads(), "seconds": round(best, 3),
            "build": "oracle as it stands: g++ -O2 -ffp-contract=off -fopenmp, threads not pinned (not the tuned -O3 -march=native build BASELINE.md section 3 sketched)",
            "sample": f"oracle O2+O8+O9 on M={m} tokens x all {len(layers)} projections of {workload} "
                      f"(best of {passes} passes, {spent:.1f} s of oracle work; the oracle parallelises over tokens only)"}


def run_reference(args, rank, world):
    """This tier's reference arm: the CPU oracle, as it stands, on the host cores."""
    if rank != 0:
        return
    import oracle
    import synth
    total = max(1, args.steps + args.warmup)
    cfg, layers = _oracle_layers(args.workload)
    m = _oracle_sample_rows(cfg, layers, 150.0 / total)
    acts = [synth.gen_act(seed + m, m, l.K) for (seed, l, _) in layers]
    for _ in range(args.warmup):
        _oracle_step(layers, acts)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_step(layers, acts)
    dt = (time.perf_counter() - t0) / args.steps
    ops = sum(algo_ops(m, l.K, l.N, L.nnz, BS) for (_, l, L) in layers)
    tops = ops / dt / 1e12
    sample = (f"oracle O2+O8+O9 on M={m} tokens x all {len(layers)} projections of {args.workload} per step "
              f"(bounded sample of the workload)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": tops, "unit": "TOPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8 values / int64 acc / f64 output", "data": "synthetic",
        "config": {"workload": f"{args.workload} (CPU oracle, sample: {sample})"},
        "cpu_baseline": {"value": tops, "unit": "TOPS", "cores": min(oracle.num_threads(), m), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": tops, "unit": "TOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="llama3_8b_decode")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep-only", action="store_true",
                    help="with --workload qwen3_8b: print only the density x block sweep of all four projections")
    ap.add_argument("--also2", default="qwen3_8b:qkv",
                    help="density x block sweep reported under \"also2\" (N=1 only): workload[:layer]; empty string = skip")
    ap.add_argument("--also", default="llama3_8b_prefill",
                    help="second workload reported under \"also\" (N=1 only); empty string = skip")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world)


if __name__ == "__main__":
    main()
