"""bench.py -- SharQ per-linear-layer hot path on B200 (BASELINE.json metric: µs/layer and effective
TFLOPS of prepare + fused sparse/dense FP4 GEMM; prep kernel HBM GB/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path (sharq_prepare -> sharq_linear) over
BASELINE.json configs[2], the configuration the north-star targets are quoted on: the four Llama-3.1-8B-shaped
prefill linears (QKV 4096->6144, O 4096->4096, gate+up 4096->28672, down 14336->4096) at T = 8192 tokens, outliers
x50: 4 prepare + 4 linear launches.  `value` = sum of the layers' nominal 2*T*K*D flop / MEAN step time (device,
CUDA events, inputs resident in HBM, the step replayed from a CUDA graph so launch latency is the GPU's, not
Python's).  `roofline` = the CTA-pair GEMM against the FP4 tensor peak (two denominators: nominal ratio x measured
bf16, and the on-box MMA issue probe), `roofline_prepare` = sharq_prepare against the HBM copy peak.
`e2e` = the same step through the public binding with the activations starting in pinned HOST memory
and every Y copied back to the host inside the timed region (three streams, two buffer sets: the copies of
neighbouring steps overlap, as in a serving loop; PCIe bound).  N > 1: one process per GPU, rows sharded
(each rank runs its own batch, no collective), time = max over ranks.
`extras`: configs[1] (decode, T <= 256: us per layer, HBM roofline of the weight stream), configs[2] at
T = 2048 / 4096, configs[3] (Qwen shapes x NVFP4 / MXFP4 / HiF4), configs[4] (MoE grouped), stream-mode host cost.

`--impl reference` times the CPU oracle (the compiled C one, oracle/sharq_oracle_c.c, as it stands) on a bounded sample
of the same workload on the host cores.  The oracle is never on the product path.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# (name, K, D, norm)  -- Llama-3.1-8B-shaped linears (BASELINE.json configs[1], configs[2])
LLAMA = [("qkv", 4096, 6144, 1), ("o", 4096, 4096, 0), ("gate_up", 4096, 28672, 1), ("down", 14336, 4096, 0)]
DECODE_T = [1, 8, 32, 128, 256]
PREFILL_T = 4096
HEADLINE_T = 8192
L2_BYTES = 126e6
BASE_SEED = 26587


def peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            m = json.load(f)
        return dict(hbm=float(m["hbm_gbs"]), bf16=float(m["bf16_tflops"]),
                    bf16_sustained=float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


def layer_flops(T, K, D):
    return 2.0 * T * K * D


def linear_bytes(T, K, D, fmt=0):
    """Algorithmic HBM bytes of one sharq_linear launch: W codes + group-32 scales read
    once, the prepared activation operands, bf16 Y written."""
    act = T * K * (0.25 + 0.5 + 1 / 32 + 1 / 16 + (1 / 16 if fmt == 0 else 1 / 32)) + 4 * T
    return K * D * (0.5 + 1 / 32) + act + 2.0 * T * D


def prepare_bytes(T, K, fmt=0):
    """Algorithmic HBM bytes of one sharq_prepare launch: 2.906 B/element NVFP4."""
    return T * K * {0: 2.90625, 1: 2.875, 2: 3.0}[fmt] + 4 * T


# ---- seeded synthetic inputs on the device -------------------------------
def device_activations(T, K, seed, outlier_mult=50.0):
    """bf16 [T, K]: N(0,1), 8 seeded outlier channels x outlier_mult, Bernoulli(1e-3) spikes x 20."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    x = torch.randn((T, K), generator=g, device="cuda", dtype=torch.float32)
    ch = torch.randperm(K, generator=g, device="cuda")[:8]
    x[:, ch] *= outlier_mult
    spikes = torch.rand((T, K), generator=g, device="cuda") < 1e-3
    x = torch.where(spikes, x * 20.0, x)
    return x.to(torch.bfloat16)


def device_weight(D, K, seed):
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    return (torch.randn((D, K), generator=g, device="cuda", dtype=torch.float32) * 0.02).to(torch.bfloat16)


def device_gamma(K, seed):
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    return (torch.rand(K, generator=g, device="cuda") + 0.5).to(torch.bfloat16)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def __enter__(self):
        fd, self.path = tempfile.mkstemp(suffix=".csv")
        os.close(fd)
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None
        t0 = time.time()                       # nvidia-smi needs a moment before its first sample
        while self.proc is not None and os.path.getsize(self.path) == 0 and time.time() - t0 < 3.0:
            time.sleep(0.05)
        return self

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            self.proc.wait()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [s.strip() for s in line.split(",")]
                if len(f) < 7:
                    continue
                sm.append(float(f[0])); mx.append(float(f[1]))
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            os.unlink(self.path)
        except (OSError, ValueError):
            pass
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    samples=len(sm), reasons=sorted(reasons))


# ---- our arm ------------------------------------------------------------------------------------
class Workload:
    """Operands of one family of layers resident in HBM: n_sets rotating quantized weight sets, and per (T, layer)
    one x / activation set / Y.  `layers` = [(name, K, D, norm)], `Ts` = token counts."""

    def __init__(self, sq, rank, layers, Ts, n_sets, outlier_mult=50.0, seed_off=0, wq=None):
        import torch
        self.sq, self.layers, self.Ts, self.n_sets = sq, layers, Ts, n_sets
        self.cfg = {n: sq.make_config(sq.NVFP4, sq.NORM_RMS if norm else sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
                    for n, _, _, norm in layers}
        seed = rank_seed(rank) + seed_off
        if wq is None:
            wq = []
            for r in range(n_sets):
                ws = {}
                for i, (n, K, D, _) in enumerate(layers):
                    w = device_weight(D, K, rank_seed(rank) + 10 * r + i)
                    ws[n] = sq.quantize_weight(self.cfg[n], w)
                    del w
                wq.append(ws)
        self.wq = wq
        self.gamma = {K: device_gamma(K, rank_seed(rank) + 5) for K in {k for _, k, _, _ in layers}}
        self.x, self.act, self.Y = {}, {}, {}
        for T in Ts:
            for i, (n, K, D, norm) in enumerate(layers):
                self.x[T, n] = device_activations(T, K, seed + 1000 + 7 * T + i, outlier_mult)
                self.act[T, n] = sq.alloc_act(self.cfg[n], T, K, "cuda")
                self.Y[T, n] = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
        torch.cuda.synchronize()

    def prepare_all(self):
        for T in self.Ts:
            for n, K, D, norm in self.layers:
                self.sq.prepare(self.cfg[n], self.x[T, n], self.gamma[K] if norm else None, out=self.act[T, n])

    def linear_all(self, r):
        for T in self.Ts:
            for n, K, D, norm in self.layers:
                self.sq.linear(self.cfg[n], self.act[T, n], self.wq[r][n], Y=self.Y[T, n])

    def step(self, r):
        for T in self.Ts:
            for n, K, D, norm in self.layers:
                self.sq.prepare(self.cfg[n], self.x[T, n], self.gamma[K] if norm else None, out=self.act[T, n])
                self.sq.linear(self.cfg[n], self.act[T, n], self.wq[r][n], Y=self.Y[T, n])

    @property
    def n_layers(self):
        return len(self.Ts) * len(self.layers)

    def flops(self):
        return sum(layer_flops(T, K, D) for T in self.Ts for _, K, D, _ in self.layers)

    def linear_bytes(self):
        return sum(linear_bytes(T, K, D) for T in self.Ts for _, K, D, _ in self.layers)

    def prepare_bytes(self):
        return sum(prepare_bytes(T, K) for T in self.Ts for _, K, _, _ in self.layers)


def capture(fn):
    """Capture fn() (kernel launches on the current stream through the C ABI) into a CUDA graph."""
    import torch
    fn()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    return g


def replays_of(fns):
    """CUDA-graph replays of the callables (plain stream launches if capture is refused)."""
    try:
        return [capture(f).replay for f in fns], "cuda_graph"
    except Exception as exc:
        return list(fns), f"stream ({type(exc).__name__})"


def timed(replays, steps, warmup, barrier):
    """W warm-up + K timed calls of replays[i % R](), CUDA events on the launching stream; MEAN ms per call."""
    import torch
    for i in range(warmup):
        replays[i % len(replays)]()
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        replays[i % len(replays)]()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1) / steps          # ms per call


def reduce_max_over_ranks(value, dist, device):
    """A step takes as long as its slowest rank: MAX all-reduce of the per-rank device time."""
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_seed(rank):
    """Rows are sharded across ranks with replicated weight SHAPES: every rank draws its own batch."""
    return BASE_SEED * 1000 + 97 * rank


def committed_traffic(name):
    """Per-launch DRAM bytes of the dominant kernel from the committed ncu --set full capture (profiles/), with the
    commit the capture was taken at; None if there is no capture."""
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        d = json.load(f)
    return d.get("traffic_bytes_per_launch"), d.get("captured_at_commit")


def run_ours(args):
    import torch
    import __graft_entry__ as ge
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    ge.build()
    import paper_2606_26587_b200 as sq                    # raises if libsharq.so is missing: no fallback

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v):
        return reduce_max_over_ranks(v, dist, "cuda")

    pk = peaks()
    n_sets = 3                                            # 3 x 116 MB of weights: > 126 MB L2 between re-reads
    steps, warmup = args.steps, max(args.warmup, 3)
    T = HEADLINE_T

    # ---- headline: BASELINE configs[2], the four Llama prefill linears at T = 8192 (the shapes the north-star
    # targets are quoted on): prepare + linear per layer, device-timed, CUDA-graph replay, MEAN of the steps ----
    wl = Workload(sq, rank, LLAMA, [T], n_sets)
    if args.decode_only:                                  # short run for ncu: the configs[1] step alone
        print(json.dumps({"decode_only": True, "decode_configs1": decode_extras(sq, wl, pk, steps, rank)}))
        return
    if args.extras_only:
        ex = prefill_extras(sq, wl, pk, steps)
        if not args.short_extras:
            ex.update(config_extras(sq, wl, pk, steps))
        print(json.dumps({"extras_only": True, "extras": ex}))
        return
    replays, launch_mode = replays_of([lambda r=r: wl.step(r) for r in range(n_sets)])
    with ClockSampler(local) as cs:
        ms_step = timed(replays, steps, warmup, barrier)
        t_end = time.time() + 0.5                         # keep the GPU under the same load until nvidia-smi has sampled
        while cs.proc is not None and time.time() < t_end:
            replays[0]()
        torch.cuda.synchronize()
    clocks = cs.summary()
    ms_step = max_over_ranks(ms_step)
    flops = wl.flops()
    value = world * flops / (ms_step * 1e-3) / 1e12

    if args.headline_only:
        if rank == 0:
            print(json.dumps({"metric": "sharq_layer_effective_tflops", "value": round(value, 2), "unit": "TFLOP/s",
                              "ms_per_step": round(ms_step, 4), "steps": steps, "warmup": warmup, "headline_only": True}))
        return

    # ---- the two kernels of the step alone, same operands and rotation (CUDA events on the launching stream) ----
    wl.prepare_all()
    lin_replays, _ = replays_of([lambda r=r: wl.linear_all(r) for r in range(n_sets)])
    ms_lin = timed(lin_replays, steps, warmup, barrier)
    prep_replays, _ = replays_of([wl.prepare_all])
    ms_prep = timed(prep_replays, steps, warmup, barrier)
    n_lin = wl.n_layers
    mp = mma_issue_peaks(sq) if rank == 0 else None
    # tensor roofline: the layer's dense path does 2TKD flop at the dense FP4 rate and its sparse path
    # 2TKD logical flop at the sparse rate; t_min = 2TKD / P_dn + 2TKD / P_sp.  As one number: achieved = 4TKD / t
    # against the combined peak 2 / (1 / P_dn + 1 / P_sp), so frac = t_min / t.
    p_dn, p_sp = 4 * pk["bf16_sustained"], 8 * pk["bf16_sustained"]              # nominal ratio x measured bf16 (TFLOP/s)
    comb = lambda a, b: 2.0 / (1.0 / a + 1.0 / b)
    ach = 2.0 * flops / (ms_lin * 1e-3) / 1e12
    traffic, traffic_commit = committed_traffic("linear_pair_traffic_r2.json")
    roofline = dict(kernel="sharq_linear_pair_kernel (CTA-pair tcgen05 tiles; the 4 sharq_linear launches of the step)",
                    bound="tensor", achieved=round(ach, 1), peak=round(comb(p_dn, p_sp), 1), unit="TFLOP/s",
                    frac=round(ach / comb(p_dn, p_sp), 4),
                    peak_definition=f"2/(1/P_dense + 1/P_sparse), P_dense = 4 x, P_sparse = 8 x the {pk['source']} sustained "
                                    "bf16 cuBLAS rate (nominal 9 / 18 PF over 2.25 PF); achieved = 4TKD / t (2TKD per path)",
                    traffic=traffic, traffic_source=("ncu --set full capture at commit " + str(traffic_commit)) if traffic else None,
                    launches_per_step=n_lin, avg_launch_us=round(ms_lin * 1e3 / n_lin, 2),
                    algorithmic_flop_per_launch=round(2.0 * flops / n_lin), share_of_step=round(ms_lin / ms_step, 3))
    if mp is not None:
        q_dn, q_sp = mp["dense"]["sustained"], mp["sparse"]["sustained"]
        r_dn, r_sp = mp["dense_random_operands"]["sustained"], mp["sparse_random_operands"]["sustained"]
        roofline.update(peak_probe=round(comb(q_dn, q_sp), 1), frac_probe=round(ach / comb(q_dn, q_sp), 4),
                        peak_probe_definition="same formula with P_dense / P_sparse measured on this GPU by the MMA issue "
                                              "probe (sharq_diag.h), sustained, CONSTANT operand bytes; SURVEY.md 8(d) names "
                                              "the probe the applicable peak",
                        peak_probe_random=round(comb(r_dn, r_sp), 1), frac_probe_random=round(ach / comb(r_dn, r_sp), 4),
                        peak_probe_random_definition="the same probe fed pseudo-random operand bits: the GPU is power capped "
                                                     "(clocks line), and a tensor pipe switching real data bits sustains a "
                                                     "lower clock than one fed constants; real FP4 activations / weights "
                                                     "lie between the two",
                        mma_issue_probe_tflops=mp)
    gbs = wl.prepare_bytes() / (ms_prep * 1e-3) / 1e9
    ptraffic, ptraffic_commit = committed_traffic("prepare_traffic_r2.json")
    roofline_prepare = dict(kernel="sharq_prepare_row_kernel (the 4 sharq_prepare launches of the step)", bound="hbm",
                            achieved=round(gbs, 1), peak=pk["hbm"], unit="GB/s", frac=round(gbs / pk["hbm"], 4),
                            traffic=ptraffic,
                            traffic_source=("ncu --set full capture at commit " + str(ptraffic_commit)) if ptraffic else None,
                            peak_source=pk["source"], launches_per_step=n_lin,
                            avg_launch_us=round(ms_prep * 1e3 / n_lin, 2),
                            algorithmic_bytes_per_launch=round(wl.prepare_bytes() / n_lin),
                            share_of_step=round(ms_prep / ms_step, 3),
                            per_launch=per_launch_prepare(sq, wl, pk, steps))

    # ---- per-layer us (BASELINE metric "us/layer"): prepare + linear, weights rotated ----
    layers = {}
    for n, K, D, norm in LLAMA:
        reps, _ = replays_of([lambda r=r, n=n, K=K, norm=norm: (
            sq.prepare(wl.cfg[n], wl.x[T, n], wl.gamma[K] if norm else None, out=wl.act[T, n]),
            sq.linear(wl.cfg[n], wl.act[T, n], wl.wq[r][n], Y=wl.Y[T, n])) for r in range(n_sets)])
        ms = timed(reps, max(steps // 2, 6), 3, lambda: None)
        layers[f"{n}_T{T}"] = dict(us=round(ms * 1e3, 1), tflops=round(layer_flops(T, K, D) / ms / 1e9, 1))

    # ---- e2e: activations start in pinned host memory, every Y is read back (C ABI, H2D + D2H inside the region) ----
    # The step moves 1.1 GB over PCIe against 1.2 ms of kernels, so it is pipelined like a serving loop: three streams
    # (host->device, compute, device->host), two sets of device x / Y buffers, plain stream launches (the launch cost is
    # noise here).  Step s + 1's inputs travel while step s computes and step s - 1's results are still going back; every
    # step still copies ITS inputs in and ITS results out, and the region ends when the last Y is on the host.
    xh = {k: v.cpu().pin_memory() for k, v in wl.x.items()}
    yh = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in wl.Y.items()}
    xs = [wl.x, {k: torch.empty_like(v) for k, v in wl.x.items()}]
    ys = [wl.Y, {k: torch.empty_like(v) for k, v in wl.Y.items()}]
    side = torch.cuda.Stream()                            # device->host copies
    up = torch.cuda.Stream()                              # host->device copies (PCIe is duplex)

    def e2e_run(n_steps):
        main = torch.cuda.current_stream()
        start = torch.cuda.Event()
        start.record(main)
        up.wait_event(start)
        side.wait_event(start)
        x_free = [None, None]                             # main: the last prepare that read x set b has been issued
        y_copied = [{}, {}]                               # side: Y set b, layer n is on the host
        for s_i in range(n_steps):
            b, r = s_i & 1, s_i % n_sets
            ready = {}
            with torch.cuda.stream(up):
                if x_free[b] is not None:
                    up.wait_event(x_free[b])
                for n, K, D, norm in LLAMA:
                    xs[b][T, n].copy_(xh[T, n], non_blocking=True)
                    ready[n] = torch.cuda.Event()
                    ready[n].record(up)
            for n, K, D, norm in LLAMA:
                main.wait_event(ready[n])
                sq.prepare(wl.cfg[n], xs[b][T, n], wl.gamma[K] if norm else None, out=wl.act[T, n])
                if n in y_copied[b]:
                    main.wait_event(y_copied[b][n])       # the copy of this buffer's previous contents has left
                sq.linear(wl.cfg[n], wl.act[T, n], wl.wq[r][n], Y=ys[b][T, n])
                done = torch.cuda.Event()
                done.record(main)
                with torch.cuda.stream(side):
                    side.wait_event(done)
                    yh[T, n].copy_(ys[b][T, n], non_blocking=True)
                    y_copied[b][n] = torch.cuda.Event()
                    y_copied[b][n].record(side)
            x_free[b] = torch.cuda.Event()
            x_free[b].record(main)
        main.wait_stream(side)                            # the region ends when every Y is on the host
        main.wait_stream(up)

    def e2e_timed(n_steps, n_warm):
        e2e_run(n_warm)
        torch.cuda.synchronize()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        e2e_run(n_steps)
        e1.record()
        torch.cuda.synchronize()
        barrier()
        return e0.elapsed_time(e1) / n_steps

    e2e_mode = "stream launches, 3 streams, 2 buffer sets (copies of neighbouring steps overlap)"
    ms_e2e = max_over_ranks(e2e_timed(max(min(steps, 10), 4), 3))
    h2d = sum(v.numel() * 2 for v in xh.values())
    d2h = sum(v.numel() * 2 for v in yh.values())
    del xh, yh, xs, ys

    extras = {}
    if rank == 0:
        extras["decode_configs1"] = decode_extras(sq, wl, pk, steps, rank)
        extras["host_cost"] = host_cost(sq, wl)
        extras.update(prefill_extras(sq, wl, pk, steps, mp))
        extras.update(config_extras(sq, wl, pk, steps, mp))

    if rank != 0:
        dist.destroy_process_group()
        return
    line = {
        "metric": "sharq_layer_effective_tflops", "value": round(value, 2), "unit": "TFLOP/s",
        "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": round(ms_step, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "fp4_e2m1(fp32 acc)",
        "data": "synthetic",
        "config": {"workload": f"BASELINE configs[2]: Llama-3.1-8B prefill linears (qkv 4096->6144, o 4096->4096, gate_up "
                               f"4096->28672, down 14336->4096) at T = {T} tokens, NVFP4, pairwise 4:8, outliers x50, "
                               "sharq_prepare + sharq_linear per layer; value = sum of the layers' nominal 2TKD / step time",
                   "l2": "inputs larger than L2: every layer streams 67-235 MB of activations, and 3 rotating weight sets",
                   "launch": launch_mode, "timing": "mean over the declared steps, CUDA events on the launching stream",
                   "parallelism": f"rows x{world} (replicated weights, no collective)"},
        "us_per_layer_mean": round(ms_step * 1e3 / n_lin, 2),
        "clocks": clocks,
        "e2e": {"value": round(world * flops / (ms_e2e * 1e-3) / 1e12, 2), "unit": "TFLOP/s",
                "ms_per_step": round(ms_e2e, 4), "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "launch": e2e_mode, "note": "PCIe-bound: the step moves 1.1 GB between host and device"},
        "gpu_launches": 2 * n_lin * steps,
        "roofline": roofline,
        "roofline_prepare": roofline_prepare,
        "cpu_baseline": cpu_baseline_sample() if world == 1 else None,
        "layers": layers,
        "layers_note": "prepare + linear per layer, weight sets rotated",
        "extras": extras,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def per_launch_prepare(sq, wl, pk, steps):
    """Each sharq_prepare launch of the headline step alone, three input sets rotated (> 126 MB between re-reads).
    Timed after a short idle: the preceding GEMM loops leave the GPU in its power-capped clock state, which the whole-step
    and prepare_all timings above include and a prepare kernel running alone does not cause."""
    import torch
    out = {}
    T = wl.Ts[0]
    torch.cuda.synchronize()
    time.sleep(0.5)
    for i, (n, K, D, norm) in enumerate(wl.layers):
        xs = [wl.x[T, n]] + [device_activations(T, K, BASE_SEED + 70 + 3 * i + j) for j in range(2)]
        acts = [wl.act[T, n]] + [sq.alloc_act(wl.cfg[n], T, K, "cuda") for _ in range(2)]
        reps = [lambda j=j: sq.prepare(wl.cfg[n], xs[j], wl.gamma[K] if norm else None, out=acts[j]) for j in range(3)]
        ms = timed(reps, max(steps, 12), 3, lambda: None)
        gbs = prepare_bytes(T, K) / (ms * 1e-3) / 1e9
        out[f"{n}_K{K}_{'rms' if norm else 'none'}"] = dict(us=round(ms * 1e3, 1), GBps=round(gbs, 1),
                                                             frac_of_hbm=round(gbs / pk["hbm"], 4))
        del xs, acts
    wl.prepare_all()                                       # act sets of the workload hold their own rows again
    return out


def decode_extras(sq, wl0, pk, steps, rank):
    """BASELINE configs[1] (last round's headline): the four Llama linears at T in {1, 8, 32, 128, 256}, 20 prepare +
    20 linear launches per step, weight-bandwidth bound: us per layer and the HBM roofline of the linear launches."""
    import torch
    wl = Workload(sq, rank, LLAMA, DECODE_T, wl0.n_sets, seed_off=31, wq=wl0.wq)
    reps, mode = replays_of([lambda r=r: wl.step(r) for r in range(wl.n_sets)])
    ms_step = timed(reps, steps, 3, lambda: None)
    wl.prepare_all()
    lin, _ = replays_of([lambda r=r: wl.linear_all(r) for r in range(wl.n_sets)])
    ms_lin = timed(lin, steps, 3, lambda: None)
    ach = wl.linear_bytes() / (ms_lin * 1e-3) / 1e9
    traffic, commit = committed_traffic("linear_decode_traffic_r2.json")
    out = dict(ms_per_step=round(ms_step, 4), effective_tflops=round(wl.flops() / ms_step / 1e9, 1),
               us_per_layer_mean=round(ms_step * 1e3 / wl.n_layers, 2), launch=mode,
               roofline=dict(kernel="sharq_linear (20 decode launches: split-K clusters, 128 x 256 tiles, CTA pairs at T = 256)",
                             bound="hbm", achieved=round(ach, 1), peak=pk["hbm"], unit="GB/s", frac=round(ach / pk["hbm"], 4),
                             traffic=traffic, traffic_source=("ncu capture at commit " + str(commit)) if traffic else None,
                             avg_launch_us=round(ms_lin * 1e3 / wl.n_layers, 2),
                             algorithmic_bytes_per_launch=round(wl.linear_bytes() / wl.n_layers)),
               layers={})
    for n, K, D, norm in LLAMA:
        for T in DECODE_T:
            reps, _ = replays_of([lambda r=r, T=T, n=n, K=K, norm=norm: (
                sq.prepare(wl.cfg[n], wl.x[T, n], wl.gamma[K] if norm else None, out=wl.act[T, n]),
                sq.linear(wl.cfg[n], wl.act[T, n], wl.wq[r][n], Y=wl.Y[T, n])) for r in range(wl.n_sets)])
            # one graph = 3 layers on 3 weight sets; the copies of one layer (<= 3 x 65 MB) plus the other traffic of the
            # chain keep the weights cold for all but the two small shapes (stated per entry)
            ms = timed(reps, max(steps, 12), 3, lambda: None)
            w_mb = K * D * (0.5 + 1 / 32 + 1 / 16) / 1e6
            out["layers"][f"{n}_T{T}"] = dict(us=round(ms * 1e3, 2), weights="cold" if 3 * w_mb > 126 else "partly L2-resident")
            if T <= 8:   # the same layer as ONE fused launch (sharq_prepare_linear single_launch = 1)
                reps1, _ = replays_of([lambda r=r, T=T, n=n, K=K, norm=norm: sq.prepare_linear(
                    wl.cfg[n], wl.x[T, n], wl.wq[r][n], wl.gamma[K] if norm else None, act=wl.act[T, n], Y=wl.Y[T, n],
                    single_launch=True) for r in range(wl.n_sets)])
                out["layers"][f"{n}_T{T}"]["single_launch_us"] = round(timed(reps1, max(steps, 12), 3, lambda: None) * 1e3, 2)
    del wl
    torch.cuda.empty_cache()
    return out


def host_cost(sq, wl):
    """Host-side cost of one sharq_linear / sharq_prepare call in STREAM mode (no CUDA graph): argument checks, tensor-map
    encodes, the launch itself.  Wall time of back-to-back calls on a shape whose kernel is shorter than the call."""
    import torch
    cfg = wl.cfg["o"]
    x = device_activations(1, 4096, BASE_SEED + 9)
    act = sq.prepare(cfg, x)
    Y = torch.empty((1, 4096), dtype=torch.bfloat16, device="cuda")
    wq = wl.wq[0]["o"]
    out = {}
    for name, fn in (("sharq_linear", lambda: sq.linear(cfg, act, wq, Y=Y)), ("sharq_prepare", lambda: sq.prepare(cfg, x, out=act))):
        for _ in range(50):
            fn()
        torch.cuda.synchronize()
        n = 2000
        t0 = time.perf_counter()
        for _ in range(n):
            fn()
        t1 = time.perf_counter()
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        out[name] = dict(us_per_call_host=round((t1 - t0) / n * 1e6, 2), us_per_call_incl_drain=round((t2 - t0) / n * 1e6, 2))
    out["note"] = ("python + ctypes + C ABI + cudaLaunchKernelEx per call, T = 1, K = D = 4096; the graph-replayed numbers "
                   "above do not pay this")
    return out


def mma_issue_peaks(sq):
    """FP4 tensor peaks measured on this GPU by the library's MMA issue-rate probe (sharq_mma_peak_launch):
    dense-only, sparse-only, and the fused per-k-block sequence with its scale-factor copies; `burst` = one
    2 ms launch, `sustained` = the last of back-to-back launches over ~1.5 s (power-capped clocks)."""
    import torch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    out = {}
    for name, mode in (("dense", 1), ("sparse", 2), ("fused_with_sf_copies", 7), ("dense_random_operands", 9),
                       ("sparse_random_operands", 10), ("fused_random_operands", 15)):
        paths = (1 if mode & 1 else 0) + (1 if mode & 2 else 0)
        res = {}
        for kind, iters, secs in (("burst", 4000, 0.0), ("sustained", 40000, 1.5)):
            sq.mma_peak_launch(mode, 100)
            torch.cuda.synchronize()
            t_end = time.time() + secs
            while True:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); sq.mma_peak_launch(mode, iters); e1.record()
                torch.cuda.synchronize()
                if time.time() >= t_end:
                    break
            ms = e0.elapsed_time(e1)
            res[kind] = round(paths * 2.0 * 128 * 256 * 256 * iters * (n_sm // 2 * 2) / ms / 1e9, 1)
        out[name] = res
    return out


def prefill_extras(sq, wl, pk, steps, mp=None):
    """configs[2] family at T = 4096 next to the T = 8192 headline: sharq_linear alone, CUDA events, rotating weight
    sets.  FP4 tensor peak = measured bf16 peak x 4 (dense, nominal ratio 9 / 2.25 PFLOP/s) and x 8 (2:4 sparse) and,
    second denominator, the on-box MMA issue probe; t_min = 2TKD / P_dense + 2TKD / P_sparse."""
    import torch
    out = {"fp4_dense_peak_tflops": round(4 * pk["bf16_sustained"], 1), "fp4_sparse_peak_tflops": round(8 * pk["bf16_sustained"], 1),
           "peak_note": f"4x / 8x the {pk['source']} sustained bf16 cuBLAS rate", "linear_T4096": {}}
    T = PREFILL_T
    p_dn, p_sp = 4 * pk["bf16_sustained"] * 1e12, 8 * pk["bf16_sustained"] * 1e12
    if mp is None:
        mp = mma_issue_peaks(sq)
    out["mma_issue_probe_tflops"] = mp
    q_dn, q_sp = mp["dense"]["sustained"] * 1e12, mp["sparse"]["sustained"] * 1e12
    for i, (n, K, D, norm) in enumerate(LLAMA):
        x = device_activations(T, K, BASE_SEED + 50 + i)
        act = sq.alloc_act(wl.cfg[n], T, K, "cuda")
        Y = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
        sq.prepare(wl.cfg[n], x, wl.gamma[K] if norm else None, out=act)
        reps = [lambda r=r: sq.linear(wl.cfg[n], act, wl.wq[r][n], Y=Y) for r in range(wl.n_sets)]
        ms = timed(reps, max(steps, 10), 3, lambda: None)
        fl = layer_flops(T, K, D)
        t_min = fl / p_dn + fl / p_sp
        out["linear_T4096"][n] = dict(us=round(ms * 1e3, 1), effective_tflops=round(fl / ms / 1e9, 1),
                                      frac_of_fp4_roofline=round(t_min / (ms * 1e-3), 4),
                                      frac_of_mma_probe=round((fl / q_dn + fl / q_sp) / (ms * 1e-3), 4),
                                      plan=sq.linear_plan(wl.cfg[n], T, D, K))
        del x, act, Y
    # residual-stream add fused into the preparation (sharq_prepare_add) against the same work
    # as two launches (a bf16 add kernel, then sharq_prepare).  Algorithmic bytes of the fused pass: the prepare
    # bytes + 2 (residual read) + 2 (new stream written) per element.
    Tp, K = 8192, 4096
    xs = [device_activations(Tp, K, BASE_SEED + 90 + j) for j in range(3)]
    rs = [device_activations(Tp, K, BASE_SEED + 95 + j, outlier_mult=10.0) for j in range(3)]
    acts = [sq.alloc_act(wl.cfg["qkv"], Tp, K, "cuda") for _ in xs]
    fused = [lambda j=j: sq.prepare_add(wl.cfg["qkv"], xs[j], rs[j], wl.gamma[K], out=acts[j]) for j in range(3)]
    ms_f = timed(fused, max(steps, 12), 3, lambda: None)

    def unfused(j):
        rs[j].add_(xs[j])
        sq.prepare(wl.cfg["qkv"], rs[j], wl.gamma[K], out=acts[j])
    ms_u = timed([lambda j=j: unfused(j) for j in range(3)], max(steps, 12), 3, lambda: None)
    by = prepare_bytes(Tp, K) + 4.0 * Tp * K
    out["prepare_add"] = {f"T{Tp}_K{K}_rms": dict(us=round(ms_f * 1e3, 1), GBps=round(by / (ms_f * 1e-3) / 1e9, 1),
                                               frac_of_hbm=round(by / (ms_f * 1e-3) / 1e9 / pk["hbm"], 4),
                                               unfused_us=round(ms_u * 1e3, 1),
                                               unfused_note="torch bf16 add_ kernel + sharq_prepare (two launches)")}
    del xs, rs, acts
    # SURVEY.md 8(f) N1, second fusion: SiLU(gate) * up in front of the down projection's preparation
    # (sharq_prepare_swiglu) against torch's silu * mul kernels + sharq_prepare.  Algorithmic bytes of the fused pass:
    # the prepare bytes + 2 (the second input) per element; h never goes to HBM.
    Tp, K = 8192, 14336
    cfg = wl.cfg["down"]
    gus = [device_activations(Tp, 2 * K, BASE_SEED + 110 + j, outlier_mult=5.0) for j in range(2)]    # [T, 2K] gate | up
    acts = [sq.alloc_act(cfg, Tp, K, "cuda") for _ in gus]
    ms_f = timed([lambda j=j: sq.prepare_swiglu(cfg, gus[j][:, :K], gus[j][:, K:], out=acts[j]) for j in range(2)],
                 max(steps, 12), 3, lambda: None)
    hbuf = torch.empty((Tp, K), dtype=torch.bfloat16, device="cuda")

    def unfused_swiglu(j):
        torch.mul(torch.nn.functional.silu(gus[j][:, :K]), gus[j][:, K:], out=hbuf)
        sq.prepare(cfg, hbuf, out=acts[j])
    ms_u = timed([lambda j=j: unfused_swiglu(j) for j in range(2)], max(steps, 12), 3, lambda: None)
    by = prepare_bytes(Tp, K) + 2.0 * Tp * K
    out["prepare_swiglu"] = {f"T{Tp}_K{K}": dict(us=round(ms_f * 1e3, 1), GBps=round(by / (ms_f * 1e-3) / 1e9, 1),
                                                 frac_of_hbm=round(by / (ms_f * 1e-3) / 1e9 / pk["hbm"], 4),
                                                 unfused_us=round(ms_u * 1e3, 1),
                                                 unfused_note="torch silu + mul kernels (MUFU exp, not bit-restatable) + sharq_prepare")}
    del gus, acts, hbuf
    return out


QWEN = [("qkv", 3584, 4608, 1), ("o", 3584, 3584, 0), ("gate_up", 3584, 37888, 1), ("down", 18944, 3584, 0)]


def config_extras(sq, wl, pk, steps, mp=None):
    """BASELINE.json configs[2] (T and outlier sweep), configs[3] (Qwen2.5-7B shapes x formats) and configs[4] (MoE
    grouped): sharq_linear alone and sharq_prepare alone, CUDA events, rotating weights / inputs."""
    import torch
    p_dn, p_sp = 4 * pk["bf16_sustained"] * 1e12, 8 * pk["bf16_sustained"] * 1e12
    out = {"config3_T_sweep": {}, "config4_qwen_formats": {}, "config5_moe": {}}
    q = (mp["dense"]["sustained"] * 1e12, mp["sparse"]["sustained"] * 1e12) if mp else None

    def lin_entry(ms, T, K, D, fmt=0):
        fl = layer_flops(T, K, D)
        e = dict(us=round(ms * 1e3, 1), effective_tflops=round(fl / ms / 1e9, 1),
                 frac_of_fp4_roofline=round((fl / p_dn + fl / p_sp) / (ms * 1e-3), 4),
                 GBps=round(linear_bytes(T, K, D, fmt) / ms / 1e6, 1))
        if q:
            e["frac_of_mma_probe"] = round((fl / q[0] + fl / q[1]) / (ms * 1e-3), 4)
        return e

    for T in (2048,):                            # T = 4096 is in linear_T4096, T = 8192 is the headline
        for i, (n, K, D, norm) in enumerate(LLAMA):
            x = device_activations(T, K, BASE_SEED + 300 + i, outlier_mult=(10.0, 50.0, 200.0)[i % 3])
            act = sq.prepare(wl.cfg[n], x, wl.gamma[K] if norm else None)
            Y = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
            reps = [lambda r=r: sq.linear(wl.cfg[n], act, wl.wq[r][n], Y=Y) for r in range(wl.n_sets)]
            out["config3_T_sweep"][f"{n}_T{T}"] = lin_entry(timed(reps, max(steps // 2, 8), 3, lambda: None), T, K, D)
            del x, act, Y
    T = 4096
    for fmt, fname in ((sq.NVFP4, "nvfp4"), (sq.MXFP4, "mxfp4"), (sq.HIF4, "hif4")):
        for i, (n, K, D, norm) in enumerate(QWEN):
            cfg = sq.make_config(fmt, sq.NORM_RMS if norm else sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
            wqs = [sq.quantize_weight(cfg, device_weight(D, K, BASE_SEED + 400 + 10 * r + i)) for r in range(2)]
            x = device_activations(T, K, BASE_SEED + 450 + i)
            g = device_gamma(K, BASE_SEED + 460)
            act = sq.alloc_act(cfg, T, K, "cuda")
            Y = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
            # prepare alone: input / output sets rotated so that every re-read follows > 126 MB of other traffic
            n_rot = max(2, int(130e6 // (T * K * 2.9)) + 1)
            xs = [x] + [device_activations(T, K, BASE_SEED + 470 + j) for j in range(n_rot - 1)]
            acts = [act] + [sq.alloc_act(cfg, T, K, "cuda") for _ in range(n_rot - 1)]
            ms_p = timed([lambda j=j: sq.prepare(cfg, xs[j], g if norm else None, out=acts[j]) for j in range(n_rot)],
                         max(steps // 2, 8), 3, lambda: None)
            sq.prepare(cfg, x, g if norm else None, out=act)
            del xs, acts
            ws = sq._bytes(sq.linear_workspace(cfg, T, D, K), "cuda") if fmt == sq.HIF4 else None
            ms_l = timed([lambda r=r: sq.linear(cfg, act, wqs[r], Y=Y, workspace=ws) for r in range(2)],
                         max(steps // 2, 8), 3, lambda: None)
            e = lin_entry(ms_l, T, K, D, fmt)
            if fmt == sq.HIF4:                   # no FP4-rate tensor path for HiF4: bf16 roofline (dense + 2:4 sparse)
                fl = layer_flops(T, K, D)
                pb = pk["bf16_sustained"] * 1e12
                del e["frac_of_fp4_roofline"]
                e.pop("frac_of_mma_probe", None)
                e["frac_of_bf16_roofline"] = round((fl / pb + fl / (2 * pb)) / (ms_l * 1e-3), 4)
                e["note"] = "dequantise A (every call; W once, by sharq_quantize_weight) + dense bf16 GEMM over 2K"
            e["prepare_us"] = round(ms_p * 1e3, 1)
            e["prepare_GBps"] = round(prepare_bytes(T, K, fmt) / ms_p / 1e6, 1)
            out["config4_qwen_formats"][f"{fname}_{n}"] = e
            del wqs, x, act, Y
    # configs[4]: 4096 tokens, 128 experts, top-8 of a seeded softmax router; rows grouped by expert into
    # 128-row-aligned slots; gate+up 2048 -> 1536 and down 768 -> 2048 as ONE grouped launch each
    E = 128
    gen = torch.Generator(device="cuda").manual_seed(BASE_SEED + 500)
    logits = torch.randn((4096, E), generator=gen, device="cuda")
    top = torch.topk(torch.softmax(logits, dim=1), 8, dim=1).indices.reshape(-1)
    counts = torch.bincount(top, minlength=E).cpu().numpy()
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    padded = int((-(-counts // 128) * 128).sum())
    for n, K, D in (("gate_up", 2048, 1536), ("down", 768, 2048)):
        cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
        parts = [sq.quantize_weight(cfg, device_weight(D, K, BASE_SEED + 510 + e % 8)) for e in range(E)]
        wq = dict(codes=torch.cat([q["codes"] for q in parts]), sf_sp=torch.cat([q["sf_sp"] for q in parts]),
                  sf_dn=torch.cat([q["sf_dn"] for q in parts]), ts_w=torch.cat([q["ts_w"] for q in parts]), D=D, K=K)
        del parts
        x = device_activations(padded, K, BASE_SEED + 520)          # every slot row filled: prepare is per row
        act = sq.alloc_act(cfg, padded, K, "cuda")
        Y = torch.empty((padded, D), dtype=torch.bfloat16, device="cuda")
        x2, act2 = device_activations(padded, K, BASE_SEED + 521), sq.alloc_act(cfg, padded, K, "cuda")
        ms_p = timed([lambda: sq.prepare(cfg, x, out=act), lambda: sq.prepare(cfg, x2, out=act2)], max(steps // 2, 8), 3,
                     lambda: None)                                   # two sets: 2 x (62-166 MB in + 28-75 MB out) > L2
        sq.prepare(cfg, x, out=act)
        del x2, act2
        offs_dev = torch.from_numpy(offsets).cuda()
        ms_l = timed([lambda: sq.linear_grouped(cfg, offs_dev, act, wq, D, Y=Y)], max(steps // 2, 8), 3, lambda: None)
        rows = int(counts.sum())
        w_bytes = E * K * D * (0.5 + 1 / 32)
        by = w_bytes + rows * K * 0.90625 + 2.0 * rows * D
        out["config5_moe"][n] = dict(us=round(ms_l * 1e3, 1), rows=rows, padded_rows=padded,
                                     effective_tflops=round(2.0 * rows * K * D / ms_l / 1e9, 1),
                                     GBps=round(by / ms_l / 1e6, 1), frac_of_hbm=round(by / ms_l / 1e6 / pk["hbm"], 4),
                                     prepare_us=round(ms_p * 1e3, 1),
                                     prepare_GBps=round(prepare_bytes(padded, K) / ms_p / 1e6, 1),
                                     note=f"all {E} experts' weights = {w_bytes / 1e6:.0f} MB per launch (the L2 holds 126 MB: "
                                          "partly resident across repeats)")
        del wq, x, act, Y
    out["config5_moe"]["rows_per_expert"] = dict(min=int(counts.min()), max=int(counts.max()))
    return out


# ---- CPU oracle legs (the only places bench.py executes oracle/) ---------------------------------------
# the baseline IS the oracle, compiled (-O2, no fast-math, no FMA contraction), rows parallel over
# the host cores: oracle/sharq_oracle_c.c, which tests/test_oracle_c.py holds byte-identical to the numpy oracle.


def sample_desc(t_prep, t_lin):
    return (f"headline workload (configs[2] shapes qkv/o/gate_up/down, T = {HEADLINE_T}): the compiled C oracle "
            f"(oracle/sharq_oracle_c.c, gcc -O2 -ffp-contract=off -fno-fast-math, OpenMP over rows) as it stands; "
            f"prepare timed on {t_prep} of the {HEADLINE_T} rows of every layer, the fp64 linear on {t_lin} seeded full "
            f"rows x all D output features of every layer; value = the whole step's nominal 2TKD / (each part's time "
            f"scaled linearly to {HEADLINE_T} rows) -- EXTRAPOLATED from the sample; weight quantization (offline) not timed")


def oracle_sample_setup(t_prep, t_lin):
    import sharq_inputs as si
    from oracle import c_oracle as co
    rng = np.random.Generator(np.random.Philox(BASE_SEED))
    items = []
    for i, (n, K, D, norm) in enumerate(LLAMA):
        x, g = si.activations(t_prep, K, config=2, extra=i), si.gamma(K, 2)
        rows = np.sort(rng.choice(t_prep, size=t_lin, replace=False))
        wq = co.quantize_weight(si.weight(D, K, config=2, extra=i))
        items.append((n, K, D, norm, x, g, rows, wq))
    return co, items


def oracle_sample_step(co, items):
    """One bounded sample of the step.  Returns (prepare seconds, linear seconds, threads used)."""
    tp = tl = 0.0
    nt = 1
    for n, K, D, norm, x, g, rows, wq in items:
        t0 = time.perf_counter()
        p = co.prepare(x, co.NVFP4, norm, g if norm else None, want_X=False)
        t1 = time.perf_counter()
        co.linear(p, wq, rows=rows)
        tl += time.perf_counter() - t1
        tp += t1 - t0
        nt = p["threads"]
    return tp, tl, nt


def oracle_value(tp, tl, t_prep, t_lin):
    """Whole-step TFLOP/s with each part scaled linearly to the full row count."""
    est = tp * HEADLINE_T / t_prep + tl * HEADLINE_T / t_lin
    fl = sum(layer_flops(HEADLINE_T, K, D) for _, K, D, _ in LLAMA)
    return fl / est / 1e12, est


def cpu_baseline_sample(t_prep=HEADLINE_T, t_lin=32):
    co, items = oracle_sample_setup(t_prep, t_lin)
    oracle_sample_step(co, items)                                    # warm
    t0 = time.perf_counter()
    acc, reps = [0.0, 0.0], 0
    while reps < 1 or time.perf_counter() - t0 < 10.0:
        tp, tl, nt = oracle_sample_step(co, items)
        acc[0] += tp
        acc[1] += tl
        reps += 1
    tp, tl = acc[0] / reps, acc[1] / reps
    v, est = oracle_value(tp, tl, t_prep, t_lin)
    return dict(value=round(v, 6), unit="TFLOP/s", cores=nt, kind="oracle", sample=sample_desc(t_prep, t_lin),
                host_cores=os.cpu_count(), prepare_s=round(tp, 3), linear_sample_s=round(tl, 3),
                extrapolated_step_s=round(est, 1), extrapolated=True)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    t_prep, t_lin = HEADLINE_T, 32                                    # the cpu_baseline leg's sample: 1.3 s per step on the box's 16 cores
    co, items = oracle_sample_setup(t_prep, t_lin)
    steps, warmup = args.steps, args.warmup
    budget = 150.0                                                    # seconds: keep the whole run to minutes
    t_all = time.perf_counter()
    for _ in range(warmup):
        oracle_sample_step(co, items)
        if time.perf_counter() - t_all > budget / 3:
            break
    t0 = time.perf_counter()
    acc, done, nt = [0.0, 0.0], 0, 1
    for _ in range(steps):
        tp, tl, nt = oracle_sample_step(co, items)
        acc[0] += tp
        acc[1] += tl
        done += 1
        if time.perf_counter() - t0 > budget:
            break
    dt = (time.perf_counter() - t0) / done
    v, est = oracle_value(acc[0] / done, acc[1] / done, t_prep, t_lin)
    v = round(v, 6)
    desc = sample_desc(t_prep, t_lin)
    print(json.dumps({
        "impl": "reference", "metric": "sharq_layer_effective_tflops", "value": v, "unit": "TFLOP/s",
        "n_gpus": world, "steps": done, "warmup": warmup, "ms_per_step": round(dt * 1e3, 3), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE configs[2] (bounded sample per step; ms_per_step is the sample's wall time, "
                               "value is extrapolated to the whole step): " + desc},
        "cpu_baseline": dict(value=v, unit="TFLOP/s", kind="oracle", cores=nt, sample=desc, host_cores=os.cpu_count(),
                             extrapolated_step_s=round(est, 1), extrapolated=True),
        "e2e": {"value": v, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--headline-only", action="store_true",
                    help="time only the whole-step region (short run for ncu launch lists / captures)")
    ap.add_argument("--decode-only", action="store_true", help="only the configs[1] decode step (short run for ncu)")
    ap.add_argument("--short-extras", action="store_true", help="with --extras-only: skip configs 3-5")
    ap.add_argument("--extras-only", action="store_true",
                    help="only the prefill (T=4096) linear and T=8192 prepare measurements (short run for ncu)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
