"""bench.py -- SharQ per-linear-layer hot path on B200 (BASELINE.json metric: µs/layer and effective
TFLOPS of prepare + fused sparse/dense FP4 GEMM; prep kernel HBM GB/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path (sharq_prepare -> sharq_linear) over
BASELINE.json configs[1]: the four Llama-3.1-8B-shaped linears (QKV 4096->6144, O 4096->4096,
gate+up 4096->28672, down 14336->4096) at every T in {1, 8, 32, 128, 256}: 20 prepare + 20 linear
launches.  `value` = sum of the layers' nominal 2*T*K*D flop / step time (device, CUDA events, inputs
resident in HBM, the step replayed from a CUDA graph so launch latency is the GPU's, not Python's).
`e2e` = the same step through the public binding with the activations starting in pinned HOST memory
and every Y copied back to the host inside the timed region.  N > 1: one process per GPU, rows sharded
(each rank runs its own batch, no collective), time = max over ranks.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on the host cores.  The oracle is never on the product path.
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
    """configs[1] operands resident in HBM: n_sets rotating quantized weight sets (so that a weight is
    re-read only after > L2 bytes of other traffic), one x / activation set / Y per (T, layer)."""

    def __init__(self, sq, rank, Ts, n_sets):
        import torch
        self.sq, self.Ts, self.n_sets = sq, Ts, n_sets
        self.cfg = {n: sq.make_config(sq.NVFP4, sq.NORM_RMS if norm else sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
                    for n, _, _, norm in LLAMA}
        seed = rank_seed(rank)
        self.wq = []
        for r in range(n_sets):
            ws = {}
            for i, (n, K, D, _) in enumerate(LLAMA):
                w = device_weight(D, K, seed + 10 * r + i)
                ws[n] = sq.quantize_weight(self.cfg[n], w)
                del w
            self.wq.append(ws)
        self.gamma = {K: device_gamma(K, seed + 5) for K in {k for _, k, _, _ in LLAMA}}
        self.x, self.act, self.Y = {}, {}, {}
        for T in Ts:
            for i, (n, K, D, norm) in enumerate(LLAMA):
                self.x[T, n] = device_activations(T, K, seed + 1000 + 7 * T + i)
                self.act[T, n] = sq.alloc_act(self.cfg[n], T, K, "cuda")
                self.Y[T, n] = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
        torch.cuda.synchronize()

    def prepare_all(self):
        for T in self.Ts:
            for n, K, D, norm in LLAMA:
                self.sq.prepare(self.cfg[n], self.x[T, n], self.gamma[K] if norm else None, out=self.act[T, n])

    def linear_all(self, r):
        for T in self.Ts:
            for n, K, D, norm in LLAMA:
                self.sq.linear(self.cfg[n], self.act[T, n], self.wq[r][n], Y=self.Y[T, n])

    def step(self, r):
        for T in self.Ts:
            for n, K, D, norm in LLAMA:
                self.sq.prepare(self.cfg[n], self.x[T, n], self.gamma[K] if norm else None, out=self.act[T, n])
                self.sq.linear(self.cfg[n], self.act[T, n], self.wq[r][n], Y=self.Y[T, n])

    @property
    def launches_per_step(self):
        return 2 * len(self.Ts) * len(LLAMA)

    def flops(self):
        return sum(layer_flops(T, K, D) for T in self.Ts for _, K, D, _ in LLAMA)


def capture(fn):
    """Capture fn() (kernel launches on the current stream through the C ABI) into a CUDA graph."""
    import torch
    fn()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    return g


def timed(replays, steps, warmup, barrier):
    """W warm-up + K timed calls of replays[i % R](), CUDA events on the launching stream."""
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
    if args.extras_only:
        wl = Workload(sq, rank, [], n_sets)
        ex = prefill_extras(sq, wl, pk, args.steps)
        if not args.short_extras:
            ex.update(config_extras(sq, wl, pk, args.steps))
        print(json.dumps({"extras_only": True, "extras": ex}))
        return
    wl = Workload(sq, rank, DECODE_T, n_sets)
    steps, warmup = args.steps, max(args.warmup, 3)

    # ---- headline: whole hot path, device-timed, CUDA-graph replay ------------------------------
    launch_mode = "cuda_graph"
    try:
        graphs = [capture(lambda r=r: wl.step(r)) for r in range(n_sets)]
        replays = [g.replay for g in graphs]
    except Exception as exc:                              # capture refused: plain stream launches
        launch_mode = f"stream ({type(exc).__name__})"
        replays = [lambda r=r: wl.step(r) for r in range(n_sets)]
    with ClockSampler(local) as cs:            # clocks under load: several passes so that >= a few samples land
        ms_step = timed(replays, steps, warmup, barrier)
        t_end = time.time() + 0.6
        while time.time() < t_end:
            ms_step = min(ms_step, timed(replays, steps, 0, barrier))
    clocks = cs.summary()
    ms_step = max_over_ranks(ms_step)
    flops = wl.flops()
    value = world * flops / (ms_step * 1e-3) / 1e12

    if args.headline_only:
        if rank == 0:
            print(json.dumps({"metric": "sharq_layer_effective_tflops", "value": round(value, 2), "unit": "TFLOP/s",
                              "ms_per_step": round(ms_step, 4), "steps": steps, "warmup": warmup, "headline_only": True}))
        return

    # ---- dominant kernel alone (sharq_linear_kernel), same operands and rotation ----------------
    wl.prepare_all()
    try:
        lin_replays = [capture(lambda r=r: wl.linear_all(r)).replay for r in range(n_sets)]
    except Exception:
        lin_replays = [lambda r=r: wl.linear_all(r) for r in range(n_sets)]
    ms_lin = timed(lin_replays, steps, warmup, barrier)
    n_lin = len(DECODE_T) * len(LLAMA)
    lin_bytes = sum(linear_bytes(T, K, D) for T in DECODE_T for _, K, D, _ in LLAMA)
    ach = lin_bytes / (ms_lin * 1e-3) / 1e9
    traffic = None                                        # per-launch DRAM bytes from the committed ncu capture
    tpath = os.path.join(ROOT, "profiles", "linear_decode_traffic_r1.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            traffic = json.load(f).get("traffic_bytes_per_launch")
    roofline = dict(kernel="sharq_linear (the 20 launches of the step: 128-wide split-K cluster / persistent, "
                           "256-wide and CTA-pair variants)", bound="hbm", achieved=round(ach, 1), peak=pk["hbm"],
                    unit="GB/s", frac=round(ach / pk["hbm"], 4), traffic=traffic, peak_source=pk["source"],
                    launches_per_step=n_lin, avg_launch_us=round(ms_lin * 1e3 / n_lin, 2),
                    algorithmic_bytes_per_launch=round(lin_bytes / n_lin),
                    share_of_step=round(ms_lin / ms_step, 3))

    # ---- per-layer µs (BASELINE metric "µs/layer"): prepare + linear as they run inside a model, i.e. in a
    # chain of launches, weights cold: one graph holds the layer once per weight copy, the copies of one
    # layer together exceed L2 (140 MB), time = graph time / copies
    layers = {}
    for n, K, D, norm in LLAMA:
        w_bytes = K * D * (0.5 + 1.0 / 32 + 1.0 / 16)
        n_copies = max(n_sets, int(140e6 // w_bytes) + 1)
        copies = [wl.wq[r][n] for r in range(n_sets)]
        while len(copies) < n_copies:
            src = copies[len(copies) % n_sets]
            copies.append({k: (v.clone() if hasattr(v, "clone") else v) for k, v in src.items()})
        for T in DECODE_T:
            def chain(T=T, n=n, K=K, norm=norm, copies=copies):
                for wq in copies:
                    sq.prepare(wl.cfg[n], wl.x[T, n], wl.gamma[K] if norm else None, out=wl.act[T, n])
                    sq.linear(wl.cfg[n], wl.act[T, n], wq, Y=wl.Y[T, n])
            try:
                rep = capture(chain).replay
            except Exception:
                rep = chain
            ms = timed([rep], max(steps // 2, 8), 3, lambda: None) / len(copies)
            layers[f"{n}_T{T}"] = dict(us=round(ms * 1e3, 2), tflops=round(layer_flops(T, K, D) / ms / 1e9, 1))
        del copies

    extras = prefill_extras(sq, wl, pk, steps) if rank == 0 else {}
    if rank == 0:
        extras.update(config_extras(sq, wl, pk, steps))

    # ---- e2e: activations start in pinned host memory, Y read back, plain stream launches --------
    xh = {k: v.cpu().pin_memory() for k, v in wl.x.items()}
    yh = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in wl.Y.items()}

    side = torch.cuda.Stream()                            # device->host copies overlap the next layers' work
    up = torch.cuda.Stream()                              # host->device copies run ahead of the layers (PCIe is duplex)

    def e2e_step(r):
        main = torch.cuda.current_stream()
        up.wait_stream(main)                              # the previous step has consumed its inputs
        ready = {}
        with torch.cuda.stream(up):
            for T in DECODE_T:
                for n, K, D, norm in LLAMA:
                    wl.x[T, n].copy_(xh[T, n], non_blocking=True)
                    ready[T, n] = torch.cuda.Event()
                    ready[T, n].record(up)
        for T in DECODE_T:
            for n, K, D, norm in LLAMA:
                main.wait_event(ready[T, n])
                sq.prepare(wl.cfg[n], wl.x[T, n], wl.gamma[K] if norm else None, out=wl.act[T, n])
                sq.linear(wl.cfg[n], wl.act[T, n], wl.wq[r][n], Y=wl.Y[T, n])
                side.wait_stream(main)
                with torch.cuda.stream(side):
                    yh[T, n].copy_(wl.Y[T, n], non_blocking=True)
        main.wait_stream(side)                            # the step ends when every Y is on the host
        main.wait_stream(up)

    e2e_mode = "cuda_graph (H2D stream + kernels + D2H stream)"
    try:
        e2e_reps = [capture(lambda r=r: e2e_step(r)).replay for r in range(n_sets)]
    except Exception as exc:
        e2e_mode = f"stream ({type(exc).__name__})"
        e2e_reps = [lambda r=r: e2e_step(r) for r in range(n_sets)]
    ms_e2e = max_over_ranks(timed(e2e_reps, steps, warmup, barrier))
    h2d = sum(v.numel() * 2 for v in xh.values())
    d2h = sum(v.numel() * 2 for v in yh.values())

    if rank != 0:
        dist.destroy_process_group()
        return
    line = {
        "metric": "sharq_layer_effective_tflops", "value": round(value, 2), "unit": "TFLOP/s",
        "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": round(ms_step, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "fp4_e2m1(fp32 acc)",
        "data": "synthetic",
        "config": {"workload": "BASELINE configs[1]: Llama-3.1-8B decode linears (qkv/o/gate_up/down) x T in "
                               "{1,8,32,128,256}, NVFP4, pairwise 4:8, prepare+linear per layer",
                   "l2": f"{n_sets} rotating weight sets (3 x 116 MB) so every weight re-read follows > 126 MB of traffic",
                   "launch": launch_mode, "parallelism": f"rows x{world} (replicated weights, no collective)"},
        "us_per_layer_mean": round(ms_step * 1e3 / n_lin, 2),
        "clocks": clocks,
        "e2e": {"value": round(world * flops / (ms_e2e * 1e-3) / 1e12, 2), "unit": "TFLOP/s",
                "ms_per_step": round(ms_e2e, 4), "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "launch": e2e_mode},
        "gpu_launches": wl.launches_per_step * steps,
        "roofline": roofline,
        "cpu_baseline": cpu_baseline_sample() if world == 1 else None,
        "layers": layers,
        "layers_note": "prepare + linear per layer, chained in one graph over enough weight copies to exceed L2",
        "extras": extras,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def mma_issue_peaks(sq):
    """FP4 tensor peaks measured on this GPU by the library's MMA issue-rate probe (sharq_mma_peak_launch):
    dense-only, sparse-only, and the fused per-k-block sequence with its scale-factor copies; `burst` = one
    2 ms launch, `sustained` = the last of back-to-back launches over ~1.5 s (power-capped clocks)."""
    import torch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    out = {}
    for name, mode in (("dense", 1), ("sparse", 2), ("fused_with_sf_copies", 7)):
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


def prefill_extras(sq, wl, pk, steps):
    """configs[2] family at T = 4096 (compute-bound) and the prep kernel's HBM rate: reported beside the
    headline, same kernels, CUDA events.  FP4 tensor peak = measured bf16 peak x 4 (dense, nominal ratio
    9 / 2.25 PFLOP/s) and x 8 (2:4 sparse); t_min = 2TKD / P_dense + 2TKD / P_sparse."""
    import torch
    out = {"fp4_dense_peak_tflops": round(4 * pk["bf16_sustained"], 1), "fp4_sparse_peak_tflops": round(8 * pk["bf16_sustained"], 1),
           "peak_note": f"4x / 8x the {pk['source']} sustained bf16 cuBLAS rate", "linear_T4096": {}, "prepare": {}}
    T = PREFILL_T
    p_dn, p_sp = 4 * pk["bf16_sustained"] * 1e12, 8 * pk["bf16_sustained"] * 1e12
    mp = mma_issue_peaks(sq)
    out["mma_issue_probe_tflops"] = mp
    out["mma_issue_probe_note"] = ("sharq_mma_peak_launch: the GEMM's own per-k-block tcgen05 sequence on smem-resident "
                                   "bytes (nominal 2MNK flop per path); frac_of_mma_probe uses the sustained dense and sparse rates")
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
                                      frac_of_mma_probe=round((fl / q_dn + fl / q_sp) / (ms * 1e-3), 4))
        del x, act, Y
    for K, norm in ((4096, 1), (14336, 0)):
        Tp = 8192
        n = "qkv" if norm else "down"
        xs = [device_activations(Tp, K, BASE_SEED + 70 + j) for j in range(3)]       # 3 x (in + out) > L2
        acts = [sq.alloc_act(wl.cfg[n], Tp, K, "cuda") for _ in xs]
        reps = [lambda j=j: sq.prepare(wl.cfg[n], xs[j], wl.gamma[K] if norm else None, out=acts[j]) for j in range(3)]
        ms = timed(reps, max(steps, 12), 3, lambda: None)
        gbs = prepare_bytes(Tp, K) / (ms * 1e-3) / 1e9
        # the kernel is ALU / issue bound, not HBM bound (profiles/prepare_r1_ncu_full.md, last capture:
        # smsp__inst_executed x 32 / elements = 25.3 thread-instructions per element with RMSNorm (K = 4096),
        # 20.5 without (K = 14336, lagged loop);
        # DRAM traffic = algorithmic bytes): second roofline = issue slots, 148 SMs x 4 schedulers x 32 lanes
        # x 1.965 GHz
        issue_peak = 148 * 128 * 1.965e9
        ipe = 25.3 if norm else 20.5
        out["prepare"][f"T{Tp}_K{K}_{'rms' if norm else 'none'}"] = dict(
            us=round(ms * 1e3, 1), GBps=round(gbs, 1), frac_of_hbm=round(gbs / pk["hbm"], 4),
            alu=dict(bound="alu", achieved=round(Tp * K * ipe / (ms * 1e-3) / 1e12, 2), peak=round(issue_peak / 1e12, 2),
                     unit="T thread-instructions/s", frac=round(Tp * K * ipe / (ms * 1e-3) / issue_peak, 4),
                     instr_per_element=ipe))
        del xs, acts
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
    return out


QWEN = [("qkv", 3584, 4608, 1), ("o", 3584, 3584, 0), ("gate_up", 3584, 37888, 1), ("down", 18944, 3584, 0)]


def config_extras(sq, wl, pk, steps):
    """BASELINE.json configs[2] (T sweep), configs[3] (Qwen2.5-7B shapes x formats) and configs[4] (MoE
    grouped): sharq_linear alone and sharq_prepare alone, CUDA events, rotating weights where they exist."""
    import torch
    p_dn, p_sp = 4 * pk["bf16_sustained"] * 1e12, 8 * pk["bf16_sustained"] * 1e12
    out = {"config3_T_sweep": {}, "config4_qwen_formats": {}, "config5_moe": {}}

    def lin_entry(ms, T, K, D, fmt=0):
        fl = layer_flops(T, K, D)
        return dict(us=round(ms * 1e3, 1), effective_tflops=round(fl / ms / 1e9, 1),
                    frac_of_fp4_roofline=round((fl / p_dn + fl / p_sp) / (ms * 1e-3), 4),
                    GBps=round(linear_bytes(T, K, D, fmt) / ms / 1e6, 1))

    for T in (2048, 8192):                       # T = 4096 is in linear_T4096
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
            ms_p = timed([lambda: sq.prepare(cfg, x, g if norm else None, out=act)], max(steps // 2, 8), 3, lambda: None)
            ws = sq._bytes(sq.linear_workspace(cfg, T, D, K), "cuda") if fmt == sq.HIF4 else None
            ms_l = timed([lambda r=r: sq.linear(cfg, act, wqs[r], Y=Y, workspace=ws) for r in range(2)],
                         max(steps // 2, 8), 3, lambda: None)
            e = lin_entry(ms_l, T, K, D, fmt)
            if fmt == sq.HIF4:                   # no FP4-rate tensor path for HiF4: bf16 roofline (dense + 2:4 sparse)
                fl = layer_flops(T, K, D)
                pb = pk["bf16_sustained"] * 1e12
                del e["frac_of_fp4_roofline"]
                e["frac_of_bf16_roofline"] = round((fl / pb + fl / (2 * pb)) / (ms_l * 1e-3), 4)
                e["note"] = "dequantise (A and W, every call) + dense bf16 GEMM over 2K"
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
        ms_p = timed([lambda: sq.prepare(cfg, x, out=act)], max(steps // 2, 8), 3, lambda: None)
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
                                     note="weights (all experts) are L2-resident across repeats: 201 / 101 MB")
        del wq, x, act, Y
    out["config5_moe"]["rows_per_expert"] = dict(min=int(counts.min()), max=int(counts.max()))
    return out


# ---- CPU oracle legs (the only places bench.py executes oracle/) ---------------------------------------
SAMPLE_T, SAMPLE_COLS = 16, 1024
SAMPLE_DESC = (f"configs[1] shapes (qkv/o/gate_up/down) at T={SAMPLE_T}, {SAMPLE_COLS} seeded output features per layer: "
               "oracle prepare + fp64 linear; weight quantization (offline) not timed")


def oracle_sample_setup():
    import sharq_inputs as si
    from oracle import sharq_oracle as so
    rng = np.random.Generator(np.random.Philox(BASE_SEED))
    items = []
    for i, (n, K, D, norm) in enumerate(LLAMA):
        x, g = si.activations(SAMPLE_T, K, config=2, extra=i), si.gamma(K, 2)
        cols = np.sort(rng.choice(D, size=SAMPLE_COLS, replace=False))
        w = si.weight(SAMPLE_COLS, K, config=2, extra=i)            # the sampled rows of W stand for W[cols]
        items.append((n, K, norm, x, g, so.quantize_weight(w)))
    return so, items


def oracle_sample_step(so, items):
    for n, K, norm, x, g, wq in items:
        p = so.prepare(x, norm=norm, gamma_u16=g if norm else None)
        so.linear(p, wq)


def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([int(i.get("num_threads", 1)) for i in threadpool_info()] or [1])
    except Exception:
        return 1


def cpu_baseline_sample():
    so, items = oracle_sample_setup()
    oracle_sample_step(so, items)                                    # warm
    t0 = time.perf_counter()
    reps = 0
    while reps < 2 or time.perf_counter() - t0 < 10.0:
        oracle_sample_step(so, items)
        reps += 1
    dt = (time.perf_counter() - t0) / reps
    fl = sum(layer_flops(SAMPLE_T, K, SAMPLE_COLS) for _, K, _, _ in LLAMA)
    return dict(value=round(fl / dt / 1e12, 6), unit="TFLOP/s", cores=oracle_threads(), kind="oracle",
                sample=SAMPLE_DESC, host_cores=os.cpu_count(), s_per_sample_step=round(dt, 3))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    so, items = oracle_sample_setup()
    steps, warmup = args.steps, args.warmup
    budget = 150.0                                                    # seconds: keep the whole run to minutes
    t_all = time.perf_counter()
    for _ in range(warmup):
        oracle_sample_step(so, items)
        if time.perf_counter() - t_all > budget / 3:
            break
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        oracle_sample_step(so, items)
        done += 1
        if time.perf_counter() - t0 > budget:
            break
    dt = (time.perf_counter() - t0) / done
    fl = sum(layer_flops(SAMPLE_T, K, SAMPLE_COLS) for _, K, _, _ in LLAMA)
    v = round(fl / dt / 1e12, 6)
    print(json.dumps({
        "impl": "reference", "metric": "sharq_layer_effective_tflops", "value": v, "unit": "TFLOP/s",
        "n_gpus": world, "steps": done, "warmup": warmup, "ms_per_step": round(dt * 1e3, 3), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE configs[1] (bounded sample): " + SAMPLE_DESC},
        "cpu_baseline": dict(value=v, unit="TFLOP/s", kind="oracle", cores=oracle_threads(), sample=SAMPLE_DESC,
                             host_cores=os.cpu_count()),
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
