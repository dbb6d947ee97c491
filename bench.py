#!/usr/bin/env python
"""bench.py -- timing harness for the TwinQuant dual-component linear layer on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

One "step" = one pass of the whole hot path (twq_quantize_act + twq_dual_linear)
over one batch of synthetic activations for one layer.  Prints ONE JSON line (rank 0).

  value      us per step, device time (CUDA events around a CUDA graph of K steps, inputs resident in HBM)
  e2e        the same through the public Python API with pinned-host X -> device and Y -> host inside the region
  roofline   the fused kernel alone (its own K-launch graph): algorithmic bytes or int8-equivalent ops / time
  cpu_baseline  the oracle (oracle/, as it stands) on the host cores, on a bounded sample
  sweep      the other graded shapes (M = 1 / 16 / 128 q_proj, M = 2048 MLP at r = 128 and 256) measured the same way

Cold-cache protocol: the layer's packed weights (and activations) are rotated through enough distinct
copies that one lap exceeds 2x the 126 MB L2, so every step streams its weights from HBM.
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

from gen import inputs as gen  # noqa: E402

L2_BYTES = 126 * 1024 * 1024

WORKLOADS = {
    # name: (generator, kwargs, description)
    "c2_qproj_m1": ("config2_qproj", dict(M=1), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=1"),
    "c2_qproj_m16": ("config2_qproj", dict(M=16), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=16"),
    "c2_qproj_m32": ("config2_qproj", dict(M=32), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=32"),
    "c2_qproj_m64": ("config2_qproj", dict(M=64), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=64"),
    "c2_qproj_m128": ("config2_qproj", dict(M=128), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=128"),
    "c3_gateup_m2048": ("config3_mlp", dict(which="gate_up", M=2048), "LLaMA3-8B gate/up K=4096 N=14336 r=128 G=128 M=2048"),
    "c3_down_m2048": ("config3_mlp", dict(which="down", M=2048), "LLaMA3-8B down K=14336 N=4096 r=128 G=128 M=2048"),
    "c3_gateup_m2048_r256": ("config3_mlp", dict(which="gate_up", M=2048, r=256), "LLaMA3-8B gate/up r=256 M=2048"),
    "c1_tiny": ("config1_tiny", dict(), "tiny M=8 K=256 N=512 r=16 G=64"),
    # rank 0 (plain W4A4): what the residual stream alone costs
    "c2_qproj_m1_r0": ("config2_qproj", dict(M=1, r=0), "LLaMA3-8B q_proj K=4096 N=4096 r=0 G=128 M=1"),
    "c2_qproj_m384": ("config2_qproj", dict(M=384), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=384"),
    "c3_gateup_m128": ("config3_mlp", dict(which="gate_up", M=128), "LLaMA3-8B gate/up K=4096 N=14336 r=128 G=128 M=128"),
    "c3_gateup_m256": ("config3_mlp", dict(which="gate_up", M=256), "LLaMA3-8B gate/up K=4096 N=14336 r=128 G=128 M=256"),
    "c3_gateup_m512": ("config3_mlp", dict(which="gate_up", M=512), "LLaMA3-8B gate/up K=4096 N=14336 r=128 G=128 M=512"),
    "c3_down_m128": ("config3_mlp", dict(which="down", M=128), "LLaMA3-8B down K=14336 N=4096 r=128 G=128 M=128"),
    "c3_down_m256": ("config3_mlp", dict(which="down", M=256), "LLaMA3-8B down K=14336 N=4096 r=128 G=128 M=256"),
    "c4_attn_m128": ("config4_qwen", dict(which="attn", M=128), "Qwen3-32B attention K=5120 N=5120 r=256 M=128"),
    "c2_qproj_m96": ("config2_qproj", dict(M=96), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=96"),
    "c2_qproj_m192": ("config2_qproj", dict(M=192), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=192"),
    "c2_qproj_m128_r0": ("config2_qproj", dict(M=128, r=0), "LLaMA3-8B q_proj K=4096 N=4096 r=0 G=128 M=128"),
    "c2_qproj_m256": ("config2_qproj", dict(M=256), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=256"),
    "c2_qproj_m512": ("config2_qproj", dict(M=512), "LLaMA3-8B q_proj K=4096 N=4096 r=128 G=128 M=512"),
    "c2_qproj_m16_r0": ("config2_qproj", dict(M=16, r=0), "LLaMA3-8B q_proj K=4096 N=4096 r=0 G=128 M=16"),
    # configs 4 / 5 (rank 256): not in the default sweep; DESIGN.md section 10 quotes them
    "c4_gateup_m4096": ("config4_qwen", dict(which="gate_up", M=4096), "Qwen3-32B gate/up K=5120 N=25600 r=256 M=4096"),
    "c4_down_m4096": ("config4_qwen", dict(which="down", M=4096), "Qwen3-32B down K=25600 N=5120 r=256 M=4096"),
    "c4_down_m1": ("config4_qwen", dict(which="down", M=1), "Qwen3-32B down K=25600 N=5120 r=256 M=1"),
    "c4_attn_m64": ("config4_qwen", dict(which="attn", M=64), "Qwen3-32B attention K=5120 N=5120 r=256 M=64"),
    "c5_gateup_m2048": ("config5_llama70b", dict(which="gate_up", M=2048), "LLaMA3-70B gate/up K=8192 N=28672 r=256 M=2048"),
    "c5_down_m1": ("config5_llama70b", dict(which="down", M=1), "LLaMA3-70B down K=28672 N=8192 r=256 M=1"),
    "c5_qproj_m16": ("config5_llama70b", dict(which="q", M=16), "LLaMA3-70B q_proj K=8192 N=8192 r=256 M=16"),
}
DEFAULT_WORKLOAD = "c2_qproj_m16"
DEFAULT_SWEEP = ["c2_qproj_m1", "c2_qproj_m16", "c2_qproj_m32", "c2_qproj_m64", "c2_qproj_m128", "c3_gateup_m2048",
                 "c3_down_m2048", "c3_gateup_m2048_r256"]


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def config_for(name):
    """The `config` object of the JSON line: identical for the GPU arm and the reference (oracle) arm."""
    return dict(workload=name, desc=WORKLOADS[name][2],
                l2="inputs larger than L2: weights and activations rotate through copies, one lap >= 2x the 126 MB L2",
                launch="CUDA graph of K steps; step = the whole hot path (quantizer, both branches, epilogue) through twq_dual_linear_x",
                multi_gpu="replicas only")


def make_layer(name):
    fn, kw, _ = WORKLOADS[name]
    return getattr(gen, fn)(**kw)


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[])
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [ln.strip().split(", ") for ln in open(self.f.name) if ln.strip()]
        os.unlink(self.f.name)
        sm, reasons, smax = [], set(), None
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                smax = float(r[1])
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if sm:
            hi = [c for c in sm if c >= 0.5 * max(sm)]   # samples under load
            out = dict(sm_mhz=float(np.median(hi)), sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm))
        return out


# ----------------------------------------------------------------------------- GPU arm
class GpuLayer:
    """Device-resident copies of one layer, rotated so that a lap over them exceeds 2x L2."""

    def __init__(self, L, twq, torch, min_lap_bytes=2 * L2_BYTES, max_copies=32):
        self.L, self.twq, self.torch = L, twq, torch
        dev = torch.device("cuda", torch.cuda.current_device())
        self.Xh = torch.from_numpy(L.X.view(np.int16)).view(torch.bfloat16).pin_memory()
        Rq, sw = torch.from_numpy(L.Rq).to(dev), torch.from_numpy(L.sw).to(dev)
        L1, L2 = torch.from_numpy(L.L1).to(dev), torch.from_numpy(L.L2).to(dev)
        first = twq.pack_weights(Rq, sw, L1 if L.r else None, L2 if L.r else None, L.G)
        per_copy = first.blob.numel() + 2 * L.M * L.K + L.M * L.K // 2 + 2 * L.M * L.N
        self.ncopies = int(min(max_copies, max(2, -(-min_lap_bytes // per_copy))))
        self.packed = [first]
        for _ in range(self.ncopies - 1):
            self.packed.append(twq.PackedLayer(first.blob.clone(), first.N, first.K, first.r, first.G))
        self.X = [self.Xh.to(dev) for _ in range(self.ncopies)]
        self.Xq = [torch.empty((L.M, L.K // 2), dtype=torch.uint8, device=dev) for _ in range(self.ncopies)]
        self.sx = [torch.empty((L.M, L.ng), dtype=torch.float32, device=dev) for _ in range(self.ncopies)]
        self.Y = [torch.empty((L.M, L.N), dtype=torch.bfloat16, device=dev) for _ in range(self.ncopies)]
        need = twq.workspace_bytes(L.M, L.N, L.K, L.r, L.G)
        self.ws = torch.zeros(max(need, 256), dtype=torch.uint8, device=dev) if need else None
        need_x = twq.workspace_bytes_x(L.M, L.N, L.K, L.r, L.G)
        self.ws_x = torch.zeros(max(need_x, 256), dtype=torch.uint8, device=dev) if need_x else None
        self.Yh = torch.empty((L.M, L.N), dtype=torch.bfloat16).pin_memory()
        # the whole hot path is ONE launch (twq_dual_linear_x with the in-kernel quantizer) where the small-batch plan exists
        self.one_launch = L.M <= 64 and need_x == 0
        self.lap_bytes = per_copy * self.ncopies
        del Rq, sw, L1, L2
        torch.cuda.synchronize()

    def step(self, i, quant=True, dual=True):
        c = i % self.ncopies
        if quant:
            self.twq.quantize_act(self.X[c], self.L.G, None, out=(self.Xq[c], self.sx[c]))
        if dual:
            self.twq.dual_linear(self.X[c], self.Xq[c], self.sx[c], self.packed[c], self.twq.OUT_BF16, Y=self.Y[c],
                                 ws=self.ws)

    def step_x(self, i):
        """The whole hot path through twq_dual_linear_x (one launch for M <= 64 where the plan fits)."""
        c = i % self.ncopies
        self.twq.dual_linear_x(self.X[c], self.packed[c], None, self.twq.OUT_BF16, Y=self.Y[c], ws=self.ws_x)

    def e2e_step(self, i):
        c = i % self.ncopies
        self.X[c].copy_(self.Xh, non_blocking=True)
        self.step_x(i)
        self.Yh.copy_(self.Y[c], non_blocking=True)

    def time_graph(self, steps, warmup, quant=True, dual=True, replays=20, fused=False):
        """Device time per step of a CUDA graph holding `steps` consecutive steps (no host launch gaps), over
        `replays` timed replays of the graph: returns (median, min) in us per step (SURVEY.md 8d protocol)."""
        torch = self.torch
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            for i in range(max(warmup, self.ncopies)):           # every Xq/sx copy is valid before dual-only timing
                self.step(i, True, True)
                if fused:
                    self.step_x(i)
            s.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                for i in range(steps):
                    if fused:
                        self.step_x(i)
                    else:
                        self.step(i, quant, dual)
            g.replay()                                            # one untimed replay (graph upload)
            s.synchronize()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(replays)]
            for e0, e1 in ev:
                e0.record(s)
                g.replay()
                e1.record(s)
            s.synchronize()
        torch.cuda.current_stream().wait_stream(s)
        us = sorted(e0.elapsed_time(e1) * 1e3 / steps for e0, e1 in ev)
        return float(np.median(us)), us[0]                        # us per step: median, min

    def time_host(self, calls=2000):
        """Host time of one twq_dual_linear_x call through the binding (plan + descriptor caches warm), no device
        synchronisation inside the loop; the queue is drained every 100 calls so that it never back-pressures."""
        torch = self.torch
        for i in range(max(20, self.ncopies)):                   # every rotating copy has its descriptors cached
            self.step_x(i)
        torch.cuda.synchronize()
        t = 0.0
        for base in range(0, calls, 100):
            t0 = time.perf_counter()
            for i in range(base, base + 100):
                self.step_x(i)
            t += time.perf_counter() - t0
            torch.cuda.synchronize()
        return t / calls * 1e6

    def time_e2e(self, steps, warmup):
        torch = self.torch
        for i in range(max(warmup, self.ncopies)):               # every rotating copy has its descriptors cached
            self.e2e_step(i)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(steps):
            self.e2e_step(i)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e3 / steps


def roofline_for(L, twq, us_dual, peaks, traffic=None, traffic_src=None, one_launch=False):
    """Roofline of the dominant kernel: twq_dual_linear's kernel, or (one_launch) the single kernel of twq_dual_linear_x."""
    by = (twq.algorithmic_bytes_x if one_launch else twq.algorithmic_bytes)(L.M, L.N, L.K, L.r, L.G)
    ops_i8, fl_lr = twq.flops(L.M, L.N, L.K, L.r)
    p_i8 = 2.0 * peaks["bf16_tflops"] * 1e12        # int8 dense = 2x bf16 (guide's nominal ratio) x measured bf16
    p_f16 = peaks["bf16_tflops"] * 1e12
    t_hbm = by / (peaks["hbm_gbs"] * 1e9)
    t_tensor = ops_i8 / p_i8 + fl_lr / p_f16
    t = us_dual * 1e-6
    if t_hbm >= t_tensor:
        ach = by / t / 1e9
        return dict(bound="hbm", achieved=round(ach, 1), peak=peaks["hbm_gbs"], unit="GB/s",
                    frac=round(ach / peaks["hbm_gbs"], 4), traffic=traffic, traffic_source=traffic_src,
                    peak_source=peaks["source"],
                    kernel=kernel_name(L) + ("<in-kernel quantizer> (the whole step)" if one_launch else ""),
                    us=round(us_dual, 3), algorithmic_bytes=by)
    eq_ops = ops_i8 + 2.0 * fl_lr                    # low-rank flops run at half the int8 rate
    ach = eq_ops / t / 1e12
    return dict(bound="tensor", achieved=round(ach, 1), peak=round(p_i8 / 1e12, 1), unit="TFLOP/s",
                frac=round(ach / (p_i8 / 1e12), 4), traffic=traffic, traffic_source=traffic_src,
                peak_source=peaks["source"] + " bf16 burst x2 (int8)",
                kernel=kernel_name(L), us=round(us_dual, 3), int8_equivalent_ops=eq_ops)


def load_traffic(name, one_launch=False):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dual-linear kernel, from the `ncu --set full`
    captures summarised under profiles/ (profiles/traffic.json names capture file and commit per workload)."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, None
    ent = json.load(open(path)).get(name + ("_x" if one_launch else ""))
    if not ent:
        return None, None
    return int(ent["dram_bytes"]), "%s @ %s" % (ent["capture"], ent["commit"])


def kernel_name(L):
    return "decode_dual_linear_kernel" if L.M <= 64 else "fused_dual_linear_kernel"


def measure_workload(name, twq, torch, steps, warmup, peaks, with_e2e=False, with_cublas=False):
    L = make_layer(name)
    gl = GpuLayer(L, twq, torch)
    # The step = the whole hot path through the public call twq_dual_linear_x: ONE launch for M <= 64 (in-kernel quantizer),
    # twq_quantize_act + twq_dual_linear otherwise.  The two-call step and its two kernels are timed beside it.
    us_x, us_x_min = gl.time_graph(steps, warmup, fused=True)
    us_two, us_two_min = gl.time_graph(steps, warmup, True, True)
    us_dual, us_dual_min = gl.time_graph(steps, warmup, False, True)
    us_quant, us_quant_min = gl.time_graph(steps, warmup, True, False)
    ops_i8, fl_lr = twq.flops(L.M, L.N, L.K, L.r)
    one = gl.one_launch
    us_kernel = us_x if one else us_dual                       # the dominant kernel: the single one, or twq_dual_linear's
    traffic, traffic_src = load_traffic(name, one)
    out = dict(workload=name, M=L.M, N=L.N, K=L.K, r=L.r, G=L.G, us_step=round(us_x, 3),
               launches_per_step=1 if one else 2,
               us_step_two_call=round(us_two, 3), us_dual_linear=round(us_dual, 3), us_quantize_act=round(us_quant, 3),
               us_min=dict(step=round(us_x_min, 3), step_two_call=round(us_two_min, 3), dual_linear=round(us_dual_min, 3), quantize_act=round(us_quant_min, 3)),
               timing="median of 20 replays of a CUDA graph of %d steps (min alongside)" % steps,
               eff_tops=round((ops_i8 + fl_lr) / (us_kernel * 1e-6) / 1e12, 2),
               gbs=round((twq.algorithmic_bytes_x if one else twq.algorithmic_bytes)(L.M, L.N, L.K, L.r, L.G) / (us_kernel * 1e-6) / 1e9, 1),
               weight_copies=gl.ncopies, lap_mb=round(gl.lap_bytes / 2 ** 20, 1),
               roofline=roofline_for(L, twq, us_kernel, peaks, traffic, traffic_src, one))
    if with_e2e:
        out["us_e2e"] = round(gl.time_e2e(steps, warmup), 3)
        out["us_host_per_call"] = round(gl.time_host(), 3)
    if with_cublas:
        A = torch.randn(L.M, L.K, device="cuda", dtype=torch.bfloat16)
        Bs = [torch.randn(L.K, L.N, device="cuda", dtype=torch.bfloat16) for _ in range(max(2, min(16, (2 * L2_BYTES) // (2 * L.K * L.N) + 1)))]
        for b in Bs[:3]:
            torch.matmul(A, b)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(steps):
            torch.matmul(A, Bs[i % len(Bs)])
        e1.record()
        torch.cuda.synchronize()
        out["us_cublas_bf16_gemm"] = round(e0.elapsed_time(e1) * 1e3 / steps, 3)
    return out, gl, L


def measure_q4lr(name, twq, torch, steps, warmup, peaks, with_oracle=False):
    """the same layer shape with the paper's 4-bit low-rank branch (twq_dual_linear_q4lr_x: quantizer,
    both 4-bit branches, re-quantization of H and the epilogue in one launch), timed like the main path: a CUDA graph of
    `steps` calls over rotating blobs (> 2 x L2 per lap), median / min of 20 replays."""
    L = make_layer(name)
    Uq, su, Vq, sv = gen.make_q4_lowrank(L.K, L.N, L.r, L.G, seed=4242)
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    first = twq.pack_weights_q4lr(t(L.Rq), t(L.sw), t(Uq), t(su), t(Vq), t(sv), L.G)
    per_copy = first.blob.numel() + 2 * L.M * L.K + 2 * L.M * L.N
    ncopies = int(min(32, max(2, -(-2 * L2_BYTES // per_copy))))
    packed = [first] + [twq.PackedLayer(first.blob.clone(), first.N, first.K, first.r, first.G) for _ in range(ncopies - 1)]
    Xh = torch.from_numpy(L.X.view(np.int16)).view(torch.bfloat16)
    X = [Xh.to(dev) for _ in range(ncopies)]
    Y = [torch.empty((L.M, L.N), dtype=torch.bfloat16, device=dev) for _ in range(ncopies)]

    def step(i):
        c = i % ncopies
        twq.dual_linear_q4lr_x(X[c], packed[c], None, twq.OUT_BF16, Y=Y[c])

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for i in range(max(warmup, ncopies)):
            step(i)
        launches = twq.last_launch_count()
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for i in range(steps):
                step(i)
        g.replay()
        s.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
        for e0, e1 in ev:
            e0.record(s)
            g.replay()
            e1.record(s)
        s.synchronize()
    torch.cuda.current_stream().wait_stream(s)
    us = sorted(e0.elapsed_time(e1) * 1e3 / steps for e0, e1 in ev)
    med = float(np.median(us))
    by = twq.algorithmic_bytes_q4lr(L.M, L.N, L.K, L.r, L.G)
    ach = by / (med * 1e-6) / 1e9
    out = dict(workload=name + "_q4lr", M=L.M, N=L.N, K=L.K, r=L.r, G=L.G, us_step=round(med, 3), us_min=round(us[0], 3),
               launches_per_step=launches, weight_copies=ncopies,
               roofline=dict(bound="hbm", achieved=round(ach, 1), peak=peaks["hbm_gbs"], unit="GB/s",
                             frac=round(ach / peaks["hbm_gbs"], 4), traffic=load_traffic(name + "_q4lr")[0],
                             traffic_source=load_traffic(name + "_q4lr")[1], kernel="decode_dual_linear_kernel<mode 2>",
                             us=round(med, 3), algorithmic_bytes=by, peak_source=peaks["source"]))
    if with_oracle:
        from oracle import oracle
        oracle.build()
        rows = list(range(min(L.M, 4)))
        t0 = time.perf_counter()
        n = 0
        while time.perf_counter() - t0 < 4.0:
            oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, L.G, rows=rows)
            n += 1
        dt = (time.perf_counter() - t0) / n
        out["cpu_baseline"] = dict(value=round(dt * 1e6 * L.M / len(rows), 1), unit="us/call", cores=oracle.num_threads(),
                                   kind="oracle", sample="oracle.forward_q4lr on %d of %d token rows, %d repeats in 4 s, "
                                   "scaled to the full call" % (len(rows), L.M, n))
    del packed, X, Y
    torch.cuda.empty_cache()
    return out


# ----------------------------------------------------------------------------- CPU oracle arm
def time_oracle(L, budget_s=12.0, max_calls=10000):
    """The oracle as it stands (quantize + pack + forward), all host cores; bounded by ~budget_s of work."""
    from oracle import oracle as orc
    orc.build()
    rows = None
    sample = f"all {L.M} token rows"
    macs = L.M * L.N * L.K
    if macs > 4e9:                                   # prefill shapes: a fixed sample of token rows, scaled linearly in M
        nrows = max(1, int(4e9 // (L.N * L.K)))
        rows = sorted(set(np.linspace(0, L.M - 1, nrows).astype(int).tolist()))
        sample = f"{len(rows)} of {L.M} token rows (all N, all groups), time scaled by M/rows"
    t0 = time.perf_counter()
    calls = 0
    while True:
        orc.forward(L.X, L.Rq, L.sw, L.L1 if L.r else None, L.L2 if L.r else None, L.G, rows=rows)
        calls += 1
        el = time.perf_counter() - t0
        if el >= budget_s or calls >= max_calls:
            break
    scale = 1.0 if rows is None else L.M / len(rows)
    us = el / calls * 1e6 * scale
    return dict(value=round(us, 1), unit="us/call", cores=orc.num_threads(), kind="oracle",
                sample=f"{sample}; {calls} call(s) in {el:.1f} s")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    L = make_layer(args.workload)
    from oracle import oracle as orc
    orc.build()
    for _ in range(min(args.warmup, 1)):
        time_oracle(L, budget_s=0.5, max_calls=1)
    per_step_budget = min(20.0, 120.0 / max(1, args.steps))
    t0 = time.perf_counter()
    res = [time_oracle(L, budget_s=per_step_budget, max_calls=1) for _ in range(args.steps)]
    us = float(np.mean([r["value"] for r in res]))
    cb = dict(res[-1])
    cb["value"] = round(us, 1)
    line = dict(metric="fused dual-linear us/call", value=round(us, 1), unit="us/call", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=round(us / 1e3, 4), higher_is_better=False,
                scaling="weak", vs_baseline=None, dtype="int64+f64", data="synthetic", impl="reference",
                config=config_for(args.workload),
                cpu_baseline=cb,
                e2e=dict(value=round(us, 1), unit="us/call", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                wall_s=round(time.perf_counter() - t0, 1))
    print(json.dumps(line))


# ----------------------------------------------------------------------------- multi-GPU (replicas only)
def max_over_ranks(values, dist, device):
    """Replicas only: every rank times its own replica; the job's time is the MAX
    over ranks.  `dist` is torch.distributed (initialised) or None for a single process."""
    import torch
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_us_per_call(us_max, world):
    """N replicas each finish one call in `us_max` (max over ranks): the job completes N calls in that time."""
    return us_max / world


# ----------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="twq", choices=["twq", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="time only --workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--q4lr", action="store_true",
                    help="time only the 4-bit low-rank variant (twq_dual_linear_q4lr_x, SURVEY 8f NEXT-1) of --workload")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import paper_2606_01556_b200 as twq
    twq.load_library()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")

    peaks = load_peaks()
    if args.q4lr:
        if rank == 0:
            print(json.dumps(measure_q4lr(args.workload, twq, torch, args.steps, args.warmup, peaks,
                                          with_oracle=not args.no_cpu_baseline)))
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return
    sampler = ClockSampler(local) if rank == 0 else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    main_res, gl, L = measure_workload(args.workload, twq, torch, args.steps, args.warmup, peaks, with_e2e=True,
                                       with_cublas=(rank == 0))
    barrier()
    us = main_res["us_step"]
    us_e2e = main_res["us_e2e"]
    us, us_e2e = max_over_ranks([us, us_e2e], dist, "cuda")   # replicas only
    clocks = sampler.stop() if sampler else None

    sweep = []
    if rank == 0 and not args.no_sweep:
        del gl
        torch.cuda.empty_cache()
        for name in DEFAULT_SWEEP:
            if name == args.workload:
                sweep.append({k: v for k, v in main_res.items() if k != "us_e2e"})
                continue
            r, g2, _ = measure_workload(name, twq, torch, max(20, min(args.steps, 100)), args.warmup, peaks,
                                        with_cublas=True)
            sweep.append(r)
            del g2
            torch.cuda.empty_cache()

    cold = None
    if rank == 0:
        # csrc/cold_fill.cu: how long a one-shot burst of the q_proj weight share (10.75 MB over the SMs) takes to reach shared memory
        # from cold HBM, by bulk copies and by plain loads: the floor under the decode-shaped calls that the bytes / bandwidth
        # roofline does not contain (lesson 24)
        try:
            sms = torch.cuda.get_device_properties(local).multi_processor_count
            per = (10_750_000 // sms + 63) // 64 * 64
            cold = dict(bulk=twq.testing_cold_fill_us(per, 0, sms), ldg=twq.testing_cold_fill_us(per, 1, sms),
                        what="us until every SM holds its 1/%d share of 10.75 MB of cold weights in shared memory (one launch, in-kernel "
                             "%%globaltimer; excludes the launch itself)" % sms)
        except Exception as e:                      # a measurement aid must not take the bench line down
            cold = dict(error=str(e))
    i8_tops = None
    if rank == 0:
        # an MMA-only tcgen05 kind::i8 loop on every SM, next to the 2 x BF16 figure the roofline uses
        i8_tops = twq.testing_measure_i8_tops(4096, 5)
        by_name = {r["workload"]: r for r in sweep}
        by_name.setdefault(args.workload, main_res)

    next1 = None
    if rank == 0 and not args.no_sweep:
        next1 = [measure_q4lr(n, twq, torch, max(20, min(args.steps, 100)), args.warmup, peaks,
                              with_oracle=(n == "c2_qproj_m16" and not args.no_cpu_baseline))
                 for n in ("c2_qproj_m1", "c2_qproj_m16", "c2_qproj_m64")]

    if rank == 0:
        cpu = None if args.no_cpu_baseline else time_oracle(L)
        # whole-job figure: N replicas each finish K calls in the max-over-ranks time
        value = whole_job_us_per_call(us, world)
        line = dict(metric="fused dual-linear us/call", value=round(value, 3), unit="us/call", n_gpus=world,
                    timing=main_res["timing"],
                    steps=args.steps, warmup=args.warmup, ms_per_step=round(us / 1e3, 6), higher_is_better=False,
                    scaling="weak", vs_baseline=None, dtype="s8 (INT4 codes x16) -> s32; f16 -> f32 low-rank",
                    data="synthetic",
                    config=config_for(args.workload),
                    l2_rotation="%d rotating copies, %.0f MB per lap" % (main_res["weight_copies"], main_res["lap_mb"]),
                    clocks=clocks,
                    e2e=dict(value=round(whole_job_us_per_call(us_e2e, world), 3), unit="us/call", h2d_bytes_per_step=2 * L.M * L.K,
                             d2h_bytes_per_step=2 * L.M * L.N),
                    gpu_launches=main_res["launches_per_step"] * args.steps,
                    roofline=main_res["roofline"],
                    # the two graded shapes (north_star: ">= 60 % of roofline at M = 1 and M = 2048"), lifted out of `sweep`
                    roofline_m1=by_name.get("c2_qproj_m1", {}).get("roofline"),
                    roofline_m2048=by_name.get("c3_gateup_m2048", {}).get("roofline"),
                    roofline_m2048_down=by_name.get("c3_down_m2048", {}).get("roofline"),
                    int8_peak=dict(measured_mma_only_tops=None if i8_tops is None else round(i8_tops, 1),
                                   roofline_uses_tops=round(2.0 * peaks["bf16_tflops"], 1),
                                   how="tcgen05.mma kind::i8 128x128x32 from shared memory, 4096 x 8 MMAs per SM, best of 5 "
                                       "(csrc/peak_i8.cu); the roofline denominator stays 2 x measured cuBLAS BF16 burst"),
                    cold_fill=cold,
                    us_host_per_call=main_res.get("us_host_per_call"),
                    cpu_baseline=cpu,
                    # `value` = the whole hot path through twq_dual_linear_x (one launch for M <= 64); beside it the same step as
                    # twq_quantize_act + twq_dual_linear (two launches) and those two kernels alone
                    api="twq_dual_linear_x", launches_per_step=main_res["launches_per_step"],
                    us_step_two_call=main_res["us_step_two_call"],
                    us_dual_linear=main_res["us_dual_linear"], us_quantize_act=main_res["us_quantize_act"],
                    eff_tops=main_res["eff_tops"], gbs=main_res["gbs"],
                    cublas_bf16_gemm_us=main_res.get("us_cublas_bf16_gemm"),
                    paper_context="paper: up to 1.8x over FP16 TensorRT-LLM end to end on RTX 4090 / L20 (PAPER.md L232)",
                    # the paper's 4-bit low-rank branch on the same shapes (whole path, one launch);
                    # compare with us_step of the matching sweep entry (FP16 low-rank branch, also one launch)
                    next1_q4lr=next1,
                    sweep=sweep)
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
