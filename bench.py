#!/usr/bin/env python
"""bench.py -- the headline measurement of the Dustin sparse-verification path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one verification pass of the whole hot path over one batch: dustin_verify_layer_fused (a1 scoring ->
a2 Eq. 5 fusion -> a3 Eq. 6 tiered top-k -> a4 sparse verification attention) in each of the L decoder layers of
the Qwen2.5-72B-shaped workload (BASELINE.json configs[2]: B=16, N=32768, Hq=64, Hkv=8, d=128, gamma=4, k=2048,
8-head subset), synthetic seeded inputs.  Rank 0 prints ONE JSON line; `value` is microseconds per layer.
The oracle is only executed by the cpu_baseline leg and by --impl reference.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2606_24957_b200 import synth  # noqa: E402

METRIC = "sparse_verify_attn_us_per_layer"
UNIT = "us/layer"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback


# --------------------------------------------------------------------------------------------------------------
# clocks: NVML sampled from a thread during the timed regions
# --------------------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, device_index: int, period_s: float = 0.02):
        self.period = period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self._h = None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            uuid = torch.cuda.get_device_properties(device_index).uuid
            try:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as e:                                    # pragma: no cover
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self._h is not None:
            self._stop.clear()
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
            self._thread = None

    def summary(self) -> dict:
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------------------------------------------
# workload
# --------------------------------------------------------------------------------------------------------------
class Workload:
    """L layers cycling over n_sets distinct seeded layer input sets (each with its own 2.1 GB K/V cache, so no
    layer finds its cache in L2).  Per-layer state: hist (in/out), out, idx, cnt.  Q / K_new / V_new live in
    stacked [L, ...] device buffers so the e2e leg can refill them from pinned host memory every step."""

    def __init__(self, cfg: synth.Config, n_sets: int, device):
        from paper_2606_24957_b200 import api
        self.api = api
        self.cfg, self.L, self.n_sets, self.device = cfg, cfg.n_layers, min(n_sets, cfg.n_layers), device
        c = cfg
        self.sets = []
        for s in range(self.n_sets):
            inp = synth.make_layer(c, s, device)
            inp.planted = None
            self.sets.append(inp)
        L, B, T, G, N = self.L, c.batch, c.n_new, c.n_lists, c.ctx
        self.q = torch.stack([self.sets[l % self.n_sets].q for l in range(L)])
        self.k_new = torch.stack([self.sets[l % self.n_sets].k_new for l in range(L)])
        self.v_new = torch.stack([self.sets[l % self.n_sets].v_new for l in range(L)])
        self.s_draft = torch.stack([s.s_draft for s in self.sets])
        self.hist = torch.stack([self.sets[l % self.n_sets].hist for l in range(L)])
        for s in self.sets:
            s.q = s.k_new = s.v_new = s.s_draft = s.hist = None
        self.k_max = self.sets[0].k_max
        self.out = torch.zeros_like(self.q)
        self.idx = torch.full((L, B, G, self.k_max), -1, dtype=torch.int32, device=device)
        self.cnt = torch.zeros((L, B, G), dtype=torch.int32, device=device)
        self.shape = api.Shape(B, c.n_q_heads, c.n_kv_heads, c.head_dim, T, N, 0.0)
        self.select = api.Select(c.budget, c.n_sink, c.n_recent, c.m_num, c.m_den, G, self.sets[0].budgets)
        self.kv = [api.KV.paged_nhd(s.k, s.v, s.page_table, s.seq_lens) if s.page_table is not None
                   else api.KV.contiguous_nhd(s.k, s.v, s.seq_lens) for s in self.sets]
        self.ws = api.alloc_workspace(self.shape, c.head_mask, 0)        # sized for the dense baseline too
        self.dense_out = torch.zeros_like(self.out[0])

    def cnt_arg(self, l: int):
        """List lengths for a stand-alone a4 call.  One budget k <= N for all sequences and no ragged lengths: every list
        holds exactly k entries, which is what cnt = NULL states (dustin.h) -- the fused call derives the same fact from
        its select parameters.  Otherwise the lengths the selection wrote."""
        s0 = self.sets[0]
        uniform = s0.seq_lens is None and s0.budgets is None and self.k_max <= self.cfg.ctx and self.cfg.budget == self.k_max
        return None if uniform else self.cnt[l]

    # -- schedules ---------------------------------------------------------------------------------------------
    def layer_fused(self, l: int):
        s = l % self.n_sets
        self.api.verify_layer_fused(self.shape, self.kv[s], self.q[l], self.k_new[l], self.v_new[l],
                                    self.cfg.head_mask, self.s_draft[s], self.hist[l], 1.0, self.select,
                                    self.out[l], self.idx[l], self.cnt[l], self.ws)

    def step_every_layer(self):
        """north_star schedule: a1..a4 in every layer."""
        for l in range(self.L):
            self.layer_fused(l)

    def step_score_once(self):
        """Paper schedule: a1-a3 in one layer, a4 in all L layers reusing that index set."""
        self.layer_fused(0)
        for l in range(1, self.L):
            s = l % self.n_sets
            self.api.sparse_verify_attn(self.shape, self.kv[s], self.q[l], self.k_new[l], self.v_new[l],
                                        self.idx[0], self.cnt_arg(0), self.out[l], self.ws)

    def step_score_only(self):
        """a1 alone in every layer (scores_now written to a scratch tensor): the estimation cost of PAPER.md:297."""
        if not hasattr(self, "scratch_scores"):
            self.scratch_scores = torch.empty_like(self.hist[0])
        T, Hq, d = self.cfg.n_new, self.cfg.n_q_heads, self.cfg.head_dim
        for l in range(self.L):
            s = l % self.n_sets
            self.api.score_heads(self.shape, self.kv[s], self.q[l][:, 0], self.cfg.head_mask, self.cfg.n_lists,
                                 self.scratch_scores, self.ws)

    def step_score_all_heads(self):
        """The Naive estimator of PAPER.md:297-299 (Fig. 8): a1 with EVERY query head in the subset, every layer."""
        c = self.cfg
        if not hasattr(self, "scratch_scores"):
            self.scratch_scores = torch.empty_like(self.hist[0])
        if not hasattr(self, "ws_all"):
            self.ws_all = self.api.alloc_workspace(self.shape, (1 << c.n_q_heads) - 1, self.k_max)
        for l in range(self.L):
            s = l % self.n_sets
            self.api.score_heads(self.shape, self.kv[s], self.q[l][:, 0], (1 << c.n_q_heads) - 1, c.n_lists,
                                 self.scratch_scores, self.ws_all)

    def quest_setup(self):
        """Page metadata of every distinct cache (built once, like after prefill) for the Quest-16 estimator leg."""
        if not hasattr(self, "quest_meta"):
            self.quest_meta = [self.api.quest_alloc_meta(self.shape, self.device) for _ in self.sets]
            n_pages = self.quest_meta[0].shape[1]
            self.quest_scores = torch.empty((self.cfg.batch, self.cfg.n_lists, n_pages), device=self.device)
            self.step_quest_build()

    def step_quest_build(self):
        """dustin_quest_build_pages for every distinct cache: one pass over K per cache."""
        for s in range(self.n_sets):
            self.api.quest_build_pages(self.shape, self.kv[s], self.quest_meta[s])

    def step_score_quest16(self):
        """The Quest-16 estimator of PAPER.md:297-299 (Fig. 8) in every layer: page scores for the SAME subset heads from
        the page min / max metadata alone (no read of K)."""
        c = self.cfg
        for l in range(self.L):
            s = l % self.n_sets
            self.api.quest_score_pages(self.shape, self.quest_meta[s], self.q[l][:, 0], c.head_mask, c.n_lists,
                                       self.quest_scores, self.ws, self.sets[s].seq_lens)

    def step_attn_only(self):
        """a4 alone in every layer, each with the index lists its own fused pass left in idx[l] / cnt[l] (kernel-only
        timing of the gathered attention: the region holds nothing but L launches of that kernel)."""
        for l in range(self.L):
            s = l % self.n_sets
            self.api.sparse_verify_attn(self.shape, self.kv[s], self.q[l], self.k_new[l], self.v_new[l],
                                        self.idx[l], self.cnt_arg(l), self.out[l], self.ws)

    def step_gather_probe(self):
        """The memory side of a4 alone: dustin_probe_gather reads the rows step_attn_only gathers, nothing else."""
        for l in range(self.L):
            s = l % self.n_sets
            self.api.probe_gather(self.shape, self.kv[s], self.idx[l], self.cnt[l], self.ws)

    def step_dense(self):
        """a5: full-cache verification attention in every layer (the baseline of PAPER.md Fig. 7/10)."""
        for l in range(self.L):
            s = l % self.n_sets
            self.api.sparse_verify_attn(self.shape, self.kv[s], self.q[l], self.k_new[l], self.v_new[l], None, None,
                                        self.dense_out, self.ws)

    # -- algorithmic bytes per layer ------------------------------------------------
    def bytes_per_layer(self) -> dict:
        c = self.cfg
        B, T, G, d, e = c.batch, c.n_new, c.n_lists, c.head_dim, 2
        s0 = self.sets[0]
        # ragged workloads: B * N stands for sum_b N_b and B * k for sum_b min(k_b, N_b)
        lens = s0.seq_lens.cpu().tolist() if s0.seq_lens is not None else [c.ctx] * B
        buds = s0.budgets.cpu().tolist() if s0.budgets is not None else [c.budget] * B
        BN = sum(lens)
        Bk = sum(min(k, n) for k, n in zip(buds, lens))
        N, k = BN / B, Bk / B
        groups = len({h // c.group for h in c.heads})
        a1_k = int(groups * BN * d * e)
        a1 = a1_k + B * len(c.heads) * d * e + 4 * G * BN
        a2 = 3 * 4 * G * BN
        a3 = 4 * BN * (G if self.s_draft.dim() == 4 else 1) + 4 * G * BN + 4 * G * Bk
        a4 = 2 * c.n_kv_heads * Bk * d * e + 2 * B * T * c.n_kv_heads * d * e + 2 * B * T * c.n_q_heads * d * e \
            + 4 * G * Bk
        a5 = 2 * c.n_kv_heads * BN * d * e + 2 * B * T * c.n_kv_heads * d * e + 2 * B * T * c.n_q_heads * d * e
        N, k = int(N), int(k)
        must_read = a1_k + 2 * 4 * G * B * N + a4          # K stream + hist, s_draft reads + a4
        return {"a1": a1, "a1_k": a1_k + B * len(c.heads) * d * e, "a2": a2, "a3": a3, "a4": a4, "a5": a5,
                "fused_must_read": must_read}


# --------------------------------------------------------------------------------------------------------------
# timing helpers
# --------------------------------------------------------------------------------------------------------------
class Dist:
    def __init__(self):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.on = self.world > 1

    def init(self, backend: str):
        if self.on:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            dist.init_process_group(backend=backend, rank=self.rank, world_size=self.world)

    def barrier(self):
        if self.on:
            import torch.distributed as dist
            dist.barrier()

    def max_float(self, x: float, device) -> float:
        if not self.on:
            return x
        import torch.distributed as dist
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def finish(self):
        if self.on:
            import torch.distributed as dist
            dist.destroy_process_group()


class CudaTimer:
    """Device-side clock: two CUDA events on the launching (current) stream."""

    def sync(self):
        torch.cuda.synchronize()

    def start(self):
        self.e0, self.e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.e0.record()

    def stop_ms(self) -> float:
        self.e1.record()
        torch.cuda.synchronize()
        return self.e0.elapsed_time(self.e1)


class HostTimer:
    """Wall clock; only for the CPU (gloo) tests of the rank plumbing and for the oracle arm."""

    def sync(self):
        pass

    def start(self):
        self.t0 = time.perf_counter()

    def stop_ms(self) -> float:
        return 1e3 * (time.perf_counter() - self.t0)


def time_steps(step_fn, steps: int, warmup: int, dist: Dist, device, timer=None) -> float:
    """ms per step: `warmup` untimed steps, then exactly `steps` steps between two CUDA events on the launching
    stream, bracketed by barrier + synchronize; max over ranks."""
    timer = timer or CudaTimer()
    for _ in range(warmup):
        step_fn()
    timer.sync()
    dist.barrier()
    timer.sync()
    timer.start()
    for _ in range(steps):
        step_fn()
    ms = timer.stop_ms()
    dist.barrier()
    return dist.max_float(ms, device) / steps


def rank_seed(cfg: synth.Config, rank: int) -> synth.Config:
    """Weak scaling: rank r draws its own batch of the same workload (independent sequences, no data-path
    collective -- DESIGN.md §9).  Rank 0 keeps the workload's base seed."""
    import dataclasses
    return dataclasses.replace(cfg, seed=cfg.seed + 104729 * rank)


def aggregate(us_per_layer_max: float, cfg: synth.Config, world: int) -> dict:
    """Whole-job figures from the max-over-ranks time: every rank verified `cfg.batch` sequences per layer in that
    time, so the job verified `world * cfg.batch`."""
    return {"global_batch": cfg.batch * world,
            "sequences_per_s": cfg.batch * world / (us_per_layer_max * 1e-6) if us_per_layer_max > 0 else 0.0}


def profile_steps(api, step_fn, steps: int) -> dict:
    """Second pass over the same steps with one CUDA event pair around every kernel launch (recorded inside the
    library on the launching stream): {kernel: (avg us per launch, launches per step)}."""
    torch.cuda.synchronize()
    api.profile_enable(True)
    for _ in range(steps):
        step_fn()
    torch.cuda.synchronize()
    rec = api.profile_collect()
    api.profile_enable(False)
    return {k: (1e3 * ms / n, n / steps) for k, (ms, n) in rec.items() if n}


class E2E:
    """The same step driven from HOST buffers: every step copies each layer's Q / K_new / V_new from pinned host
    memory, runs the layer, and copies the layer's output (and the last layer's index lists) back to pinned host
    memory.  Copies run on their own streams and overlap the kernels layer by layer.  The KV cache, the historical
    scores and the draft scores are device-resident state of the decode loop, not step inputs: S_Draft is what
    dustin_draft_aggregate leaves on the device (Eq. 5, first line), like the cache the draft model wrote."""

    def __init__(self, w: Workload):
        self.w = w
        pin = lambda t: torch.empty(t.shape, dtype=t.dtype, device="cpu", pin_memory=True).copy_(t)
        self.h_q, self.h_kn, self.h_vn = pin(w.q), pin(w.k_new), pin(w.v_new)
        self.h_out = torch.empty(w.out.shape, dtype=w.out.dtype, device="cpu", pin_memory=True)
        self.h_idx = torch.empty(w.idx[0].shape, dtype=torch.int32, device="cpu", pin_memory=True)
        self.h_cnt = torch.empty(w.cnt[0].shape, dtype=torch.int32, device="cpu", pin_memory=True)
        self.s_in, self.s_out = torch.cuda.Stream(), torch.cuda.Stream()
        nb = lambda t: t.numel() * t.element_size()
        self.h2d = nb(self.h_q) + nb(self.h_kn) + nb(self.h_vn)
        self.d2h = nb(self.h_out) + nb(self.h_idx) + nb(self.h_cnt)

    def step(self):
        w, main = self.w, torch.cuda.current_stream()
        start = torch.cuda.Event()
        start.record(main)
        self.s_in.wait_event(start)
        self.s_out.wait_event(start)
        ready = []
        with torch.cuda.stream(self.s_in):
            for l in range(w.L):
                w.q[l].copy_(self.h_q[l], non_blocking=True)
                w.k_new[l].copy_(self.h_kn[l], non_blocking=True)
                w.v_new[l].copy_(self.h_vn[l], non_blocking=True)
                ev = torch.cuda.Event()
                ev.record(self.s_in)
                ready.append(ev)
        for l in range(w.L):
            main.wait_event(ready[l])
            w.layer_fused(l)
            done = torch.cuda.Event()
            done.record(main)
            self.s_out.wait_event(done)
            with torch.cuda.stream(self.s_out):
                self.h_out[l].copy_(w.out[l], non_blocking=True)
        with torch.cuda.stream(self.s_out):
            self.h_idx.copy_(w.idx[w.L - 1], non_blocking=True)
            self.h_cnt.copy_(w.cnt[w.L - 1], non_blocking=True)
            fin = torch.cuda.Event()
            fin.record(self.s_out)
        main.wait_event(fin)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel: str):
    """(DRAM bytes per launch of `kernel`, commit the capture was taken at) from the committed ncu --set full summary
    (profiles/traffic.json: dram__bytes_read.sum + dram__bytes_write.sum of one capture; stale once the kernel changes,
    hence the commit stamp that travels with it)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            d = json.load(f)
        return d.get(kernel), d.get("captured_at_commit")
    except Exception:
        return None, None


def graphed(step_fn):
    """Captures one step (all L layers' launches on the current stream) into a CUDA graph; returns its replay."""
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step_fn()
    return g.replay


# --------------------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands, on the host cores, on a bounded sample of the same workload
# --------------------------------------------------------------------------------------------------------------
def oracle_layer(ref, cfg: synth.Config, inp: synth.LayerInputs, stage_s: dict = None):
    """One layer of the path through oracle/ (O1 -> O2 -> O3 -> O4).  `inp` on the CPU.  stage_s (optional) receives the
    wall time of each stage in seconds (appended to lists)."""
    def timed(name, fn):
        t0 = time.perf_counter()
        r = fn()
        if stage_s is not None:
            stage_s.setdefault(name, []).append(time.perf_counter() - t0)
        return r
    kv = ref.KV.contiguous_nhd(inp.k, inp.v, inp.seq_lens)
    a = timed("O1_score_heads", lambda: ref.score_heads(kv, inp.q[:, 0], cfg.head_mask, cfg.n_lists, cfg.n_kv_heads, cfg.ctx))
    h = timed("O2_fuse_scores", lambda: ref.fuse_scores(a, inp.hist, 1.0, inp.seq_lens))
    idx, cnt = timed("O3_topk_select", lambda: ref.topk_select(inp.s_draft, h, cfg.budget, cfg.n_sink, cfg.n_recent,
                                                               cfg.m_num, cfg.m_den, inp.k_max, inp.seq_lens, inp.budgets))
    out, _ = timed("O4_sparse_verify_attn", lambda: ref.sparse_verify_attn(kv, inp.q, inp.k_new, inp.v_new, idx, cnt, cfg.ctx))
    return out


def cpu_baseline(cfg: synth.Config, inp_cpu: synth.LayerInputs, budget_s: float = 15.0) -> dict:
    """The oracle as it stands on the host cores: ONE full-size layer, repeated within ~budget_s, median; per-stage
    medians beside it; the dense full-cache oracle (a5) once (SURVEY.md section 8d "Oracle timing")."""
    from oracle import ref
    stage_s = {}
    t0 = time.perf_counter()
    oracle_layer(ref, cfg, inp_cpu, stage_s)
    t1 = time.perf_counter() - t0
    n = max(1, min(8, int(budget_s / max(t1, 1e-3)) - 1))
    times = [t1]
    for _ in range(n):
        t0 = time.perf_counter()
        oracle_layer(ref, cfg, inp_cpu, stage_s)
        times.append(time.perf_counter() - t0)
    us = 1e6 * statistics.median(times)
    kv = ref.KV.contiguous_nhd(inp_cpu.k, inp_cpu.v, inp_cpu.seq_lens)
    t0 = time.perf_counter()
    ref.sparse_verify_attn(kv, inp_cpu.q, inp_cpu.k_new, inp_cpu.v_new, None, None, cfg.ctx)
    dense_us = 1e6 * (time.perf_counter() - t0)
    return {"value": us, "unit": UNIT, "cores": ref.threads(), "kind": "oracle",
            "sample": f"{len(times)} repetitions of ONE full-size layer (all {cfg.batch} sequences, N={cfg.ctx}; "
                      f"O1 scoring -> O2 fusion -> O3 selection -> O4 attention), median; a step is "
                      f"{cfg.n_layers} such layers",
            "stages_us_per_layer": {k: round(1e6 * statistics.median(v), 1) for k, v in stage_s.items()},
            "dense_us_per_layer": round(dense_us, 1),
            "dense_sample": "the dense full-cache oracle (O4 with idx = NULL) on the same layer, timed once",
            "build": "g++ -O2 -fopenmp (oracle/ref.py), fp64, as it stands"}


def run_reference(args, dist: Dist):
    """--impl reference: the oracle timed on this box's host cores, same config / metric / unit; each step is a
    bounded sample (one layer of the workload).  Rank 0 only."""
    if dist.rank != 0:
        return
    from oracle import ref
    cfg = headline_config(args)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    inp = synth.make_layer(cfg, 0, dev).to("cpu")
    inp.planted = None
    for _ in range(args.warmup):
        oracle_layer(ref, cfg, inp)
    times = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        oracle_layer(ref, cfg, inp)
        times.append(time.perf_counter() - t0)
    us = 1e6 * sum(times) / len(times)
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, 1),
        "run": {"sample": "oracle: ONE full-size layer per step (a bounded sample of the L-layer step)",
                "world": dist.world, "launcher": os.environ.get("DUSTIN_BENCH_LAUNCHER", "torchrun" if dist.on else "single process")},
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": ref.threads(), "kind": "oracle",
                         "sample": "each step = ONE full-size layer of the workload through oracle/ (O1..O4)"},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def headline_config(args) -> synth.Config:
    cfg = synth.config_qwen72b(batch=args.batch, ctx=args.ctx, n_layers=args.layers, spread=not args.packed,
                               gamma=getattr(args, "gamma", 4))
    return cfg


def workload_config(cfg: synth.Config, world: int = 1) -> dict:
    """What is measured -- the same dict in both arms (ours and --impl reference); how each arm runs it is in `run`."""
    return {"workload": "BASELINE.json configs[2]: Qwen2.5-72B-shaped verification step "
                        f"(B={cfg.batch}, N={cfg.ctx}, Hq={cfg.n_q_heads}, Hkv={cfg.n_kv_heads}, d={cfg.head_dim}, "
                        f"gamma={cfg.gamma}, k={cfg.budget} incl. {cfg.n_sink} sink + {cfg.n_recent} recent, "
                        f"|H|={len(cfg.heads)} subset heads {'spread one per KV group' if cfg.n_lists > 1 else 'packed in one KV group'}, "
                        f"G={cfg.n_lists} lists per sequence, L={cfg.n_layers} layers)",
            "schedule": "every layer runs a1 scoring -> a2 fusion -> a3 top-k -> a4 sparse attention (north_star)",
            "global_batch": cfg.batch * world, "batch_per_gpu": cfg.batch, "seq_len": cfg.ctx, "layers": cfg.n_layers,
            "budget": cfg.budget,
            "l2": "inputs exceed L2: every layer has a 2.1 GB K/V cache, none is re-read within 126 MB"}


def run_info(n_sets: int, world: int, ranks=None) -> dict:
    return {"launcher": os.environ.get("DUSTIN_BENCH_LAUNCHER", "torchrun" if world > 1 else "single process"),
            "ranks": ranks,
            "scaling_bearing_number": "aggregate.sequences_per_s (value is max-over-ranks us per layer at a fixed per-GPU "
                                      "batch, flat by construction under weak scaling)",
            "distinct_kv_caches": n_sets,
            "launch": "one CUDA graph replay per step (the L fused C-ABI calls captured once)",
            "scaling": "weak: every rank runs this workload on its own batch (value = max-over-ranks us per layer of the "
                       "whole job's global batch)", "world": world}


def measure_workload(api, cfg: synth.Config, n_sets: int, steps: int, warmup: int, dist: Dist, device,
                     with_dense: bool, with_score_once: bool, profile: bool = True):
    """Builds the workload and times its schedules.  Returns (workload, dict of results)."""
    w = Workload(cfg, n_sets, device)
    w.step_every_layer()                                  # first-launch setup (function attributes) before capture
    n0 = api.launch_count()
    replay = graphed(w.step_every_layer)
    launches_per_step = api.launch_count() - n0
    r = {"launches_per_step": launches_per_step}
    sampler = ClockSampler(dist.local_rank)
    with sampler:
        r["ms_per_step"] = time_steps(replay, steps, warmup, dist, device)
    r["clocks"] = sampler.summary()
    r["us_per_layer"] = 1e3 * r["ms_per_step"] / cfg.n_layers
    if profile:
        r["kernels"] = profile_steps(api, w.step_every_layer, min(steps, 3))
    if with_score_once:
        rp = graphed(w.step_attn_only)
        r["attn_only_us_per_launch"] = 1e3 * time_steps(rp, max(3, steps // 2), warmup, dist, device) / cfg.n_layers
        w.step_gather_probe()
        rp = graphed(w.step_gather_probe)
        r["gather_probe_us_per_launch"] = 1e3 * time_steps(rp, max(3, steps // 2), warmup, dist, device) / cfg.n_layers
        rp = graphed(w.step_score_once)
        r["score_once_us_per_layer"] = 1e3 * time_steps(rp, max(3, steps // 2), warmup, dist, device) / cfg.n_layers
    if with_dense:
        w.step_dense()
        rp = graphed(w.step_dense)
        r["dense_us_per_layer"] = 1e3 * time_steps(rp, max(3, steps // 3), warmup, dist, device) / cfg.n_layers
        if profile:
            r["dense_kernels"] = profile_steps(api, w.step_dense, 2)
    return w, r


def run_sweep(api, args, dist: Dist, device):
    """BASELINE.json configs[3] (context sweep on the Qwen2.5-72B-shaped layer: N in 4k..128k, batch reduced so the
    cache fits, budget 2048 and 6.25 % of N, gamma 2 / 4 / 8) and configs[4] (paged, ragged, Llama-3-8B-shaped).  Per
    point, graph-replayed regions that hold one kind of launch each: scoring (a1) and sparse verification (a4)
    separately, the fused layer (a1..a4) and the dense baseline (a5).  Rank 0 prints ONE JSON line {"sweep": [...]}."""
    peak, _ = measured_peak()
    points = []
    grid = []
    for ctx, batch in ((4096, 16), (8192, 16), (16384, 16), (32768, 16), (65536, 8), (131072, 4)):
        for gamma in (2, 4, 8):
            grid.append(("fixed-2048", ctx, batch, gamma, 2048))
        grid.append(("6.25%", ctx, batch, 4, ctx // 16))
    # the paper's own efficiency budget (PAPER.md:443, :470: k = 512 with S = 4 sink + W = 16 recent; :570 quotes 27.85x /
    # 15.58x self-attention speed-up at 32k / 16k, B = 16 on other hardware -- context only)
    for ctx in (16384, 32768):
        grid.append(("paper-512", ctx, 16, 4, 512))
    L, n_sets = 8, 4
    for label, ctx, batch, gamma, budget in grid:
        cfg = synth.config_qwen72b(batch=batch, ctx=ctx, n_layers=L, gamma=gamma, budget=budget)
        if label == "paper-512":
            cfg = synth.shrink(cfg, n_sink=4, n_recent=16)
        points.append(sweep_point(api, cfg, n_sets, dist, device, peak,
                                  {"series": label, "ctx": ctx, "batch": batch, "gamma": gamma, "budget": budget},
                                  naive=(label == "fixed-2048" and gamma == 4)))
        torch.cuda.empty_cache()
    cfg = synth.config_paged(n_layers=4)
    points.append(sweep_point(api, cfg, 2, dist, device, peak,
                              {"series": "paged-ragged (configs[4])", "ctx": "U[8192,65536]", "batch": cfg.batch,
                               "gamma": cfg.gamma, "budget": "6.25% of N_b", "page_size": cfg.page_size}))
    if dist.rank == 0:
        print(json.dumps({"sweep": points, "unit": "us per layer (graph-replayed, CUDA events)",
                          "peak_gbs": peak, "layers_per_point": L, "crossover": crossover(points)}), flush=True)


def crossover(points) -> dict:
    """Context length at which the fused sparse layer costs what the dense baseline costs (log-linear interpolation of
    dense/fused over the context points of one series at gamma = 4): below it the method's fixed costs lose."""
    out = {}
    for series in ("fixed-2048", "6.25%"):
        pts = sorted((p["ctx"], p["speedup_vs_dense"]) for p in points
                     if p.get("series") == series and p.get("gamma") == 4 and isinstance(p.get("ctx"), int))
        x = None
        for (c0, r0), (c1, r1) in zip(pts, pts[1:]):
            if (r0 - 1.0) * (r1 - 1.0) <= 0 and r0 != r1:
                import math
                x = int(round(math.exp(math.log(c0) + (1.0 - r0) / (r1 - r0) * (math.log(c1) - math.log(c0)))))
                break
        out[series] = {"fused_equals_dense_at_ctx": x,
                       "note": None if x else ("fused faster than dense at every point" if pts and pts[0][1] > 1
                                               else "no crossing inside the sweep")}
    return out


def sweep_point(api, cfg: synth.Config, n_sets: int, dist: Dist, device, peak: float, tag: dict,
                naive: bool = False) -> dict:
    """One workload point: graph-replayed regions that hold one kind of launch each -- the fused layer (a1..a4), scoring
    alone (a1), sparse verification alone (a4, on the lists of the fused pass), the dense baseline (a5) and, with
    naive=True, scoring with EVERY head in the subset (the Naive estimator of PAPER.md:297-299)."""
    w = Workload(cfg, n_sets, device)
    w.step_every_layer()
    w.step_dense()
    w.step_score_only()
    by = w.bytes_per_layer()
    t = {}
    legs = [("fused", w.step_every_layer), ("score", w.step_score_only), ("attn", w.step_attn_only),
            ("dense", w.step_dense)]
    if naive:
        w.step_score_all_heads()
        legs.append(("score_all_heads", w.step_score_all_heads))
        w.quest_setup()
        w.step_score_quest16()
        legs.append(("score_quest16", w.step_score_quest16))
    for name, fn in legs:
        t[name] = 1e3 * time_steps(graphed(fn), 3, 3, dist, device) / cfg.n_layers
    # the streaming kernel of a1 alone (event pairs inside the library): "score" above is the whole staged a1 stage --
    # score_logits_kernel + the stats and normalise launches that write scores_now
    kern = profile_steps(api, w.step_score_only, 2).get("score_logits_kernel")
    out = dict(tag)
    if kern:
        out["score_logits_kernel_us"] = round(kern[0], 2)
        out["score_logits_kernel_gbs"] = round(by["a1_k"] / kern[0] / 1e3, 1)
    if naive:
        out["score_all_heads_us"] = round(t["score_all_heads"], 2)
        out["score_all_heads_over_dense"] = round(t["score_all_heads"] / t["dense"], 3)
        # Fig. 8's third estimator: Quest with 16-token pages on the same subset heads (metadata bytes = 1/8 of the K bytes
        # of the scored groups), and the one-off cost of building that metadata (one pass over K per cache)
        out["score_quest16_us"] = round(t["score_quest16"], 2)
        out["score_quest16_over_dense"] = round(t["score_quest16"] / t["dense"], 3)
        out["score_subset_over_dense"] = round(t["score"] / t["dense"], 3)
        meta_bytes = by["a1_k"] / 8.0
        out["score_quest16_gbs"] = round(meta_bytes / t["score_quest16"] / 1e3, 1)
        tb = 1e3 * time_steps(graphed(w.step_quest_build), 3, 3, dist, device) / w.n_sets
        out["quest16_build_us_per_cache"] = round(tb, 2)
        out["quest16_build_gbs"] = round((cfg.batch * cfg.ctx * cfg.n_kv_heads * cfg.head_dim * 2 * 1.125) / tb / 1e3, 1)
    out.update({
        "fused_us": round(t["fused"], 2), "score_us": round(t["score"], 2), "sparse_attn_us": round(t["attn"], 2),
        "dense_us": round(t["dense"], 2), "speedup_vs_dense": round(t["dense"] / t["fused"], 2),
        "attn_speedup_vs_dense": round(t["dense"] / t["attn"], 2),
        "score_gbs": round(by["a1_k"] / t["score"] / 1e3, 1), "sparse_attn_gbs": round(by["a4"] / t["attn"] / 1e3, 1),
        "dense_gbs": round(by["a5"] / t["dense"] / 1e3, 1),
        "fused_frac_of_peak": round(by["fused_must_read"] / t["fused"] / 1e3 / peak, 3),
    })
    del w
    return out


def run_loop(api, args, dist: Dist, device):
    """Multi-step decode loop (PAPER.md:153 accept -> append -> next step): per speculative
    step, on the device with no host synchronisation inside a step,
      dustin_draft_aggregate (S_Draft from a Qwen2.5-0.5B-shaped draft: 14 / 2 heads, d = 64, 3 layers x 4 heads, Gamma
      lookahead queries -- PAPER.md:395)  ->  dustin_verify_layer_fused in each of L target layers (history H carried per
      layer)  ->  dustin_append_kv of the accepted rows into every target-layer cache and every draft-layer cache.
    Accept lengths are seeded synthetic draws with mean ~2.2 tokens per step (tau of PAPER.md:315-319, Table 2); the
    context N_b grows by them.  Reports attention-path us per step, per layer and per accepted token."""
    L, n_steps, B = args.loop_layers, args.loop_steps, args.batch
    cfg = synth.config_qwen72b(B, args.ctx, L)
    T, G, Hkv, d = cfg.n_new, cfg.n_lists, cfg.n_kv_heads, cfg.head_dim
    N0 = args.ctx - n_steps * T                              # room for every step's appends below max_ctx
    g = torch.Generator(device=device)
    g.manual_seed(cfg.seed + 77)
    layers = []
    for l in range(L):
        inp = synth.make_layer(cfg, l, device)
        inp.planted = None
        layers.append(inp)
    shape = api.Shape(B, cfg.n_q_heads, Hkv, d, T, cfg.ctx, 0.0)
    select = api.Select(cfg.budget, cfg.n_sink, cfg.n_recent, cfg.m_num, cfg.m_den, G, None)
    seq_lens = torch.full((B,), N0, dtype=torch.int32, device=device)
    kvs = [api.KV.contiguous_nhd(x.k, x.v, seq_lens) for x in layers]
    hist = torch.stack([x.hist for x in layers])
    for x in layers:
        x.hist = None
    ws = api.alloc_workspace(shape, cfg.head_mask, layers[0].k_max)
    out = torch.zeros_like(layers[0].q)
    idx = torch.full((B, G, layers[0].k_max), -1, dtype=torch.int32, device=device)
    cnt = torch.zeros((B, G), dtype=torch.int32, device=device)
    # draft model: 3 selected layers x 4 heads, Gamma lookahead queries, its own K caches
    dHq, dHkv, dd, dL, dmask = 14, 2, 64, 3, 0b00101000100010
    dshape = api.Shape(B, dHq, dHkv, dd, cfg.gamma, cfg.ctx, 0.0)
    dk = [torch.randn(B, cfg.ctx, dHkv, dd, device=device, generator=g).bfloat16() for _ in range(dL)]
    dq = [torch.randn(B, cfg.gamma, dHq, dd, device=device, generator=g).bfloat16() for _ in range(dL)]
    dkn = torch.randn(B, T, dHkv, dd, device=device, generator=g).bfloat16()
    dkvs = [api.KV.contiguous_nhd(k, k, seq_lens) for k in dk]          # V of the draft is not read by this path
    dws = api.alloc_draft_workspace(dshape, dmask)
    s_draft = torch.zeros(B, cfg.ctx, device=device)
    # accept lengths: 1 + Binomial(Gamma, p) with mean 2.2 accepted tokens per step (the bonus token always lands)
    p_acc = (2.2 - 1.0) / cfg.gamma
    accepts = (1 + (torch.rand(n_steps, B, cfg.gamma, device=device, generator=g) < p_acc).sum(-1)).to(torch.int32)
    n_app = torch.zeros(B, dtype=torch.int32, device=device)
    scratch = torch.zeros_like(seq_lens)
    dshape_T = api.Shape(B, dHq, dHkv, dd, T, cfg.ctx, 0.0)      # the draft's verify block has T rows too

    def step():
        api.draft_aggregate(dshape, dkvs, dq, dmask, s_draft, dws)
        for l in range(L):
            x = layers[l]
            api.verify_layer_fused(shape, kvs[l], x.q, x.k_new, x.v_new, cfg.head_mask, s_draft, hist[l], 1.0, select,
                                   out, idx, cnt, ws)
        # accept -> append.  dustin_append_kv advances the lengths it is given; all caches share one set of
        # lengths, so every call but the last works on a scratch copy and the last one advances the live lengths.
        caches = [(shape, api.KV.contiguous_nhd(x.k, x.v, None), x.k_new, x.v_new, hist[l]) for l, x in enumerate(layers)]
        caches += [(dshape_T, api.KV.contiguous_nhd(k, k, None), dkn, dkn, None) for k in dk]
        for i, (sh_, kv_, kn_, vn_, h_) in enumerate(caches):
            if i < len(caches) - 1:
                scratch.copy_(seq_lens)
                api.append_kv(sh_, kv_, scratch, kn_, vn_, n_app, h_)
            else:
                api.append_kv(sh_, kv_, seq_lens, kn_, vn_, n_app, h_)

    # warm-up step on a scratch copy of the lengths is not possible without touching the caches: the first step is
    # simply not timed
    # Steps 1 .. n/2 run eagerly (one C-ABI call after the other from Python), the rest replay ONE CUDA graph of the whole
    # step, captured once: lengths, history and accept counts live on the device and every pointer is fixed, so the step
    # is the same graph whatever the lengths have grown to.  Both read-outs are reported.
    per_step, per_step_eager = [], []
    total_acc = 0
    n_eager = max(2, n_steps // 2)
    replay = None
    for sidx in range(n_steps):
        n_app.copy_(accepts[sidx])
        if sidx == n_eager:
            replay = graphed(step)                 # capture only: nothing runs, the state is untouched
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        (replay or step)()
        e1.record()
        torch.cuda.synchronize()
        if sidx >= 1:
            (per_step if replay else per_step_eager).append(1e3 * e0.elapsed_time(e1))
        if replay:
            total_acc += int(accepts[sidx].sum())
    lens_end = seq_lens.cpu().tolist()
    med = statistics.median(per_step)
    med_eager = statistics.median(per_step_eager)
    res = {"decode_loop": {
        "workload": f"Qwen2.5-72B-shaped target ({L} layers with their own caches), Qwen2.5-0.5B-shaped draft (3 layers x 4 "
                    f"heads, Gamma={cfg.gamma}), B={B}, N_b {N0} -> {lens_end[0]}..{max(lens_end)}, k={cfg.budget}",
        "steps_timed": len(per_step), "accepted_tokens_per_step_per_sequence": round(total_acc / len(per_step) / B, 3),
        "us_per_step": round(med, 1), "us_per_step_min_max": [round(min(per_step), 1), round(max(per_step), 1)],
        "us_per_layer": round(med / L, 2),
        "us_per_accepted_token": round(med * len(per_step) / max(total_acc / B, 1e-9), 1),
        "eager": {"steps_timed": len(per_step_eager), "us_per_step": round(med_eager, 1),
                  "us_per_layer": round(med_eager / L, 2)},
        "what": "draft_aggregate + L x verify_layer_fused + (L + 3) x append_kv per step on one stream, CUDA events around "
                "each step, the first step untimed; us_per_step / us_per_layer: the whole step replayed as ONE CUDA graph "
                "(captured once; lengths, history and accept counts are device state); `eager`: the same step as "
                "back-to-back C-ABI calls from Python; acceptance is a seeded draw (no models here)"}}
    if dist.rank == 0:
        print(json.dumps(res), flush=True)
    return res


def run_quest(api, args, dist: Dist, device):
    """Quest-16 estimator alone at the headline shape (Fig. 8): the metadata build of one K cache and the
    page scoring of the subset heads, each replayed as a CUDA graph over 4 distinct caches, beside the subset a1 on the same
    caches.  This is also the command the ncu capture of the Quest kernels runs (profiles/r03_ncu.md)."""
    cfg = synth.config_qwen72b(batch=args.batch, ctx=args.ctx, n_layers=4, gamma=args.gamma)
    w = Workload(cfg, 4, device)
    w.quest_setup()
    w.step_score_quest16()
    w.step_score_only()
    by = w.bytes_per_layer()
    t_score = 1e3 * time_steps(graphed(w.step_score_quest16), args.steps, args.warmup, dist, device) / cfg.n_layers
    t_build = 1e3 * time_steps(graphed(w.step_quest_build), args.steps, args.warmup, dist, device) / w.n_sets
    t_a1 = 1e3 * time_steps(graphed(w.step_score_only), args.steps, args.warmup, dist, device) / cfg.n_layers
    kern = profile_steps(api, lambda: (w.step_quest_build(), w.step_score_quest16()), 2)
    peak, _ = measured_peak()
    k_bytes = cfg.batch * cfg.ctx * cfg.n_kv_heads * cfg.head_dim * 2
    res = {"quest16": {
        "workload": f"Qwen2.5-72B-shaped layer, B={cfg.batch}, N={cfg.ctx}, {len(cfg.heads)} subset heads, page 16",
        "score_pages_us": round(t_score, 2), "score_pages_gbs": round(by["a1_k"] / 8 / t_score / 1e3, 1),
        "score_pages_frac_of_peak": round(by["a1_k"] / 8 / t_score / 1e3 / peak, 3),
        "build_us_per_cache": round(t_build, 2), "build_gbs": round(1.125 * k_bytes / t_build / 1e3, 1),
        "build_frac_of_peak": round(1.125 * k_bytes / t_build / 1e3 / peak, 3),
        "subset_a1_us": round(t_a1, 2),
        "kernels_us_per_launch": {k: round(v[0], 2) for k, v in kern.items()},
        "what": "graph-replayed, CUDA events; bytes: metadata = 1/8 of the K bytes of the scored groups (scoring), K + "
                "metadata (build); kernels_us_per_launch: eager event pairs inside the library"}}
    if dist.rank == 0:
        print(json.dumps(res), flush=True)
    return res


def run_arr(api, args, dist: Dist, device):
    """Quality read-out on the synthetic saliency-drift workload (shape of PAPER.md Table 3 /
    Fig. 4, no datasets): lists are selected at drift step l (history = step l-1's scores, draft = noisy step-l scores)
    with Dustin-T (m = 0), Dustin-H (m = 1/2) and Dustin-D (m = all), and scored by the Attention Recovery Rate (Eq. 1)
    against the attention of step l+1; the SD-oracle bound (Eq. 3-4, w = 1) is TopK_k of that future attention itself."""
    cfg0 = synth.config_qwen72b(batch=args.batch, ctx=args.ctx, n_layers=1)
    out = {"workload": f"Qwen2.5-72B-shaped, B={cfg0.batch}, N={cfg0.ctx}, k={cfg0.budget}, drift 10 % per step", "steps": []}
    n_steps = 4
    acc = {}
    for l in range(n_steps):
        cur = synth.make_layer(cfg0, l, device)
        nxt = synth.make_layer(cfg0, l + 1, device, want_hist_draft=False)
        B, G, N = cfg0.batch, cfg0.n_lists, cfg0.ctx
        shape = api.Shape(B, cfg0.n_q_heads, cfg0.n_kv_heads, cfg0.head_dim, cfg0.n_new, N, 0.0)
        ws = api.alloc_workspace(shape, cfg0.head_mask, cur.k_max)
        truth = torch.empty(B, G, N, device=device)
        api.score_heads(shape, api.KV.contiguous_nhd(nxt.k, nxt.v, None), nxt.q[:, 0], cfg0.head_mask, G, truth, ws)
        idx = torch.empty(B, G, cur.k_max, dtype=torch.int32, device=device)
        cnt = torch.empty(B, G, dtype=torch.int32, device=device)
        arr = torch.empty(B, G, device=device)
        outb = torch.empty_like(cur.q)
        row = {}
        for name, (num, den) in (("dustin_T (m=0)", (0, 1)), ("dustin_H (m=1/2)", (1, 2)), ("dustin_D (m=all)", (1, 1))):
            hist = cur.hist.clone()
            sel = api.Select(cfg0.budget, cfg0.n_sink, cfg0.n_recent, num, den, G, None)
            api.verify_layer_fused(shape, api.KV.contiguous_nhd(cur.k, cur.v, None), cur.q, cur.k_new, cur.v_new,
                                   cfg0.head_mask, cur.s_draft, hist, 1.0, sel, outb, idx, cnt, ws)
            api.arr(truth, idx, cnt, arr)
            row[name] = float(arr.mean())
        sel = api.Select(cfg0.budget, 0, 0, 0, 1, G, None)                      # Eq. 3: TopK_k of the future attention
        api.topk_select(sel, truth, truth, idx, cnt)
        api.arr(truth, idx, cnt, arr)
        row["sd_oracle (Eq. 4)"] = float(arr.mean())
        out["steps"].append({k: round(v, 4) for k, v in row.items()})
        for k, v in row.items():
            acc[k] = acc.get(k, 0.0) + v / n_steps
        del cur, nxt
        torch.cuda.empty_cache()
    out["mean_arr"] = {k: round(v, 4) for k, v in acc.items()}
    if dist.rank == 0:
        print(json.dumps({"arr_readout": out}), flush=True)


def stage_table(kernels: dict, layers: int) -> dict:
    """us per layer per kernel: avg launch duration x launches per step / layers."""
    return {k: round(us * n / layers, 3) for k, (us, n) in kernels.items()}


def spawn_ranks(n: int, argv=None) -> int:
    """`python bench.py --gpus N` without a launcher: re-executes this script under torch.distributed.run with one rank
    per GPU (the launch line the docstring gives, on a free port) and returns its exit code.  The ranks find WORLD_SIZE
    in their environment and take the normal multi-rank path; rank 0 prints the one JSON line."""
    import socket
    import subprocess
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *(sys.argv[1:] if argv is None else argv)]
    env = dict(os.environ, DUSTIN_BENCH_LAUNCHER="self-spawned torch.distributed.run")
    return subprocess.call(cmd, env=env)


def rank_table(dist: Dist, device) -> list:
    """Which process runs on which GPU, gathered over the process group: the evidence that N ranks on N distinct devices
    took part (the path has no data collective whose NCCL log would show it)."""
    me = {"rank": dist.rank, "local_rank": dist.local_rank, "pid": os.getpid()}
    if torch.cuda.is_available() and str(device).startswith("cuda"):
        pr = torch.cuda.get_device_properties(device)
        me.update(device=torch.cuda.current_device(), name=pr.name, uuid=str(getattr(pr, "uuid", "")))
    if not dist.on:
        return [me]
    import torch.distributed as td
    out = [None] * dist.world
    td.all_gather_object(out, me)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=16)
    ap.add_argument("--ctx", type=int, default=32768)
    ap.add_argument("--layers", type=int, default=80)
    ap.add_argument("--gamma", type=int, default=4, help="draft depth (T = gamma + 1 verify positions)")
    ap.add_argument("--sets", type=int, default=20, help="distinct K/V caches the layers cycle over")
    ap.add_argument("--packed", action="store_true", help="headline on the packed/G=1 subset placement")
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary workloads and the CPU baseline")
    ap.add_argument("--arr", action="store_true", help="ARR read-out of the selection policies on the drift workload")
    ap.add_argument("--sweep", action="store_true", help="context / gamma / budget sweep (configs[3]) + paged (configs[4])")
    ap.add_argument("--loop", action="store_true", help="multi-step decode loop: draft aggregate -> L fused layers -> append")
    ap.add_argument("--quest", action="store_true", help="Quest-16 estimator alone: metadata build + page scoring at the headline shape")
    ap.add_argument("--loop-layers", type=int, default=8)
    ap.add_argument("--loop-steps", type=int, default=12)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: never report N GPUs from one process -- start the N ranks ourselves
        raise SystemExit(spawn_ranks(args.gpus))
    dist = Dist()
    if args.impl == "reference":
        run_reference(args, dist)
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if dist.on and dist.world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={dist.world}")
    torch.cuda.set_device(dist.local_rank)
    device = torch.device("cuda", dist.local_rank)
    dist.init("nccl")
    from paper_2606_24957_b200 import api, build as cuda_build
    if not os.path.exists(api.LIB_PATH):
        if dist.rank == 0:
            cuda_build.build()
        dist.barrier()
    api.lib()

    if args.sweep or args.arr or args.loop or args.quest:
        (run_sweep if args.sweep else (run_arr if args.arr else (run_loop if args.loop else run_quest)))(api, args, dist, device)
        dist.finish()
        return
    cfg = rank_seed(headline_config(args), dist.rank)
    w, r = measure_workload(api, cfg, args.sets, args.steps, args.warmup, dist, device, True, True)
    by = w.bytes_per_layer()
    peak, peak_src = measured_peak()
    L = cfg.n_layers
    us_layer = r["us_per_layer"]

    # e2e: same step from host buffers
    e2e = E2E(w)
    e2e.step()                                            # once eagerly, then the whole step (copies on their own
    e2e_step = graphed(e2e.step)                          # streams included) as one CUDA graph, like the device-only leg
    e2e_ms = time_steps(e2e_step, max(3, args.steps // 2), args.warmup, dist, device)

    # roofline of the dominant kernel (largest share of the step in the per-kernel event pass)
    kern = r["kernels"]
    share = {k: us * n for k, (us, n) in kern.items()}
    dom = max(share, key=share.get)
    kbytes = {"score_logits_kernel": by["a1_k"], "attn_kernel": by["a4"]}
    def roof(kernel, nbytes, us=None, how="CUDA event pair around each launch, second pass over the same steps"):
        us = kern[kernel][0] if us is None else us
        ach = nbytes / us / 1e3
        traffic, traffic_commit = ncu_traffic(kernel)
        return {"kernel": kernel, "bound": "hbm", "achieved": round(ach, 1), "peak": peak, "unit": "GB/s",
                "frac": round(ach / peak, 4), "traffic": traffic, "traffic_commit": traffic_commit,
                # the measured peak is a COPY (read + write) bandwidth; a read-only stream can run a few per cent above it
                **({"frac_note": "above 1: the peak is the measured copy (read+write) bandwidth, this kernel only reads"}
                   if ach > peak else {}),
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": nbytes, "avg_launch_us": round(us, 3),
                # share of the GRAPH-timed step: this kernel's launches x its average duration over the step time
                "share_of_step": round(kern[kernel][0] * kern[kernel][1] / (1e3 * r["ms_per_step"]), 4),
                "timed_with": how,
                "definition": "kernel-v2 (since round 2): per-kernel times come from a second, EAGER pass with an event pair "
                              "around every launch, which serialises the kernels -- no programmatic-dependent-launch overlap, "
                              "the hoisted draft tier shows as exposed time -- so shares can sum above 1; `value` and "
                              "`ms_per_step` come from the graph-replayed pass with the overlap"}
    roofline = roof(dom, kbytes.get(dom, by["a1_k"]))
    fused_gbs = by["fused_must_read"] / us_layer / 1e3

    line = {
        "metric": METRIC, "value": round(us_layer, 3), "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(r["ms_per_step"], 4), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": workload_config(cfg, dist.world),
        "run": run_info(w.n_sets, dist.world, rank_table(dist, device)),
        "aggregate": aggregate(us_layer, cfg, dist.world),
        "clocks": r["clocks"],
        "e2e": {"value": round(1e3 * e2e_ms / L, 3), "unit": UNIT, "h2d_bytes_per_step": e2e.h2d,
                "d2h_bytes_per_step": e2e.d2h, "ms_per_step": round(e2e_ms, 4),
                "definition": "e2e-v2 (since round 2): S_Draft is device-resident state and is no longer copied H2D per "
                              "layer; round-1 lines (e2e-v1) copied it and are not comparable",
                "what": "Q/K_new/V_new of every layer copied from pinned host memory, outputs of every layer + last "
                        "index lists copied back, copy streams overlapped with the kernels; KV cache, history and draft "
                        "scores (what dustin_draft_aggregate leaves on the device) are device-resident state"},
        "gpu_launches": int(r["launches_per_step"] * args.steps),
        "roofline": roofline,
        "roofline_attn": roof("attn_kernel", by["a4"], r["attn_only_us_per_launch"],
                              "CUDA events around graph replays that hold only this kernel (L launches, one per "
                              "layer, each on its own K/V cache and index lists; cnt = NULL: one budget <= N for all "
                              "sequences, so every list holds k entries -- the fact the fused call derives from its select "
                              "parameters); time / launches"),
        "gather_probe": {"us_per_launch": round(r["gather_probe_us_per_launch"], 3),
                         "gbs": round(by["a4"] / r["gather_probe_us_per_launch"] / 1e3, 1),
                         "attn_time_over_probe": round(r["attn_only_us_per_launch"] / r["gather_probe_us_per_launch"], 3),
                         "what": "dustin_probe_gather: plain 16-byte loads of exactly the K/V rows a4 gathers (same lists, "
                                 "same caches, graph-replayed), no arithmetic -- the practical floor of the 256-byte row "
                                 "gather on this memory system"},
        "fused_path": {"bytes_it_must_read_per_layer": by["fused_must_read"], "achieved_gbs": round(fused_gbs, 1),
                       "frac_of_measured_peak": round(fused_gbs / peak, 4),
                       "frac_of_8000_nominal": round(fused_gbs / 8000.0, 4)},
        "stages_us_per_layer": stage_table(kern, L),
        "dense_us_per_layer": round(r["dense_us_per_layer"], 3),
        "speedup_vs_dense": round(r["dense_us_per_layer"] / us_layer, 3),
        "score_once": {"us_per_layer": round(r["score_once_us_per_layer"], 3),
                       "speedup_vs_dense": round(r["dense_us_per_layer"] / r["score_once_us_per_layer"], 3),
                       "what": "paper schedule: a1-a3 in one layer, a4 in all layers with that index set"},
        "dense_roofline": None,
        "paper_context": "PAPER.md:570 27.85x self-attention, :319 9.17x end-to-end at 32k/B=16 on Qwen2.5-72B, "
                         "4x H200, k=512 -- other hardware and budget, context only",
    }
    if "dense_kernels" in r and "attn_kernel" in r["dense_kernels"]:
        us = r["dense_kernels"]["attn_kernel"][0]
        line["dense_roofline"] = {"kernel": "attn_kernel (idx=NULL)", "achieved": round(by["a5"] / us / 1e3, 1),
                                  "peak": peak, "unit": "GB/s", "frac": round(by["a5"] / us / 1e3 / peak, 4)}

    if dist.rank == 0 and args.gpus == 1 and not args.no_extras:
        s0 = w.sets[0]
        inp_cpu = synth.LayerInputs(cfg=cfg, q=w.q[0].cpu(), k_new=w.k_new[0].cpu(), v_new=w.v_new[0].cpu(),
                                    k=s0.k.cpu(), v=s0.v.cpu(), s_draft=w.s_draft[0].cpu(), hist=w.hist[0].cpu(),
                                    k_max=w.k_max)
        line["cpu_baseline"] = cpu_baseline(cfg, inp_cpu)
        del inp_cpu
    elif dist.rank == 0:
        line["cpu_baseline"] = None

    if not args.no_extras and args.gpus == 1:
        del e2e, w
        torch.cuda.empty_cache()
        extras = {}
        other = ("qwen2.5-72b spread subset, G=Hkv (one subset head and one list per KV head)" if args.packed else
                 "qwen2.5-72b packed subset, G=1 (paper's global list)")   # the placement the headline did NOT run
        for name, c in ((other, synth.config_qwen72b(args.batch, args.ctx, args.layers, spread=args.packed)),
                        ("llama3-8b spread subset, G=Hkv (BASELINE.json configs[1])",
                         synth.config_llama8b(args.batch, args.ctx, 32, spread=True))):
            w2, r2 = measure_workload(api, c, 8, max(3, args.steps // 2), args.warmup, dist, device, True, True)
            b2 = w2.bytes_per_layer()
            extras[name] = {
                "us_per_layer": round(r2["us_per_layer"], 3), "dense_us_per_layer": round(r2["dense_us_per_layer"], 3),
                "speedup_vs_dense": round(r2["dense_us_per_layer"] / r2["us_per_layer"], 3),
                "score_once_us_per_layer": round(r2["score_once_us_per_layer"], 3),
                "stages_us_per_layer": stage_table(r2["kernels"], c.n_layers),
                "fused_must_read_gbs": round(b2["fused_must_read"] / r2["us_per_layer"] / 1e3, 1),
                "fused_frac_of_measured_peak": round(b2["fused_must_read"] / r2["us_per_layer"] / 1e3 / peak, 4),
                "attn_kernel_gbs": round(b2["a4"] / r2["attn_only_us_per_launch"] / 1e3, 1),
                "attn_only_us_per_launch": round(r2["attn_only_us_per_launch"], 3),
                "score_logits_kernel_gbs": round(b2["a1_k"] / r2["kernels"]["score_logits_kernel"][0] / 1e3, 1),
            }
            del w2
            torch.cuda.empty_cache()
        # BASELINE.json configs[3] (the two ends of the context sweep, gamma 8 once, the Naive all-head estimator at 4k
        # and 32k) and configs[4] (paged, ragged): 8 layers over 4 distinct caches each, graph-replayed per leg.
        # The full grid is `bench.py --sweep` (profiles/r02_sweep.json).
        pts = []
        for tag, c, naive in (
                ({"point": "configs[3] 4k, B=16, gamma 4, k=2048"}, synth.config_qwen72b(16, 4096, 8), True),
                ({"point": "configs[3] 32k, B=16, gamma 8, k=2048"}, synth.config_qwen72b(16, 32768, 8, gamma=8), False),
                ({"point": "configs[3] 32k, B=16, gamma 4, k=2048 (+ all-head scoring)"}, synth.config_qwen72b(16, 32768, 8), True),
                ({"point": "paper budget 32k, B=16, gamma 4, k=512 (S=4, W=16; PAPER.md:443, :570 quotes 27.85x attention speed-up on 4x H200)"},
                 synth.shrink(synth.config_qwen72b(16, 32768, 8, budget=512), n_sink=4, n_recent=16), False),
                ({"point": "configs[3] 128k, B=4, gamma 4, k=2048"}, synth.config_qwen72b(4, 131072, 8), False),
                ({"point": "configs[3] 128k, B=4, gamma 4, k=8192 (6.25 %)"}, synth.config_qwen72b(4, 131072, 8, budget=8192), False)):
            pts.append(sweep_point(api, c, 4, dist, device, peak, tag, naive=naive))
            torch.cuda.empty_cache()
        pts.append(sweep_point(api, synth.config_paged(n_layers=4), 2, dist, device, peak,
                               {"point": "configs[4] paged (page 16) ragged U[8k,64k], B=32, Llama-3-8B-shaped, k_b = 6.25 % of N_b"}))
        torch.cuda.empty_cache()
        extras["sweep_points"] = pts
        line["other_workloads"] = extras

    if dist.rank == 0:
        print(json.dumps(line), flush=True)
    dist.finish()


if __name__ == "__main__":
    main()
