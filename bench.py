#!/usr/bin/env python
"""bench.py - the Kamera hot path on BASELINE.json configs[1] (GQA Qwen2-VL-7B-like, bf16), one JSON line.

    python bench.py --gpus N --steps K --warmup W [--impl reference]

A STEP is one pass of the whole hot path over one batch of synthetic input:
  phase A  kam_relocate_patch_batch : 8 chunks x 1024 tokens x 28 layers relocated to p ~ U[0, 32768) with their rank-16
                                      patches into one request's pages, ONE launch           (A1-A5)   <- the headline metric
  phase B  kam_slide                : the request's window slides: oldest chunk out (its 7 survivors re-rotate in place by
                                      -1024), one evicted chunk recalled by relocate+patch, ONE launch (A6, A7)
  phase C  kam_window_plan + 28 x kam_window_decode : fused paged decode over every request's 8192-token window, all
                                      layers, LSE merge (A8, A9).  The 28 per-layer calls (2 kernels each) are captured once
                                      into a CUDA graph and replayed; the plan is rebuilt eagerly every step (the window slid)
Inputs are resident in HBM before the timed region; every step touches > 1 GB of fresh source and destination memory
(the B200 L2 is 126 MB), and the request / canonical set rotate from step to step.

metric = relocate+patch GB/s: ALGORITHMIC bytes of phase A (page read + page write + U + W + block table)
divided by the device time of phase A.  The other two headline figures (us per 1024-token chunk, decode tokens/s) and all
three kernels' roofline fractions ride along in the same line.  N > 1: requests are sharded over ranks (rank_requests),
no data-path collective (the path partitions by request), time = max over ranks, value = all ranks'
bytes / that.  The rank-aware part (timed loop, reductions, the rank-0 line) is `run()`; tests/test_multirank.py drives it
with a stub workload over gloo.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CFG_ID = 2
N_REQ = 32              # requests per GPU = decode batch (configs[1] names none; 32 is configs[3]'s); each owns an 8-chunk window
N_SETS = 2              # canonical chunk sets cycled so that sources miss L2
CPU_SAMPLE_CHUNKS = 12  # cpu_baseline sample: ~10 s of oracle work on the GPU box's host


def algorithmic_bytes_relocate(T, H, D, m, P, has_v=True):
    """bytes(chunk, layer) = 2*nkv*T*H*D*2 + nkv*H*T*m*2 + nkv*H*m*D*2 + 4*T/P."""
    nkv = 2 if has_v else 1
    return 2 * nkv * T * H * D * 2 + nkv * H * T * m * 2 + nkv * H * m * D * 2 + 4 * (T // P)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: NVML polled from a thread every ~2 ms (a 60 ms region
    still yields tens of samples); `nvidia-smi -lms 20` as the fallback when the NVML binding is missing."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.idx = [], None, gpu_index
        self.t0 = self.t1 = None                      # host times bracketing the timed region: only samples inside count
        self.nvml, self.stop_flag, self.sm_max = None, False, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[self.idx]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else self.idx
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.nvml = (pynvml, h)
            self.th = threading.Thread(target=self._poll, daemon=True)
            self.th.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _poll(self):
        pynvml, h = self.nvml
        bits = {"hw_slowdown": pynvml.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": pynvml.nvmlClocksEventReasonHwThermalSlowdown,
                "sw_thermal_slowdown": pynvml.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": pynvml.nvmlClocksEventReasonSwPowerCap}
        while not self.stop_flag:
            try:
                sm = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
                rs = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                self.rows.append((time.time(), float(sm), [n for n, b in bits.items() if rs & b]))
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")] + [time.time()])

    def stop(self):
        inside = lambda t: self.t0 is None or self.t1 is None or self.t0 <= t <= self.t1 + 0.02
        if self.nvml:
            self.stop_flag = True
            self.th.join(timeout=1)
            rows = [r for r in self.rows if inside(r[0])]
            sm = [r[1] for r in rows]
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.sm_max, "reasons": sorted({n for r in rows for n in r[2]}),
                    "samples": len(sm), "how": "NVML polled every ~2 ms inside the timed region"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for r in self.rows if len(r) >= 10 and r[1].replace(".", "").isdigit() and inside(r[-1])]
        sm = [float(r[1]) for r in rows]
        mx = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in rows for n, v in zip(names, r[5:9]) if v.lower().startswith("active")})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm), "how": "nvidia-smi -lms 20"}


# ------------------------------------------------------------------------------------------------------- the workload
def tensor_peak():
    """Dense bf16 tensor peak in TFLOP/s: the sustained cuBLAS figure of MEASURED_PEAKS.json, else the profiling guide's nominal."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d.get("bf16_tflops_sustained") or d.get("bf16_tflops") or 2250.0)
    return 2250.0


class DeviceClock:
    """Phase boundaries as CUDA events on the launching stream (torch's current stream, which the binding passes on)."""

    def __init__(self, torch):
        self.torch = torch

    def mark(self):
        e = self.torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def ms(self, a, b):
        return a.elapsed_time(b)

    def sync(self):
        self.torch.cuda.synchronize()


class Workload:
    def __init__(self, device, rank, use_graph=True, world=1):
        import numpy as np
        import torch

        import paper_2606_23581_b200 as kam
        from paper_2606_23581_b200 import binding as B
        from synth import CONFIGS, randn_device
        self.torch, self.kam, self.B = torch, kam, B
        cfg = self.cfg = CONFIGS[CFG_ID]
        L, H, D, P, T, m = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.chunk_tokens, cfg.rank
        self.n_chunks = cfg.chunks_per_step
        # the job serves world * N_REQ requests; this rank owns the block rank_requests() names.  A request's content (which
        # canonical set it recalls from) follows its GLOBAL id, so the ranks do different work of the same shape.
        self.global_ids = rank_requests(rank, world)
        self.rng = np.random.Generator(np.random.PCG64(cfg.seed + 1000 * rank))
        seed = [cfg.seed * 100003 + 7919 * rank]

        def rnd(shape, std):
            seed[0] += 1
            return randn_device(shape, seed[0], std, torch.bfloat16, device)

        # canonical store: N_SETS x 8 position-free chunks + rank-16 factors, resident in HBM (K,V ~ N(0,1); U ~ N(0,1); W ~ N(0,.05))
        self.sets = []
        for _ in range(N_SETS):
            cs = []
            for _ in range(self.n_chunks):
                ch = kam.Chunk([rnd((T, H, D), 1.0) for _ in range(L)], [rnd((T, H, D), 1.0) for _ in range(L)])
                pa = kam.Patch([rnd((T, H, m), 1.0) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)],
                               [rnd((T, H, m), 1.0) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)])
                cs.append((ch, pa))
            self.sets.append(cs)
        ppc = T // P
        lay = kam.make_layout(B.KAM_GQA, L, cfg.n_q_heads, H, D, cfg.rope_off, cfg.rope_dim, True, P, cfg.theta)
        # pool A: target of the stateless batched operator (phase A); block table = random permutation of its pages
        npa = N_REQ * self.n_chunks * ppc
        self.pool_a = kam.Pool([torch.zeros((npa, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)],
                               [torch.zeros((npa, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)])
        self.ctx_a = kam.Context(lay, self.pool_a)
        self.bt_a = torch.from_numpy(self.rng.permutation(npa).astype(np.int32)).to(device)
        # pool B: the window store (phases B, C): N_REQ windows of 8 chunks (+1 chunk of slack while sliding)
        npb = N_REQ * (self.n_chunks + 1) * ppc
        self.pool_b = kam.Pool([torch.zeros((npb, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)],
                               [torch.zeros((npb, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)])
        self.ctx_b = kam.Context(lay, self.pool_b, max_requests=N_REQ, max_chunks_per_request=self.n_chunks + 1,
                                 max_pages_per_chunk=ppc)
        for r in range(N_REQ):
            self.ctx_b.kam_window_open(r, 0)
            for c in range(self.n_chunks):
                ch, pa = self.sets[self.global_ids[r] % N_SETS][c]
                self.ctx_b.kam_admit(r, B.KAM_BACK, ch, pa, m, 1)
        self.q = rnd((N_REQ, cfg.n_q_heads, D), 1.0)
        self.out = torch.zeros((N_REQ, cfg.n_q_heads, D), dtype=torch.bfloat16, device=device)
        self.lse = torch.zeros((N_REQ, cfg.n_q_heads), dtype=torch.float32, device=device)
        self.sm_scale = D ** -0.5
        self.req_ids = list(range(N_REQ))
        # algorithmic bytes
        self.bytes_a = self.n_chunks * L * algorithmic_bytes_relocate(T, H, D, m, P)
        self.bytes_b = (self.n_chunks - 1) * L * (2 * T * H * D * 2) + L * algorithmic_bytes_relocate(T, H, D, m, P)
        self.bytes_c_layer = N_REQ * 2 * self.n_chunks * T * H * D * 2
        self.bytes_c = L * self.bytes_c_layer
        torch.cuda.synchronize()
        # phase C as a CUDA graph: with a valid plan kam_window_decode launches exactly two kernels and nothing else
        self.graph, self.graph_replays, self.launches_per_replay = None, 0, 0
        if use_graph:
            self.ctx_b.kam_window_plan(self.req_ids)
            k0 = self.ctx_b.kam_get_stats()["kernels_launched"]
            self.decode_layers()                                   # eager once: workspace sized, kernels loaded
            self.launches_per_replay = self.ctx_b.kam_get_stats()["kernels_launched"] - k0     # what one graph replay launches
            torch.cuda.synchronize()
            self.graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(self.graph):
                self.decode_layers()
            torch.cuda.synchronize()

    def decode_layers(self):
        for l in range(self.cfg.n_layers):
            self.ctx_b.kam_window_decode(self.q, self.req_ids, l, self.sm_scale, self.out, self.lse)

    def launches(self):
        """Kernels launched so far: the contexts' own counters + what every graph replay launches (counted on the eager pass)."""
        return (self.ctx_a.kam_get_stats()["kernels_launched"] + self.ctx_b.kam_get_stats()["kernels_launched"]
                + self.graph_replays * self.launches_per_replay)

    def step(self, i, mark=None):
        """One pass of the hot path.  mark(k): phase boundary k (0 .. 3), recorded by the caller's clock."""
        cfg, B, T, m = self.cfg, self.B, self.cfg.chunk_tokens, self.cfg.rank
        r, cs = i % N_REQ, self.sets[(i + self.global_ids[0]) % N_SETS]
        rec = mark if mark is not None else (lambda k: None)
        rec(0)
        # phase A: 8 chunks relocated+patched to random offsets, one launch
        p = self.rng.integers(0, cfg.max_pos, size=self.n_chunks)
        base = r * self.n_chunks * T
        self.ctx_a.kam_relocate_patch_batch([(self.bt_a, base + c * T, cs[c][0], int(p[c]), cs[c][1], m) for c in range(self.n_chunks)])
        rec(1)
        # phase B: the window of request r slides by one chunk
        ch, pa = cs[i % self.n_chunks]
        self.ctx_b.kam_slide(r, B.KAM_FRONT, B.KAM_BACK, ch, pa, m, 1)
        rec(2)
        # phase C: every request decodes one token over its window, all layers
        self.ctx_b.kam_window_plan(self.req_ids)
        if self.graph is not None:
            self.graph.replay()
            self.graph_replays += 1
        else:
            self.decode_layers()
        rec(3)


class E2E:
    """The same path through the C-ABI entries that take HOST buffers: canonical chunks and factors live in pinned host
    memory (an off-device canonical store), H2D inside kam_relocate_patch_host; the decode query comes from the host
    and out / lse go back to it inside kam_paged_decode_merge_host.  Pipelined (the library's default): the copy of chunk
    c + 1 runs on the library's copy stream under the kernel of chunk c, the 28 decode calls share one pinned plan and the
    step ends with ONE synchronise, after which the host reads out / lse.  Serial (options host_copy_overlap = 0,
    host_entries_sync = 1): round 1's behaviour, every decode call synchronises."""

    def __init__(self, wl, device):
        torch = wl.torch
        cfg = wl.cfg
        L, T = cfg.n_layers, cfg.chunk_tokens
        self.wl = wl

        def slab(ch, pa):
            """One pinned host slab per chunk, per layer K | V | U_k | W_k | U_v | W_v (how an off-device canonical store would keep
            a chunk); the per-layer tensors handed to the library are views into it."""
            parts = [ch.k_layers, ch.v_layers, pa.t[0], pa.t[1], pa.t[2], pa.t[3]]
            n = sum(t.numel() for grp in parts for t in grp)
            buf = torch.empty(n, dtype=torch.bfloat16).pin_memory()
            views, off = [[] for _ in parts], 0
            for l in range(L):
                for k, grp in enumerate(parts):
                    t = grp[l]
                    v = buf[off:off + t.numel()].view(t.shape)
                    v.copy_(t)
                    views[k].append(v)
                    off += t.numel()
            return tuple(views) + (buf,)
        self.chunks = [slab(ch, pa) for ch, pa in wl.sets[0]]
        self.h2d = sum(c[6].numel() * 2 for c in self.chunks)
        P = cfg.page_size
        n_pages = wl.n_chunks * T // P
        self.bt = wl.bt_a[:n_pages].contiguous().reshape(1, -1)
        self.starts = torch.arange(0, (wl.n_chunks + 1) * T, T, dtype=torch.int32, device=device).reshape(1, -1)
        self.nc = torch.tensor([wl.n_chunks], dtype=torch.int32, device=device)
        self.q_h = wl.q[:1].to("cpu").pin_memory()
        self.out_h = torch.zeros((L, 1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16).pin_memory()
        self.lse_h = torch.zeros((L, 1, cfg.n_q_heads), dtype=torch.float32).pin_memory()
        self.h2d += L * self.q_h.numel() * 2
        self.d2h = self.out_h.numel() * 2 + self.lse_h.numel() * 4

    def step(self, i, pipelined=True):
        wl, cfg = self.wl, self.wl.cfg
        T, m = cfg.chunk_tokens, cfg.rank
        p = wl.rng.integers(0, cfg.max_pos, size=wl.n_chunks)
        for c, (k, v, uk, wk, uv, wv, _slab) in enumerate(self.chunks):
            wl.ctx_a.kam_relocate_patch_host(self.bt.reshape(-1), c * T, T, 0, int(p[c]), k, v, uk, wk, uv, wv, m)
        if pipelined:
            wl.ctx_a.kam_paged_decode_plan(self.bt, self.starts, None, self.nc)
        for l in range(cfg.n_layers):
            wl.ctx_a.kam_paged_decode_merge_host(self.q_h, self.bt, self.starts, None, self.nc, l, wl.sm_scale, self.out_h[l], self.lse_h[l])
        wl.torch.cuda.synchronize()                  # the step's result (out, lse of every layer) is now readable on the host
        return float(self.lse_h[-1, 0, 0])


# ------------------------------------------------------------------------------------------------------- CPU oracle legs
_ORACLE_CORES = 1


def _timed_oracle(fn):
    """Runs fn() once; returns (seconds, cores it kept busy = process CPU time / wall time)."""
    global _ORACLE_CORES
    t0, c0 = time.perf_counter(), time.process_time()
    fn()
    dt = time.perf_counter() - t0
    _ORACLE_CORES = max(1, int(round((time.process_time() - c0) / dt)))
    return dt, _ORACLE_CORES


def oracle_sample(n_chunks, n_layers, seed=1):
    """Times oracle/reuse.py (as it stands) on n_chunks x n_layers (chunk, layer) units of config 2.  Returns (GB/s, seconds)."""
    import numpy as np
    import torch

    from oracle import reuse
    from synth import CONFIGS, make_chunk
    cfg = CONFIGS[CFG_ID]
    rng = np.random.Generator(np.random.PCG64(seed))
    T, H, D, P, m = cfg.chunk_tokens, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.rank
    chunks = [make_chunk(cfg, rng, n_layers=n_layers) for _ in range(n_chunks)]
    f = lambda t: t.to(torch.float64).numpy()
    pool_k = np.zeros((T // P, P, H, D), np.uint16); pool_v = np.zeros_like(pool_k)
    bt = rng.permutation(T // P).astype(np.int32)

    def work():
        for ch in chunks:
            p = int(rng.integers(0, cfg.max_pos))
            for l in range(n_layers):
                reuse.relocate_patch_layer(pool_k, pool_v, bt, 0, f(ch["K"][l]), f(ch["V"][l]), p, f(ch["Uk"][l]), f(ch["Wk"][l]),
                                           f(ch["Uv"][l]), f(ch["Wv"][l]), theta=cfg.theta, rope_off=cfg.rope_off, d_r=cfg.rope_dim)
    dt, _ = _timed_oracle(work)
    nbytes = n_chunks * n_layers * algorithmic_bytes_relocate(T, H, D, m, P)
    return nbytes / dt / 1e9, dt


def oracle_inplace_sample(n_chunks, n_layers, seed=2):
    """oracle/reuse.rotate_inplace_layer (row A6) on n_chunks x n_layers survivors of config 2's shape.  (GB/s, seconds, cores)."""
    import numpy as np

    from oracle import reuse
    from synth import CONFIGS
    cfg = CONFIGS[CFG_ID]
    rng = np.random.Generator(np.random.PCG64(seed))
    T, H, D, P = cfg.chunk_tokens, cfg.n_kv_heads, cfg.row_dim, cfg.page_size
    pools = [rng.integers(0x3c00, 0x4000, size=(T // P, P, H, D)).astype(np.uint16) for _ in range(n_layers)]     # bf16 bits in [~0.008, 2)
    bt = rng.permutation(T // P).astype(np.int32)

    def work():
        for _ in range(n_chunks):
            for l in range(n_layers):
                reuse.rotate_inplace_layer(pools[l], bt, 0, T, -T, theta=cfg.theta, rope_off=cfg.rope_off, d_r=cfg.rope_dim)
    dt, cores = _timed_oracle(work)
    return n_chunks * n_layers * (2 * T * H * D * 2) / dt / 1e9, dt, cores


def oracle_decode_sample(n_layers, seed=3):
    """oracle/attention.attend_bruteforce (rows A8 + A9 by their definition) for ONE request of config 2 (8 chunks x 1024 tokens,
    28 query heads) over n_layers layers.  (GB/s of K+V read, tokens/s for a batch of 1, seconds, cores)."""
    import numpy as np

    from oracle import attention as att
    from synth import CONFIGS
    cfg = CONFIGS[CFG_ID]
    rng = np.random.Generator(np.random.PCG64(seed))
    T, H, D, n = cfg.chunk_tokens, cfg.n_kv_heads, cfg.row_dim, cfg.chunks_per_step
    layers = [[{"k": rng.standard_normal((T, H, D)), "v": rng.standard_normal((T, H, D)), "delta": int(rng.integers(-4096, 4096))} for _ in range(n)]
              for _ in range(n_layers)]
    q = rng.standard_normal((cfg.n_q_heads, D))
    rope = dict(theta=cfg.theta, rope_off=cfg.rope_off, d_r=cfg.rope_dim)

    def work():
        for chunks in layers:
            att.attend_bruteforce(q, chunks, D ** -0.5, rope)
    dt, cores = _timed_oracle(work)
    nbytes = n_layers * n * T * H * 2 * D * 2
    return nbytes / dt / 1e9, 1.0 / (dt / n_layers * cfg.n_layers), dt, cores


def cpu_threads():
    """Cores the last oracle leg actually used: process CPU time / wall time (the numpy fp64 oracle is mostly one thread)."""
    return _ORACLE_CORES


def run_reference(args):
    """--impl reference: this tier has no reference implementation; the arm is the fp64 CPU oracle, as it stands, on the
    host cores, each step a bounded sample (1 chunk x 2 layers) of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    for i in range(args.warmup + args.steps):
        gbs, dt = oracle_sample(1, 2, seed=i)
        if i >= args.warmup:
            vals.append((gbs, dt))
    tot_t = sum(d for _, d in vals)
    value = sum(g * d for g, d in vals) / tot_t
    sample = "1 chunk x 2 layers of config 2 per step (of 8 chunks x 28 layers)"
    print(json.dumps({
        "impl": "reference", "metric": "relocate+patch GB/s", "value": value, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, len(vals)), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": "BASELINE.json configs[1] GQA Qwen2-VL-7B-like", "sample": sample},
        "cpu_baseline": {"value": value, "unit": "GB/s", "cores": cpu_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------------- extras (outside the step)
def _time_ms(torch, fn, reps):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fn(); torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record(); torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def extras(wl, device, peak):
    """Measured after the timed region, NOT part of the step or of `value`.  Every figure is algorithmic bytes / device time
    (CUDA events around back-to-back launches) as a fraction of the measured HBM peak:
      * the paper's "rank-invariant in latency" claim as a rank sweep m in {0, 4, 16, 32, 48, 64} of the relocate kernel
        on config 2's shape, and kam_rotate_inplace alone (row A6);
      * relocate+patch on the shapes of configs 4 (MHA-32, m = 16, T = 1280) and 5 (GQA-8, m = 32, T = 2048), every launch
        reading sources no other launch of the loop reads (no L2 reuse), and config 3's stated launch of 96 relocations;
      * the stateless decode call (plan + decode + merge per call; with the plan pinned once for all layers; with the rank-16
        patch applied ON READ, row A8's second form) and the decode on the shapes of configs 4 and 5;
      * the MLA instantiation (config 3's shape): relocate+patch, absorbed decode without and with the on-read patch."""
    import torch
    kam, B, cfg = wl.kam, wl.B, wl.cfg
    from synth import CONFIGS, randn_device
    L, H, D, P, T, n = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.chunk_tokens, wl.n_chunks
    out, seed = {}, [987654]

    def rnd(shape, std=1.0):
        seed[0] += 1
        return randn_device(shape, seed[0], std, torch.bfloat16, device)

    def entry(nbytes, ms, **kw):
        d = {"ms": ms, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak}
        d.update(kw)
        return d

    # ---- T11: rank sweep, one launch of 8 chunks x 28 layers per rank; sources/destinations rotate over the request slots
    sweep = {}
    for m in (0, 4, 16, 32, 48, 64):
        pats = None
        if m:
            pats = [kam.Patch([rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)],
                              [rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)]) for _ in range(n)]
        it = [0]

        def launch():
            r, cs = it[0] % N_REQ, wl.sets[it[0] % N_SETS]
            it[0] += 1
            wl.ctx_a.kam_relocate_patch_batch([(wl.bt_a, (r * n + c) * T, cs[c][0], 1000 + 37 * c + it[0], pats[c] if pats else None, m) for c in range(n)])
        g0 = wl.ctx_a.kam_get_stats()["generic_launches"]
        ms = _time_ms(torch, launch, 10)
        nbytes = n * L * algorithmic_bytes_relocate(T, H, D, m, P) if m else n * L * (2 * 2 * T * H * D * 2 + 4 * (T // P))
        sweep["m=%d" % m] = entry(nbytes, ms, us_per_1024tok_chunk=1e3 * ms / n, tiled_kernel=wl.ctx_a.kam_get_stats()["generic_launches"] == g0)
        del pats
    out["relocate_rank_sweep"] = sweep

    # ---- row A6 alone: kam_rotate_inplace over one request's 8 chunks (8192 tokens x 28 layers, K only), rotating requests
    it = [0]

    def launch():
        r = it[0] % N_REQ
        it[0] += 1
        wl.ctx_a.kam_rotate_inplace(wl.bt_a, r * n * T, n * T, -T)
    ms = _time_ms(torch, launch, 10)
    out["rotate_inplace_alone"] = entry(n * L * 2 * T * H * D * 2, ms, bytes="K rows read + written, V untouched")

    # ---- relocate+patch on the shapes of configs 4 and 5: a few resident layers, distinct sources and destinations per launch
    for name, cid, Lx, n_src, per_launch in (("relocate_config4_shape_mha32_m16_T1280", 4, 4, 16, 4), ("relocate_config5_shape_gqa8_m32_T2048", 5, 4, 32, 8)):
        cx = CONFIGS[cid]
        Hx, Dx, Px, Tx, mx = cx.n_kv_heads, cx.row_dim, cx.page_size, cx.chunk_tokens, cx.rank
        srcs = [(kam.Chunk([rnd((Tx, Hx, Dx)) for _ in range(Lx)], [rnd((Tx, Hx, Dx)) for _ in range(Lx)]),
                 kam.Patch([rnd((Tx, Hx, mx)) for _ in range(Lx)], [rnd((Hx, mx, Dx), cx.w_std) for _ in range(Lx)],
                           [rnd((Tx, Hx, mx)) for _ in range(Lx)], [rnd((Hx, mx, Dx), cx.w_std) for _ in range(Lx)])) for _ in range(n_src)]
        npx = n_src * Tx // Px
        poolx = kam.Pool([torch.zeros((npx, Px, Hx, Dx), dtype=torch.bfloat16, device=device) for _ in range(Lx)],
                         [torch.zeros((npx, Px, Hx, Dx), dtype=torch.bfloat16, device=device) for _ in range(Lx)])
        ctxx = kam.Context(kam.make_layout(B.KAM_MHA if cx.n_q_heads == Hx else B.KAM_GQA, Lx, cx.n_q_heads, Hx, Dx, 0, Dx, True, Px, cx.theta), poolx)
        btx = torch.randperm(npx, device=device, dtype=torch.int32)
        it = [0]

        def launch():
            i0 = (it[0] * per_launch) % n_src
            it[0] += 1
            ctxx.kam_relocate_patch_batch([(btx, (i0 + c) * Tx, srcs[i0 + c][0], 777 + 1000 * c + it[0], srcs[i0 + c][1], mx) for c in range(per_launch)])
        reps = 3 * (n_src // per_launch)                     # three passes over the sources: 2 GB of them, so no launch finds its rows in L2
        ms = _time_ms(torch, launch, reps)
        nbytes = per_launch * Lx * algorithmic_bytes_relocate(Tx, Hx, Dx, mx, Px)
        out[name] = entry(nbytes, ms, us_per_1024tok_chunk=1e3 * ms / per_launch * 1024 / Tx * cx.n_layers / Lx, layers_resident=Lx,
                          chunks_per_launch=per_launch, note="us per 1024 tokens scaled to the config's %d layers; the launches cycle through %d distinct source chunks (%.1f GB), so no launch finds its rows in L2" % (cx.n_layers, n_src, n_src * Lx * 2 * Tx * Hx * Dx * 2 / 1e9),
                          tiled_kernel=ctxx.kam_get_stats()["generic_launches"] == 0)
        ctxx.close()
        del srcs, poolx, ctxx, btx

    # ---- A8: the stateless decode call on config 2's shape: per-call plan | plan pinned once | rank-16 patch on read
    Ld = 4
    ppr = n * T // P
    npages = N_REQ * ppr
    bt = torch.randperm(npages, device=device, dtype=torch.int32).reshape(N_REQ, ppr)
    starts = torch.arange(0, (n + 1) * T, T, dtype=torch.int32, device=device).repeat(N_REQ, 1)
    offs = torch.full((N_REQ, n), 4321, dtype=torch.int64, device=device)
    nc = torch.full((N_REQ,), n, dtype=torch.int32, device=device)
    m = cfg.rank
    wl.ctx_a.kam_decode_set_max_patch_rank(16)
    refs = [B.patch_refs([[(rnd((T, H, m)), rnd((H, m, D), cfg.w_std), rnd((T, H, m)), rnd((H, m, D), cfg.w_std), m) for _ in range(n)]
                          for _ in range(N_REQ)], device) for _ in range(Ld)]
    for name, pr, pin in (("decode_stateless_no_patch", None, False), ("decode_stateless_pinned_plan", None, True),
                          ("decode_stateless_on_read_patch_m16", refs, False), ("decode_stateless_on_read_patch_m16_pinned_plan", refs, True)):
        it = [0]
        wl.ctx_a.kam_paged_decode_plan(bt if pin else None, starts, offs, nc, has_patches=pr is not None)

        def launch():
            l = it[0] % Ld
            it[0] += 1
            wl.ctx_a.kam_paged_decode_merge(wl.q, bt, starts, offs, nc, l, wl.sm_scale, wl.out, wl.lse, patches=pr[l] if pr else None)
        ms = _time_ms(torch, launch, 12)
        nbytes = N_REQ * n * T * H * (2 * D + (2 * m if pr else 0)) * 2
        out[name] = entry(nbytes, ms, bytes="K + V" + (" + U_k + U_v" if pr else "") + " once; on-read rotation by a pending offset in both",
                          what="kam_paged_decode_plan once, then decode + merge per layer" if pin else "plan + decode + merge per call")
    wl.ctx_a.kam_paged_decode_plan(None, None, None, None)
    del refs

    # ---- the decode kernel on the other configs' shapes (stateless call, no patch, two resident layers): a layer of config 2 is
    # 0.54 GB, so plan / ramp / merge weigh ~15 %; configs 4 and 5 read 2.3 and 4.3 GB per layer
    for name, cid, nreq, nch, Tc in (("decode_config4_shape_b32_4352tok", 4, 32, 4, 1088), ("decode_config5_shape_b64_16384tok", 5, 64, 8, 2048)):
        cx = CONFIGS[cid]
        Hx, Dx, Px, Lx = cx.n_kv_heads, cx.row_dim, cx.page_size, 2
        pprx = nch * Tc // Px
        poolx = kam.Pool([rnd((nreq * pprx, Px, Hx, Dx)) for _ in range(Lx)], [rnd((nreq * pprx, Px, Hx, Dx)) for _ in range(Lx)])
        ctxx = kam.Context(kam.make_layout(B.KAM_MHA if cx.n_q_heads == Hx else B.KAM_GQA, Lx, cx.n_q_heads, Hx, Dx, 0, Dx, True, Px, cx.theta), poolx)
        btx = torch.randperm(nreq * pprx, device=device, dtype=torch.int32).reshape(nreq, pprx)
        stx = torch.arange(0, (nch + 1) * Tc, Tc, dtype=torch.int32, device=device).repeat(nreq, 1)
        ncx = torch.full((nreq,), nch, dtype=torch.int32, device=device)
        qx = rnd((nreq, cx.n_q_heads, Dx))
        ox, lx = torch.zeros_like(qx), torch.zeros((nreq, cx.n_q_heads), dtype=torch.float32, device=device)
        it = [0]

        def launch():
            it[0] += 1
            ctxx.kam_paged_decode_merge(qx, btx, stx, None, ncx, it[0] % Lx, Dx ** -0.5, ox, lx)
        ms = _time_ms(torch, launch, 6)
        nbytes = nreq * nch * Tc * Hx * 2 * Dx * 2
        out[name] = entry(nbytes, ms, bytes="K + V once", what="stateless call = plan + kam_paged_decode_kernel + merge; %d q / %d kv heads" % (cx.n_q_heads, Hx))
        ctxx.close()
        del poolx, ctxx, btx, qx, ox

    # ---- f4: chunked prefill - a 512-token text turn of 8 requests over their 8192-token recalled windows (config 2's shape,
    # the TTFT path of P:105 / P:349), causal over the appended tokens, recalled chunks read at a pending offset
    nbp, Tq = 8, 512
    Lp = 2
    pprp = (n * T + Tq) // P
    poolp = kam.Pool([rnd((nbp * pprp, P, H, D)) for _ in range(Lp)], [rnd((nbp * pprp, P, H, D)) for _ in range(Lp)])
    ctxp = kam.Context(kam.make_layout(B.KAM_GQA, Lp, cfg.n_q_heads, H, D, 0, D, True, P, cfg.theta), poolp)
    btp = torch.randperm(nbp * pprp, device=device, dtype=torch.int32).reshape(nbp, pprp)
    stp = torch.tensor([[c * T for c in range(n + 1)] + [n * T + Tq]] * nbp, dtype=torch.int32, device=device)
    ofp = torch.tensor([[4321] * n + [0]] * nbp, dtype=torch.int64, device=device)
    ncp = torch.full((nbp,), n + 1, dtype=torch.int32, device=device)
    qp = rnd((nbp, Tq, cfg.n_q_heads, D))
    op, lp = torch.zeros_like(qp), torch.zeros((nbp, Tq, cfg.n_q_heads), dtype=torch.float32, device=device)
    it = [0]

    def launch():
        it[0] += 1
        ctxp.kam_paged_prefill_merge(qp, btp, stp, ofp, ncp, it[0] % Lp, 1, wl.sm_scale, op, lp)
    ms = _time_ms(torch, launch, 6)
    ctxp.kam_set_option("prefill_tcgen05", 0)
    ms_legacy = _time_ms(torch, launch, 4)
    ctxp.kam_set_option("prefill_tcgen05", 1)
    Nkv = n * T + Tq
    flops = 4.0 * nbp * cfg.n_q_heads * D * (Tq * (Nkv - Tq) + Tq * (Tq + 1) / 2)          # visible (row, token) pairs x 4 D
    flops_issued = flops * 2 * (n * T) / Nkv + flops * Tq / Nkv                               # rotated chunks run the q~ lo products too
    tf_peak = tensor_peak()
    out["prefill_config2_shape_b8_512rows_over_8192"] = {
        "ms": ms, "tflops": flops / ms / 1e9, "frac_of_dense_bf16_peak": flops / ms / 1e9 / tf_peak, "tflops_issued": flops_issued / ms / 1e9,
        "tensor_peak_tflops": tf_peak, "GB/s": nbp * Nkv * H * 2 * D * 2 / ms / 1e6, "frac_of_hbm_peak": nbp * Nkv * H * 2 * D * 2 / ms / 1e6 / peak,
        "bound": "tensor", "mma_sync_kernel": {"ms": ms_legacy, "tflops": flops / ms_legacy / 1e9, "what": "option prefill_tcgen05 = 0: kam_paged_prefill_kernel<128>, FlashAttention-2 shape on mma.sync"},
        "what": "kam_paged_prefill_tc_kernel<128> (tcgen05.mma M128 N64/128 K16, S and O in tensor memory); flops = 4 D per visible (row, token) "
        "pair; tflops_issued counts the second (lo) QK^T product of chunks read at a pending offset; bytes = K + V once per request"}
    ctxp.close()
    del poolp, ctxp, btp, qp, op

    # ---- MLA (config 3 shape): relocate+patch - 4 chunks x 27 layers, and config 3's stated launch (every ordering of the 4
    # cached chunks = 96 relocations, one launch); absorbed decode, batch 64 x 8192 tokens, without and with the on-read patch
    c3 = CONFIGS[3]
    L3, D3, P3, T3, m3 = c3.n_layers, c3.row_dim, c3.page_size, c3.chunk_tokens, c3.rank
    lay3 = kam.make_layout(B.KAM_MLA, L3, c3.n_q_heads, 1, D3, c3.rope_off, c3.rope_dim, False, P3, c3.theta, v_dim=c3.v_dim)
    nb3, nch3 = 64, 8
    np3 = nb3 * nch3 * T3 // P3
    pool3 = kam.Pool([rnd((np3, P3, 1, D3)) for _ in range(L3)], None)
    ctx3 = kam.Context(lay3, pool3)
    ch3 = [(kam.Chunk([rnd((T3, 1, D3)) for _ in range(L3)], None), kam.Patch([rnd((T3, 1, m3)) for _ in range(L3)], [rnd((1, m3, D3), c3.w_std) for _ in range(L3)]))
           for _ in range(8)]
    bt3 = torch.randperm(np3, device=device, dtype=torch.int32)
    it = [0]

    def launch():
        i = it[0]
        it[0] += 1
        ctx3.kam_relocate_patch_batch([(bt3, ((4 * i + c) % (nb3 * nch3)) * T3, ch3[(4 * i + c) % 8][0], 1024 * c, ch3[(4 * i + c) % 8][1], m3) for c in range(4)])
    ms = _time_ms(torch, launch, 10)
    out["mla_relocate_patch"] = entry(4 * L3 * algorithmic_bytes_relocate(T3, 1, D3, m3, P3, has_v=False), ms, us_per_1024tok_chunk=1e3 * ms / 4)
    import itertools
    perms = list(itertools.permutations(range(4)))
    it = [0]

    def launch():
        base = (it[0] % 5) * 96
        it[0] += 1
        ctx3.kam_relocate_patch_batch([(bt3, (base + 4 * pi + slot) * T3, ch3[c][0], 1024 * slot, ch3[c][1], m3)
                                       for pi, perm in enumerate(perms) for slot, c in enumerate(perm)])
    ms = _time_ms(torch, launch, 5)
    out["mla_config3_96_relocations_one_launch"] = entry(96 * L3 * algorithmic_bytes_relocate(T3, 1, D3, m3, P3, has_v=False), ms, us_per_1024tok_chunk=1e3 * ms / 96,
                                                         note="BASELINE.json configs[2] as stated: 4 cached chunks in all 24 orders; each source is read 24 times per launch, "
                                                              "so most source reads hit L2 - an algorithmic rate, the DRAM traffic is the 3.1 GB of page writes")
    q3 = rnd((nb3, c3.n_q_heads, D3))
    o3 = torch.zeros((nb3, c3.n_q_heads, c3.v_dim), dtype=torch.bfloat16, device=device)
    l3 = torch.zeros((nb3, c3.n_q_heads), dtype=torch.float32, device=device)
    st3 = torch.arange(0, (nch3 + 1) * T3, T3, dtype=torch.int32, device=device).repeat(nb3, 1)
    nc3 = torch.full((nb3,), nch3, dtype=torch.int32, device=device)
    bt3b = bt3.reshape(nb3, -1)
    ctx3.kam_decode_set_max_patch_rank(16)
    Lr = 2
    refs3 = [B.patch_refs([[(rnd((T3, 1, m3)), rnd((1, m3, D3), c3.w_std), None, None, m3) for _ in range(nch3)] for _ in range(nb3)], device) for _ in range(Lr)]
    # (the two per-call-plan entries first: profiles/ncu_extras_r02.md counts launches of this kernel from the start of the extras)
    for name, pr, pin in (("mla_decode_absorbed", None, False), ("mla_decode_on_read_patch_m16", refs3, False),
                          ("mla_decode_absorbed_pinned_plan", None, True), ("mla_decode_on_read_patch_m16_pinned_plan", refs3, True)):
        it = [0]
        ctx3.kam_paged_decode_plan(bt3b if pin else None, st3, None, nc3, has_patches=pr is not None)

        def launch():
            l = it[0] % L3
            it[0] += 1
            ctx3.kam_paged_decode_merge(q3, bt3b, st3, None, nc3, l, 192 ** -0.5, o3, l3, patches=pr[l % Lr] if pr else None)
        ms = _time_ms(torch, launch, 27)
        nbytes = nb3 * nch3 * T3 * (D3 + (m3 if pr else 0)) * 2
        out[name] = entry(nbytes, ms, bytes="every latent+rope row once (it is both key and value)" + (" + its U row" if pr else ""), batch=nb3, tokens=nch3 * T3,
                          what=("kam_paged_decode_plan once, then " if pin else "stateless call = plan + ") + "kam_mla_ts_decode_kernel (token-split) + merge",
                          tflops=nb3 * nch3 * T3 * c3.n_q_heads * (D3 + c3.v_dim) * 2 / ms / 1e9)
    ctx3.kam_paged_decode_plan(None, None, None, None)
    ctx3.close()
    del pool3, ctx3, ch3, refs3, q3, o3
    return out


_PROFILE_LEGS = False            # --profile-legs: one representative call of every as-stated phase runs between cudaProfilerStart / Stop


def _prof(torch, fn):
    if _PROFILE_LEGS:
        torch.cuda.synchronize(); torch.cuda.profiler.start()
        fn()
        torch.cuda.synchronize(); torch.cuda.profiler.stop()


def as_stated_legs(wl, device, peak):
    """After the extras: kam_form_patch timed (f3), and BASELINE.json configs[3] / configs[4] at their stated sizes (not reduced
    shapes).  Each leg frees what it allocated; a leg that cannot run (memory) says so instead of taking the line down."""
    import torch
    from synth import randn_device
    out, seed = {}, [192837]

    def rnd(shape, std=1.0):
        seed[0] += 1
        return randn_device(shape, seed[0], std, torch.bfloat16, device)
    for name, leg in (("form_patch_config2_chunk_m16", lambda: _form_patch_leg(wl, device, rnd)),
                      ("config5_as_stated", lambda: _config5_leg(wl, device, peak, rnd)),
                      ("config4_as_stated", lambda: _config4_leg(wl, device, peak, rnd))):
        torch.cuda.synchronize(); torch.cuda.empty_cache()
        try:
            out[name] = leg()
        except Exception as e:
            out[name] = {"error": repr(e)[:300]}
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    out["note_on_frac"] = ("frac = algorithmic bytes / device time / MEASURED_PEAKS.json hbm_gbs, which is a COPY rate (read + write); a stream that mostly "
                           "reads (decode) or runs for milliseconds (no ramp, no tail) can exceed it: ncu's dram__throughput %% in profiles/ncu_legs_r03.md "
                           "is the figure to hold against the hardware")
    return out


def _time_queued_ms(torch, fn, reps, sleep_cycles=120_000_000):
    """Device time of `reps` calls of fn whose HOST side (marshalling a few hundred descriptors in Python) is slower than their
    kernels: the calls are enqueued while the GPU sits in a sleep kernel, so the events bracket back-to-back device work."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fn(); torch.cuda.synchronize()
    torch.cuda._sleep(sleep_cycles)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record(); torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def _form_patch_leg(wl, device, rnd):
    import torch
    cfg = wl.cfg
    L, H, D, T, m = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.chunk_tokens, cfg.rank
    solo = [rnd((T, H, D)) for _ in range(L)]
    # conditioned rows = rotated solo rows + an exactly rank-m perturbation would need the oracle; for TIMING any rows do
    cond = [rnd((T, H, D)) for _ in range(L)]
    ms = _time_ms(torch, lambda: wl.ctx_a.kam_form_patch(cond, solo, 4096, 1, m), 3)
    _prof(torch, lambda: wl.ctx_a.kam_form_patch(cond, solo, 4096, 1, m))
    sweeps = 6
    b = m + 8
    flops = L * H * (2.0 * T * D * D + sweeps * 2 * (2.0 * D * D * b)) + L * H * 2.0 * T * D * b       # Gram + sweeps on D x D + U = Delta V
    return {"ms": ms, "ms_per_chunk_k_and_v": 2 * ms, "gflops": flops / ms / 1e6,
            "what": "kam_form_patch(is_key = 1) for one 1024-token chunk x 28 layers x 4 KV heads, rank 16 (+8 oversampling), 6 sweeps of block "
                    "subspace iteration on Delta^T Delta; flops = Gram product + sweeps + U = Delta V; CUDA cores (fp32), not tuned: paid once per chunk at "
                    "compile time (P:56), not on the serve path"}


def _config5_leg(wl, device, peak, rnd):
    """BASELINE.json configs[4]: GQA 64 q / 8 kv heads, head_dim 128, chunks of 2048 tokens, m = 32, page size 16; 64 requests x 32
    chunks.  The stated pool (~150 GB) holds 8 of the 80 layers at a time; the bench keeps 2 layers resident (34 GB) beside its own
    workload: ONE launch relocates 256 chunks (8 requests x 32 chunks) from 256 distinct canonical chunks (5.4 GB; with fewer sources
    than relocations two CTAs read the same source at the same moment and the second read is an L2 hit - measured: DRAM reads fell to
    half the algorithmic bytes), and the fused decode reads batch 64 x 65536 tokens (17.2 GB per layer)."""
    import torch
    kam, B = wl.kam, wl.B
    from synth import CONFIGS
    cx = CONFIGS[5]
    H, D, P, T, m, Hq = cx.n_kv_heads, cx.row_dim, cx.page_size, cx.chunk_tokens, cx.rank, cx.n_q_heads
    Lx, NREQ, NCH, NSRC, PER = 2, 64, 32, 256, 256
    ppr = NCH * T // P
    need = 2 * Lx * NREQ * ppr * P * H * D * 2 + NSRC * Lx * 2 * (T * H * D * 2 + T * H * m * 2) + 2e9
    free = torch.cuda.mem_get_info()[0]
    if free < need:
        return {"skipped": "needs %.0f GB of free HBM, %.0f GB free" % (need / 1e9, free / 1e9)}
    pool = kam.Pool([torch.zeros((NREQ * ppr, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(Lx)],
                    [torch.zeros((NREQ * ppr, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(Lx)])
    ctx = kam.Context(kam.make_layout(B.KAM_GQA, Lx, Hq, H, D, 0, D, True, P, cx.theta), pool)
    srcs = [(kam.Chunk([rnd((T, H, D)) for _ in range(Lx)], [rnd((T, H, D)) for _ in range(Lx)]),
             kam.Patch([rnd((T, H, m)) for _ in range(Lx)], [rnd((H, m, D), cx.w_std) for _ in range(Lx)],
                       [rnd((T, H, m)) for _ in range(Lx)], [rnd((H, m, D), cx.w_std) for _ in range(Lx)])) for _ in range(NSRC)]
    bt = torch.randperm(NREQ * ppr, device=device, dtype=torch.int32)
    gen = torch.Generator().manual_seed(5)
    targets = torch.randint(0, cx.max_pos, (NREQ * NCH,), generator=gen).tolist()
    it = [0]

    def launch():
        g0 = (it[0] * PER) % (NREQ * NCH)
        it[0] += 1
        ctx.kam_relocate_patch_batch([(bt, (g0 + c) * T, srcs[(g0 + c) % NSRC][0], targets[g0 + c], srcs[(g0 + c) % NSRC][1], m) for c in range(PER)])
    for _ in range(NREQ * NCH // PER):                            # fill the whole pool once (8 launches): the decode reads relocated rows
        launch()
    ms = _time_queued_ms(torch, launch, 4)
    _prof(torch, launch)
    nbytes = PER * Lx * algorithmic_bytes_relocate(T, H, D, m, P)
    res = {"relocate": {"ms_per_launch": ms, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak, "chunks_per_launch": PER, "layers_resident": Lx,
                        "us_per_1024tok_chunk_80_layers": 1e3 * ms / PER * 1024 / T * cx.n_layers / Lx,
                        "ms_all_2048_chunks_80_layers_extrapolated": ms * (NREQ * NCH / PER) * cx.n_layers / Lx,
                        "tiled_kernel": ctx.kam_get_stats()["generic_launches"] == 0,
                        "what": "one kam_relocate_patch_batch of 256 chunk-relocations (m = 32) into 2 resident layers; 256 distinct sources (5.4 GB), every launch reads each once"}}
    btd = bt.reshape(NREQ, ppr)
    starts = torch.arange(0, (NCH + 1) * T, T, dtype=torch.int32, device=device).repeat(NREQ, 1)
    nc = torch.full((NREQ,), NCH, dtype=torch.int32, device=device)
    q = rnd((NREQ, Hq, D))
    o, l = torch.zeros_like(q), torch.zeros((NREQ, Hq), dtype=torch.float32, device=device)
    jt = [0]

    def dec():
        jt[0] += 1
        ctx.kam_paged_decode_merge(q, btd, starts, None, nc, jt[0] % Lx, D ** -0.5, o, l)
    msd = _time_ms(torch, dec, 4)
    _prof(torch, dec)
    nb = NREQ * NCH * T * H * 2 * D * 2
    res["decode"] = {"ms_per_layer": msd, "GB/s": nb / msd / 1e6, "frac": nb / msd / 1e6 / peak, "batch": NREQ, "tokens_per_request": NCH * T,
                     "tok_per_s_80_layers_extrapolated": NREQ / (msd * cx.n_layers / 1e3),
                     "roofline_tok_per_s_80_layers": NREQ / (nb * cx.n_layers / (peak * 1e9)),
                     "what": "kam_paged_decode_merge (plan + decode + merge per call), batch 64 over 32 chunks x 2048 tokens, one layer = 17.2 GB"}
    ctx.close()
    return res


def _config4_leg(wl, device, peak, rnd):
    """BASELINE.json configs[3] at its stated size: MHA 32 layers x 32 heads x 128, 32 requests, each a pinned 512-token text prefix + a
    window of 3 screenshots of 1280 tokens (pool 73 GB).  One slide step = every request evicts its oldest screenshot and recalls
    one by relocate+patch (m = 16) from 8 canonical chunks (5.5 GB) while the two survivors rotate in place by -1280; then
    the fused decode, batch 32, over window + prefix (4352 tokens) x 32 layers."""
    import torch
    kam, B = wl.kam, wl.B
    from synth import CONFIGS
    cx = CONFIGS[4]
    L, H, D, P, T, m = cx.n_layers, cx.n_kv_heads, cx.row_dim, cx.page_size, cx.chunk_tokens, cx.rank
    NREQ, TP, NCAN = 32, 512, 8
    ppc = T // P
    n_pages = NREQ * (TP // P + 4 * ppc)
    need = 2 * L * n_pages * P * H * D * 2 + NCAN * L * 2 * (T * H * D * 2 + T * H * m * 2) + 3e9
    free = torch.cuda.mem_get_info()[0]
    if free < need:
        return {"skipped": "needs %.0f GB of free HBM, %.0f GB free" % (need / 1e9, free / 1e9)}
    pool = kam.Pool([torch.zeros((n_pages, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)],
                    [torch.zeros((n_pages, P, H, D), dtype=torch.bfloat16, device=device) for _ in range(L)])
    ctx = kam.Context(kam.make_layout(B.KAM_MHA, L, cx.n_q_heads, H, D, 0, D, True, P, cx.theta), pool, max_requests=NREQ,
                      max_chunks_per_request=5, max_pages_per_chunk=ppc)
    canon = [(kam.Chunk([rnd((T, H, D)) for _ in range(L)], [rnd((T, H, D)) for _ in range(L)]),
              kam.Patch([rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cx.w_std) for _ in range(L)],
                        [rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cx.w_std) for _ in range(L)])) for _ in range(NCAN)]
    prefix = kam.Chunk([rnd((TP, H, D)) for _ in range(L)], [rnd((TP, H, D)) for _ in range(L)])
    for r in range(NREQ):
        ctx.kam_window_open(r, 0)
        ctx.kam_admit(r, B.KAM_BACK, prefix, None, 0, 1)
        ctx.kam_window_pin(r, 1)
        for c in range(3):
            ctx.kam_admit(r, B.KAM_BACK, canon[(r + c) % NCAN][0], canon[(r + c) % NCAN][1], m, 1)
    torch.cuda.synchronize()
    it = [0]

    def slide_step():                                            # ONE launch per request: 2 survivors in place + the recalled chunk
        s = it[0]
        it[0] += 1
        for r in range(NREQ):
            ci = (r + 3 + s) % NCAN
            ctx.kam_slide(r, B.KAM_FRONT, B.KAM_BACK, canon[ci][0], canon[ci][1], m, 1)
    ms_slide = _time_ms(torch, slide_step, 3)
    _prof(torch, lambda: ctx.kam_slide(0, B.KAM_FRONT, B.KAM_BACK, canon[1][0], canon[1][1], m, 1))
    _prof(torch, lambda: ctx.kam_evict(1, B.KAM_FRONT, 1))
    _prof(torch, lambda: ctx.kam_admit(1, B.KAM_BACK, canon[2][0], canon[2][1], m, 1))
    b_surv = 2 * L * (2 * T * H * D * 2)                           # two survivors: K rows read + written, V untouched
    b_rec = L * algorithmic_bytes_relocate(T, H, D, m, P)
    # the two halves separately (the two-call form: kam_evict rotates the survivors, kam_admit recalls)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ms_e = ms_a = 0.0
    for rep in range(3):
        ev[0].record()
        for r in range(NREQ):
            ctx.kam_evict(r, B.KAM_FRONT, 1)
        ev[1].record()
        for r in range(NREQ):
            ci = (r + 5 + rep) % NCAN
            ctx.kam_admit(r, B.KAM_BACK, canon[ci][0], canon[ci][1], m, 1)
        ev[2].record(); torch.cuda.synchronize()
        if rep:                                                   # the first repetition warms up
            ms_e += ev[0].elapsed_time(ev[1]) / 2; ms_a += ev[1].elapsed_time(ev[2]) / 2
    res = {"slide_step": {"ms": ms_slide, "GB/s": NREQ * (b_surv + b_rec) / ms_slide / 1e6, "frac": NREQ * (b_surv + b_rec) / ms_slide / 1e6 / peak,
                          "roofline_ms": NREQ * (b_surv + b_rec) / (peak * 1e6), "launches": NREQ,
                          "what": "32 x kam_slide(FRONT, BACK, m = 16): per request 2 x 1280 survivor tokens rotated in place (K only) + 1280 tokens recalled by Eq. 1, 32 layers"},
           "survivors_alone": {"ms": ms_e, "GB/s": NREQ * b_surv / ms_e / 1e6, "frac": NREQ * b_surv / ms_e / 1e6 / peak,
                               "us_per_1024tok_chunk": 1e3 * ms_e / (NREQ * 2 * T / 1024), "what": "32 x kam_evict(FRONT, materialize = 1)"},
           "recall_alone": {"ms": ms_a, "GB/s": NREQ * b_rec / ms_a / 1e6, "frac": NREQ * b_rec / ms_a / 1e6 / peak,
                            "us_per_1024tok_chunk": 1e3 * ms_a / (NREQ * T / 1024), "what": "32 x kam_admit(BACK, m = 16)"}}
    q = rnd((NREQ, cx.n_q_heads, D))
    o, l = torch.zeros_like(q), torch.zeros((NREQ, cx.n_q_heads), dtype=torch.float32, device=device)
    reqs = list(range(NREQ))

    def decode_step():
        ctx.kam_window_plan(reqs)
        for layer in range(L):
            ctx.kam_window_decode(q, reqs, layer, D ** -0.5, o, l)
    ms_d = _time_ms(torch, decode_step, 3)
    _prof(torch, lambda: ctx.kam_window_decode(q, reqs, 7, D ** -0.5, o, l))
    nb = NREQ * (TP + 3 * T) * H * 2 * D * 2 * L
    res["decode_step"] = {"ms": ms_d, "GB/s": nb / ms_d / 1e6, "frac": nb / ms_d / 1e6 / peak, "tok_per_s": NREQ / (ms_d / 1e3),
                          "roofline_tok_per_s": NREQ / (nb / (peak * 1e9)), "batch": NREQ, "tokens_per_request": TP + 3 * T,
                          "what": "kam_window_plan + 32 x kam_window_decode (eager), 73 GB read per step"}
    res["pool_GB"] = 2 * L * n_pages * P * H * D * 2 / 1e9
    ctx.close()
    return res


# ------------------------------------------------------------------------------------------------------- ncu evidence
NCU_SUMMARY = "profiles/ncu_step_r03.json"


def ncu_evidence(kernel_key):
    """DRAM bytes per launch and ncu's own dram__throughput % for the named kernel, from the committed summary of ONE
    `ncu --set full` capture of a bench step (profiles/ncu_step_r03.md names the command and the commit).  None if absent."""
    path = os.path.join(ROOT, NCU_SUMMARY)
    if not os.path.exists(path):
        return None
    d = json.load(open(path))
    k = d.get("kernels", {}).get(kernel_key)
    if k is None:
        return None
    return {"traffic": k.get("dram_bytes"), "ncu_dram_pct": k.get("dram_throughput_pct"), "source": "%s (%s)" % (NCU_SUMMARY, d.get("capture", ""))}


# ------------------------------------------------------------------------------------------------------- main
def rank_requests(rank, world, per_gpu=N_REQ):
    """Global request ids rank `rank` owns: the path partitions by request with no exchange; per-GPU
    work is fixed as N grows (weak scaling), so the job serves world * per_gpu requests and rank r the r-th block of them."""
    return list(range(rank * per_gpu, (rank + 1) * per_gpu))


def _reduce(x, world, op):
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op))
    return float(t.item())


def max_over_ranks(x, world):
    """Largest value of x over all ranks (device timing is reduced this way; works on NCCL and gloo alike)."""
    return _reduce(x, world, "MAX")


def sum_over_ranks(x, world):
    return _reduce(x, world, "SUM")


def barrier(world, clock):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    clock.sync()


def timed_steps(wl, steps, warmup, world, clock, profile=None):
    """W untimed warm-up steps, then EXACTLY `steps` steps bracketed by barrier + synchronise on both sides; device time of
    the whole region and of each phase, each the MAX over ranks; bytes summed over ranks.  wl needs step(i, mark),
    launches(), bytes_a / bytes_b / bytes_c.  clock: DeviceClock (CUDA events) - or a host clock in the gloo test."""
    for i in range(warmup):
        wl.step(i)
    barrier(world, clock)
    marks = [[None] * 4 for _ in range(steps)]
    l0 = wl.launches()
    t_host0 = time.time()
    t_start = clock.mark()
    for i in range(steps):
        if profile and i == 0:
            profile(True)
        wl.step(warmup + i, lambda k, row=marks[i]: row.__setitem__(k, clock.mark()))
        if profile and i == 0:
            profile(False)
    t_end = clock.mark()
    barrier(world, clock)
    t_host1 = time.time()
    ms_local = [sum(clock.ms(m[k], m[k + 1]) for m in marks) / steps for k in range(3)]
    return {
        "total_ms": max_over_ranks(clock.ms(t_start, t_end), world),
        "phase_ms": [max_over_ranks(x, world) for x in ms_local], "phase_ms_local": ms_local,
        "launches_per_step": (wl.launches() - l0) // steps,
        "bytes": [sum_over_ranks(b, world) for b in (wl.bytes_a, wl.bytes_b, wl.bytes_c)],
        "host_window": (t_host0, t_host1),
    }


def assemble_line(args, world, tm, peak, peak_src, wl_info, cpu=None, e2e=None, clocks=None, ex=None):
    """The one JSON line rank 0 prints.  value = ALL ranks' relocate+patch bytes / the slowest rank's device time."""
    steps = args.steps
    ms_a, ms_b, ms_c = tm["phase_ms"]
    by_a, by_b, by_c = tm["bytes"]
    la, lb, lc = tm["phase_ms_local"]
    gb = lambda b, t_ms: b / (t_ms * 1e-3) / 1e9
    L, n_req = wl_info["n_layers"], wl_info["n_req"]
    tot = la + lb + lc
    kernels = {
        "kam_relocate_patch_kernel": {"bound": "hbm", "achieved": gb(wl_info["bytes_a"], la), "bytes_per_launch": wl_info["bytes_a"], "ms_per_launch": la, "share_of_step": la / tot},
        "window_slide(kam_slide)": {"bound": "hbm", "achieved": gb(wl_info["bytes_b"], lb), "bytes_per_launch": wl_info["bytes_b"], "ms_per_launch": lb, "share_of_step": lb / tot},
        "kam_paged_decode_kernel(+merge)": {"bound": "hbm", "achieved": gb(wl_info["bytes_c"], lc), "bytes_per_launch": wl_info["bytes_c"] / L, "ms_per_launch": lc / L, "share_of_step": lc / tot},
    }
    for name, k in kernels.items():
        k.update({"peak": peak, "unit": "GB/s", "frac": k["achieved"] / peak})
        ev = ncu_evidence(name)
        if ev:
            k.update({"traffic": ev["traffic"], "ncu_dram_pct": ev["ncu_dram_pct"], "traffic_source": ev["source"]})
    dom = max(kernels, key=lambda k: kernels[k]["share_of_step"])
    roofline = {"kernel": dom, "bound": "hbm", "achieved": kernels[dom]["achieved"], "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "traffic": kernels[dom].get("traffic"), "ncu_dram_pct": kernels[dom].get("ncu_dram_pct"),
                "traffic_source": kernels[dom].get("traffic_source", "no ncu summary committed: traffic is null"),
                "denominators": "frac = achieved / MEASURED_PEAKS.json hbm_gbs (a copy: read + write); ncu_dram_pct = ncu's "
                                "dram__throughput.avg.pct_of_peak_sustained_elapsed of the same kernel (BASELINE.json's 'per ncu')"}
    return {
        "metric": "relocate+patch GB/s", "value": by_a / (ms_a * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": world, "steps": steps, "warmup": args.warmup,
        "ms_per_step": tm["total_ms"] / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: GQA Qwen2-VL-7B-like, 28 layers, 28q/4kv heads, head_dim 128, theta 1e6, "
                               "8 chunks x 1024 tokens per slide, rank-16 patch, page 16, offsets U[0,32768)",
                   "requests_per_gpu": n_req, "decode_batch": n_req, "window_tokens": wl_info["window_tokens"],
                   "decode_launch": wl_info["decode_launch"],
                   "l2": "inputs larger than L2: each step streams >1 GB of fresh source and destination; request and canonical set rotate",
                   "parallelism": "requests sharded over ranks (rank r serves global requests [r*%d, (r+1)*%d)), no collective" % (n_req, n_req)},
        "phases_ms": {"relocate_patch_batch": ms_a, "window_slide": ms_b, "decode_all_layers": ms_c},
        "us_per_1024tok_chunk": 1e3 * ms_a / wl_info["n_chunks"],
        "decode_tok_per_s": world * n_req / (ms_c * 1e-3),
        "decode_note": "attention only: batch / (per-layer attention time x 28 layers); projections and MLP are not part of the method",
        "step_gbs": (by_a + by_b + by_c) / (tm["total_ms"] / steps * 1e-3) / 1e9,
        "roofline": roofline, "roofline_all": kernels, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": tm["launches_per_step"], "clocks": clocks,
        "extras_outside_the_step": ex,
    }


def run(args, world, rank, wl, clock, wl_info, sampler=None, after=None):
    """The rank-aware part of the bench: timed region (barrier + sync on both sides, max over ranks), then rank 0 assembles and
    prints the line.  `after(tm)` (rank 0, single GPU) returns the extra legs measured outside the timed region."""
    prof = None
    if getattr(args, "profile_step", False):
        import torch
        prof = lambda on: torch.cuda.profiler.start() if on else torch.cuda.profiler.stop()
    if sampler is not None and rank == 0:
        sampler.start()                              # already streaming when the timed region starts
    tm = timed_steps(wl, args.steps, args.warmup, world, clock, prof)
    clocks = None
    if sampler is not None and rank == 0:
        sampler.t0, sampler.t1 = tm["host_window"]
        clocks = sampler.stop()
    legs = after(tm) if after is not None else {}
    line = None
    if rank == 0:
        peak, peak_src = peaks()
        line = assemble_line(args, world, tm, peak, peak_src, wl_info, cpu=legs.get("cpu"), e2e=legs.get("e2e"), clocks=clocks, ex=legs.get("extras"))
        print(json.dumps(line))
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the measurements outside the step (rank sweep, on-read patch, MLA)")
    ap.add_argument("--profile-step", action="store_true",
                    help="bracket the first timed step with cudaProfilerStart/Stop (for `ncu --profile-from-start off`)")
    ap.add_argument("--profile-extras", action="store_true",
                    help="bracket the extras leg with cudaProfilerStart/Stop instead of a timed step")
    ap.add_argument("--profile-legs", action="store_true",
                    help="skip the other extras and bracket ONE call of every phase of the as-stated config 4 / 5 legs with cudaProfilerStart/Stop")
    ap.add_argument("--no-graph", action="store_true", help="launch the per-layer decode calls eagerly instead of replaying a CUDA graph")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(3, args.warmup)
    global _PROFILE_LEGS
    _PROFILE_LEGS = args.profile_legs

    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libkamera has no CPU fallback")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)

    wl = Workload(device, rank, use_graph=not args.no_graph, world=world)
    peak, _ = peaks()
    cfg = wl.cfg
    wl_info = {"n_layers": cfg.n_layers, "n_req": N_REQ, "n_chunks": wl.n_chunks, "window_tokens": wl.n_chunks * cfg.chunk_tokens,
               "bytes_a": wl.bytes_a, "bytes_b": wl.bytes_b, "bytes_c": wl.bytes_c,
               "decode_launch": "eager" if args.no_graph else "CUDA graph of 28 x (decode, merge), plan rebuilt eagerly per step"}
    clock = DeviceClock(torch)

    def after(tm):
        legs = {}
        # e2e: the same path through the host-buffer entries, H2D and D2H inside the timed region
        if not args.no_e2e:
            ee = E2E(wl, device)
            res = {}
            for mode, pipelined in (("serial", False), ("pipelined", True)):
                wl.ctx_a.kam_set_option("host_copy_overlap", int(pipelined))
                wl.ctx_a.kam_set_option("host_entries_sync", int(not pipelined))
                for i in range(2):
                    ee.step(i, pipelined)
                barrier(world, clock)
                n_e = max(2, min(args.steps, 5))
                t0 = time.perf_counter()
                for i in range(n_e):
                    ee.step(i, pipelined)
                torch.cuda.synchronize()
                res[mode] = max_over_ranks((time.perf_counter() - t0) / n_e, world)
            by = sum_over_ranks(wl.bytes_a, world)
            legs["e2e"] = {"value": by / res["pipelined"] / 1e9, "unit": "GB/s", "h2d_bytes_per_step": ee.h2d, "d2h_bytes_per_step": ee.d2h,
                           "ms_per_step": res["pipelined"] * 1e3, "serial_value": by / res["serial"] / 1e9, "serial_ms_per_step": res["serial"] * 1e3,
                           "what": "8 x kam_relocate_patch_host (one pinned host slab per chunk: rows + factors of 28 layers -> one merged H2D on the "
                                   "library's copy stream (option host_copy_overlap = 1, opt-in: the slabs are final before the call) -> kernel; the copy of chunk c+1 runs under the kernel of chunk c) + kam_paged_decode_plan + 28 x "
                                   "kam_paged_decode_merge_host (q H2D, out/lse D2H) + ONE synchronise per step, after which the host reads out/lse; "
                                   "relocate+patch bytes / whole region.  serial_*: options host_copy_overlap=0, host_entries_sync=1 (a synchronise per decode call)"}
        if rank == 0 and world == 1 and not args.no_cpu:
            gbs, dt = oracle_sample(CPU_SAMPLE_CHUNKS, cfg.n_layers)
            cores = cpu_threads()
            ig, idt, icores = oracle_inplace_sample(4, cfg.n_layers)
            dg, dtok, ddt, dcores = oracle_decode_sample(4)
            legs["cpu"] = {"value": gbs, "unit": "GB/s", "cores": cores, "host_cores": os.cpu_count(), "kind": "oracle", "seconds": dt,
                           "sample": "relocate+patch of %d chunks x 28 layers of config 2 (1.5 steps' worth; a step has 8 chunks), "
                                     "oracle/reuse.py in numpy fp64" % CPU_SAMPLE_CHUNKS,
                           "legs": {"rotate_inplace": {"value": ig, "unit": "GB/s", "seconds": idt, "cores": icores,
                                                       "sample": "oracle/reuse.rotate_inplace_layer on 4 survivors x 28 layers (a slide has 7)"},
                                    "decode_bruteforce": {"value": dg, "unit": "GB/s", "tok_per_s_batch1_28_layers": dtok, "seconds": ddt, "cores": dcores,
                                                          "sample": "oracle/attention.attend_bruteforce for ONE request (8 x 1024 tokens, 28 query heads) x 4 layers (a step has 32 requests x 28 layers)"}}}
        if rank == 0 and world == 1 and not args.no_extras and not args.profile_step:
            if args.profile_extras:
                torch.cuda.profiler.start()
            legs["extras"] = {} if args.profile_legs else extras(wl, device, peak)
            if args.profile_extras:
                torch.cuda.profiler.stop()
            legs["extras"].update(as_stated_legs(wl, device, peak))
        return legs

    run(args, world, rank, wl, clock, wl_info, sampler=ClockSampler(local), after=after)
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
