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
three kernels' roofline fractions ride along in the same line.  N > 1: requests are sharded over ranks, no data-path
collective (the path partitions by request), time = max over ranks, value = all ranks' bytes / that.
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
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.idx = [], None, gpu_index
        self.t0 = self.t1 = None                      # host times bracketing the timed region: only samples inside count

    def mark_begin(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")] + [time.time()])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for r in self.rows if len(r) >= 10 and r[1].replace(".", "").isdigit()]
        if self.t0 is not None and self.t1 is not None:
            rows = [r for r in rows if self.t0 <= r[-1] <= self.t1 + 0.02]
        sm = [float(r[1]) for r in rows]
        mx = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in rows for n, v in zip(names, r[5:9]) if v.lower().startswith("active")})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------------- the workload
class Workload:
    def __init__(self, device, rank, use_graph=True):
        import numpy as np
        import torch

        import paper_2606_23581_b200 as kam
        from paper_2606_23581_b200 import binding as B
        from synth import CONFIGS, randn_device
        self.torch, self.kam, self.B = torch, kam, B
        cfg = self.cfg = CONFIGS[CFG_ID]
        L, H, D, P, T, m = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.chunk_tokens, cfg.rank
        self.n_chunks = cfg.chunks_per_step
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
                ch, pa = self.sets[r % N_SETS][c]
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

    def step(self, i, ev=None):
        cfg, B, T, m = self.cfg, self.B, self.cfg.chunk_tokens, self.cfg.rank
        r, cs = i % N_REQ, self.sets[i % N_SETS]
        rec = (lambda k: ev[k].record()) if ev is not None else (lambda k: None)
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
    and out / lse go back to it inside kam_paged_decode_merge_host."""

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
        self.out_h = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16).pin_memory()
        self.lse_h = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32).pin_memory()
        self.h2d += L * self.q_h.numel() * 2
        self.d2h = L * (self.out_h.numel() * 2 + self.lse_h.numel() * 4)

    def step(self, i):
        wl, cfg = self.wl, self.wl.cfg
        T, m = cfg.chunk_tokens, cfg.rank
        p = wl.rng.integers(0, cfg.max_pos, size=wl.n_chunks)
        for c, (k, v, uk, wk, uv, wv, _slab) in enumerate(self.chunks):
            wl.ctx_a.kam_relocate_patch_host(self.bt.reshape(-1), c * T, T, 0, int(p[c]), k, v, uk, wk, uv, wv, m)
        for l in range(cfg.n_layers):
            wl.ctx_a.kam_paged_decode_merge_host(self.q_h, self.bt, self.starts, None, self.nc, l, wl.sm_scale, self.out_h, self.lse_h)


# ------------------------------------------------------------------------------------------------------- CPU oracle legs
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
    t0, c0 = time.perf_counter(), time.process_time()
    for ch in chunks:
        p = int(rng.integers(0, cfg.max_pos))
        for l in range(n_layers):
            reuse.relocate_patch_layer(pool_k, pool_v, bt, 0, f(ch["K"][l]), f(ch["V"][l]), p, f(ch["Uk"][l]), f(ch["Wk"][l]),
                                       f(ch["Uv"][l]), f(ch["Wv"][l]), theta=cfg.theta, rope_off=cfg.rope_off, d_r=cfg.rope_dim)
    dt = time.perf_counter() - t0
    global _ORACLE_CORES
    _ORACLE_CORES = max(1, int(round((time.process_time() - c0) / dt)))       # threads the oracle actually kept busy
    nbytes = n_chunks * n_layers * algorithmic_bytes_relocate(T, H, D, m, P)
    return nbytes / dt / 1e9, dt


_ORACLE_CORES = 1


def cpu_threads():
    """Cores the last oracle_sample() actually used: process CPU time / wall time (the numpy fp64 oracle is mostly one thread)."""
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
    """Measured after the timed region, NOT part of the step or of `value`: the paper's "rank-invariant in latency" claim
     as a rank sweep of the relocate kernel on config 2's shape, the rank-m patch applied ON READ inside the decode
    (row A8's second form), the decode on the shapes of configs 4 and 5 (2.3 / 4.3 GB per layer instead of config 2's 0.54 GB),
    and the MLA instantiation (config 3's shape): relocate+patch and absorbed decode.  Every
    figure is algorithmic bytes / device time, as a fraction of the measured HBM peak."""
    import torch
    kam, B, cfg = wl.kam, wl.B, wl.cfg
    from synth import CONFIGS, randn_device
    L, H, D, P, T, n = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.chunk_tokens, wl.n_chunks
    out, seed = {}, [987654]

    def rnd(shape, std=1.0):
        seed[0] += 1
        return randn_device(shape, seed[0], std, torch.bfloat16, device)

    # ---- T11: rank sweep, one launch of 8 chunks x 28 layers per rank; sources/destinations rotate over 4 request slots
    sweep = {}
    for m in (0, 16, 32, 64):
        pats = None
        if m:
            pats = [kam.Patch([rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)],
                              [rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)]) for _ in range(n)]
        it = [0]

        def launch():
            r, cs = it[0] % bench_slots, wl.sets[it[0] % N_SETS]
            it[0] += 1
            wl.ctx_a.kam_relocate_patch_batch([(wl.bt_a, (r * n + c) * T, cs[c][0], 1000 + 37 * c + it[0], pats[c] if pats else None, m) for c in range(n)])
        bench_slots = N_REQ
        ms = _time_ms(torch, launch, 10)
        nbytes = n * L * algorithmic_bytes_relocate(T, H, D, m, P) if m else n * L * (2 * 2 * T * H * D * 2 + 4 * (T // P))
        sweep["m=%d" % m] = {"ms": ms, "us_per_1024tok_chunk": 1e3 * ms / n, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak}
        del pats
    out["relocate_rank_sweep"] = sweep

    # ---- A8, second form: decode with the rank-16 patch applied on read (stateless call: plan + decode + merge per layer)
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
    for name, pr in (("decode_stateless_no_patch", None), ("decode_stateless_on_read_patch_m16", refs)):
        it = [0]

        def launch():
            l = it[0] % Ld
            it[0] += 1
            wl.ctx_a.kam_paged_decode_merge(wl.q, bt, starts, offs, nc, l, wl.sm_scale, wl.out, wl.lse, patches=pr[l] if pr else None)
        ms = _time_ms(torch, launch, 12)
        nbytes = N_REQ * n * T * H * (2 * D + (2 * m if pr else 0)) * 2
        out[name] = {"ms_per_layer": ms, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak,
                     "bytes": "K + V" + (" + U_k + U_v" if pr else "") + " once; on-read rotation by a pending offset in both"}
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
        out[name] = {"ms_per_layer": ms, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak, "bytes": "K + V once",
                     "what": "stateless call = plan + kam_paged_decode_kernel + merge; %d q / %d kv heads" % (cx.n_q_heads, Hx)}
        ctxx.close()
        del poolx, ctxx, btx, qx, ox

    # ---- MLA (config 3 shape): relocate+patch of 4 chunks x 27 layers in one launch; absorbed decode, batch 64 x 8192 tokens
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
    nbytes = 4 * L3 * algorithmic_bytes_relocate(T3, 1, D3, m3, P3, has_v=False)
    out["mla_relocate_patch"] = {"ms": ms, "us_per_1024tok_chunk": 1e3 * ms / 4, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak}
    q3 = rnd((nb3, c3.n_q_heads, D3))
    o3 = torch.zeros((nb3, c3.n_q_heads, c3.v_dim), dtype=torch.bfloat16, device=device)
    l3 = torch.zeros((nb3, c3.n_q_heads), dtype=torch.float32, device=device)
    st3 = torch.arange(0, (nch3 + 1) * T3, T3, dtype=torch.int32, device=device).repeat(nb3, 1)
    nc3 = torch.full((nb3,), nch3, dtype=torch.int32, device=device)
    bt3b = bt3.reshape(nb3, -1)
    it = [0]

    def launch():
        l = it[0] % L3
        it[0] += 1
        ctx3.kam_paged_decode_merge(q3, bt3b, st3, None, nc3, l, 192 ** -0.5, o3, l3)
    ms = _time_ms(torch, launch, 27)
    nbytes = nb3 * nch3 * T3 * D3 * 2
    out["mla_decode_absorbed"] = {"ms_per_layer": ms, "GB/s": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peak,
                                  "bytes": "every latent+rope row once (it is both key and value)", "batch": nb3, "tokens": nch3 * T3,
                                  "what": "stateless call = plan + kam_mla_ts_decode_kernel (token-split) + merge",
                                  "tflops": nb3 * nch3 * T3 * c3.n_q_heads * (D3 + c3.v_dim) * 2 / ms / 1e9}
    ctx3.close()
    return out

# ------------------------------------------------------------------------------------------------------- main
def rank_requests(rank, world, per_gpu=N_REQ):
    """Global request ids rank `rank` owns: the path partitions by request with no exchange; per-GPU
    work is fixed as N grows (weak scaling), so the job serves world * per_gpu requests and rank r the r-th block of them."""
    return list(range(rank * per_gpu, (rank + 1) * per_gpu))


def max_over_ranks(x, world):
    """Largest value of x over all ranks (device timing is reduced this way; works on NCCL and gloo alike)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x, world):
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


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
    ap.add_argument("--no-graph", action="store_true", help="launch the per-layer decode calls eagerly instead of replaying a CUDA graph")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(3, args.warmup)

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

    wl = Workload(device, rank, use_graph=not args.no_graph)
    peak, peak_src = peaks()

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()                              # already streaming when the timed region starts
    for i in range(args.warmup):
        wl.step(i)
    barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    l0 = wl.launches()
    sampler.mark_begin()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    for i in range(args.steps):
        if args.profile_step and i == 0:
            torch.cuda.profiler.start()
        wl.step(args.warmup + i, ev[i])
        if args.profile_step and i == 0:
            torch.cuda.profiler.stop()
    t_end.record()
    barrier()
    sampler.mark_end()
    clocks = sampler.stop() if rank == 0 else None
    launches = (wl.launches() - l0) // args.steps
    total_ms = max_over_ranks(t_start.elapsed_time(t_end), world)
    ms = {k: sum(e[k].elapsed_time(e[k + 1]) for e in ev) / args.steps for k in range(3)}
    ms_a = max_over_ranks(ms[0], world); ms_b = max_over_ranks(ms[1], world); ms_c = max_over_ranks(ms[2], world)
    n_ranks_bytes_a = sum_over_ranks(wl.bytes_a, world)
    value = n_ranks_bytes_a / (ms_a * 1e-3) / 1e9

    # e2e: same path through the host-buffer entries
    e2e = None
    if not args.no_e2e:
        ee = E2E(wl, device)
        for i in range(2):
            ee.step(i)
        barrier()
        n_e = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for i in range(n_e):
            ee.step(i)
        torch.cuda.synchronize()
        dt = max_over_ranks((time.perf_counter() - t0) / n_e, world)
        e2e = {"value": sum_over_ranks(wl.bytes_a, world) / dt / 1e9, "unit": "GB/s", "h2d_bytes_per_step": ee.h2d, "d2h_bytes_per_step": ee.d2h,
               "ms_per_step": dt * 1e3, "what": "8 x kam_relocate_patch_host (one pinned host slab per chunk: rows + factors of 28 layers -> one merged H2D -> kernel) + 28 x "
               "kam_paged_decode_merge_host (q H2D, out/lse D2H) per step; relocate+patch bytes / whole region"}

    cfg = wl.cfg
    L, T = cfg.n_layers, cfg.chunk_tokens
    gb = lambda b, t_ms: b / (t_ms * 1e-3) / 1e9
    kernels = {
        "kam_relocate_patch_kernel": {"bound": "hbm", "achieved": gb(wl.bytes_a, ms[0]), "bytes_per_launch": wl.bytes_a, "ms_per_launch": ms[0],
                                      "share_of_step": ms[0] / (ms[0] + ms[1] + ms[2])},
        "window_slide(kam_slide)": {"bound": "hbm", "achieved": gb(wl.bytes_b, ms[1]), "bytes_per_launch": wl.bytes_b, "ms_per_launch": ms[1],
                                      "share_of_step": ms[1] / (ms[0] + ms[1] + ms[2])},
        "kam_paged_decode_kernel(+merge)": {"bound": "hbm", "achieved": gb(wl.bytes_c, ms[2]), "bytes_per_launch": wl.bytes_c_layer, "ms_per_launch": ms[2] / L,
                                            "share_of_step": ms[2] / (ms[0] + ms[1] + ms[2])},
    }
    for k in kernels.values():
        k.update({"peak": peak, "unit": "GB/s", "frac": k["achieved"] / peak})
    dom = max(kernels, key=lambda k: kernels[k]["share_of_step"])
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic_r01.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(dom.split("(")[0])
    roofline = {"kernel": dom, "bound": "hbm", "achieved": kernels[dom]["achieved"], "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "traffic": traffic}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        gbs, dt = oracle_sample(CPU_SAMPLE_CHUNKS, L)
        cpu = {"value": gbs, "unit": "GB/s", "cores": cpu_threads(), "host_cores": os.cpu_count(), "kind": "oracle", "seconds": dt,
               "sample": "relocate+patch of %d chunks x 28 layers of config 2 (1.5 steps' worth; a step has 8 chunks), "
                         "oracle/reuse.py in numpy fp64" % CPU_SAMPLE_CHUNKS}

    ex = None
    if rank == 0 and world == 1 and not args.no_extras and not args.profile_step:
        if args.profile_extras:
            torch.cuda.profiler.start()
        ex = extras(wl, device, peak)
        if args.profile_extras:
            torch.cuda.profiler.stop()

    if rank == 0:
        out = {
            "metric": "relocate+patch GB/s", "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1]: GQA Qwen2-VL-7B-like, 28 layers, 28q/4kv heads, head_dim 128, theta 1e6, "
                                   "8 chunks x 1024 tokens per slide, rank-16 patch, page 16, offsets U[0,32768)",
                       "requests_per_gpu": N_REQ, "decode_batch": N_REQ, "window_tokens": wl.n_chunks * T,
                       "decode_launch": "eager" if args.no_graph else "CUDA graph of 28 x (decode, merge), plan rebuilt eagerly per step",
                       "l2": "inputs larger than L2: each step streams >1 GB of fresh source and destination; request and canonical set rotate",
                       "parallelism": "requests sharded over ranks, no collective"},
            "phases_ms": {"relocate_patch_batch": ms_a, "window_slide": ms_b, "decode_all_layers": ms_c},
            "us_per_1024tok_chunk": 1e3 * ms_a / wl.n_chunks,
            "decode_tok_per_s": world * N_REQ / (ms_c * 1e-3),
            "decode_note": "attention only: batch / (per-layer attention time x 28 layers); projections and MLP are not part of the method",
            "step_gbs": sum_over_ranks(wl.bytes_a + wl.bytes_b + wl.bytes_c, world) / (total_ms / args.steps * 1e-3) / 1e9 if world == 1 else None,
            "roofline": roofline, "roofline_all": kernels, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "extras_outside_the_step": ex,
        }
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
