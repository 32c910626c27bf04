"""Parity at BASELINE.json's FULL sizes: configs[1] in the launch configuration bench.py times (the bench workload), configs[2]
(MLA, all 24 orderings x 27 layers) and configs[3] (MHA sliding window, 32 requests x 64 slides, ~73 GB pool); configs[4] at
scale is tests/test_gpu_config5_scale.py and configs[0] is full-size everywhere.

The test builds bench.py's own `Workload` (28 layers, 8 chunks x 1024 tokens per launch, 32 requests with 8192-token
windows, decode through the captured CUDA graph), runs steps of it and checks SAMPLED outputs against the oracle:
the inputs of every verified unit are read back from the device (the bits on the device are the ground truth, DESIGN.md
"Input recipe"); the oracle computes that unit alone.  Integer work (window block tables) is compared in full.
"""
import numpy as np
import pytest
import torch

import bench
from oracle import attention as att
from oracle import reuse
from oracle.window import BACK, FRONT, WindowStore
from tests import parity as par
from tests.test_gpu_decode import check_attention

pytestmark = pytest.mark.gpu


def _chunk_layer(ch, pa, l):
    """One layer of a device-resident canonical chunk + factors as the dict layout of synth.make_chunk (CPU tensors)."""
    g = lambda ts: ts[l].detach().cpu()[None]
    return {"K": g(ch.k_layers), "V": g(ch.v_layers), "Uk": g(pa.t[0]), "Wk": g(pa.t[1]), "Uv": g(pa.t[2]), "Wv": g(pa.t[3])}


def _check_unit(cfg, pool, l, ch, pa, bt, dst0, delta, m):
    d = _chunk_layer(ch, pa, l)
    ko, vo, Sk, Sv = par.oracle_layer(cfg, d, 0, delta)
    T = d["K"].shape[1]
    a = par.compare_bf16(par.pool_rows(pool.k_layers[l], bt, dst0, T), ko, Sk, m, "K layer %d" % l)
    b = par.compare_bf16(par.pool_rows(pool.v_layers[l], bt, dst0, T), vo, Sv, m, "V layer %d" % l)
    return {k: a[k] + b[k] for k in a}


def test_bench_workload_full_size_sampled():
    dev = torch.device("cuda", 0)
    wl = bench.Workload(dev, 0, use_graph=True)
    cfg = wl.cfg
    L, T, P, m, n = cfg.n_layers, cfg.chunk_tokens, cfg.page_size, cfg.rank, wl.n_chunks
    assert (L, T, n, bench.N_REQ) == (28, 1024, 8, 32)

    # the oracle's window model follows every admit / evict the workload makes (R-13: LIFO free list)
    npb = bench.N_REQ * (n + 1) * (T // P)
    ws = WindowStore(npb, P)
    for r in range(bench.N_REQ):
        ws.open(r, 0)
        for c in range(n):
            ws.admit(r, BACK, T, 1)

    steps = 3
    for i in range(steps):
        # the random offsets of phase A come from wl.rng: replay the stream on a copy to know them
        rng_copy = np.random.Generator(np.random.PCG64())
        rng_copy.bit_generator.state = wl.rng.bit_generator.state
        p = rng_copy.integers(0, cfg.max_pos, size=n)
        wl.step(i)
        r = i % bench.N_REQ
        ws.evict(r, FRONT, 1); ws.admit(r, BACK, T, 1)
    torch.cuda.synchronize()

    # ---- phase A of the LAST step: one launch, 8 chunks x 28 layers.  Sample: chunk 0 at every layer, every chunk at
    # the first and last layer.
    i = steps - 1
    r, cs = i % bench.N_REQ, wl.sets[i % bench.N_SETS]
    bt_a = wl.bt_a.cpu().numpy()
    tot = {}
    units = [(0, l) for l in range(L)] + [(c, l) for c in range(1, n) for l in (0, L - 1)]
    for c, l in units:
        st = _check_unit(cfg, wl.pool_a, l, cs[c][0], cs[c][1], bt_a, r * n * T + c * T, int(p[c]), m)
        for k, v in st.items():
            tot[k] = tot.get(k, 0) + v
    assert tot["fail"] == 0 and tot["within_1ulp"] >= 0.9999 * tot["n"], tot

    # ---- phase B: integer state of every request, bit for bit; the recalled chunk of the last slide sits where Eq. 1 puts it
    for rq in range(bench.N_REQ):
        got, want = wl.ctx_b.kam_window_export(rq), ws.export(rq)
        for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets"):
            assert got[key] == want[key], (rq, key)
    want = ws.export(r)
    ch, pa = cs[i % n]
    for l in (0, L // 2, L - 1):
        st = _check_unit(cfg, wl.pool_b, l, ch, pa, want["block_table"], want["chunk_starts"][-2], ws.positions(r)[-1], m)
        assert st["fail"] == 0

    # ---- phase C: the graph's last layer left out / lse of all 32 requests; sample 4 requests x all 28 query heads
    # (the slid request among them).  The oracle reads the pool rows the kernel read.
    l = L - 1
    out_g, lse_g = par.to_f64(wl.out), par.to_f64(wl.lse)
    q = par.to_f64(wl.q)
    for rq in (r, 0, 13, bench.N_REQ - 1):
        w = ws.export(rq)
        bt, st_, of = w["block_table"], w["chunk_starts"], w["chunk_offsets"]
        chunks = [{"k": par.pool_rows(wl.pool_b.k_layers[l], bt, st_[c], st_[c + 1] - st_[c]),
                   "v": par.pool_rows(wl.pool_b.v_layers[l], bt, st_[c], st_[c + 1] - st_[c]), "delta": of[c]}
                  for c in range(len(of))]
        o, ls = att.attend_bruteforce(q[rq], chunks, wl.sm_scale, par.rope_kw(cfg))
        check_attention(out_g[rq], lse_g[rq], o, ls, "request %d" % rq)

    # ---- every other request: finite, and identical on a second replay (fixed merge order => deterministic)
    assert np.isfinite(out_g).all() and np.isfinite(lse_g).all()
    out1, lse1 = wl.out.clone(), wl.lse.clone()
    wl.graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(out1, wl.out) and torch.equal(lse1, wl.lse)


def test_config3_full_size_all_permutations_sampled():
    """BASELINE.json configs[2] at full size: 27 layers, 4 cached chunks of 1024 tokens, all 24 orderings (96 relocations with
    one patch per chunk, ONE launch).  Oracle on a sample (every (chunk, offset) pair at 3 layers); across permutations the
    result of a (chunk, offset) pair must be bit-identical at EVERY layer (T10); the latent of a rank-0 relocation is untouched."""
    import itertools

    import paper_2606_23581_b200 as kam
    from synth import CONFIGS, randn_device
    cfg = CONFIGS[3]
    L, T, m, P, D = cfg.n_layers, cfg.chunk_tokens, cfg.rank, cfg.page_size, cfg.row_dim
    assert (L, T, m, P, D) == (27, 1024, 16, 64, 576)
    sd = [333]

    def rnd(shape, std=1.0):
        sd[0] += 1
        return randn_device(shape, sd[0], std, torch.bfloat16, "cuda")
    canon = [(kam.Chunk([rnd((T, 1, D)) for _ in range(L)], None),
              kam.Patch([rnd((T, 1, m)) for _ in range(L)], [rnd((1, m, D), cfg.w_std) for _ in range(L)])) for _ in range(4)]
    perms = list(itertools.permutations(range(4)))
    ppc = T // P
    n_pages = len(perms) * 4 * ppc
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    bt_h = rng.permutation(n_pages + 5)[:n_pages].astype(np.int32)
    bt_d = torch.from_numpy(bt_h).cuda()
    pool = par.make_pool(cfg, L, n_pages + 5, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    ctx.kam_relocate_patch_batch([(bt_d, (pi * 4 + slot) * T, canon[c][0], 1024 * slot, canon[c][1], m)
                                  for pi, perm in enumerate(perms) for slot, c in enumerate(perm)])
    torch.cuda.synchronize()
    assert ctx.kam_get_stats()["kernels_launched"] == 1
    first = {}
    for pi, perm in enumerate(perms):
        for slot, c in enumerate(perm):
            dst0 = (pi * 4 + slot) * T
            if (c, slot) not in first:
                first[(c, slot)] = dst0
                for l in (0, 13, 26):
                    d = {"K": canon[c][0].k_layers[l].cpu()[None], "V": None, "Uk": canon[c][1].t[0][l].cpu()[None],
                         "Wk": canon[c][1].t[1][l].cpu()[None], "Uv": None, "Wv": None}
                    ko, _, Sk, _ = par.oracle_layer(cfg, d, 0, 1024 * slot)
                    assert par.compare_bf16(par.pool_rows(pool.k_layers[l], bt_h, dst0, T), ko, Sk, m, "MLA (%d,%d,%d)" % (c, slot, l))["fail"] == 0
            else:                                                  # same (chunk, offset) under another permutation: same bits, every layer
                a0 = first[(c, slot)]
                ia = torch.from_numpy(bt_h[a0 // P:(a0 + T) // P].astype(np.int64)).cuda()
                ib = torch.from_numpy(bt_h[dst0 // P:(dst0 + T) // P].astype(np.int64)).cuda()
                for l in range(L):
                    assert torch.equal(pool.k_layers[l][ia], pool.k_layers[l][ib]), (c, slot, l)
    assert len(first) == 16
    assert par.untouched_pages_intact(pool, bt_h, L)
    ctx.close()


def test_config4_full_size_sliding_window_sampled():
    """BASELINE.json configs[3] at full size: MHA 32 layers x 32 heads x 128, 32 requests, each a pinned 512-token text prefix
    plus a window of 3 chunks of 1280 tokens (pool ~73 GB), 64 slides per request: evict FRONT (the two survivors rotate in
    place by -1280, rank 0) + recall BACK by relocate+patch (m = 16) from 8 canonical chunks cycled round-robin; then the fused
    decode, batch 32, over window + prefix.  Sampled, teacher-forced parity (R-10): for two requests and four slides the
    survivors' keys after the slide are compared with the oracle's rotation of the GPU's OWN keys before it, and the recalled
    chunk with Eq. 1; the integer state of every request is compared with the oracle's deque model after all slides."""
    import paper_2606_23581_b200 as kam
    from paper_2606_23581_b200 import binding as B
    from synth import CONFIGS, randn_device
    cfg = CONFIGS[4]
    free, _ = torch.cuda.mem_get_info()
    if free < 100e9:
        pytest.skip("config 4 at scale needs ~85 GB of free HBM")
    L, H, D, P, T, m = cfg.n_layers, cfg.n_kv_heads, cfg.row_dim, cfg.page_size, cfg.chunk_tokens, cfg.rank
    assert (L, H, D, T, m) == (32, 32, 128, 1280, 16)
    NREQ, TP, NCAN, SLIDES = 32, 512, 8, 64
    ppc = T // P
    n_pages = NREQ * (TP // P + 4 * ppc)
    sd = [4444]

    def rnd(shape, std=1.0):
        sd[0] += 1
        return randn_device(shape, sd[0], std, torch.bfloat16, "cuda")
    pool = kam.Pool([torch.zeros((n_pages, P, H, D), dtype=torch.bfloat16, device="cuda") for _ in range(L)],
                    [torch.zeros((n_pages, P, H, D), dtype=torch.bfloat16, device="cuda") for _ in range(L)])
    ctx = kam.Context(par.layout_of(cfg, L), pool, max_requests=NREQ, max_chunks_per_request=5, max_pages_per_chunk=ppc)
    canon = [(kam.Chunk([rnd((T, H, D)) for _ in range(L)], [rnd((T, H, D)) for _ in range(L)]),
              kam.Patch([rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)],
                        [rnd((T, H, m)) for _ in range(L)], [rnd((H, m, D), cfg.w_std) for _ in range(L)])) for _ in range(NCAN)]
    prefix = kam.Chunk([rnd((TP, H, D)) for _ in range(L)], [rnd((TP, H, D)) for _ in range(L)])
    ws = WindowStore(n_pages, P)
    for r in range(NREQ):
        ctx.kam_window_open(r, 0); ws.open(r, 0)
        ctx.kam_admit(r, BACK, prefix, None, 0, 1); ws.admit(r, BACK, TP, 1)
        ctx.kam_window_pin(r, 1); ws.pin(r, 1)
        for c in range(3):
            ctx.kam_admit(r, BACK, canon[(r + c) % NCAN][0], canon[(r + c) % NCAN][1], m, 1); ws.admit(r, BACK, T, 1)
    sample_req, sample_slides, sample_layers = (3, 30), (0, 1, 31, 63), (0, 31)
    checked = 0
    for s in range(SLIDES):
        for r in range(NREQ):
            probe = r in sample_req and s in sample_slides
            if probe:                                            # the GPU's own keys of the two survivors before the slide
                w = ws.export(r)
                before = {l: par.pool_rows(pool.k_layers[l], w["block_table"], w["chunk_starts"][2], 2 * T) for l in sample_layers}
                v_before = par.pool_rows(pool.v_layers[0], w["block_table"], w["chunk_starts"][2], 2 * T)
            ci = (r + 3 + s) % NCAN
            if s % 2:                                            # the two-call form ...
                ctx.kam_evict(r, FRONT, 1); ws.evict(r, FRONT, 1)
                ctx.kam_admit(r, BACK, canon[ci][0], canon[ci][1], m, 1); ws.admit(r, BACK, T, 1)
            else:                                                # ... and the slide as ONE call and ONE launch
                ctx.kam_slide(r, FRONT, BACK, canon[ci][0], canon[ci][1], m, 1); ws.evict(r, FRONT, 0); ws.admit(r, BACK, T, 1)
            if probe:
                torch.cuda.synchronize()
                w = ws.export(r)
                assert ctx.kam_window_export(r)["block_table"] == w["block_table"]
                for l in sample_layers:
                    after = par.pool_rows(pool.k_layers[l], w["block_table"], w["chunk_starts"][1], 2 * T)
                    want = reuse.relocate(before[l], -T, **par.rope_kw(cfg))
                    assert par.compare_bf16(after, want, par.abs_sum_k(before[l], -T, None, None, cfg), 0, "survivors")["fail"] == 0
                    d = {"K": canon[ci][0].k_layers[l].cpu()[None], "V": canon[ci][0].v_layers[l].cpu()[None],
                         "Uk": canon[ci][1].t[0][l].cpu()[None], "Wk": canon[ci][1].t[1][l].cpu()[None],
                         "Uv": canon[ci][1].t[2][l].cpu()[None], "Wv": canon[ci][1].t[3][l].cpu()[None]}
                    ko, vo, Sk, Sv = par.oracle_layer(cfg, d, 0, ws.positions(r)[-1])
                    assert par.compare_bf16(par.pool_rows(pool.k_layers[l], w["block_table"], w["chunk_starts"][3], T), ko, Sk, m, "recall K")["fail"] == 0
                    assert par.compare_bf16(par.pool_rows(pool.v_layers[l], w["block_table"], w["chunk_starts"][3], T), vo, Sv, m, "recall V")["fail"] == 0
                assert np.array_equal(par.pool_rows(pool.v_layers[0], w["block_table"], w["chunk_starts"][1], 2 * T), v_before)   # V untouched
                checked += 1
    assert checked == len(sample_req) * len(sample_slides)
    for r in range(NREQ):                                        # integer state of every request after 64 slides, bit for bit
        got, want = ctx.kam_window_export(r), ws.export(r)
        for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets"):
            assert got[key] == want[key], (r, key)
    # ---- fused decode, batch 32, window + prefix (4352 tokens), last layer; two requests against the brute-force softmax
    q = rnd((NREQ, cfg.n_q_heads, D))
    out = torch.zeros((NREQ, cfg.n_q_heads, D), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((NREQ, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    ctx.kam_window_decode(q, list(range(NREQ)), L - 1, D ** -0.5, out, lse)
    torch.cuda.synchronize()
    for r in (3, 17):
        w = ws.export(r)
        bt, st_, of = w["block_table"], w["chunk_starts"], w["chunk_offsets"]
        chunks = [{"k": par.pool_rows(pool.k_layers[L - 1], bt, st_[c], st_[c + 1] - st_[c]),
                   "v": par.pool_rows(pool.v_layers[L - 1], bt, st_[c], st_[c + 1] - st_[c]), "delta": of[c]} for c in range(len(of))]
        o, ls = att.attend_bruteforce(par.to_f64(q[r]), chunks, D ** -0.5, par.rope_kw(cfg))
        check_attention(par.to_f64(out)[r], par.to_f64(lse)[r], o, ls, "config 4 request %d" % r)
    ctx.close()
