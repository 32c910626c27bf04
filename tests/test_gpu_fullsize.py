"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (configs[1], the bench workload).

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
