"""GPU parity of kam_paged_prefill_merge (the P:44 readout for a block of query rows over relocated chunks)
against oracle.attention.attend_prefill_bruteforce.  Bar as for the decode (BASELINE.json; reading R-11): per (row, head)
max-abs <= 2e-2, ||g-o||inf / ||o||inf <= 1e-2, |lse_g - lse_o| <= 1e-3.  The oracle reads the SAME pool bits the kernel reads.
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import attention as att
from oracle import reuse
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table
from tests import parity as par
from tests.test_gpu_decode import _fill_pool, check_attention

pytestmark = pytest.mark.gpu


KERNELS = {"tcgen05": 1, "mma.sync": 0}       # option prefill_tcgen05: both formulations must meet the same bar


def _run(cfg, lens, deltas, Tq, causal, seed, style=reuse.HALF, rows=None, layer=0, L=1, kernel="tcgen05"):
    """lens[b]: chunk lengths of request b (its cached tokens, the appended block included when causal); every request gets a
    block of Tq query rows.  rows: the query rows the oracle evaluates (None = all)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    P, D, Hq = cfg.page_size, cfg.row_dim, cfg.n_q_heads
    batch = len(lens)
    max_chunks = max(1, max(len(x) for x in lens))
    max_pages = max(1, max((sum(x) + P - 1) // P for x in lens))
    num_pages = batch * max_pages + 3
    pool = _fill_pool(cfg, L, num_pages, seed)
    ctx = kam.Context(par.layout_of(cfg, L, B.KAM_ROPE_HALF if style == reuse.HALF else B.KAM_ROPE_INTERLEAVED), pool)
    ctx.kam_set_option("prefill_tcgen05", KERNELS[kernel])
    perm = make_block_table(rng, batch * max_pages, num_pages).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32)
    offs = np.zeros((batch, max_chunks), np.int64)
    base = rng.integers(0, 40, size=batch)
    for b in range(batch):
        starts[b, 0] = base[b]
        for c, n in enumerate(lens[b]):
            starts[b, c + 1] = starts[b, c] + n
            offs[b, c] = deltas[b][c]
        starts[b, len(lens[b]) + 1:] = starts[b, len(lens[b])]
    ncs = torch.tensor([len(x) for x in lens], dtype=torch.int32, device="cuda")
    q = torch.from_numpy(rng.standard_normal((batch, Tq, Hq, D), dtype=np.float32)).to(torch.bfloat16)
    out = torch.full((batch, Tq, Hq, D), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((batch, Tq, Hq), 7.0, dtype=torch.float32, device="cuda")
    scale = D ** -0.5
    args = (q.cuda(), torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(), ncs, layer, causal, scale)
    ctx.kam_paged_prefill_merge(*args, out, lse)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.kam_paged_prefill_merge(*args, out2, lse2)
    torch.cuda.synchronize()
    assert torch.equal(out, out2) and torch.equal(lse, lse2)            # run-to-run deterministic
    assert ctx.kam_get_stats()["kernels_launched"] == 2
    out_g, lse_g = par.to_f64(out), par.to_f64(lse)
    worst = (0.0, 0.0)
    sel = list(range(Tq)) if rows is None else rows
    for b in range(batch):
        chunks, t0 = [], 0
        for c, n in enumerate(lens[b]):
            chunks.append({"k": par.pool_rows(pool.k_layers[layer], perm[b], t0, n), "v": par.pool_rows(pool.v_layers[layer], perm[b], t0, n),
                           "delta": int(deltas[b][c])})
            t0 += n
        if not chunks:
            chunks = [{"k": np.zeros((0, cfg.n_kv_heads, D)), "v": np.zeros((0, cfg.n_kv_heads, D))}]
        o, l = att.attend_prefill_bruteforce(par.to_f64(q[b]), chunks, scale, par.rope_kw(cfg, style), causal=bool(causal), rows=sel)
        for i, t in enumerate(sel):
            r = check_attention(out_g[b, t], lse_g[b, t], o[i], l[i], "request %d row %d" % (b, t))
            worst = (max(worst[0], r[0]), max(worst[1], r[1]))
    ctx.close()
    return worst


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_config2_gqa_64_rows_over_relocated_chunks(kernel):
    """GQA 28 / 4: the appended 64-token turn (last chunk, offset 0) over recalled chunks read at pending offsets; ragged chunk
    lengths, tiles cut by chunk ends, 64 x 7 = 448 rows per KV head = 7 row tiles."""
    cfg = CONFIGS[2]
    _run(cfg, [[300, 1024, 37, 64], [100, 64]], [[3100, -77, 5, 0], [0, 0]], 64, 1, 501, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_config2_gqa_512_rows_sampled(kernel):
    """A 512-token text turn (P:105 TTFT path) over three recalled chunks; the oracle evaluates 40 of the 512 rows."""
    cfg = CONFIGS[2]
    rows = sorted(set([0, 1, 63, 64, 255, 256, 510, 511] + list(range(5, 512, 16))))
    _run(cfg, [[1024, 700, 200, 512]], [[-20000, 1, 32767, 0]], 512, 1, 502, rows=rows, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_config4_mha_64_and_512_rows(kernel):
    """MHA (G = 1: one row tile per 64 tokens and head), config 4's window + prefix shape scaled to 8 heads."""
    cfg = CONFIGS[4].scaled(n_layers=2, n_q_heads=8, n_kv_heads=8)
    _run(cfg, [[512, 1280, 64]], [[0, -1280, 0]], 64, 1, 503, layer=1, L=2, kernel=kernel)
    _run(cfg, [[160, 1280, 512]], [[0, 4096, 0]], 512, 1, 504, rows=[0, 7, 100, 300, 511], layer=0, L=2, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_not_causal_every_row_is_the_decode_readout(kernel):
    cfg = CONFIGS[2].scaled(n_q_heads=8, n_kv_heads=4)
    _run(cfg, [[130, 70], [16]], [[9, -9], [123]], 24, 0, 505, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_edge_cases(kernel):
    """Rows x G not a multiple of the 64-row tile; more query rows than cached tokens (the first rows see nothing: out = 0,
    lse = -inf); a request with no cached tokens; single-token chunks; an empty chunk in the middle."""
    cfg = CONFIGS[2].scaled(n_q_heads=12, n_kv_heads=4)           # G = 3
    _run(cfg, [[5, 0, 1, 30], [3], []], [[7, 0, -1, 0], [0], []], 10, 1, 506, kernel=kernel)
    _run(cfg, [[17]], [[0]], 1, 1, 507, kernel=kernel)           # one query row = a decode step


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_head_dim_64_and_interleaved_pairs(kernel):
    cfg = CONFIGS[1].scaled(elem_dtype="bf16", factor_dtype="bf16", n_layers=1)      # MHA 4 heads, head_dim 64
    _run(cfg, [[200, 64]], [[1000, 0]], 64, 1, 508, kernel=kernel)
    _run(CONFIGS[2].scaled(n_q_heads=8, n_kv_heads=4), [[90, 40]], [[-555, 0]], 40, 1, 509, style=reuse.INTERLEAVED, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_bench_shape_many_waves_sampled(kernel):
    """The shape bench.py's extras time (8 requests x 512 appended rows over 8 recalled 1024-token chunks + the turn, config 2's
    28 / 4 heads): 896 CTAs of the tcgen05 kernel (one per SM: 6 waves, so tensor memory is allocated after an earlier CTA's
    dealloc and the barrier words are re-initialised over used shared memory), 1792 of the mma.sync kernel.  The oracle evaluates
    8 rows of EVERY request (first / last row tiles included): 64 (request, row) pairs."""
    cfg = CONFIGS[2]
    lens = [[1024] * 8 + [512] for _ in range(8)]
    deltas = [[(-1) ** c * (1000 * b + 37 * c) for c in range(8)] + [0] for b in range(8)]
    rows = [0, 1, 17, 18, 255, 300, 493, 511]                     # G = 7: rows 0-18 sit in row tile 0, 493-511 in the last one
    _run(cfg, lens, deltas, 512, 1, 510, rows=rows, kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_three_waves_with_chunk_ends_inside_tiles(kernel):
    """11 requests x 200 rows x 7 query heads per KV head = 11 row tiles x 4 KV heads x 11 requests = 484 CTAs (> 3 x 148), ragged
    chunks whose ends fall inside 64-token tiles in every request, offsets pending on most of them."""
    cfg = CONFIGS[2]
    rng = np.random.Generator(np.random.PCG64(511))
    lens, deltas = [], []
    for b in range(11):
        n = [int(x) for x in rng.integers(1, 400, size=4)] + [200]
        lens.append(n)
        deltas.append([int(x) for x in rng.integers(-30000, 30000, size=4)] + [0])
    _run(cfg, lens, deltas, 200, 1, 512, rows=[0, 9, 10, 100, 191, 199], kernel=kernel)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_out_of_range_block_table_entries_read_as_zero_rows(kernel):
    """Inconsistent paging metadata must never be dereferenced (kamera.h): a block-table entry outside [0, num_pages) - here far
    beyond the pool and negative - reads as zero key / value rows and is counted in kam_stats.device_errors.  Checked without the
    oracle: the result must carry the bits of the same call with those entries pointing at a page that IS all zeros."""
    cfg = CONFIGS[2].scaled(n_q_heads=8, n_kv_heads=4)
    P, D, Hq, Tq = cfg.page_size, cfg.row_dim, cfg.n_q_heads, 40
    rng = np.random.Generator(np.random.PCG64(513))
    n_tok, max_pages = 300, 20                                    # 19 pages used
    num_pages = max_pages + 2
    pool = _fill_pool(cfg, 1, num_pages, 513)
    zero_page = num_pages - 1
    pool.k_layers[0][zero_page].zero_(); pool.v_layers[0][zero_page].zero_()
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    ctx.kam_set_option("prefill_tcgen05", KERNELS[kernel])
    perm = make_block_table(rng, max_pages, num_pages - 1).reshape(1, max_pages)
    starts = torch.tensor([[0, 130, n_tok]], dtype=torch.int32, device="cuda")
    offs = torch.tensor([[777, 0]], dtype=torch.int64, device="cuda")
    ncs = torch.tensor([2], dtype=torch.int32, device="cuda")
    q = torch.from_numpy(rng.standard_normal((1, Tq, Hq, D), dtype=np.float32)).to(torch.bfloat16).cuda()
    res = []
    for bad in ((zero_page, zero_page), (num_pages + 1000, -3)):
        bt = perm.copy()
        bt[0, 2], bt[0, 11] = bad
        out = torch.full((1, Tq, Hq, D), 7.0, dtype=torch.bfloat16, device="cuda")
        lse = torch.full((1, Tq, Hq), 7.0, dtype=torch.float32, device="cuda")
        ctx.kam_paged_prefill_merge(q, torch.from_numpy(bt).cuda(), starts, offs, ncs, 0, 1, D ** -0.5, out, lse)
        torch.cuda.synchronize()
        res.append((out, lse, ctx.kam_get_stats()["device_errors"]))
    assert res[0][2] == 0 and res[1][2] >= 2
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])
    ctx.close()


def test_unsupported_and_invalid_arguments():
    cfg = CONFIGS[3]                                              # MLA: not covered by the multi-query kernel
    pool = kam.Pool([torch.zeros((4, cfg.page_size, 1, cfg.row_dim), dtype=torch.bfloat16, device="cuda")], None)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    z = lambda *s, dt=torch.int32: torch.zeros(s, dtype=dt, device="cuda")
    q = torch.zeros((1, 4, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_paged_prefill_merge(q, z(1, 4), z(1, 2), None, z(1), 0, 1, 0.1, torch.zeros_like(q), z(1, 4, cfg.n_q_heads, dt=torch.float32))
    assert e.value.status == B.KAM_ERR_UNSUPPORTED and ctx.kam_get_stats()["kernels_launched"] == 0
    ctx.close()
