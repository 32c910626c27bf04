"""GPU parity of the absorbed MLA decode (kam_paged_decode_merge over a latent pool) against
the oracle: a cached token is one row [c_KV 512 | k_pe 64]; the score is the 576-wide dot product, the value is the row's
first 512 columns; relocation on read rotates only the 64-wide rope band; the on-read patch is the key's U, W (its latent
columns patch the value).  Same bar as the GQA decode: max-abs 2e-2, per-(request, head) max-rel 1e-2, lse 1e-3.
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import attention as att
from oracle import reuse
from oracle.window import BACK, FRONT, WindowStore
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table, make_chunk, randn_device
from tests import parity as par
from tests.test_gpu_decode import check_attention

pytestmark = pytest.mark.gpu


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _latent_pool(cfg, L, num_pages, seed):
    shape = (num_pages, cfg.page_size, 1, cfg.row_dim)
    return kam.Pool([randn_device(shape, seed + l, 1.0, torch.bfloat16, "cuda") for l in range(L)], None)


def _run(cfg, lens, deltas, seed, ranks=None, frame=reuse.TARGET_FRAME, style=reuse.HALF, layer=0, L=1, u_pad=0):
    rng = _rng(seed)
    P, D, Dv, Hq = cfg.page_size, cfg.row_dim, cfg.v_dim, cfg.n_q_heads
    batch = len(lens)
    max_chunks = max(1, max(len(x) for x in lens))
    max_pages = max(1, max((sum(x) + P - 1) // P for x in lens))
    num_pages = batch * max_pages + 3
    pool = _latent_pool(cfg, L, num_pages, seed)
    ctx = kam.Context(par.layout_of(cfg, L, style), pool)
    perm = make_block_table(rng, batch * max_pages, num_pages).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32)
    offs = np.zeros((batch, max_chunks), np.int64)
    ncs = np.array([len(x) for x in lens], np.int32)
    refs, host = [], {}
    for b in range(batch):
        row = []
        for c, n in enumerate(lens[b]):
            starts[b, c + 1] = starts[b, c] + n
            offs[b, c] = deltas[b][c]
            m = ranks[b][c] if ranks else 0
            if m == 0:
                row.append(None)
                continue
            f = make_chunk(cfg.scaled(n_layers=1), rng, n_tokens=n, n_layers=1, rank=m)
            Uk, Wk = f["Uk"][0], f["Wk"][0]
            host[(b, c)] = (Uk, Wk)
            Ud = Uk.cuda()
            if u_pad:                                            # token stride m + u_pad: the U rows of a tile are not one run
                wide = torch.zeros((n, 1, m + u_pad), dtype=Ud.dtype, device="cuda")
                wide[:, :, :m] = Ud
                Ud = wide[:, :, :m]
            row.append((Ud, Wk.cuda(), None, None, m, frame))
        starts[b, len(lens[b]) + 1:] = starts[b, len(lens[b])]
        refs.append(row)
    patches = None
    if ranks:
        ctx.kam_decode_set_max_patch_rank(16 if max(max(r) for r in ranks if r) <= 16 else 32 if max(max(r) for r in ranks if r) <= 32 else 64)
        patches = B.patch_refs(refs, "cuda", max_chunks=max_chunks)
    q = torch.from_numpy(rng.standard_normal((batch, Hq, D), dtype=np.float32)).to(torch.bfloat16)
    out = torch.full((batch, Hq, Dv), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((batch, Hq), 7.0, dtype=torch.float32, device="cuda")
    scale = (128 + 64) ** -0.5                                  # DeepSeek-V2's softmax scale: qk_nope 128 + rope 64
    args = (q.cuda(), torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(),
            torch.from_numpy(ncs).cuda(), layer, scale)
    ctx.kam_paged_decode_merge(*args, out, lse, patches=patches)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.kam_paged_decode_merge(*args, out2, lse2, patches=patches)
    torch.cuda.synchronize()
    assert torch.equal(out, out2) and torch.equal(lse, lse2)
    out_g, lse_g = par.to_f64(out), par.to_f64(lse)
    rope = dict(par.rope_kw(cfg, style), frame=frame)
    for b in range(batch):
        chunks, t0 = [], 0
        for c, n in enumerate(lens[b]):
            ch = {"k": par.pool_rows(pool.k_layers[layer], perm[b], t0, n), "v": None, "delta": int(deltas[b][c])}
            if (b, c) in host:
                ch.update(Uk=par.to_f64(host[(b, c)][0]), Wk=par.to_f64(host[(b, c)][1]))
            chunks.append(ch)
            t0 += n
        if not chunks:
            chunks = [{"k": np.zeros((0, 1, D)), "v": None}]
        o, l = att.attend_bruteforce(par.to_f64(q[b]), chunks, scale, rope, v_dim=Dv)
        check_attention(out_g[b], lse_g[b], o, l, "MLA request %d" % b)
    assert ctx.kam_get_stats()["device_errors"] == 0
    ctx.close()


def test_config3_shape_ragged_chunks_on_read_rotation():
    """DeepSeek-V2-Lite-like: 16 heads, rows of 512 + 64, page 64; ragged chunks, tiles straddling chunk boundaries."""
    lens = [[100, 1024, 37], [1024], [5, 16, 300, 700]]
    deltas = [[0, 3100, -77], [1024], [0, 0, -1024, 2048]]
    _run(CONFIGS[3], lens, deltas, 61)


def test_config3_four_chunks_in_every_order_give_the_same_readout():
    """The reorder workload read on the fly: chunk pi(i) read at offset 1024 i for two different permutations."""
    lens = [[1024] * 4, [1024] * 4]
    deltas = [[0, 1024, 2048, 3072], [3072, 0, 1024, 2048]]
    _run(CONFIGS[3], lens, deltas, 62, L=2, layer=1)


def test_more_and_fewer_heads_than_one_tile():
    _run(CONFIGS[3].scaled(n_q_heads=32), [[200, 64]], [[17, 0]], 63)
    _run(CONFIGS[3].scaled(n_q_heads=8), [[70], [130, 3]], [[-5], [0, 999]], 64)


def test_interleaved_rope_pairs():
    _run(CONFIGS[3], [[256, 31]], [[1234, -1]], 65, style=reuse.INTERLEAVED)


def test_edge_cases():
    _run(CONFIGS[3], [[], [0, 1], [16, 0, 16], [1]], [[], [5, 7], [0, 3, -3], [4000]], 66)


def test_on_read_patch_rank16_and_rank32():
    lens = [[100, 512, 37], [300]]
    deltas = [[0, 3100, -77], [1024]]
    _run(CONFIGS[3], lens, deltas, 67, ranks=[[16, 16, 0], [16]])
    _run(CONFIGS[3], lens, deltas, 68, ranks=[[32, 16, 32], [32]])
    _run(CONFIGS[3], lens, deltas, 69, ranks=[[64, 16, 48], [0]])


def test_on_read_patch_canonical_frame():
    _run(CONFIGS[3], [[200, 64]], [[777, -3]], 70, ranks=[[16, 16]], frame=reuse.CANONICAL_FRAME)


def test_window_decode_over_mla_pool_lazy_slides():
    """kam_admit / kam_evict / kam_window_decode on an MLA layout: relocate+patch writes the latent pool, a lazy FRONT evict
    leaves a pending offset that the decode applies to q_pe on read."""
    cfg = CONFIGS[3].scaled(n_layers=1)
    rng = _rng(71)
    P, m, Tc = cfg.page_size, 16, 192
    n_pages = 4 * (Tc // P) + 2
    canon = [make_chunk(cfg, rng, n_tokens=Tc, n_layers=1) for _ in range(4)]
    up = [par.upload_chunk(c) for c in canon]
    pool = par.make_pool(cfg, 1, n_pages, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool, max_requests=1, max_chunks_per_request=4, max_pages_per_chunk=Tc // P)
    ws = WindowStore(n_pages, P)
    ctx.kam_window_open(0, 0); ws.open(0, 0)
    for i in range(3):
        ctx.kam_admit(0, BACK, up[i][0], up[i][1], m, 0); ws.admit(0, BACK, Tc, 0)
    ctx.kam_evict(0, FRONT, 0); ws.evict(0, FRONT, 0)
    ctx.kam_admit(0, BACK, up[3][0], up[3][1], m, 0); ws.admit(0, BACK, Tc, 0)
    got, want = ctx.kam_window_export(0), ws.export(0)
    for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets"):
        assert got[key] == want[key], key
    assert want["chunk_offsets"][0] == -Tc
    q = torch.from_numpy(rng.standard_normal((1, cfg.n_q_heads, cfg.row_dim), dtype=np.float32)).to(torch.bfloat16)
    out = torch.zeros((1, cfg.n_q_heads, cfg.v_dim), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    scale = 192 ** -0.5
    ctx.kam_window_decode(q.cuda(), [0], 0, scale, out, lse)
    torch.cuda.synchronize()
    bt, st, of = want["block_table"], want["chunk_starts"], want["chunk_offsets"]
    chunks = [{"k": par.pool_rows(pool.k_layers[0], bt, st[c], st[c + 1] - st[c]), "v": None, "delta": of[c]} for c in range(len(of))]
    o, l = att.attend_bruteforce(par.to_f64(q[0]), chunks, scale, par.rope_kw(cfg), v_dim=cfg.v_dim)
    check_attention(par.to_f64(out)[0], par.to_f64(lse)[0], o, l, "MLA window")
    ctx.close()


def test_on_read_patch_shapes_that_stress_the_ring():
    """The patch rides in the token-split kernel's box ring (W iterations around every patched segment, U rows behind their
    boxes): mixed ranks and unpatched chunks in one call, chunks shorter than one iteration, 16-token pages, more and fewer
    heads than one tile, long segments (many ring wraps), both pair layouts, U rows that are not one run per tile."""
    _run(CONFIGS[3], [[16, 33, 48, 7, 64, 20, 16, 95, 1, 40] * 2, [48] * 6], [[(7 * i) % 5 - 2 for i in range(20)], [0, 3] * 3], 110,
         ranks=[[16, 0, 32, 16, 0, 16, 48, 16, 16, 64] * 2, [16] * 6])
    _run(CONFIGS[3].scaled(page_size=16), [[100, 500, 64, 48], [77]], [[9, -9, 0, 3], [0]], 111, ranks=[[16, 16, 0, 16], [16]])
    _run(CONFIGS[3].scaled(n_q_heads=32), [[200, 64]], [[17, 0]], 112, ranks=[[16, 32]])
    _run(CONFIGS[3].scaled(n_q_heads=24), [[70], [130, 3]], [[-5], [0, 999]], 113, ranks=[[16], [16, 16]])
    _run(CONFIGS[3].scaled(n_q_heads=8), [[70], [130, 3]], [[-5], [0, 999]], 114, ranks=[[32], [16, 64]])
    _run(CONFIGS[3], [[4096 + 50], [3000, 3000]], [[123], [0, -3000]], 115, ranks=[[16], [16, 16]])
    _run(CONFIGS[3], [[256, 31]], [[1234, -1]], 116, ranks=[[16, 16]], style=reuse.INTERLEAVED)
    _run(CONFIGS[3], [[256, 31]], [[1234, -1]], 117, ranks=[[32, 16]], style=reuse.INTERLEAVED, frame=reuse.CANONICAL_FRAME)
    _run(CONFIGS[3], [[300, 100, 37]], [[5, 0, -9]], 118, ranks=[[16, 32, 16]], u_pad=8)
    _run(CONFIGS[3], [[], [0, 1], [16, 0, 16], [1]], [[], [5, 7], [0, 3, -3], [4000]], 119, ranks=[[], [16, 16], [16, 16, 0], [16]])


def test_token_split_kernel_shapes_its_iterations_do_not_divide():
    """Shapes that stress the token-split kernel's own structure (64-token iterations over a ring of 11 boxes, q staged per
    segment): a second head tile with 8 live rows of 16, 16-token pages (every box its own page), and runs of segments
    shorter than one iteration - the producer then stages the next q while the previous segment's boxes are still unread."""
    _run(CONFIGS[3].scaled(n_q_heads=24), [[200, 64, 1000], [333]], [[17, 0, -4], [5]], 101)
    _run(CONFIGS[3].scaled(page_size=16), [[100, 500, 64, 48], [77]], [[9, -9, 0, 3], [0]], 102)
    tiny = [[16, 33, 48, 7, 64, 20, 16, 95, 1, 40] * 3, [48] * 12]
    _run(CONFIGS[3], tiny, [[(7 * i) % 5 - 2 for i in range(30)], [0] * 12], 103)
    _run(CONFIGS[3], [[4096 + 50], [3000, 3000]], [[123], [0, -3000]], 104)          # long segments: many ring wraps


def test_misaligned_query_is_refused():
    """q rows travel as 16-byte-granular bulk copies: a query pointer off a 16-byte boundary is INVALID_ARG, not a fault."""
    cfg = CONFIGS[3]
    pool = _latent_pool(cfg, 1, 4, 7)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    qbuf = torch.zeros(cfg.n_q_heads * cfg.row_dim + 8, dtype=torch.bfloat16, device="cuda")
    q = qbuf[1:1 + cfg.n_q_heads * cfg.row_dim].view(1, cfg.n_q_heads, cfg.row_dim)      # 2 bytes off
    bt = torch.zeros((1, 4), dtype=torch.int32, device="cuda")
    st = torch.tensor([[0, 64]], dtype=torch.int32, device="cuda")
    nc = torch.ones(1, dtype=torch.int32, device="cuda")
    out = torch.zeros((1, cfg.n_q_heads, cfg.v_dim), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    with pytest.raises(B.KameraError) as e:
        ctx.kam_paged_decode_merge(q, bt, st, None, nc, 0, 0.1, out, lse)
    assert e.value.status == B.KAM_ERR_INVALID_ARG
    ctx.close()
