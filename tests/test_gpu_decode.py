"""GPU parity of kam_paged_decode_merge / kam_window_decode against the oracle.

Bar (BASELINE.json north_star; reading R-11): per (request, head) max-abs <= 2e-2, ||g-o||inf / ||o||inf <= 1e-2,
|lse_g - lse_o| <= 1e-3 (natural log).  The oracle reads the SAME pool bits the kernel reads (copied back from the
device), applies the pending relocation on read in fp64 and takes the brute-force softmax over the concatenation.
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import attention as att
from oracle import reuse
from oracle.window import BACK, FRONT, WindowStore
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table, make_chunk, make_offsets, make_query, randn_device
from tests import parity as par

pytestmark = pytest.mark.gpu


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def check_attention(out_g, lse_g, out_o, lse_o, what=""):
    """out [Hq, Dv], lse [Hq] for one request."""
    fin = np.isfinite(lse_o)
    assert np.array_equal(np.isfinite(lse_g), fin), what
    assert np.all(np.isneginf(lse_g[~fin])) and np.all(out_g[~fin] == 0), what
    if not fin.any():
        return 0.0, 0.0
    err = np.abs(out_g[fin] - out_o[fin])
    mabs = float(err.max())
    rel = float((err.max(axis=1) / np.abs(out_o[fin]).max(axis=1)).max())
    dl = float(np.abs(lse_g[fin] - lse_o[fin]).max())
    assert mabs <= 2e-2, (what, "max-abs", mabs)
    assert rel <= 1e-2, (what, "max-rel", rel)
    assert dl <= 1e-3, (what, "lse", dl)
    return mabs, dl


def _fill_pool(cfg, L, num_pages, seed):
    shape = (num_pages, cfg.page_size, cfg.n_kv_heads, cfg.row_dim)
    k = [randn_device(shape, seed + 2 * l, 1.0, torch.bfloat16, "cuda") for l in range(L)]
    v = [randn_device(shape, seed + 2 * l + 1, 1.0, torch.bfloat16, "cuda") for l in range(L)]
    return kam.Pool(k, v)


def _run_stateless(cfg, lens, deltas, seed, L=1, layer=0, sm_scale=None):
    """lens[b] = list of chunk lengths; deltas[b] = list of on-read offsets.  Everything verified vs the oracle."""
    rng = _rng(seed)
    P = cfg.page_size
    batch = len(lens)
    max_chunks = max(1, max(len(x) for x in lens))
    tot = [sum(x) for x in lens]
    max_pages = max(1, max((t + P - 1) // P for t in tot))
    num_pages = batch * max_pages + 3
    pool = _fill_pool(cfg, L, num_pages, seed)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    perm = make_block_table(rng, batch * max_pages, num_pages).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32)
    offs = np.zeros((batch, max_chunks), np.int64)
    ncs = np.zeros(batch, np.int32)
    base = rng.integers(0, 50, size=batch)                        # CSR need not start at 0: only differences count
    for b in range(batch):
        ncs[b] = len(lens[b])
        starts[b, 0] = base[b]
        for c, n in enumerate(lens[b]):
            starts[b, c + 1] = starts[b, c] + n
            offs[b, c] = deltas[b][c]
        starts[b, len(lens[b]) + 1:] = starts[b, len(lens[b])]
    q = make_query(cfg, rng, batch)
    qd = q.cuda()
    out = torch.full((batch, cfg.n_q_heads, cfg.row_dim), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((batch, cfg.n_q_heads), 7.0, dtype=torch.float32, device="cuda")
    scale = sm_scale if sm_scale is not None else cfg.row_dim ** -0.5
    args = (qd, torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(),
            torch.from_numpy(ncs).cuda(), layer, scale, out, lse)
    ctx.kam_paged_decode_merge(*args)
    torch.cuda.synchronize()
    out_g, lse_g = par.to_f64(out), par.to_f64(lse)
    # determinism: a second run gives the same bits (fixed merge order, R-17)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.kam_paged_decode_merge(*args[:-2], out2, lse2)
    torch.cuda.synchronize()
    assert torch.equal(out, out2) and torch.equal(lse, lse2)
    worst = (0.0, 0.0)
    for b in range(batch):
        chunks, t0 = [], 0
        for c, n in enumerate(lens[b]):
            chunks.append({"k": par.pool_rows(pool.k_layers[layer], perm[b], t0, n),
                           "v": par.pool_rows(pool.v_layers[layer], perm[b], t0, n), "delta": int(deltas[b][c])})
            t0 += n
        if not chunks:
            chunks = [{"k": np.zeros((0, cfg.n_kv_heads, cfg.row_dim)), "v": np.zeros((0, cfg.n_kv_heads, cfg.row_dim))}]
        o, l = att.attend_bruteforce(par.to_f64(q[b]), chunks, scale, par.rope_kw(cfg))
        r = check_attention(out_g[b], lse_g[b], o, l, "request %d" % b)
        worst = (max(worst[0], r[0]), max(worst[1], r[1]))
    ctx.close()
    return worst


def test_config1_two_relocated_chunks_end_to_end():
    """BASELINE.json configs[0]: one query ~ N(0,1) over 2 chunks that were relocated+patched (rank 4) by the GPU; the
    oracle runs the WHOLE pipeline itself (its own Eq. 1, its own rounding to the bf16 pool, its own attention)."""
    cfg = CONFIGS[1].scaled(elem_dtype="bf16")
    rng = _rng(cfg.seed)
    T, m, P = cfg.chunk_tokens, cfg.rank, cfg.page_size
    chunks = [make_chunk(cfg, rng) for _ in range(2)]
    p = make_offsets(cfg, rng, 2)
    bt_h = make_block_table(rng, 2 * T // P, 2 * T // P + 4)
    bt_d = torch.from_numpy(bt_h).cuda()
    pool = par.make_pool(cfg, 1, 2 * T // P + 4, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    up = [par.upload_chunk(c) for c in chunks]
    ctx.kam_relocate_patch_batch([(bt_d, i * T, up[i][0], int(p[i]), up[i][1], m) for i in range(2)])
    q = make_query(cfg, rng, 1)
    out = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    starts = torch.tensor([[0, T, 2 * T]], dtype=torch.int32, device="cuda")
    scale = cfg.row_dim ** -0.5
    ctx.kam_paged_decode_merge(q.cuda(), bt_d.reshape(1, -1), starts, None, torch.tensor([2], dtype=torch.int32, device="cuda"),
                               0, scale, out, lse)
    torch.cuda.synchronize()
    from oracle.bf16 import bf16_rne
    oc = []
    for i in range(2):
        ko, vo, _, _ = par.oracle_layer(cfg, chunks[i], 0, int(p[i]))
        oc.append({"k": bf16_rne(ko), "v": bf16_rne(vo), "delta": 0})          # the oracle's own pool write
    o, l = att.attend_chunks_merge(par.to_f64(q[0]), oc, scale, par.rope_kw(cfg))
    check_attention(par.to_f64(out)[0], par.to_f64(lse)[0], o, l, "config 1")
    ctx.close()


def test_config2_gqa_ragged_chunks_on_read_rotation():
    """GQA 28/4 (G = 7, padded to the 16-row MMA): ragged chunk lengths, several splits, deltas pending on read."""
    lens = [[100, 1024, 37], [1024], [5, 16, 300, 2000]]
    deltas = [[0, 31000, -77], [12345], [0, 0, -1280, 99999]]
    _run_stateless(CONFIGS[2], lens, deltas, 11)


def test_config4_mha_window_plus_prefix():
    """MHA 32 heads: 512-token text prefix + 3 x 1280 window, survivors carrying a pending -1280 (lazy slide)."""
    lens = [[512, 1280, 1280, 1280]] * 2
    deltas = [[0, -1280, -1280, 0], [0, 0, 0, 0]]
    _run_stateless(CONFIGS[4], lens, deltas, 12)


def test_config5_gqa8_many_chunks():
    """GQA 64/8 (G = 8): 32 chunks per request (shortened), random offsets up to 131072, LSE merge across all of them."""
    rng = _rng(5)
    lens = [[int(x) for x in rng.integers(40, 200, size=32)] for _ in range(2)]
    deltas = [[int(x) for x in rng.integers(-131072, 131072, size=32)] for _ in range(2)]
    _run_stateless(CONFIGS[5], lens, deltas, 13)


def test_head_dim_64_and_interleaved_scale():
    cfg = CONFIGS[1].scaled(elem_dtype="bf16")
    _run_stateless(cfg, [[256, 256], [33]], [[17, 4000], [-5]], 14, sm_scale=0.2)


def test_edge_cases_empty_request_empty_chunk_single_token():
    cfg = CONFIGS[2]
    lens = [[], [0, 1], [16, 0, 16], [1]]
    deltas = [[], [5, 7], [0, 3, -3], [100000]]
    _run_stateless(cfg, lens, deltas, 15)


def test_on_read_rotation_equals_materialised_rotation():
    """Lazy (offset applied on read) and materialised (kam_rotate_inplace, then delta = 0) decode agree; the lazy one
    has no re-rounding drift (reading R-10)."""
    cfg = CONFIGS[2]
    rng = _rng(21)
    T, P = 640, cfg.page_size
    pool = _fill_pool(cfg, 1, T // P + 2, 77)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    bt_h = make_block_table(rng, T // P, T // P + 2)
    bt = torch.from_numpy(bt_h).cuda().reshape(1, -1)
    q = make_query(cfg, rng, 1).cuda()
    starts = torch.tensor([[0, T]], dtype=torch.int32, device="cuda")
    nc = torch.tensor([1], dtype=torch.int32, device="cuda")
    res = []
    for lazy in (True, False):
        out = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
        lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
        if not lazy:
            ctx.kam_rotate_inplace(bt.reshape(-1), 0, T, -1280)
        offs = torch.tensor([[-1280 if lazy else 0]], dtype=torch.int64, device="cuda")
        ctx.kam_paged_decode_merge(q, bt, starts, offs, nc, 0, cfg.row_dim ** -0.5, out, lse)
        torch.cuda.synchronize()
        res.append((par.to_f64(out)[0], par.to_f64(lse)[0]))
    check_attention(res[1][0], res[1][1], res[0][0], res[0][1], "lazy vs materialised")
    ctx.close()


def test_window_store_slides_lazy_and_materialised_match_oracle():
    """kam_admit / kam_evict / kam_window_decode on the GPU against oracle.window + oracle.reuse + oracle.attention:
    a pinned prefix and a 3-chunk window slide 4 times, once materialising survivors in place (teacher-forced against
    the GPU's own pool state, R-10) and once lazily; block tables are compared bit for bit at every step."""
    cfg = CONFIGS[4].scaled(n_layers=1, n_q_heads=8, n_kv_heads=8)           # MHA, 8 heads to keep the oracle quick
    rng = _rng(31)
    P, L, m = cfg.page_size, 1, 16
    Tp, Tc = 64, 160
    n_pages = 2 * ((Tp + 4 * Tc) // P) + 4
    canon = [make_chunk(cfg, rng, n_tokens=Tc, n_layers=L) for _ in range(5)]
    prefix = make_chunk(cfg, rng, n_tokens=Tp, n_layers=L, rank=0)
    up = [par.upload_chunk(c) for c in canon]
    up_prefix = par.upload_chunk(prefix)
    scale = cfg.row_dim ** -0.5
    for lazy in (False, True):
        pool = par.make_pool(cfg, L, n_pages, torch.bfloat16)
        ctx = kam.Context(par.layout_of(cfg, L), pool, max_requests=2, max_chunks_per_request=6, max_pages_per_chunk=Tc // P)
        ws = WindowStore(n_pages, P)
        mat = 0 if lazy else 1
        ctx.kam_window_open(1, 0); ws.open(1, 0)
        ctx.kam_admit(1, BACK, up_prefix[0], None, 0, mat); ws.admit(1, BACK, Tp, mat)
        ctx.kam_window_pin(1, 1); ws.pin(1, 1)
        live = []                                                  # canonical index of each window chunk, in order
        for i in range(3):
            ctx.kam_admit(1, BACK, up[i][0], up[i][1], m, mat); ws.admit(1, BACK, Tc, mat); live.append(i)
        q = make_query(cfg, rng, 1)
        for slide in range(4):
            ctx.kam_evict(1, FRONT, mat); ws.evict(1, FRONT, mat); live.pop(0)
            nxt = (3 + slide) % 5
            ctx.kam_admit(1, BACK, up[nxt][0], up[nxt][1], m, mat); ws.admit(1, BACK, Tc, mat); live.append(nxt)
            got, want = ctx.kam_window_export(1), ws.export(1)
            for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets", "handles"):
                assert got[key] == want[key], (lazy, slide, key)
            out = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
            lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
            ctx.kam_window_decode(q.cuda(), [1], 0, scale, out, lse)
            torch.cuda.synchronize()
            # oracle readout over what is in the pool now, offsets pending on read in lazy mode
            bt, st, of = want["block_table"], want["chunk_starts"], want["chunk_offsets"]
            chunks = [{"k": par.pool_rows(pool.k_layers[0], bt, st[c], st[c + 1] - st[c]),
                       "v": par.pool_rows(pool.v_layers[0], bt, st[c], st[c + 1] - st[c]), "delta": of[c]}
                      for c in range(len(of))]
            o, l = att.attend_bruteforce(par.to_f64(q[0]), chunks, scale, par.rope_kw(cfg))
            check_attention(par.to_f64(out)[0], par.to_f64(lse)[0], o, l, "slide %d lazy=%s" % (slide, lazy))
        # the newest chunk sits exactly where Eq. 1 puts it: position = prefix + 2 chunks
        pos = ws.positions(1)
        last = want["chunk_starts"][-2]
        st_ = par.check_relocated(cfg, pool, canon[live[-1]], want["block_table"], last, pos[-1], m)
        assert st_["fail"] == 0
        if lazy:                                                   # survivors were never rewritten: offsets carry the slides
            assert want["chunk_offsets"][0] == 0 and want["chunk_offsets"][-1] == 0 and want["chunk_offsets"][1] < 0
        else:
            assert all(x == 0 for x in want["chunk_offsets"])
        ctx.kam_window_close(1)
        assert ctx.kam_get_stats()["pages_free"] == n_pages
        ctx.close()


# ------------------------------------------------------------------------------------------------ on-read patch (A8)
def _run_patched(cfg, lens, deltas, ranks, seed, max_rank=None, shared_u=False, frame=reuse.TARGET_FRAME, other_pool=False,
                 bad=None):
    """Stateless decode with the rank-m patch applied ON READ: ranks[b][c] = rank of chunk (b, c) (0 = no patch).  The oracle
    attends over k^ = R(delta) k + U_k W_k, v^ = v + U_v W_v formed in fp64 from the same pool bits and factor bits (O8).
    bad = (b, c, rank): that ref is given a malformed rank; the kernel must ignore it and count it."""
    rng = _rng(seed)
    P, H, D = cfg.page_size, cfg.n_kv_heads, cfg.row_dim
    batch = len(lens)
    max_chunks = max(1, max(len(x) for x in lens))
    max_pages = max(1, max((sum(x) + P - 1) // P for x in lens))
    num_pages = batch * max_pages + 3
    pool = _fill_pool(cfg, 1, num_pages, seed)
    ctx_pool = _fill_pool(cfg, 1, 2, seed + 1) if other_pool else pool       # other_pool: the bulk-copy (non tensor-map) path
    ctx = kam.Context(par.layout_of(cfg, 1), ctx_pool)
    if max_rank:
        ctx.kam_decode_set_max_patch_rank(max_rank)
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
            m = ranks[b][c]
            if m == 0:
                row.append(None)
                continue
            f = make_chunk(cfg.scaled(n_layers=1), rng, n_tokens=n, n_layers=1, rank=m)      # only the factors are used
            Uk, Wk, Uv, Wv = f["Uk"][0], f["Wk"][0], f["Uv"][0], f["Wv"][0]
            if shared_u:
                Uk, Uv = Uk[:, 0, :].contiguous(), Uv[:, 0, :].contiguous()
            host[(b, c)] = (Uk, Wk, Uv, Wv)
            mm = bad[2] if bad is not None and bad[:2] == (b, c) else m
            row.append((Uk.cuda(), Wk.cuda(), Uv.cuda(), Wv.cuda(), mm, frame))
        starts[b, len(lens[b]) + 1:] = starts[b, len(lens[b])]
        refs.append(row)
    patches = B.patch_refs(refs, "cuda", max_chunks=max_chunks)
    q = make_query(cfg, rng, batch)
    out = torch.full((batch, cfg.n_q_heads, D), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((batch, cfg.n_q_heads), 7.0, dtype=torch.float32, device="cuda")
    scale = D ** -0.5
    args = (q.cuda(), torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(),
            torch.from_numpy(ncs).cuda(), 0, scale)
    ctx.kam_paged_decode_merge(*args, out, lse, patches=patches, pool=pool if other_pool else None)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.kam_paged_decode_merge(*args, out2, lse2, patches=patches, pool=pool if other_pool else None)
    torch.cuda.synchronize()
    assert torch.equal(out, out2) and torch.equal(lse, lse2)                 # deterministic
    out_g, lse_g = par.to_f64(out), par.to_f64(lse)
    rope = dict(par.rope_kw(cfg), frame=frame)
    for b in range(batch):
        chunks, t0 = [], 0
        for c, n in enumerate(lens[b]):
            ch = {"k": par.pool_rows(pool.k_layers[0], perm[b], t0, n), "v": par.pool_rows(pool.v_layers[0], perm[b], t0, n),
                  "delta": int(deltas[b][c])}
            if (b, c) in host and not (bad is not None and bad[:2] == (b, c)):
                Uk, Wk, Uv, Wv = [par.to_f64(x) for x in host[(b, c)]]
                if shared_u:
                    Uk = np.repeat(Uk[:, None, :], H, axis=1); Uv = np.repeat(Uv[:, None, :], H, axis=1)
                ch.update(Uk=Uk, Wk=Wk, Uv=Uv, Wv=Wv)
            chunks.append(ch)
            t0 += n
        o, l = att.attend_bruteforce(par.to_f64(q[b]), chunks, scale, rope)
        check_attention(out_g[b], lse_g[b], o, l, "patched request %d" % b)
    errs = ctx.kam_get_stats()["device_errors"]
    ctx.close()
    return errs


def test_on_read_patch_config2_rank16_ragged_with_rotation():
    """GQA 28/4, rank 16: ragged chunks (tiles that straddle chunk boundaries), pending offsets AND patches on read, one
    chunk without a patch."""
    lens = [[100, 1024, 37], [1024], [5, 16, 300, 700]]
    deltas = [[0, 31000, -77], [12345], [0, 0, -1280, 99999]]
    ranks = [[16, 16, 16], [16], [16, 0, 16, 16]]
    assert _run_patched(CONFIGS[2], lens, deltas, ranks, 41, max_rank=16) == 0


def test_on_read_patch_config5_rank32_mixed_ranks_two_head_groups():
    """GQA 64/8 (two head groups of 4 KV heads): ranks 32 and 16 mixed in one call, kernel specialised for 32."""
    rng = _rng(42)
    lens = [[int(x) for x in rng.integers(40, 200, size=6)] for _ in range(2)]
    deltas = [[int(x) for x in rng.integers(-131072, 131072, size=6)] for _ in range(2)]
    ranks = [[32, 16, 32, 0, 32, 16], [16, 32, 32, 32, 0, 32]]
    assert _run_patched(CONFIGS[5], lens, deltas, ranks, 42, max_rank=32) == 0


def test_on_read_patch_rank64_default_max_rank_mha():
    """MHA (config 4 shape, 32 heads): the rank-64 removal patch with the default specialisation (KAM_MAX_RANK)."""
    assert _run_patched(CONFIGS[4], [[160, 96]], [[-1280, 0]], [[64, 48]], 43) == 0


def test_on_read_patch_shared_u_and_canonical_frame():
    """The paper's per-layer form (one U for all KV heads, R-6) and the CANONICAL frame R(delta)(k + U W) (R-4)."""
    lens, deltas, ranks = [[200, 64]], [[777, -3]], [[16, 16]]
    assert _run_patched(CONFIGS[2], lens, deltas, ranks, 44, max_rank=16, shared_u=True) == 0
    assert _run_patched(CONFIGS[2], lens, deltas, ranks, 45, max_rank=16, frame=reuse.CANONICAL_FRAME) == 0


def test_on_read_patch_head_dim_64_and_bulk_copy_path():
    cfg = CONFIGS[1].scaled(elem_dtype="bf16", factor_dtype="bf16")
    assert _run_patched(cfg, [[256, 40]], [[17, 4000]], [[16, 16]], 46, max_rank=16) == 0
    assert _run_patched(CONFIGS[2], [[300, 33]], [[5, 0]], [[16, 16]], 47, max_rank=16, other_pool=True) == 0


def test_on_read_patch_equals_materialised_patch():
    """Patching on read and materialising the same patch with kam_relocate_patch give the same readout within the decode
    tolerance (the materialised one rounds k^, v^ to bf16 once; the on-read one never rounds them)."""
    cfg = CONFIGS[2]
    rng = _rng(48)
    T, P, m = 512, cfg.page_size, 16
    ch = make_chunk(cfg, rng, n_tokens=T, n_layers=1, rank=m)
    bt_h = make_block_table(rng, 2 * T // P, 2 * T // P + 2)
    bt = torch.from_numpy(bt_h).cuda()
    pool = par.make_pool(cfg, 1, 2 * T // P + 2, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    ctx.kam_decode_set_max_patch_rank(16)
    chunk, patch = par.upload_chunk(ch)
    p_t = 20000
    ctx.kam_relocate_patch(bt, 0, chunk, p_t, patch, m)              # tokens [0, T): rotated + patched in the pool
    ctx.kam_relocate_patch(bt, T, chunk, 0, None, 0)                 # tokens [T, 2T): the canonical rows, untouched
    q = make_query(cfg, rng, 1).cuda()
    nc = torch.tensor([1], dtype=torch.int32, device="cuda")
    res = []
    for on_read in (False, True):
        out = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
        lse = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
        starts = torch.tensor([[0, T]], dtype=torch.int32, device="cuda")
        table = (bt[T // P:] if on_read else bt[:T // P]).contiguous().reshape(1, -1)
        offs = torch.tensor([[p_t if on_read else 0]], dtype=torch.int64, device="cuda")
        pr = B.patch_refs([[(patch.t[0][0], patch.t[1][0], patch.t[2][0], patch.t[3][0], m)]], "cuda") if on_read else None
        ctx.kam_paged_decode_merge(q, table, starts, offs, nc, 0, cfg.row_dim ** -0.5, out, lse, patches=pr)
        torch.cuda.synchronize()
        res.append((par.to_f64(out)[0], par.to_f64(lse)[0]))
    check_attention(res[1][0], res[1][1], res[0][0], res[0][1], "on-read vs materialised patch")
    ctx.close()


def test_on_read_patch_malformed_ref_is_ignored_and_counted():
    lens, deltas, ranks = [[64, 64]], [[0, 9]], [[16, 16]]
    assert _run_patched(CONFIGS[2], lens, deltas, ranks, 49, max_rank=16, bad=(0, 1, 8)) == 2      # rank 8: not a multiple of 16; the helper calls decode twice
    assert _run_patched(CONFIGS[2], lens, deltas, ranks, 50, max_rank=16, bad=(0, 0, 32)) == 2     # above the specialisation
