"""GPU tests of what round 2 added around the kernels: the one-launch window slide (kam_slide; kam_admit with survivors),
a CUDA graph over kam_window_decode that survives a change of the windows' chunk count, the pinned plan of the stateless
decode (kam_paged_decode_plan), and decode over a caller's pool.  All through the C ABI, all against the oracle.
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import attention as att
from oracle import reuse
from oracle.window import BACK, FRONT, WindowStore
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table, make_chunk, make_query
from tests import parity as par
from tests.test_gpu_decode import _fill_pool, check_attention

pytestmark = pytest.mark.gpu


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _window_rows(pool, view, layer, kv="k"):
    layers = pool.k_layers if kv == "k" else pool.v_layers
    st = view["chunk_starts"]
    return [par.pool_rows(layers[layer], view["block_table"], st[c], st[c + 1] - st[c]) for c in range(len(st) - 1)]


@pytest.mark.parametrize("cfg_id,evict_end,admit_end", [(2, FRONT, BACK), (4, FRONT, BACK), (2, BACK, FRONT), (2, FRONT, FRONT)])
def test_slide_is_one_launch_and_matches_oracle(cfg_id, evict_end, admit_end):
    """kam_slide(evict_end, admit_end): ONE kernel launch in which the survivors rotate in place by their net displacement
    (teacher-forced against the GPU's own keys before the slide, R-10), V of the survivors keeps its bits, and the admitted
    chunk holds Eq. 1 at its position; integer state bit for bit against oracle.window (evict lazily, admit materialising).
    P:97: "as the oldest frame leaves, survivors re-rotate by the slide offset and a later recall rehydrates the dropped frame"."""
    cfg = CONFIGS[cfg_id].scaled(n_layers=2) if cfg_id == 2 else CONFIGS[4].scaled(n_layers=2, n_q_heads=8, n_kv_heads=8)
    P, L, m, T = cfg.page_size, 2, 16, 176                      # 176 tokens: 5.5 double tiles of 32, a ragged in-place tail
    rng = _rng(900 + cfg_id + 10 * evict_end + admit_end)
    canon = [make_chunk(cfg, rng, n_tokens=T, n_layers=L) for _ in range(5)]
    up = [par.upload_chunk(c) for c in canon]
    n_pages = 6 * (T // P)
    pool = par.make_pool(cfg, L, n_pages, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool, max_requests=1, max_chunks_per_request=5, max_pages_per_chunk=T // P)
    ws = WindowStore(n_pages, P)
    ctx.kam_window_open(0, 1000); ws.open(0, 1000)
    live = []
    for i in range(4):
        ctx.kam_admit(0, BACK, up[i][0], up[i][1], m, 1); ws.admit(0, BACK, T, 1); live.append(i)
    torch.cuda.synchronize()
    for step in range(3):
        before_view = ws.export(0)
        k_before = [_window_rows(pool, before_view, l) for l in range(L)]
        v_before = [_window_rows(pool, before_view, l, "v") for l in range(L)]
        pos_before = ws.positions(0)
        launched = ctx.kam_get_stats()["kernels_launched"]
        nxt = (4 + step) % 5
        h = ctx.kam_slide(0, evict_end, admit_end, up[nxt][0], up[nxt][1], m, 1)
        ws.evict(0, evict_end, 0)
        h2, _, p_new, _ = ws.admit(0, admit_end, T, 1)
        torch.cuda.synchronize()
        assert h == h2 and ctx.kam_get_stats()["kernels_launched"] - launched == 1
        gone = live.pop(0 if evict_end == FRONT else -1)
        live.insert(0 if admit_end == FRONT else len(live), nxt)
        got, want = ctx.kam_window_export(0), ws.export(0)
        for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets", "handles"):
            assert got[key] == want[key], (step, key)
        assert all(o == 0 for o in want["chunk_offsets"])
        pos_after = ws.positions(0)
        old_index = [i for i in range(4) if i != (0 if evict_end == FRONT else 3)]        # survivors, in order, in the old view
        new_index = [i for i in range(4) if i != (0 if admit_end == FRONT else 3)]        # where they sit in the new view
        for l in range(L):
            k_after, v_after = _window_rows(pool, want, l), _window_rows(pool, want, l, "v")
            for oi, ni in zip(old_index, new_index):
                delta = pos_after[ni] - pos_before[oi]
                expect = reuse.relocate(k_before[l][oi], delta, **par.rope_kw(cfg))
                if delta == 0:
                    assert np.array_equal(k_after[ni], k_before[l][oi])
                else:
                    assert par.compare_bf16(k_after[ni], expect, par.abs_sum_k(k_before[l][oi], delta, None, None, cfg), 0, "survivor")["fail"] == 0
                assert np.array_equal(v_after[ni], v_before[l][oi])                        # V is never touched
        ai = 0 if admit_end == FRONT else 3
        st = par.check_relocated(cfg, pool, canon[nxt], want["block_table"], want["chunk_starts"][ai], p_new, m)
        assert st["fail"] == 0 and p_new == pos_after[ai]
        del gone
    # a slide that cannot admit fails as a whole: nothing is evicted
    big = B.kam_chunk(up[0][0].c.k_layers, up[0][0].c.v_layers, T + P, 0)
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_slide(0, FRONT, BACK, big, None, 0, 1)
    assert e.value.status == B.KAM_ERR_INVALID_ARG and ctx.kam_window_export(0) == got
    assert ctx.kam_get_stats()["device_errors"] == 0
    ctx.close()


def test_front_admit_moves_survivors_in_the_same_launch():
    cfg = CONFIGS[2].scaled(n_layers=1)
    P, T, m = cfg.page_size, 64, 16
    rng = _rng(77)
    canon = [make_chunk(cfg, rng, n_tokens=T, n_layers=1) for _ in range(3)]
    up = [par.upload_chunk(c) for c in canon]
    pool = par.make_pool(cfg, 1, 12, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool, max_requests=1, max_chunks_per_request=3, max_pages_per_chunk=T // P)
    ws = WindowStore(12, P)
    ctx.kam_window_open(0, 0); ws.open(0, 0)
    for i in range(2):
        ctx.kam_admit(0, BACK, up[i][0], up[i][1], m, 1); ws.admit(0, BACK, T, 1)
    torch.cuda.synchronize()
    view = ws.export(0)
    before = _window_rows(pool, view, 0)
    launched = ctx.kam_get_stats()["kernels_launched"]
    ctx.kam_admit(0, FRONT, up[2][0], up[2][1], m, 1); ws.admit(0, FRONT, T, 1)
    torch.cuda.synchronize()
    assert ctx.kam_get_stats()["kernels_launched"] - launched == 1
    view = ws.export(0)
    assert ctx.kam_window_export(0)["block_table"] == view["block_table"]
    after = _window_rows(pool, view, 0)
    for i in range(2):
        want = reuse.relocate(before[i], T, **par.rope_kw(cfg))
        assert par.compare_bf16(after[i + 1], want, par.abs_sum_k(before[i], T, None, None, cfg), 0, "survivor")["fail"] == 0
    assert par.check_relocated(cfg, pool, canon[2], view["block_table"], 0, 0, m)["fail"] == 0
    ctx.close()


def test_graph_over_window_decode_survives_a_change_of_the_chunk_count():
    """A CUDA graph captured over kam_window_decode while the windows hold 5 chunks in total is replayed after they grew to 7
    and after they shrank to 4 (each time after an eager kam_window_plan): the window workspace never moves and the kernels
    read the plan's sizes from it, so every replay must equal the oracle over the windows as they are then."""
    cfg = CONFIGS[2].scaled(n_layers=1)
    P, T, m = cfg.page_size, 96, 16
    rng = _rng(55)
    canon = [make_chunk(cfg, rng, n_tokens=T, n_layers=1) for _ in range(4)]
    up = [par.upload_chunk(c) for c in canon]
    n_pages = 2 * 6 * (T // P)
    pool = par.make_pool(cfg, 1, n_pages, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool, max_requests=2, max_chunks_per_request=6, max_pages_per_chunk=T // P)
    ws = WindowStore(n_pages, P)
    q = make_query(cfg, rng, 2)
    qd = q.cuda()
    out = torch.zeros((2, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((2, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    scale = cfg.row_dim ** -0.5
    for r in range(2):
        ctx.kam_window_open(r, 0); ws.open(r, 0)

    def admit(r, i, lazy=False):
        ctx.kam_admit(r, BACK, up[i][0], up[i][1], m, 0 if lazy else 1); ws.admit(r, BACK, T, 0 if lazy else 1)

    def check(what):
        torch.cuda.synchronize()
        for r in range(2):
            w = ws.export(r)
            chunks = [{"k": par.pool_rows(pool.k_layers[0], w["block_table"], w["chunk_starts"][c], T),
                       "v": par.pool_rows(pool.v_layers[0], w["block_table"], w["chunk_starts"][c], T), "delta": w["chunk_offsets"][c]}
                      for c in range(len(w["chunk_offsets"]))]
            o, l = att.attend_bruteforce(par.to_f64(q[r]), chunks, scale, par.rope_kw(cfg))
            check_attention(par.to_f64(out)[r], par.to_f64(lse)[r], o, l, "%s request %d" % (what, r))

    for r, i in ((0, 0), (0, 1), (0, 2), (1, 3), (1, 0)):
        admit(r, i)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ctx.kam_window_plan([0, 1])
        ctx.kam_window_decode(qd, [0, 1], 0, scale, out, lse)      # eager once: the workspace exists before the capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ctx.kam_window_decode(qd, [0, 1], 0, scale, out, lse)
        g.replay()
        check("captured state")
        admit(0, 3); admit(1, 1)                                   # 7 chunks
        ctx.kam_window_plan([0, 1])
        out.zero_(); g.replay()
        check("grown")
        for _ in range(2):
            ctx.kam_evict(0, FRONT, 0); ws.evict(0, FRONT, 0)      # lazy: pending offsets ride in the plan
        ctx.kam_evict(1, BACK, 1); ws.evict(1, BACK, 1)            # 4 chunks
        ctx.kam_window_plan([0, 1])
        out.zero_(); g.replay()
        check("shrunk, with pending offsets")
    ctx.close()


def test_pinned_plan_is_reused_across_layers_and_gives_the_same_bits():
    """kam_paged_decode_plan pins the work split of a metadata set: the per-layer calls then launch two kernels instead of
    three and return the bits of the unpinned call; other metadata drops the pin; re-planning follows changed content."""
    cfg = CONFIGS[2].scaled(n_layers=3)
    L, P = 3, cfg.page_size
    rng = _rng(66)
    lens = [[200, 37, 512], [64], [300, 300]]
    batch, max_chunks, max_pages = 3, 3, 48
    pool = _fill_pool(cfg, L, batch * max_pages + 2, 1234)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    perm = make_block_table(rng, batch * max_pages, batch * max_pages + 2).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32); offs = np.zeros((batch, max_chunks), np.int64)
    for b, row in enumerate(lens):
        for c, n in enumerate(row):
            starts[b, c + 1] = starts[b, c] + n; offs[b, c] = 100 * b - 7 * c
        starts[b, len(row) + 1:] = starts[b, len(row)]
    ncs = torch.tensor([len(r) for r in lens], dtype=torch.int32, device="cuda")
    bt_d, st_d, of_d = torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda()
    q = make_query(cfg, rng, batch).cuda()
    scale = cfg.row_dim ** -0.5
    ref = []
    for l in range(L):
        o = torch.zeros((batch, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
        s = torch.zeros((batch, cfg.n_q_heads), dtype=torch.float32, device="cuda")
        ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, l, scale, o, s)
        ref.append((o, s))
    k0 = ctx.kam_get_stats()["kernels_launched"]
    assert k0 == 3 * L
    ctx.kam_paged_decode_plan(bt_d, st_d, of_d, ncs)
    for l in range(L):
        o, s = torch.zeros_like(ref[0][0]), torch.zeros_like(ref[0][1])
        ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, l, scale, o, s)
        torch.cuda.synchronize()
        assert torch.equal(o, ref[l][0]) and torch.equal(s, ref[l][1])
    assert ctx.kam_get_stats()["kernels_launched"] - k0 == 1 + 2 * L
    # content changed in place -> the caller re-plans; the result follows the new offsets (vs the oracle)
    of_d.add_(5)
    ctx.kam_paged_decode_plan(bt_d, st_d, of_d, ncs)
    o, s = torch.zeros_like(ref[0][0]), torch.zeros_like(ref[0][1])
    ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, 1, scale, o, s)
    torch.cuda.synchronize()
    for b, row in enumerate(lens):
        chunks, t0 = [], 0
        for c, n in enumerate(row):
            chunks.append({"k": par.pool_rows(pool.k_layers[1], perm[b], t0, n), "v": par.pool_rows(pool.v_layers[1], perm[b], t0, n),
                           "delta": int(offs[b, c]) + 5})
            t0 += n
        oo, ll = att.attend_bruteforce(par.to_f64(q[b]), chunks, scale, par.rope_kw(cfg))
        check_attention(par.to_f64(o)[b], par.to_f64(s)[b], oo, ll, "re-planned request %d" % b)
    # a call with other metadata builds its own plan and drops the pin
    k1 = ctx.kam_get_stats()["kernels_launched"]
    st2 = st_d.clone()
    ctx.kam_paged_decode_merge(q, bt_d, st2, of_d, ncs, 0, scale, o, s)
    ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, 0, scale, o, s)
    assert ctx.kam_get_stats()["kernels_launched"] - k1 == 6
    ctx.close()


def test_decode_over_a_callers_pool_gqa_and_mla():
    """kam_paged_decode_merge's `pool` argument: a pool other than the context's gets its own TMA tensor maps (cached per pool);
    GQA and absorbed MLA, against the oracle; the context's own pool still works afterwards."""
    for cfg in (CONFIGS[2].scaled(n_layers=1), CONFIGS[3].scaled(n_layers=1)):
        mla = not cfg.has_v
        rng = _rng(88 + mla)
        P, D = cfg.page_size, cfg.row_dim
        Dv = cfg.v_dim if mla else D
        lens = [[150, 64], [300]]
        max_pages = (300 + P - 1) // P + 1
        num_pages = 2 * max_pages + 1

        def mk(seed):
            shape = (num_pages, P, cfg.n_kv_heads, D)
            from synth import randn_device
            k = [randn_device(shape, seed, 1.0, torch.bfloat16, "cuda")]
            return kam.Pool(k, None if mla else [randn_device(shape, seed + 1, 1.0, torch.bfloat16, "cuda")])
        own, other = mk(500), mk(600)
        ctx = kam.Context(par.layout_of(cfg, 1), own)
        perm = make_block_table(rng, 2 * max_pages, num_pages).reshape(2, max_pages)
        starts = np.array([[0, 150, 214], [0, 300, 300]], np.int32)
        offs = np.array([[12, -900], [4000, 0]], np.int64)
        ncs = torch.tensor([2, 1], dtype=torch.int32, device="cuda")
        q = torch.from_numpy(rng.standard_normal((2, cfg.n_q_heads, D), dtype=np.float32)).to(torch.bfloat16)
        scale = 192 ** -0.5 if mla else D ** -0.5
        for pool, arg in ((other, other), (own, None), (other, other)):
            out = torch.zeros((2, cfg.n_q_heads, Dv), dtype=torch.bfloat16, device="cuda")
            lse = torch.zeros((2, cfg.n_q_heads), dtype=torch.float32, device="cuda")
            ctx.kam_paged_decode_merge(q.cuda(), torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(),
                                       ncs, 0, scale, out, lse, pool=arg)
            torch.cuda.synchronize()
            for b in range(2):
                chunks, t0 = [], 0
                for c, n in enumerate(lens[b]):
                    chunks.append({"k": par.pool_rows(pool.k_layers[0], perm[b], t0, n),
                                   "v": None if mla else par.pool_rows(pool.v_layers[0], perm[b], t0, n), "delta": int(offs[b, c])})
                    t0 += n
                kw = dict(v_dim=Dv) if mla else {}
                o, l = att.attend_bruteforce(par.to_f64(q[b]), chunks, scale, par.rope_kw(cfg), **kw)
                check_attention(par.to_f64(out)[b], par.to_f64(lse)[b], o, l, "%s request %d" % ("MLA" if mla else "GQA", b))
        ctx.close()


@pytest.mark.parametrize("cfg_id", [2, 3])
def test_first_decode_right_behind_the_plan_kernel(cfg_id):
    """kam_paged_decode_plan followed AT ONCE by kam_paged_decode_merge on a fresh context (fresh workspace, no kernel between the
    two): the plan kernel releases its dependents at its first instruction, so the decode launched behind it with programmatic
    dependent launch must still not read the plan before it is complete.  Many chunks make the plan kernel long.  The result must
    carry the bits of an unpinned call on another context, for GQA and for absorbed MLA, on repeated fresh contexts."""
    cfg = CONFIGS[cfg_id].scaled(n_layers=1)
    mla = not cfg.has_v
    rng = _rng(70 + cfg_id)
    P, D = cfg.page_size, cfg.row_dim
    Dv = cfg.v_dim if mla else D
    batch, max_chunks = 24, 40
    lens = [[int(x) for x in rng.integers(1, 90, size=int(rng.integers(1, max_chunks + 1)))] for _ in range(batch)]
    max_pages = max((sum(r) + P - 1) // P for r in lens) + 1
    num_pages = batch * max_pages + 2
    from synth import randn_device
    shape = (num_pages, P, cfg.n_kv_heads, D)
    pool = kam.Pool([randn_device(shape, 77, 1.0, torch.bfloat16, "cuda")], None if mla else [randn_device(shape, 78, 1.0, torch.bfloat16, "cuda")])
    perm = make_block_table(rng, batch * max_pages, num_pages).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32); offs = np.zeros((batch, max_chunks), np.int64)
    for b, row in enumerate(lens):
        for c, n in enumerate(row):
            starts[b, c + 1] = starts[b, c] + n; offs[b, c] = int(rng.integers(-5000, 5000)) * (c % 3 != 0)
        starts[b, len(row) + 1:] = starts[b, len(row)]
    ncs = torch.tensor([len(r) for r in lens], dtype=torch.int32, device="cuda")
    bt_d, st_d, of_d = torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda()
    q = torch.from_numpy(rng.standard_normal((batch, cfg.n_q_heads, D), dtype=np.float32)).to(torch.bfloat16).cuda()
    scale = 192 ** -0.5 if mla else D ** -0.5
    ref_o = torch.zeros((batch, cfg.n_q_heads, Dv), dtype=torch.bfloat16, device="cuda")
    ref_s = torch.zeros((batch, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, 0, scale, ref_o, ref_s)      # unpinned: plan, decode and merge in one call
    torch.cuda.synchronize()
    ctx.close()
    b0 = int(np.argmax([len(r) for r in lens]))                                       # and the reference itself against the oracle
    chunks, t0 = [], 0
    for c, n in enumerate(lens[b0]):
        chunks.append({"k": par.pool_rows(pool.k_layers[0], perm[b0], t0, n),
                       "v": None if mla else par.pool_rows(pool.v_layers[0], perm[b0], t0, n), "delta": int(offs[b0, c])})
        t0 += n
    o, l = att.attend_bruteforce(par.to_f64(q[b0].cpu()), chunks, scale, par.rope_kw(cfg), **(dict(v_dim=Dv) if mla else {}))
    check_attention(par.to_f64(ref_o)[b0], par.to_f64(ref_s)[b0], o, l, "reference request %d" % b0)
    for rep in range(6):
        ctx = kam.Context(par.layout_of(cfg, 1), pool)                                # fresh context: its workspace holds no older plan
        out = torch.full_like(ref_o, 7.0); lse = torch.full_like(ref_s, 7.0)
        torch.cuda.synchronize()
        ctx.kam_paged_decode_plan(bt_d, st_d, of_d, ncs)
        ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, 0, scale, out, lse)      # nothing between the plan kernel and this
        torch.cuda.synchronize()
        assert torch.equal(out, ref_o) and torch.equal(lse, ref_s), "repetition %d" % rep
        ctx.kam_paged_decode_merge(q, bt_d, st_d, of_d, ncs, 0, scale, out, lse)      # the settled plan: same bits again
        torch.cuda.synchronize()
        assert torch.equal(out, ref_o) and torch.equal(lse, ref_s)
        ctx.close()


def test_first_window_decode_right_behind_kam_window_plan():
    """The same sequence on the window path: an explicit kam_window_plan followed at once by kam_window_decode (the plan counts as
    cached there, so the decode used to start under the plan kernel); against the oracle, on fresh contexts."""
    cfg = CONFIGS[2].scaled(n_layers=1)
    P, T, m, R, C = cfg.page_size, 64, 16, 8, 12
    rng = _rng(91)
    canon = [make_chunk(cfg, rng, n_tokens=T, n_layers=1) for _ in range(3)]
    up = [par.upload_chunk(c) for c in canon]
    n_pages = R * C * (T // P)
    q = make_query(cfg, rng, R)
    qd = q.cuda()
    scale = cfg.row_dim ** -0.5
    for rep in range(3):
        pool = par.make_pool(cfg, 1, n_pages, torch.bfloat16)
        ctx = kam.Context(par.layout_of(cfg, 1), pool, max_requests=R, max_chunks_per_request=C, max_pages_per_chunk=T // P)
        ws = WindowStore(n_pages, P)
        for r in range(R):
            ctx.kam_window_open(r, 0); ws.open(r, 0)
            for i in range(C - (r % 3)):
                ctx.kam_admit(r, BACK, up[(r + i) % 3][0], up[(r + i) % 3][1], m, 1); ws.admit(r, BACK, T, 1)
            ctx.kam_evict(r, FRONT, 0); ws.evict(r, FRONT, 0)                         # lazy: a pending offset rides in the plan
        out = torch.full((R, cfg.n_q_heads, cfg.row_dim), 7.0, dtype=torch.bfloat16, device="cuda")
        lse = torch.full((R, cfg.n_q_heads), 7.0, dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        ctx.kam_window_plan(list(range(R)))
        ctx.kam_window_decode(qd, list(range(R)), 0, scale, out, lse)
        torch.cuda.synchronize()
        for r in (0, R - 1):
            w = ws.export(r)
            chunks = [{"k": par.pool_rows(pool.k_layers[0], w["block_table"], w["chunk_starts"][c], T),
                       "v": par.pool_rows(pool.v_layers[0], w["block_table"], w["chunk_starts"][c], T), "delta": w["chunk_offsets"][c]}
                      for c in range(len(w["chunk_offsets"]))]
            o, l = att.attend_bruteforce(par.to_f64(q[r]), chunks, scale, par.rope_kw(cfg))
            check_attention(par.to_f64(out)[r], par.to_f64(lse)[r], o, l, "repetition %d request %d" % (rep, r))
        assert not bool((lse == 7.0).any())                                           # every (request, head) was written
        ctx.close()
