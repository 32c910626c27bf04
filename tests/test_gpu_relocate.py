"""GPU parity of kam_relocate_patch / kam_relocate_patch_batch / kam_rotate_inplace against the oracle (Eq. 1).

Every case runs through the C ABI (ctypes) on cuda:0 and is compared element by element with oracle/reuse.py on
the same seeded inputs.  Sizes span several tiles, several pages and a ragged tail.  Integer work (slot mapping:
which pool rows were written) is checked bit-exactly via sentinels; bf16 results by the 1-ulp rule in tests/parity.py.
"""
import itertools

import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import reuse
from oracle.bf16 import bf16_bits
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table, make_chunk, make_offsets
from tests import parity as par

pytestmark = pytest.mark.gpu


def _rng(cfg, salt=0):
    return np.random.Generator(np.random.PCG64(cfg.seed * 1000 + salt))


def _bt(rng, n_pages, num_pages):
    host = make_block_table(rng, n_pages, num_pages)
    return host, torch.from_numpy(host).cuda()


def _run_single(cfg, L, T, m, dst0=0, style=B.KAM_ROPE_HALF, frame=B.KAM_PATCH_TARGET_FRAME, delta=None, salt=0,
                shared_u=False, rank_per_layer=None, elem=None, factor=None, options=None):
    """One stateless kam_relocate_patch call, everything verified.  Returns the comparison stats (+ the context's launch
    counters: "generic_launches" says whether the element-wise fallback kernel ran)."""
    rng = _rng(cfg, salt)
    c = cfg.scaled(elem_dtype=elem or cfg.elem_dtype, factor_dtype=factor or cfg.factor_dtype)
    ch = make_chunk(c, rng, n_tokens=T, n_layers=L, rank=m)
    p_target = int(make_offsets(c, rng, 1)[0]) if delta is None else delta
    n_pages = (dst0 + T + c.page_size - 1) // c.page_size
    num_pages = n_pages + 5
    bt_h, bt_d = _bt(rng, n_pages, num_pages)
    dt = torch.bfloat16 if c.elem_dtype == "bf16" else torch.float32
    pool = par.make_pool(c, L, num_pages, dt)
    ctx = kam.Context(par.layout_of(c, L, style), pool)
    for key, val in (options or {}).items():
        ctx.kam_set_option(key, val)
    chunk, patch = par.upload_chunk(ch, shared_u=shared_u, rank_per_layer=rank_per_layer)
    if patch is not None:
        patch.c.frame = frame
        if rank_per_layer is not None:
            patch._rpl = (B.i32 * L)(*rank_per_layer)
            patch.c.rank_per_layer = patch._rpl
    ctx.kam_relocate_patch(bt_d, dst0, chunk, p_target, patch, m, layout=ctx.layout)
    torch.cuda.synchronize()
    st = par.check_relocated(c, pool, ch, bt_h, dst0, p_target, m, style=style, frame=frame,
                             rank_per_layer=rank_per_layer, shared_u=shared_u, elem=c.elem_dtype)
    stats = ctx.kam_get_stats()
    st["generic_launches"], st["device_errors"] = stats["generic_launches"], stats["device_errors"]
    assert stats["kernels_launched"] == 1 and stats["device_errors"] == 0
    assert par.untouched_pages_intact(pool, bt_h, L)
    # rows of the first/last page outside [dst0, dst0+T) must still hold the sentinel (slot mapping is exact)
    P = c.page_size
    if dst0 > 0:
        head = par.pool_rows(pool.k_layers[0], bt_h, 0, dst0)
        assert np.all(head == par.SENTINEL)
    tail_n = n_pages * P - (dst0 + T)
    if tail_n:
        tail = par.pool_rows(pool.k_layers[0], bt_h, dst0 + T, tail_n)
        assert np.all(tail == par.SENTINEL)
    ctx.close()
    return st


# ---------------------------------------------------------------------------------------------- config 1 (tiny MHA)
def test_config1_fp32_as_written():
    """BASELINE.json configs[0]: fp32 K/V/U/W, rank 4, one chunk of 256 tokens, p uniform in [0, 4096).  fp32 tensors are the
    element-wise kernel's job (the tiled kernel moves bf16)."""
    st = _run_single(CONFIGS[1], 1, 256, 4)
    assert st["fail"] == 0 and st["generic_launches"] == 1


def test_config1_bf16_elements():
    st = _run_single(CONFIGS[1], 1, 256, 4, elem="bf16")
    assert st["fail"] == 0 and st["within_1ulp"] >= 0.999 * st["n"]


def test_config1_all_bf16_rank4_runs_on_the_tiled_kernel():
    """Rank 4 is padded to one 16-wide rank tile in shared memory (zero U columns, zero W rows): no fallback kernel."""
    st = _run_single(CONFIGS[1], 1, 256, 4, elem="bf16", factor="bf16")
    assert st["fail"] == 0 and st["generic_launches"] == 0


# ---------------------------------------------------------------------------------------------- config 2 (GQA)
def test_config2_batch_of_8_chunks():
    """8 chunks of 1024 tokens relocated in ONE launch to offsets in [0, 32768), rank 16, 3 of the 28 layers."""
    cfg = CONFIGS[2]; L, T, m, n = 3, cfg.chunk_tokens, cfg.rank, cfg.chunks_per_step
    rng = _rng(cfg)
    chunks = [make_chunk(cfg, rng, n_layers=L) for _ in range(n)]
    p = make_offsets(cfg, rng, n)
    ppc = T // cfg.page_size
    bt_h, bt_d = _bt(rng, n * ppc, n * ppc + 7)
    pool = par.make_pool(cfg, L, n * ppc + 7, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    up = [par.upload_chunk(c) for c in chunks]
    ctx.kam_relocate_patch_batch([(bt_d, i * T, up[i][0], int(p[i]), up[i][1], m) for i in range(n)])
    torch.cuda.synchronize()
    tot = {}
    for i in range(n):
        st = par.check_relocated(cfg, pool, chunks[i], bt_h, i * T, int(p[i]), m)
        for k, v in st.items():
            tot[k] = tot.get(k, 0) + v
    assert tot["fail"] == 0 and tot["within_1ulp"] >= 0.9999 * tot["n"]
    assert par.untouched_pages_intact(pool, bt_h, L)
    assert ctx.kam_get_stats()["kernels_launched"] == 1
    ctx.close()


@pytest.mark.parametrize("T,dst0", [(1000, 0), (1024, 5), (17, 30), (1, 15), (16, 16)])
def test_config2_ragged_and_unaligned(T, dst0):
    st = _run_single(CONFIGS[2], 2, T, 16, dst0=dst0, salt=T + dst0)
    assert st["fail"] == 0


def test_zero_tokens_is_a_noop():
    cfg = CONFIGS[2]
    pool = par.make_pool(cfg, 1, 4, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    ch = make_chunk(cfg, _rng(cfg), n_tokens=16, n_layers=1)
    chunk, patch = par.upload_chunk(ch)
    chunk.c.n_tokens = 0
    ctx.kam_relocate_patch(torch.zeros(4, dtype=torch.int32, device="cuda"), 0, chunk, 5, patch, 16)
    torch.cuda.synchronize()
    assert par.untouched_pages_intact(pool, [], 1)
    assert ctx.kam_get_stats()["kernels_launched"] == 0
    ctx.close()


@pytest.mark.parametrize("m", [0, 16, 32, 48, 64, 4, 8, 24, 40, 5, 63, 1])
def test_rank_sweep(m):
    """Every rank in [0, 64] runs on the tensor-core tiled kernel ("rank-invariant in latency"; P:216 / P:297 free-form
    ranks per layer): multiples of 16 directly, anything else padded to the next multiple in shared memory.  323 tokens: a
    ragged last tile, whose U rows of an odd rank end off a 16-byte boundary."""
    st = _run_single(CONFIGS[2], 2, 323, m, salt=m)
    assert st["fail"] == 0 and st["generic_launches"] == 0


@pytest.mark.parametrize("m,kw", [(16, {}), (32, dict(style=B.KAM_ROPE_INTERLEAVED)), (40, dict(frame=B.KAM_PATCH_CANONICAL_FRAME)),
                                  (64, dict(shared_u=True)), (64, dict(rank_per_layer=[64, 0, 24])), (0, {})])
def test_kv_split_geometry(m, kw):
    """The tile form ranks 48 / 64 select on their own (a tile carries K rows OR V rows, so only one of W_k / W_v is resident),
    forced here for every rank, both pair styles, both frames, shared U and mixed per-layer ranks; ragged tail, unaligned start."""
    L = 3 if "rank_per_layer" in kw else 2
    st = _run_single(CONFIGS[2], L, 1000, m, dst0=7, salt=100 + m, options={"reloc_kv_split": 2}, **kw)
    assert st["fail"] == 0 and st["generic_launches"] == 0
    if m >= 48:                                                  # and with the head group forced down: slices of one head
        st = _run_single(CONFIGS[2], L, 200, m, salt=300 + m, options={"reloc_kv_split": 2, "reloc_head_group": 1}, **kw)
        assert st["fail"] == 0


def test_free_form_ranks_shared_u_and_mha():
    cfg = CONFIGS[2]
    assert _run_single(cfg, 2, 200, 4, shared_u=True, salt=41)["generic_launches"] == 0       # [T][4] bf16: 8 bytes per token
    assert _run_single(cfg, 4, 200, 24, rank_per_layer=[4, 8, 24, 0], salt=42)["generic_launches"] == 0
    assert _run_single(CONFIGS[4], 1, 100, 4, salt=43)["generic_launches"] == 0              # MHA 32 heads: 4-head slices of U
    assert _run_single(CONFIGS[3], 2, 300, 12, salt=44)["generic_launches"] == 0             # MLA, one latent head


def test_block_table_entry_outside_the_pool_is_skipped_and_counted():
    """A block-table entry >= num_pages (or negative) is never dereferenced: its 16 tokens are skipped in every layer, the
    other pages are written as usual, no page outside the table is touched, and kam_stats.device_errors counts the entry once.
    Tiled kernel (stateless and in place) and the element-wise kernel (fp32 layout)."""
    for elem, factor in (("bf16", "bf16"), ("f32", "f32")):
        cfg = CONFIGS[2].scaled(elem_dtype=elem, factor_dtype=factor)
        L, T, m = 2, 96, 16
        rng = _rng(cfg, 77)
        ch = make_chunk(cfg, rng, n_tokens=T, n_layers=L, rank=m)
        n_pages = T // cfg.page_size
        bt_h, _ = _bt(rng, n_pages, 16)
        bad = bt_h.copy()
        bad[2] = 16 if elem == "bf16" else -3                       # one entry outside [0, 16)
        pool = par.make_pool(cfg, L, 16, torch.bfloat16 if elem == "bf16" else torch.float32)
        ctx = kam.Context(par.layout_of(cfg, L), pool)
        chunk, patch = par.upload_chunk(ch)
        ctx.kam_relocate_patch(torch.from_numpy(bad).cuda(), 0, chunk, 999, patch, m)
        torch.cuda.synchronize()
        st = ctx.kam_get_stats()
        assert st["device_errors"] == 1 and st["generic_launches"] == (0 if elem == "bf16" else 1)
        good_pages = [int(p) for i, p in enumerate(bt_h) if i != 2]
        assert par.untouched_pages_intact(pool, good_pages, L)      # incl. the page the valid table would have named
        for l in range(L):                                          # the five good pages hold Eq. 1
            ko, vo, Sk, Sv = par.oracle_layer(cfg, ch, l, 999)
            rows = np.r_[0:32, 48:96]
            got = np.concatenate([par.pool_rows(pool.k_layers[l], bt_h, 0, 32), par.pool_rows(pool.k_layers[l], bt_h, 48, 48)])
            cmp = par.compare_bf16 if elem == "bf16" else par.compare_f32
            assert cmp(got, ko[rows], Sk[rows], m, "K")["fail"] == 0
        if elem == "bf16":                                          # in place over the same table: the bad page is skipped again
            before = par.pool_rows(pool.k_layers[0], bt_h, 0, 32)
            ctx.kam_rotate_inplace(torch.from_numpy(bad).cuda(), 0, T, -7)
            torch.cuda.synchronize()
            assert ctx.kam_get_stats()["device_errors"] == 2
            want = reuse.relocate(before, -7, **par.rope_kw(cfg))
            assert par.compare_bf16(par.pool_rows(pool.k_layers[0], bt_h, 0, 32), want, par.abs_sum_k(before, -7, None, None, cfg), 0, "in place")["fail"] == 0
            assert par.untouched_pages_intact(pool, good_pages, L)
        ctx.close()


@pytest.mark.parametrize("delta", [0, 1, -1280, 131071, -131071, 32767])
def test_offsets_including_negative_and_huge(delta):
    """fp64 angles: a position of 1e5 must not cost accuracy (an fp32 angle would be off by ~2 bf16 ulp)."""
    st = _run_single(CONFIGS[2], 1, 128, 16, delta=delta, salt=abs(delta) % 97)
    assert st["fail"] == 0


def test_interleaved_pairs_canonical_frame_shared_u_and_layer_sparse():
    cfg = CONFIGS[2]
    assert _run_single(cfg, 2, 200, 16, style=B.KAM_ROPE_INTERLEAVED, salt=1)["fail"] == 0
    assert _run_single(cfg, 2, 200, 16, frame=B.KAM_PATCH_CANONICAL_FRAME, salt=2)["fail"] == 0
    assert _run_single(cfg, 2, 200, 16, style=B.KAM_ROPE_INTERLEAVED, frame=B.KAM_PATCH_CANONICAL_FRAME, salt=3)["fail"] == 0
    assert _run_single(cfg, 2, 200, 32, shared_u=True, salt=4)["fail"] == 0              # paper's per-layer U (R-6)
    assert _run_single(cfg, 4, 200, 16, rank_per_layer=[0, 0, 16, 16], salt=5)["fail"] == 0   # deep-half patch


def test_copy_identities():
    """delta = 0, m = 0 is a bit-exact copy; with m = 0 V is bit-identical for any delta."""
    cfg = CONFIGS[2]; L, T = 2, 160
    rng = _rng(cfg, 9)
    ch = make_chunk(cfg, rng, n_tokens=T, n_layers=L, rank=0)
    bt_h, bt_d = _bt(rng, T // 16, 16)
    pool = par.make_pool(cfg, L, 16, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    chunk, _ = par.upload_chunk(ch)
    ctx.kam_relocate_patch(bt_d, 0, chunk, 0, None, 0)
    torch.cuda.synchronize()
    for l in range(L):
        assert np.array_equal(bf16_bits(par.pool_rows(pool.k_layers[l], bt_h, 0, T)), bf16_bits(par.to_f64(ch["K"][l])))
        assert np.array_equal(bf16_bits(par.pool_rows(pool.v_layers[l], bt_h, 0, T)), bf16_bits(par.to_f64(ch["V"][l])))
    ctx.kam_relocate_patch(bt_d, 0, chunk, 4097, None, 0)
    torch.cuda.synchronize()
    for l in range(L):
        assert np.array_equal(bf16_bits(par.pool_rows(pool.v_layers[l], bt_h, 0, T)), bf16_bits(par.to_f64(ch["V"][l])))
    ctx.close()


# ---------------------------------------------------------------------------------------------- config 3 (MLA)
def test_config3_mla_all_permutations():
    """4 cached chunks, every permutation places chunk pi(i) at p = 1024 i with ONE stored patch per chunk.
    The latent (first 512 columns) is position-free: rank-0 relocation leaves it bit-identical.  The result for
    a given (chunk, offset) pair must be bit-identical whichever permutation produced it (T10)."""
    cfg = CONFIGS[3]; L, T, m, P = 2, cfg.chunk_tokens, cfg.rank, cfg.page_size
    rng = _rng(cfg)
    chunks = [make_chunk(cfg, rng, n_layers=L) for _ in range(4)]
    up = [par.upload_chunk(c) for c in chunks]
    perms = list(itertools.permutations(range(4)))
    ppc = T // P
    n_pages = len(perms) * 4 * ppc
    bt_h, bt_d = _bt(rng, n_pages, n_pages + 3)
    pool = par.make_pool(cfg, L, n_pages + 3, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    descs = []
    for pi, perm in enumerate(perms):
        for slot, c in enumerate(perm):
            descs.append((bt_d, (pi * 4 + slot) * T, up[c][0], 1024 * slot, up[c][1], m))
    ctx.kam_relocate_patch_batch(descs)                          # 96 relocations, one launch
    torch.cuda.synchronize()
    seen = {}
    checked = 0
    for pi, perm in enumerate(perms):
        for slot, c in enumerate(perm):
            rows = [par.pool_rows(pool.k_layers[l], bt_h, (pi * 4 + slot) * T, T) for l in range(L)]
            key = (c, slot)
            if key not in seen:
                seen[key] = rows
                st = par.check_relocated(cfg, pool, chunks[c], bt_h, (pi * 4 + slot) * T, 1024 * slot, m)
                assert st["fail"] == 0
                checked += 1
            else:
                for a, b in zip(seen[key], rows):
                    assert np.array_equal(a, b)
    assert checked == 16
    # rank-0: latent untouched bit for bit, rope band rotated
    ctx.kam_relocate_patch(bt_d, 0, up[0][0], 2048, None, 0)
    torch.cuda.synchronize()
    got = par.pool_rows(pool.k_layers[0], bt_h, 0, T)
    src = par.to_f64(chunks[0]["K"][0])
    assert np.array_equal(got[..., :512], src[..., :512]) and not np.array_equal(got[..., 512:], src[..., 512:])
    ctx.close()


# ---------------------------------------------------------------------------------------------- configs 4 / 5 shapes
def test_config4_shape_relocate_and_inplace_slide():
    """MHA 32 heads: recall by relocate+patch (m=16), then survivors rotate in place by delta = -1280, twice;
    each in-place step is checked against the oracle started from the GPU's own previous pool state (R-10)."""
    cfg = CONFIGS[4]; L, T, m = 1, cfg.chunk_tokens, cfg.rank
    rng = _rng(cfg)
    ch = make_chunk(cfg, rng, n_layers=L)
    bt_h, bt_d = _bt(rng, T // 16 + 2, T // 16 + 6)
    pool = par.make_pool(cfg, L, T // 16 + 6, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    chunk, patch = par.upload_chunk(ch)
    ctx.kam_relocate_patch(bt_d, 16, chunk, 3072, patch, m)
    torch.cuda.synchronize()
    assert par.check_relocated(cfg, pool, ch, bt_h, 16, 3072, m)["fail"] == 0
    v_before = par.pool_rows(pool.v_layers[0], bt_h, 16, T)
    for _ in range(2):
        before = par.pool_rows(pool.k_layers[0], bt_h, 16, T)
        ctx.kam_rotate_inplace(bt_d, 16, T, -1280)
        torch.cuda.synchronize()
        after = par.pool_rows(pool.k_layers[0], bt_h, 16, T)
        want = reuse.relocate(before, -1280, **par.rope_kw(cfg))
        S = par.abs_sum_k(before, -1280, None, None, cfg)
        assert par.compare_bf16(after, want, S, 0, "in-place")["fail"] == 0
    assert np.array_equal(par.pool_rows(pool.v_layers[0], bt_h, 16, T), v_before)       # V is not touched
    assert par.untouched_pages_intact(pool, bt_h, L)
    ctx.close()


def test_config5_shape_rank32():
    st = _run_single(CONFIGS[5], 1, 2048, 32, delta=131072 - 2048 - 1)
    assert st["fail"] == 0


def test_rank0_equals_rotate_inplace_path():
    """T5: relocating with m = 0 and rotating a verbatim copy in place give the same bits."""
    cfg = CONFIGS[2]; L, T = 1, 96
    rng = _rng(cfg, 21)
    ch = make_chunk(cfg, rng, n_tokens=T, n_layers=L, rank=0)
    bt_h, bt_d = _bt(rng, 12, 12)
    pool = par.make_pool(cfg, L, 12, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    chunk, _ = par.upload_chunk(ch)
    ctx.kam_relocate_patch(bt_d, 0, chunk, 777, None, 0)         # pages 0..5: rotated on the way in
    ctx.kam_relocate_patch(bt_d, 96, chunk, 0, None, 0)          # pages 6..11: verbatim copy ...
    ctx.kam_rotate_inplace(bt_d, 96, T, 777)                     # ... rotated where it sits
    torch.cuda.synchronize()
    a = par.pool_rows(pool.k_layers[0], bt_h, 0, T); b = par.pool_rows(pool.k_layers[0], bt_h, 96, T)
    assert np.array_equal(a, b)
    ctx.close()


def test_invalid_arguments_are_rejected_before_any_launch():
    cfg = CONFIGS[2]
    pool = par.make_pool(cfg, 1, 4, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    ch = make_chunk(cfg, _rng(cfg), n_tokens=16, n_layers=1)
    chunk, patch = par.upload_chunk(ch)
    bt = torch.zeros(4, dtype=torch.int32, device="cuda")
    for kwargs in (dict(rank=65), dict(rank=-1)):
        with pytest.raises(kam.KameraError) as e:
            ctx.kam_relocate_patch(bt, 0, chunk, 0, patch, **kwargs)
        assert e.value.status == B.KAM_ERR_INVALID_ARG
    with pytest.raises(kam.KameraError):
        ctx.kam_relocate_patch(None, 0, chunk, 0, patch, 16)
    with pytest.raises(kam.KameraError):
        ctx.kam_relocate_patch(bt, -1, chunk, 0, patch, 16)
    with pytest.raises(kam.KameraError) as e:                     # token range beyond int32
        ctx.kam_relocate_patch(bt, 2 ** 31 - 8, chunk, 0, patch, 16)
    assert e.value.status == B.KAM_ERR_INVALID_ARG
    with pytest.raises(kam.KameraError) as e:                     # a layout that is not the context's
        ctx.kam_relocate_patch(bt, 0, chunk, 0, patch, 16, layout=par.layout_of(CONFIGS[5], 1))
    assert e.value.status == B.KAM_ERR_INVALID_ARG
    assert ctx.kam_get_stats()["kernels_launched"] == 0
    assert par.untouched_pages_intact(pool, [], 1)
    ctx.close()
