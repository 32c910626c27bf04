"""CPU-side checks of the boundary: the library loads, exports every symbol include/kamera.h declares, validates
arguments, and its host bookkeeping (window deque + free list) matches the oracle model bit for bit.  No compute
call is made here (there is no GPU and the library has no CPU fallback)."""
import ctypes as C
import os
import random
import re

import pytest

import paper_2606_23581_b200 as kam
from paper_2606_23581_b200 import binding as B
from oracle.window import BACK, FRONT, WindowStore

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _layout(**kw):
    a = dict(kind=B.KAM_GQA, n_layers=2, n_q_heads=8, n_kv_heads=4, row_dim=128, rope_off=0, rope_dim=128, has_v=True,
             page_size=16, rope_theta=1e6)
    a.update(kw)
    return kam.make_layout(**a)


def test_every_declared_symbol_is_exported_and_bound():
    hdr = open(os.path.join(ROOT, "include", "kamera.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(kam_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.SIGNATURES), declared ^ set(B.SIGNATURES)
    lib = kam.lib()
    for name in declared:
        assert hasattr(lib, name)
    assert b"sm_100a" in lib.kam_version()


def test_struct_sizes_match_the_header_layout():
    assert C.sizeof(B.kam_layout) == 13 * 4 + 4 + 8          # 13 int32, padding, double
    assert C.sizeof(B.kam_pool) == 24 and C.sizeof(B.kam_chunk) == 32
    assert C.sizeof(B.kam_patch) == 64 and C.sizeof(B.kam_reloc_desc) == 48 and C.sizeof(B.kam_patch_ref) == 56


def test_create_rejects_bad_layouts():
    for bad in (dict(n_layers=0), dict(n_q_heads=7), dict(row_dim=12), dict(rope_dim=3), dict(rope_off=64),
                dict(page_size=0), dict(rope_theta=0.0), dict(n_layers=129)):
        with pytest.raises(kam.KameraError) as e:
            kam.Context(_layout(**bad), None, 1, 1, 1)
        assert e.value.status == B.KAM_ERR_INVALID_ARG


def test_compute_entries_fail_loudly_without_cuda():
    ctx = kam.Context(_layout(), None, 2, 4, 8)
    # no pool, no device: the stateless operator must refuse, not fall back
    ch = B.kam_chunk(None, None, 16, 0)
    st = kam.lib().kam_relocate_patch(ctx.h, None, None, 0, C.byref(ch), 0, None, 0, None)
    assert st == B.KAM_ERR_INVALID_ARG
    st = kam.lib().kam_rotate_inplace(ctx.h, None, None, 0, 16, 5, None)
    assert st == B.KAM_ERR_INVALID_ARG and b"pool" in kam.lib().kam_last_error(ctx.h)
    # the newer entries too: valid-looking arguments, but no device -> KAM_ERR_CUDA (never a CPU computation)
    fake = (B.vp * 1)(0x1000)
    st = kam.lib().kam_form_patch(ctx.h, C.cast(fake, B.vp), C.cast(fake, B.vp), 16, 0, 1, 16, 0, C.cast(fake, B.vp), C.cast(fake, B.vp), None, None)
    assert st == B.KAM_ERR_CUDA and b"no CPU fallback" in kam.lib().kam_last_error(ctx.h)
    st = kam.lib().kam_lse_merge_states(ctx.h, 1, fake, fake, 2, B.vp(0x1000), B.vp(0x1000), None)
    assert st == B.KAM_ERR_CUDA
    assert kam.lib().kam_lse_merge_states(ctx.h, 17, fake, fake, 2, B.vp(0x1000), B.vp(0x1000), None) == B.KAM_ERR_INVALID_ARG
    assert kam.lib().kam_decode_set_max_patch_rank(ctx.h, 48) == B.KAM_ERR_INVALID_ARG
    assert kam.lib().kam_decode_set_max_patch_rank(ctx.h, 32) == B.KAM_OK


def _chunk(n):
    return B.kam_chunk(None, None, n, 0)


def test_window_errors_leave_state_unchanged():
    ctx = kam.Context(_layout(), None, 2, 3, 4)               # 2 req x 3 chunks x 4 pages = 24 pages
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_admit(0, BACK, _chunk(16))
    assert e.value.status == B.KAM_ERR_STATE                  # not open
    ctx.kam_window_open(0, 7)
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_window_open(0, 7)
    assert e.value.status == B.KAM_ERR_STATE
    for bad_n in (17, 0, 16 * 5):                             # not a page multiple / empty / more pages than a chunk may hold
        with pytest.raises(kam.KameraError) as e:
            ctx.kam_admit(0, BACK, _chunk(bad_n))
        assert e.value.status == B.KAM_ERR_INVALID_ARG
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_admit(0, BACK, _chunk(16), rank=65)
    assert e.value.status == B.KAM_ERR_INVALID_ARG
    with pytest.raises(kam.KameraError) as e:
        ctx.kam_evict(0, FRONT)
    assert e.value.status == B.KAM_ERR_STATE
    s = ctx.kam_get_stats()
    assert s["pages_free"] == 24 and s["chunks_live"] == 0 and s["table_entries_written"] == 0
    assert ctx.kam_window_export(0)["block_table"] == []
    for _ in range(3):
        ctx.kam_admit(0, BACK, _chunk(64))
    with pytest.raises(kam.KameraError) as e:                 # window full
        ctx.kam_admit(0, BACK, _chunk(16))
    assert e.value.status == B.KAM_ERR_STATE


def test_free_list_exhaustion_is_no_pages():
    lay = _layout()
    ctx = kam.Context(lay, None, 1, 4, 2)                     # 8 pages in total
    ctx.kam_window_open(0)
    for _ in range(4):
        ctx.kam_admit(0, BACK, _chunk(32))
    assert ctx.kam_get_stats()["pages_free"] == 0
    ctx.kam_evict(0, FRONT)
    ctx.kam_admit(0, BACK, _chunk(32))
    ctx.kam_evict(0, BACK)
    ctx.kam_evict(0, BACK)
    assert ctx.kam_get_stats()["pages_free"] == 4


def test_window_matches_oracle_model_bit_for_bit_and_is_O1():
    """Random admit/evict at both ends, 3 requests, lazy and materialising: the exported linear view (block table,
    slot mapping, chunk starts, pending offsets, handles) equals oracle/window.py after every operation, and the
    number of page-table entries written per operation is the page count of ONE chunk."""
    rnd = random.Random(2)
    P, R, CH, PPC = 16, 3, 12, 6
    ctx = kam.Context(_layout(), None, R, CH, PPC)
    ws = WindowStore(R * CH * PPC, P)
    for r in range(R):
        ctx.kam_window_open(r, 100 * r); ws.open(r, 100 * r)
    ctx.kam_admit(1, BACK, _chunk(32)); ws.admit(1, BACK, 32)
    ctx.kam_window_pin(1, 1); ws.pin(1, 1)                    # request 1 keeps a pinned prefix
    live = {r: len(ws.req[r]["chunks"]) for r in range(R)}
    for step in range(1500):
        r, end, mat = rnd.randrange(R), rnd.choice((FRONT, BACK)), rnd.randrange(2)
        before = ctx.kam_get_stats()["table_entries_written"]
        if live[r] > ws.req[r]["pinned"] and (rnd.random() < 0.45 or live[r] == CH):
            ctx.kam_evict(r, end, mat); ws.evict(r, end, mat)
            live[r] -= 1
            assert ctx.kam_get_stats()["table_entries_written"] == before
        else:
            n = P * rnd.randrange(1, PPC + 1)
            h = ctx.kam_admit(r, end, _chunk(n), materialize=mat)
            h2, _, _, _ = ws.admit(r, end, n, mat)
            assert h == h2
            live[r] += 1
            assert ctx.kam_get_stats()["table_entries_written"] - before == n // P      # O(1) in the window length
        got, want = ctx.kam_window_export(r), ws.export(r)
        for key in ("block_table", "slot_mapping", "chunk_starts", "chunk_offsets", "handles"):
            assert got[key] == want[key], (step, key)
        assert ctx.kam_get_stats()["pages_free"] == len(ws.free)
    for r in range(R):
        ctx.kam_window_close(r); ws.close(r)
    assert ctx.kam_get_stats()["pages_free"] == R * CH * PPC
