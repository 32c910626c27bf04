"""CPU-side checks of the boundary: the library loads, exports every symbol include/kamera.h declares, validates
arguments, and its host bookkeeping (window deque + free list) matches the oracle model bit for bit.  No compute
call is made here (there is no GPU and the library has no CPU fallback)."""
import ctypes as C
import os
import random
import re
import subprocess

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


def test_c_program_against_the_header_agrees_with_the_ctypes_mirror(tmp_path):
    """tests/abi_check.c is compiled with `cc -I include` and linked against libkamera.so: every struct size and field offset
    the C compiler derives from include/kamera.h must equal binding.py's ctypes mirror, the constants must agree, and the
    bookkeeping-only entries (create / set_option / window open / admit / export / slide / stats / destroy) work through the
    header's own prototypes."""
    lib_path = kam.build.build()
    exe = str(tmp_path / "abi_check")
    cc = subprocess.run(["cc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), os.path.join(ROOT, "tests", "abi_check.c"),
                         "-o", exe, lib_path, "-Wl,-rpath," + os.path.dirname(lib_path)], capture_output=True, text=True)
    assert cc.returncode == 0, cc.stdout + cc.stderr
    run = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert run.returncode == 0 and run.stdout.strip().endswith("OK"), run.stdout + run.stderr
    lines = [l.split() for l in run.stdout.splitlines()]
    structs = {n: getattr(B, n) for n in ("kam_layout", "kam_pool", "kam_chunk", "kam_patch", "kam_reloc_desc", "kam_patch_ref", "kam_stats")}
    seen = {n: set() for n in structs}
    for l in lines:
        if l[0] == "sizeof":
            assert C.sizeof(structs[l[1]]) == int(l[2]), l
        elif l[0] == "offsetof":
            assert getattr(structs[l[1]], l[2]).offset == int(l[3]), l
            seen[l[1]].add(l[2])
        elif l[0] in ("const", "enum"):
            assert getattr(B, l[1]) == int(l[2]), l
    for n, st in structs.items():                                   # the C program lists every field the mirror has
        assert seen[n] == {f[0] for f in st._fields_}, n
    exp = [l for l in lines if l[0] == "export"][0]
    # front-admitted 48-token chunk (pages 2,3,4) precedes the 32-token one (pages 0,1); lazily admitted, so the older chunk
    # carries a pending offset of +48
    assert exp[1:] == "n_pages 5 n_chunks 2 bt 2 3 4 0 1 starts 0 48 80 offs 0 48 handles 1 0".split()
    st = [l for l in lines if l[0] == "stats"][0]
    assert st[1:] == "free 61 total 64 written 6 live 2 launched 0".split()


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
    st = kam.lib().kam_relocate_patch(ctx.h, None, None, 0, C.byref(ch), 0, None, 0, None, None)
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
    # a layout argument that differs from the context's is refused (north_star's `layout` is a check, not a dispatch)
    other = _layout(row_dim=64, rope_dim=64)
    st = kam.lib().kam_relocate_patch(ctx.h, None, None, 0, C.byref(ch), 0, None, 0, C.byref(other), None)
    assert st == B.KAM_ERR_INVALID_ARG and b"layout" in kam.lib().kam_last_error(ctx.h)
    # options: known keys in range only; the library reads no environment variable
    ctx.kam_set_option("reloc_kv_split", 2)
    for key, val in (("reloc_kv_split", 3), ("nonsense", 1)):
        with pytest.raises(kam.KameraError) as e:
            ctx.kam_set_option(key, val)
        assert e.value.status == B.KAM_ERR_INVALID_ARG
    srcs = "".join(open(os.path.join(ROOT, "paper_2606_23581_b200", "csrc", f)).read() for f in os.listdir(os.path.join(ROOT, "paper_2606_23581_b200", "csrc")))
    assert "getenv" not in srcs


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
        if live[r] > ws.req[r]["pinned"] and rnd.random() < 0.25:
            # kam_slide = evict (lazy) + admit (materialize) as one call; fails as a whole, before evicting, when it cannot admit
            end2, n = rnd.choice((FRONT, BACK)), P * rnd.randrange(1, PPC + 2)
            if n > P * PPC:
                with pytest.raises(kam.KameraError) as e:
                    ctx.kam_slide(r, end, end2, _chunk(n), materialize=mat)
                assert e.value.status == B.KAM_ERR_INVALID_ARG
                assert ctx.kam_get_stats()["table_entries_written"] == before
            else:
                h = ctx.kam_slide(r, end, end2, _chunk(n), materialize=mat)
                ws.evict(r, end, 0)
                h2, _, _, _ = ws.admit(r, end2, n, mat)
                assert h == h2
                assert ctx.kam_get_stats()["table_entries_written"] - before == n // P
        elif live[r] > ws.req[r]["pinned"] and (rnd.random() < 0.45 or live[r] == CH):
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
