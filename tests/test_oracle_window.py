"""Pins for oracle/window.py: brute-force rebuilds and invariants of the deque/page model."""
import random

import pytest

from oracle.window import BACK, FRONT, WindowStore


def _check_invariants(ws, num_pages):
    owned = [p for r in ws.req.values() for c in r["chunks"] for p in c.pages]
    assert len(owned) == len(set(owned)), "page owned twice"
    assert sorted(owned + ws.free) == list(range(num_pages)), "pages leaked or duplicated"


def test_first_pops_are_0_1_2_and_logical_order():
    ws = WindowStore(32, 16)
    ws.open(0, window_base=100)
    h, pages, p, rot = ws.admit(0, BACK, 48)
    assert (h, pages, p, rot) == (0, [0, 1, 2], 100, [])
    h, pages, p, rot = ws.admit(0, BACK, 32)
    assert (h, pages, p, rot) == (1, [3, 4], 148, [])
    e = ws.export(0)
    assert e["block_table"] == [0, 1, 2, 3, 4]
    assert e["chunk_starts"] == [0, 48, 80] and e["chunk_offsets"] == [0, 0]
    assert e["slot_mapping"][47] == 2 * 16 + 15 and e["slot_mapping"][48] == 3 * 16


def test_evict_then_readmit_restores_identical_table():
    ws = WindowStore(64, 16)
    ws.open(0)
    for _ in range(3):
        ws.admit(0, BACK, 64)
    before = ws.export(0)
    _, pages, _ = ws.evict(0, BACK)
    _, pages2, _, _ = ws.admit(0, BACK, 64)
    assert pages2 == pages and ws.export(0)["block_table"] == before["block_table"]
    _, pages, _ = ws.evict(0, FRONT, materialize=0)
    _, pages2, _, _ = ws.admit(0, FRONT, 64, materialize=0)
    assert pages2 == pages and ws.export(0)["block_table"] == before["block_table"]
    assert ws.export(0)["chunk_offsets"] == [0, 0, 0]


def test_front_evict_shifts_survivors_by_minus_Te():
    """Config 4: window of 3 x 1280 behind a pinned 512-token prefix; survivors get delta = -1280."""
    ws = WindowStore(1024, 16)
    ws.open(0)
    ws.admit(0, BACK, 512)
    ws.pin(0, 1)
    hs = [ws.admit(0, BACK, 1280)[0] for _ in range(3)]
    assert ws.positions(0) == [0, 512, 1792, 3072]
    h, _, rot = ws.evict(0, FRONT, materialize=1)
    assert h == hs[0] and rot == [(hs[1], -1280), (hs[2], -1280)]       # prefix does not move
    assert ws.positions(0) == [0, 512, 1792]
    h4, _, p, rot = ws.admit(0, BACK, 1280)
    assert p == 3072 and rot == []
    # lazy mode: nothing rotates, the offsets accumulate instead
    ws.evict(0, FRONT, materialize=0)
    assert ws.export(0)["chunk_offsets"] == [0, -1280, -1280]
    ws.evict(0, FRONT, materialize=0)
    assert ws.export(0)["chunk_offsets"] == [0, -2560]
    # a later materialising op settles the whole pending delta at once
    _, _, _, rot = ws.admit(0, BACK, 1280, materialize=1)
    assert rot == [(h4, -2560)] and ws.export(0)["chunk_offsets"] == [0, 0, 0]


def test_front_admit_shifts_survivors_by_plus_Ta_and_back_ops_move_nothing():
    ws = WindowStore(256, 16)
    ws.open(3, window_base=1000)
    a = ws.admit(3, BACK, 160)[0]
    b, _, p, rot = ws.admit(3, FRONT, 320)
    assert p == 1000 and rot == [(a, +320)]
    _, _, rot = ws.evict(3, BACK)
    assert rot == [] and ws.export(3)["handles"] == [b]


def test_errors_leave_state_unchanged():
    ws = WindowStore(4, 16)
    ws.open(0)
    with pytest.raises(ValueError):
        ws.admit(0, BACK, 17)
    with pytest.raises(MemoryError):
        ws.admit(0, BACK, 16 * 5)
    with pytest.raises(IndexError):
        ws.evict(0, FRONT)
    assert ws.free == [3, 2, 1, 0] and ws.export(0)["block_table"] == []


def test_random_ops_against_a_from_scratch_rebuild():
    """Brute force: an independent flat log of (req, chunk order) is replayed from scratch after
    every operation; only page identities are shared with the model."""
    rnd = random.Random(5)
    N, P = 512, 16
    ws = WindowStore(N, P)
    shadow = {}                                   # req -> list of (handle, n_tokens, pages)
    for r in range(3):
        ws.open(r, window_base=10 * r); shadow[r] = []
    for step in range(600):
        r = rnd.randrange(3)
        end = rnd.choice((FRONT, BACK))
        if shadow[r] and rnd.random() < 0.45:
            h, pages, _ = ws.evict(r, end, materialize=rnd.randrange(2))
            gone = shadow[r].pop(0 if end == FRONT else -1)
            assert (h, pages) == (gone[0], gone[2])
        else:
            n = P * rnd.randrange(1, 6)
            if n // P > len(ws.free):
                continue
            expect_pages = list(reversed(ws.free[-(n // P):]))
            h, pages, p, _ = ws.admit(r, end, n, materialize=rnd.randrange(2))
            assert pages == expect_pages
            shadow[r].insert(0 if end == FRONT else len(shadow[r]), (h, n, pages))
        _check_invariants(ws, N)
        for rr in range(3):
            e = ws.export(rr)
            bt = [p for _, _, pg in shadow[rr] for p in pg]
            assert e["block_table"] == bt
            assert e["handles"] == [h for h, _, _ in shadow[rr]]
            pos, acc = [], 10 * rr
            for _, n, _ in shadow[rr]:
                pos.append(acc); acc += n
            assert e["positions"] == pos
            tot = sum(n for _, n, _ in shadow[rr])
            assert e["slot_mapping"] == [bt[g // P] * P + g % P for g in range(tot)]
    for r in range(3):
        ws.close(r)
    assert sorted(ws.free) == list(range(N))
