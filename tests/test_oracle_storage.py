"""Pins oracle/storage.py to the only numbers the paper prints about this path (tests/golden/patch_storage.txt)."""
import os

from oracle import storage

GOLD = os.path.join(os.path.dirname(__file__), "golden", "patch_storage.txt")


def test_paper_storage_figures():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 2
    for rank, tok, lo, hi in rows:
        m = int(rank)
        te = storage.shared_u_token_equivalents(m, 480, 4, 128)       # Qwen2.5-VL: F = 4 x 128, n_B = 480 (R-6)
        assert round(te) == int(tok)
        assert float(lo) <= 100 * storage.shared_u_fraction(m, 480, 4, 128) <= float(hi)


def test_per_head_accounting_matches_direct_count():
    T, H, D, m = 1024, 4, 128, 16
    direct = (T * H * m + H * m * D) / (T * H * D)
    assert abs(storage.per_head_fraction(m, T, D) - direct) < 1e-15
    assert abs(direct - 0.140625) < 1e-12                            # config 2: 14 % of page bytes
