"""Byte accounting of a stored patch (test infrastructure; see oracle/__init__.py).

The paper states the patch size only as ratios: top-m factors "~2 % of the page",
"rank-16 ~ 6 %, rank-64 ~ 25 % of the segment's KV bytes", and as token
equivalents "rank-16 = 31 tokens, rank-64 = 124 tokens" (Table 6).  Those figures fit
ONE factor pair per layer for K and one for V over the concatenated KV-head features
(F = H*D columns) of a segment of n_B tokens - reading R-6 of DESIGN.md:

    factor elements per layer  = 2 * (n_B*m + m*F)         (U and V_m^T, for K and for V)
    segment elements per layer = 2 * n_B * F
    fraction                   = m * (1/F + 1/n_B)
    token equivalents          = fraction * n_B = m * (1 + n_B/F)

BASELINE.json instead fixes per-KV-head factors (U [T,H,m], W [H,m,D]); both accountings are
given so that bench.py can report either.
"""


def shared_u_fraction(m, n_tokens, n_kv_heads, head_dim):
    """Paper-style (one U per layer shared by all heads): factor bytes / segment KV bytes."""
    F = n_kv_heads * head_dim
    return m * (1.0 / F + 1.0 / n_tokens)


def shared_u_token_equivalents(m, n_tokens, n_kv_heads, head_dim):
    return shared_u_fraction(m, n_tokens, n_kv_heads, head_dim) * n_tokens


def per_head_fraction(m, n_tokens, head_dim):
    """BASELINE.json form (U per KV head): (T*H*m + H*m*D) / (T*H*D) = m * (1/D + 1/T)."""
    return m * (1.0 / head_dim + 1.0 / n_tokens)
