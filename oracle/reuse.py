"""Eq. 1 of the paper, step by step, in fp64 (test infrastructure; see oracle/__init__.py).

    KV^(B|A) = R(delta) . KV(B|0)  +  U_m V_m^T                      (Eq. 1)
               relocate (exact)       rank-m patch (conditioning)

"Relocate: re-rotate B's keys by delta = p1 - p0. Because RoPE composes,
R(delta)R(p0) = R(p1) exactly; V is untouched.".  "MLA ... relocation only
re-rotates the 64-dim decoupled k_pe ... GQA ... relocate the full key ... patch both
K and V per KV-head. MHA is GQA with one KV head per query head".
Serve step (`apply_reuse`): rotate the rope band by delta, K += U.K @ V.K^T,
V += U.V @ V.V^T, assemble into the paged KV cache.

Array conventions (one layer):
  k, v   [T, H, D]   rows of one chunk (H KV heads; MLA: H = 1, D = 576, no v)
  U      [T, H, m]   left factors with the singular values folded in
  W      [H, m, D]   the paper's V_m^T, per KV head (BASELINE.json: "per layer and KV head")
  pool   [num_pages, P, H, D]  paged KV pool of one layer, as bf16 bit patterns (uint16)
         or as float32 (config 1's fp32 variant)

Readings of the paper used here are listed in DESIGN.md (R-1 ... R-12).
"""
import numpy as np

from .bf16 import bf16_bits

HALF, INTERLEAVED = 0, 1                     # RoPE pair layout (reading R-1)
TARGET_FRAME, CANONICAL_FRAME = 0, 1         # where the K patch lives (reading R-4)


def rope_frequencies(theta, d_r):
    """O1: f_i = theta^(-2i/d_r), i = 0 .. d_r/2-1  (RoFormer's schedule, cited at P:52)."""
    return np.array([float(theta) ** (-2.0 * i / d_r) for i in range(d_r // 2)], dtype=np.float64)


def rope_pair_columns(style, rope_off, d_r):
    """O2: the two columns rotated together by frequency i."""
    i = np.arange(d_r // 2)
    if style == HALF:
        return rope_off + i, rope_off + i + d_r // 2
    if style == INTERLEAVED:
        return rope_off + 2 * i, rope_off + 2 * i + 1
    raise ValueError("unknown rope style")


def relocate(k, delta, theta, rope_off, d_r, style=HALF):
    """O3: R(delta) on the rope band of every row of k; other columns copied.

    The rotation angle of pair i is delta * f_i for EVERY token of the chunk: the stored
    keys already carry their intra-chunk phase, and M-RoPE coordinates advance together
    (P:66), so relocation is one uniform phase advance (reading R-3).
    """
    k = np.array(k, dtype=np.float64, copy=True)
    phi = float(int(delta)) * rope_frequencies(theta, d_r)
    c, s = np.cos(phi), np.sin(phi)
    ia, ib = rope_pair_columns(style, rope_off, d_r)
    a, b = k[..., ia].copy(), k[..., ib].copy()
    k[..., ia] = a * c - b * s
    k[..., ib] = a * s + b * c
    return k


def patch_term(U, W):
    """U_m V_m^T per KV head: [T,H,m] x [H,m,D] -> [T,H,D]  (one GEMM per head)."""
    return np.einsum("thj,hjc->thc", np.asarray(U, np.float64), np.asarray(W, np.float64))


def reuse_k(k, delta, Uk, Wk, theta, rope_off, d_r, style=HALF, frame=TARGET_FRAME):
    """O3+O4 for keys: Eq. 1 in fp64, no rounding.  Uk/Wk None or rank 0 => pure rotation."""
    k = np.asarray(k, np.float64)
    has_patch = Uk is not None and np.asarray(Uk).shape[-1] > 0
    if has_patch and frame == CANONICAL_FRAME:       # patch stored in the chunk's own frame
        k = k + patch_term(Uk, Wk)
    k = relocate(k, delta, theta, rope_off, d_r, style)
    if has_patch and frame == TARGET_FRAME:          # Eq. 1 literally: rotate, then add
        k = k + patch_term(Uk, Wk)
    return k


def reuse_v(v, Uv, Wv):
    """O4 for values: V is untouched by relocation; only the patch is added."""
    v = np.array(v, dtype=np.float64, copy=True)
    if Uv is not None and np.asarray(Uv).shape[-1] > 0:
        v = v + patch_term(Uv, Wv)
    return v


def slot_mapping(block_table, dst_token_start, n_tokens, page_size):
    """O5: logical token g = dst_token_start + t -> (physical page, slot in page)."""
    g = int(dst_token_start) + np.arange(int(n_tokens), dtype=np.int64)
    page = np.asarray(block_table, dtype=np.int64)[g // page_size]
    return page, g % page_size


def scatter(pool, block_table, dst_token_start, rows):
    """O5: one rounding (fp64 -> pool dtype) and the paged store.  pool is modified in place."""
    T = rows.shape[0]
    page, slot = slot_mapping(block_table, dst_token_start, T, pool.shape[1])
    if pool.dtype == np.uint16:
        pool[page, slot] = bf16_bits(rows)
    elif pool.dtype == np.float32:
        pool[page, slot] = rows.astype(np.float32)
    else:
        raise TypeError("pool must be uint16 (bf16 bits) or float32")


def relocate_patch_layer(pool_k, pool_v, block_table, dst_token_start, k, v, delta,
                         Uk, Wk, Uv, Wv, theta, rope_off, d_r, style=HALF, frame=TARGET_FRAME):
    """One layer of `apply_reuse` written into the paged pool.  v/pool_v None for MLA."""
    scatter(pool_k, block_table, dst_token_start,
            reuse_k(k, delta, Uk, Wk, theta, rope_off, d_r, style, frame))
    if v is not None:
        scatter(pool_v, block_table, dst_token_start, reuse_v(v, Uv, Wv))


def gather(pool, block_table, token_start, n_tokens):
    """Rows [n_tokens, H, D] currently in the pool, as fp64."""
    from .bf16 import bf16_from_bits
    page, slot = slot_mapping(block_table, token_start, n_tokens, pool.shape[1])
    rows = pool[page, slot]
    return bf16_from_bits(rows) if pool.dtype == np.uint16 else rows.astype(np.float64)


def rotate_inplace_layer(pool_k, block_table, token_start, n_tokens, delta, theta, rope_off, d_r,
                         style=HALF):
    """O6: a survivor's keys re-rotated where they sit ("survivors cost only R(delta)").
    Read pool -> fp64 -> rotate -> round -> same slots.  V is not read."""
    rows = gather(pool_k, block_table, token_start, n_tokens)
    scatter(pool_k, block_table, token_start, relocate(rows, delta, theta, rope_off, d_r, style))


def form_patch(kv_cond, kv_solo_relocated, m):
    """O10: Delta = KV(B|A) - R(delta)KV(B|0) per head; top-m SVD; S folded into U.

    kv_* are [T, H, D]; returns U [T, H, m], W [H, m, D], and the singular values [H, min(T,D)].
    """
    delta = np.asarray(kv_cond, np.float64) - np.asarray(kv_solo_relocated, np.float64)
    T, H, D = delta.shape
    U = np.zeros((T, H, m)); W = np.zeros((H, m, D)); S = np.zeros((H, min(T, D)))
    for h in range(H):
        u, s, vt = np.linalg.svd(delta[:, h, :], full_matrices=False)
        U[:, h, :] = u[:, :m] * s[:m]
        W[h] = vt[:m]
        S[h] = s
    return U, W, S
