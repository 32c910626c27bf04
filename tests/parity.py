"""Shared machinery of the GPU parity tests: runs the CUDA path through the C ABI and the oracle on the same
seeded inputs and compares element by element.  Test infrastructure only.

Tolerance ("Parity bar"; BASELINE.json: "within 1 bf16 ulp of the oracle value rounded to bf16"):
    bf16 pool:  |g - bf16(o)| <= max( ulp_bf16(bf16(o)), (m + 4) * 2^-24 * S )
    fp32 pool:  |g - o|       <= (m + 4) * 2^-24 * S + ulp_fp32(o)
with S = sum of |terms| of the element (|a cos| + |b sin| + sum_j |U_j W_j|).  The second clause of the bf16 rule
is the worst-case fp32 accumulation error of the m + 2 terms; it only matters where the terms cancel to less than
~1e-4 of their size, and the number of elements that needed it is reported.
"""
import numpy as np
import torch

import paper_2606_23581_b200 as kam
from oracle import reuse
from oracle.bf16 import bf16_bits, bf16_from_bits, bf16_rne, ulp_bf16
from paper_2606_23581_b200 import binding as B

SENTINEL = 1248.0          # exactly representable in bf16
# every compare_bf16 call of the session adds its counts here; tests/conftest.py prints the totals at the end of the run, so
# that the second clause of the 1-ulp rule (the fp32-accumulation floor) stays visible: how many elements needed it
TOTALS = {"n": 0, "exact": 0, "within_1ulp": 0, "needed_floor": 0, "fail": 0}


def layout_of(cfg, n_layers=None, style=B.KAM_ROPE_HALF, elem=None, factor=None):
    kind = {"MHA": B.KAM_MHA, "GQA": B.KAM_GQA, "MLA": B.KAM_MLA}[cfg.kind]
    dt = {"bf16": B.KAM_BF16, "f32": B.KAM_F32}
    return kam.make_layout(kind, n_layers or cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, cfg.row_dim, cfg.rope_off,
                           cfg.rope_dim, cfg.has_v, cfg.page_size, cfg.theta, rope_style=style,
                           elem_dtype=dt[elem or cfg.elem_dtype], factor_dtype=dt[factor or cfg.factor_dtype],
                           v_dim=cfg.v_dim)


def rope_kw(cfg, style=reuse.HALF):
    return dict(theta=cfg.theta, rope_off=cfg.rope_off, d_r=cfg.rope_dim, style=style)


def make_pool(cfg, n_layers, num_pages, dtype, device="cuda"):
    shape = (num_pages, cfg.page_size, cfg.n_kv_heads, cfg.row_dim)
    k = [torch.full(shape, SENTINEL, dtype=dtype, device=device) for _ in range(n_layers)]
    v = [torch.full(shape, SENTINEL, dtype=dtype, device=device) for _ in range(n_layers)] if cfg.has_v else None
    return kam.Pool(k, v)


def to_f64(t):
    return t.detach().to("cpu").to(torch.float64).numpy()


def pool_rows(pool_layer, block_table, token_start, n_tokens):
    """Rows [n_tokens, H, D] of one pool layer (torch, on device) as fp64 numpy, through the block table."""
    P = pool_layer.shape[1]
    g = token_start + np.arange(n_tokens)
    page = np.asarray(block_table)[g // P]
    idx = torch.from_numpy(page * P + g % P).to(pool_layer.device)
    flat = pool_layer.reshape(-1, pool_layer.shape[2], pool_layer.shape[3])
    return to_f64(flat[idx])


def abs_sum_k(k, delta, U, W, cfg, style=reuse.HALF):
    """S for keys: |a||cos| + |b||sin| on the band, |k| elsewhere, + |U| |W|."""
    k = np.abs(np.asarray(k, np.float64))
    S = k.copy()
    phi = float(int(delta)) * reuse.rope_frequencies(cfg.theta, cfg.rope_dim)
    c, s = np.abs(np.cos(phi)), np.abs(np.sin(phi))
    ia, ib = reuse.rope_pair_columns(style, cfg.rope_off, cfg.rope_dim)
    S[..., ia] = k[..., ia] * c + k[..., ib] * s
    S[..., ib] = k[..., ia] * s + k[..., ib] * c
    if U is not None and np.asarray(U).shape[-1]:
        S = S + reuse.patch_term(np.abs(U), np.abs(W))
    return S


def abs_sum_v(v, U, W):
    S = np.abs(np.asarray(v, np.float64))
    if U is not None and np.asarray(U).shape[-1]:
        S = S + reuse.patch_term(np.abs(U), np.abs(W))
    return S


def compare_bf16(g, o, S, m, what=""):
    """g: GPU values (fp64 of the stored bf16), o: oracle fp64 (unrounded).  Returns stats; asserts the rule."""
    ob = bf16_rne(o)
    err = np.abs(g - ob)
    ulp = ulp_bf16(ob)
    floor = (m + 4) * 2.0 ** -24 * S
    ok = err <= np.maximum(ulp, floor)
    stats = {"n": int(err.size), "exact": int(np.sum(err == 0)), "within_1ulp": int(np.sum(err <= ulp)),
             "needed_floor": int(np.sum((err > ulp) & ok)), "fail": int(np.sum(~ok))}
    for k_, v_ in stats.items():
        TOTALS[k_] += v_
    if stats["fail"]:
        bad = np.argwhere(~ok)[:5]
        detail = [(tuple(i), g[tuple(i)], ob[tuple(i)], o[tuple(i)]) for i in bad]
        raise AssertionError("%s: %d / %d elements outside 1 bf16 ulp: %s" % (what, stats["fail"], stats["n"], detail))
    return stats


def compare_f32(g, o, S, m, what=""):
    ulp32 = np.ldexp(1.0, np.frexp(np.abs(o))[1] - 24)
    ok = np.abs(g - o) <= (m + 4) * 2.0 ** -24 * S + ulp32
    if not np.all(ok):
        raise AssertionError("%s: %d / %d fp32 elements outside tolerance" % (what, int(np.sum(~ok)), ok.size))
    return {"n": int(ok.size), "fail": 0}


def upload_chunk(ch, device="cuda", shared_u=False, rank_per_layer=None):
    """synth.make_chunk output -> kam.Chunk / kam.Patch over per-layer device tensors.  rank_per_layer: layer l uses the first
    r_l columns of its stored U (strides unchanged) and a contiguous W[l] of r_l rows (kamera.h: W[l] is [H][rank_l][D])."""
    L = ch["K"].shape[0]
    K = [ch["K"][l].to(device).contiguous() for l in range(L)]
    V = [ch["V"][l].to(device).contiguous() for l in range(L)] if ch["V"] is not None else None
    chunk = kam.Chunk(K, V)
    patch = None
    if ch["Uk"] is not None and ch["Uk"].shape[-1] > 0:
        def U(x):
            if x is None:
                return None
            return [(x[l][:, 0, :] if shared_u else x[l]).to(device).contiguous() for l in range(L)]

        def W(x):
            if x is None:
                return None
            r = rank_per_layer if rank_per_layer is not None else [x.shape[2]] * L
            return [x[l][:, :max(1, r[l])].to(device).contiguous() for l in range(L)]
        patch = kam.Patch(U(ch["Uk"]), W(ch["Wk"]), U(ch["Uv"]), W(ch["Wv"]))
    return chunk, patch


def oracle_layer(cfg, ch, l, delta, style=reuse.HALF, frame=reuse.TARGET_FRAME, rank=None, shared_u=False):
    """Unrounded fp64 Eq. 1 for one layer of a synth chunk, plus the S arrays.  rank=0 => rotation only."""
    k = to_f64(ch["K"][l]); v = to_f64(ch["V"][l]) if ch["V"] is not None else None
    use = ch["Uk"] is not None and ch["Uk"].shape[-1] > 0 and (rank is None or rank > 0)
    Uk = to_f64(ch["Uk"][l]) if use else None; Wk = to_f64(ch["Wk"][l]) if use else None
    Uv = to_f64(ch["Uv"][l]) if use and v is not None else None; Wv = to_f64(ch["Wv"][l]) if use and v is not None else None
    if use and rank is not None:                     # a layer whose rank is below the stored one: leading columns / rows
        Uk, Wk = Uk[..., :rank], Wk[:, :rank]
        if Uv is not None:
            Uv, Wv = Uv[..., :rank], Wv[:, :rank]
    if use and shared_u:
        Uk = np.repeat(Uk[:, :1, :], Uk.shape[1], axis=1)
        if Uv is not None:
            Uv = np.repeat(Uv[:, :1, :], Uv.shape[1], axis=1)
    ko = reuse.reuse_k(k, delta, Uk, Wk, frame=frame, **rope_kw(cfg, style))
    Sk = abs_sum_k(k, delta, Uk, Wk, cfg, style)
    if frame == reuse.CANONICAL_FRAME and use:       # patched first, rotated after: bound via the patched magnitudes
        Sk = abs_sum_k(np.abs(k) + reuse.patch_term(np.abs(Uk), np.abs(Wk)), delta, None, None, cfg, style)
    vo = reuse.reuse_v(v, Uv, Wv) if v is not None else None
    Sv = abs_sum_v(v, Uv, Wv) if v is not None else None
    return ko, vo, Sk, Sv


def check_relocated(cfg, pool, ch, bt, dst0, delta, m, style=reuse.HALF, frame=reuse.TARGET_FRAME, layers=None,
                    rank_per_layer=None, shared_u=False, elem="bf16"):
    """Compare every element the call wrote, for the given layers.  Returns merged stats."""
    T = ch["K"].shape[1]
    tot = {}
    cmp = compare_bf16 if elem == "bf16" else compare_f32
    for l in (layers if layers is not None else range(ch["K"].shape[0])):
        ml = m if rank_per_layer is None else rank_per_layer[l]
        ko, vo, Sk, Sv = oracle_layer(cfg, ch, l, delta, style, frame, rank=ml, shared_u=shared_u)
        st = cmp(pool_rows(pool.k_layers[l], bt, dst0, T), ko, Sk, ml, "K layer %d" % l)
        for k_, v_ in st.items():
            tot[k_] = tot.get(k_, 0) + v_
        if vo is not None:
            st = cmp(pool_rows(pool.v_layers[l], bt, dst0, T), vo, Sv, ml, "V layer %d" % l)
            for k_, v_ in st.items():
                tot[k_] = tot.get(k_, 0) + v_
    return tot


def untouched_pages_intact(pool, used_pages, n_layers):
    """No page outside the block table was written."""
    for l in range(n_layers):
        for layer in ([pool.k_layers[l]] + ([pool.v_layers[l]] if pool.v_layers is not None else [])):
            mask = torch.ones(layer.shape[0], dtype=torch.bool, device=layer.device)
            mask[torch.as_tensor(np.asarray(used_pages, dtype=np.int64), device=layer.device)] = False
            if not bool((layer[mask].float() == SENTINEL).all()):
                return False
    return True
