"""Decode readout over cached chunks (test infrastructure; see oracle/__init__.py).

"Readout is the value a query pulls out: attention over the union of two key sets equals
attending each separately and merging by softmax mass, o = (1 - mu) o_B + mu o_A, the
log-sum-exp state merge already used by FlashAttention and ring/star attention".

Two independent routines:
  attend_bruteforce   O8: softmax over the concatenation of all chunks' keys - the definition.
  attend_chunks_merge O9: per-chunk (o_c, lse_c), then the LSE merge.
and a third that evaluates the same quantity the way a fused-on-read kernel may (rotation moved
onto the query, the rank-m patch contracted in O(m) per token):
  attend_on_read_factorized

A chunk is a dict with
  k [T,H,D], v [T,H,D] or None   rows as they sit in the pool (fp64 values of the stored bf16)
  delta                          RoPE offset still to be applied on read (0 if materialised)
  Uk,Wk,Uv,Wv (optional)         rank-m patch still to be applied on read (None if materialised)
If v is None (MLA, absorbed form) the value of a token is the first `v_dim` columns of its
(patched) key row - the latent c_KV.

Conventions (reading R-12): natural log, sm_scale inside the exponent, query head hq reads KV
head hq // G with G = Hq // H, no mask (the decode query is the newest token).

Multi-query readout ("chunked-prefill (multi-query) attention over relocated
chunks"; the TTFT path of P:105 / P:349: after `apply_reuse` has placed the recalled
chunks, the appended text turn is prefilled over them):
  attend_prefill_bruteforce   the same readout for Tq query rows.  With causal=True the
                              query rows ARE the last Tq cached tokens (reading R-19 in DESIGN.md):
                              row t sees cached token j iff j <= N - Tq + t, N = all cached tokens
                              of the request.  It is the single-query definition applied row by
                              row to the visible prefix - nothing else.
"""
import numpy as np

from . import reuse


def _effective_kv(ch, rope, v_dim):
    k = reuse.reuse_k(ch["k"], ch.get("delta", 0), ch.get("Uk"), ch.get("Wk"), **rope)
    if ch.get("v") is None:
        v = k[..., :v_dim]
    else:
        v = reuse.reuse_v(ch["v"], ch.get("Uv"), ch.get("Wv"))
    return k, v


def _softmax_readout(q_h, k_h, v_h, sm_scale):
    """(out [Dv], lse) of one query vector over rows k_h [N,D], v_h [N,Dv]; N = 0 allowed."""
    if k_h.shape[0] == 0:
        return np.zeros(v_h.shape[1]), -np.inf
    s = sm_scale * (k_h @ q_h)
    m = s.max()
    w = np.exp(s - m)
    l = w.sum()
    return (w @ v_h) / l, m + np.log(l)


def attend_bruteforce(q, chunks, sm_scale, rope, v_dim=None):
    """O8.  q [Hq, D]; returns out [Hq, Dv], lse [Hq]."""
    kv = [_effective_kv(c, rope, v_dim) for c in chunks]
    H = chunks[0]["k"].shape[1]
    Hq = q.shape[0]
    G = Hq // H
    K = np.concatenate([k for k, _ in kv], axis=0)
    V = np.concatenate([v for _, v in kv], axis=0)
    out = np.zeros((Hq, V.shape[2])); lse = np.zeros(Hq)
    for hq in range(Hq):
        out[hq], lse[hq] = _softmax_readout(np.asarray(q[hq], np.float64), K[:, hq // G], V[:, hq // G], sm_scale)
    return out, lse


def chunk_partials(q, chunks, sm_scale, rope, v_dim=None):
    """Per-chunk softmax states: o [C, Hq, Dv], lse [C, Hq] (lse = -inf, o = 0 for an empty chunk)."""
    H = chunks[0]["k"].shape[1]
    Hq = q.shape[0]
    G = Hq // H
    o, l = [], []
    for c in chunks:
        k, v = _effective_kv(c, rope, v_dim)
        oc = np.zeros((Hq, v.shape[2])); lc = np.zeros(Hq)
        for hq in range(Hq):
            oc[hq], lc[hq] = _softmax_readout(np.asarray(q[hq], np.float64), k[:, hq // G], v[:, hq // G], sm_scale)
        o.append(oc); l.append(lc)
    return np.stack(o), np.stack(l)


def lse_merge(o, lse):
    """O9: lse = ln sum_c e^{lse_c};  out = sum_c e^{lse_c - lse} o_c.   o [C,Hq,Dv], lse [C,Hq].
    All chunks empty => out = 0, lse = -inf (no NaN)."""
    m = lse.max(axis=0)
    safe_m = np.where(np.isfinite(m), m, 0.0)
    w = np.exp(lse - safe_m)                       # exp(-inf) = 0 for empty chunks
    tot = w.sum(axis=0)
    with np.errstate(divide="ignore", invalid="ignore"):
        merged_lse = np.where(tot > 0, safe_m + np.log(tot), -np.inf)
        mu = np.where(tot > 0, w / tot, 0.0)       # softmax mass of each chunk
    return np.einsum("ch,chd->hd", mu, o), merged_lse


def attend_chunks_merge(q, chunks, sm_scale, rope, v_dim=None):
    return lse_merge(*chunk_partials(q, chunks, sm_scale, rope, v_dim))


def attend_on_read_factorized(q, chunks, sm_scale, rope, v_dim=None):
    """Same readout with the operator folded into the read (TARGET frame only):
         q.(R(d)k_t)            = (R(-d)q).k_t
         q.(U_k[t,:] W_k)       = U_k[t,:].(W_k q)
         sum_t p_t (U_v[t,:] W_v) = (sum_t p_t U_v[t,:]) W_v
    MLA (v is None): the value patch is the latent columns of the key patch."""
    H = chunks[0]["k"].shape[1]
    Hq = q.shape[0]
    G = Hq // H
    q = np.asarray(q, np.float64)
    o, l = [], []
    for c in chunks:
        k = np.asarray(c["k"], np.float64)
        T = k.shape[0]
        qrot = reuse.relocate(q, -int(c.get("delta", 0)), **rope)        # rotation moved to the query
        mla = c.get("v") is None
        v = k[..., :v_dim] if mla else np.asarray(c["v"], np.float64)
        Uk, Wk = c.get("Uk"), c.get("Wk")
        Uv, Wv = (Uk, None if Wk is None else np.asarray(Wk)[..., :v_dim]) if mla else (c.get("Uv"), c.get("Wv"))
        oc = np.zeros((Hq, v.shape[2])); lc = np.full(Hq, -np.inf)
        for hq in range(Hq):
            h = hq // G
            if T == 0:
                continue
            s = k[:, h] @ qrot[hq]
            if Uk is not None:
                s = s + np.asarray(Uk, np.float64)[:, h] @ (np.asarray(Wk, np.float64)[h] @ q[hq])
            s = sm_scale * s
            m = s.max(); w = np.exp(s - m); lsum = w.sum()
            acc = w @ v[:, h]
            if Uv is not None:
                acc = acc + (w @ np.asarray(Uv, np.float64)[:, h]) @ np.asarray(Wv, np.float64)[h]
            oc[hq], lc[hq] = acc / lsum, m + np.log(lsum)
        o.append(oc); l.append(lc)
    return lse_merge(np.stack(o), np.stack(l))


def attend_prefill_bruteforce(q, chunks, sm_scale, rope, causal=True, v_dim=None, rows=None):
    """q [Tq, Hq, D] -> out [Tq, Hq, Dv], lse [Tq, Hq] (rows: evaluate only these query rows, in this order).  Row t = attend_bruteforce(q[t]) over the cached tokens it may see:
    all N of them (causal=False), or tokens 0 .. N - Tq + t (causal=True: the rows are the last Tq cached tokens, each
    seeing the recalled context, the appended tokens before it, and itself).  A row that sees nothing (Tq > N, its index
    before the first cached token) gives out = 0, lse = -inf."""
    q = np.asarray(q, np.float64)
    Tq = q.shape[0]
    N = sum(c["k"].shape[0] for c in chunks)
    outs, lses = [], []
    for t in (range(Tq) if rows is None else rows):
        n_vis = N if not causal else N - Tq + t + 1
        vis, left = [], max(n_vis, 0)
        for c in chunks:                                      # the visible prefix, chunk by chunk (a chunk may be cut)
            take = min(left, c["k"].shape[0])
            cut = dict(c, k=c["k"][:take], v=None if c.get("v") is None else c["v"][:take])
            for name in ("Uk", "Uv"):
                if c.get(name) is not None:
                    cut[name] = np.asarray(c[name])[:take]
            vis.append(cut)
            left -= take
        o, l = attend_bruteforce(q[t], vis, sm_scale, rope, v_dim)
        outs.append(o); lses.append(l)
    return np.stack(outs), np.stack(lses)
