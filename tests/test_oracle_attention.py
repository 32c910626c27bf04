"""Pins for oracle/attention.py: the LSE merge equals softmax over the concatenation,
the paper's two-set formula, closed forms, permutation invariance, and the on-read factorisations."""
import numpy as np
import pytest

from oracle import attention as att
from oracle import reuse
from oracle.bf16 import bf16_rne

RNG = np.random.default_rng(11)
ROPE = dict(theta=1e4, rope_off=0, d_r=64, style=reuse.HALF)


def _chunks(n, T, H, D, m=0, deltas=None, with_v=True):
    out = []
    for i in range(n):
        c = {"k": bf16_rne(RNG.standard_normal((T, H, D))), "delta": 0 if deltas is None else deltas[i]}
        c["v"] = bf16_rne(RNG.standard_normal((T, H, D))) if with_v else None
        if m:
            c["Uk"] = RNG.standard_normal((T, H, m)); c["Wk"] = 0.1 * RNG.standard_normal((H, m, D))
            if with_v:
                c["Uv"] = RNG.standard_normal((T, H, m)); c["Wv"] = 0.1 * RNG.standard_normal((H, m, D))
        out.append(c)
    return out


def test_bruteforce_against_plain_loops():
    """O8 against the definition written as scalar loops (tiny)."""
    H, Hq, D, T = 2, 4, 64, 5
    ch = _chunks(2, T, H, D)
    q = RNG.standard_normal((Hq, D))
    out, lse = att.attend_bruteforce(q, ch, 0.125, ROPE)
    for hq in range(Hq):
        h = hq // 2
        ks = [c["k"][t, h] for c in ch for t in range(T)]
        vs = [c["v"][t, h] for c in ch for t in range(T)]
        s = [0.125 * sum(q[hq, d] * k[d] for d in range(D)) for k in ks]
        Z = sum(np.exp(x) for x in s)
        want = sum(np.exp(x) / Z * v for x, v in zip(s, vs))
        assert np.allclose(out[hq], want, atol=1e-13) and np.isclose(lse[hq], np.log(Z), atol=1e-13)


def test_uniform_keys_closed_form():
    """All keys equal => weights uniform: out = mean(v), lse = ln N + s."""
    H, D, T = 1, 64, 12
    k = np.tile(RNG.standard_normal((1, H, D)), (T, 1, 1))
    v = RNG.standard_normal((T, H, D))
    q = RNG.standard_normal((1, D))
    out, lse = att.attend_bruteforce(q, [{"k": k, "v": v}], 0.3, ROPE)
    assert np.allclose(out[0], v[:, 0].mean(axis=0), atol=1e-13)
    assert np.isclose(lse[0], np.log(T) + 0.3 * (k[0, 0] @ q[0]), atol=1e-12)


@pytest.mark.parametrize("m", [0, 4])
def test_lse_merge_equals_softmax_over_concatenation(m):
    """BASELINE.json: 'the LSE-merge of per-chunk attention equals brute-force softmax over the
    concatenation on tiny inputs' - with relocation and patch pending on read."""
    ch = _chunks(3, 7, 2, 64, m=m, deltas=[0, 300, -41])
    q = RNG.standard_normal((4, 64))
    o1, l1 = att.attend_bruteforce(q, ch, 0.125, ROPE)
    o2, l2 = att.attend_chunks_merge(q, ch, 0.125, ROPE)
    assert np.max(np.abs(o1 - o2)) < 1e-12 and np.max(np.abs(l1 - l2)) < 1e-12


def test_paper_two_set_formula():
    """o = (1 - mu) o_B + mu o_A with mu = mass_A / (mass_A + mass_B)."""
    A, B = _chunks(2, 9, 1, 64)
    q = RNG.standard_normal((1, 64))
    o, lse = att.chunk_partials(q, [A, B], 0.125, ROPE)
    massA, massB = np.exp(lse[0, 0]), np.exp(lse[1, 0])
    mu = massA / (massA + massB)
    want = (1 - mu) * o[1, 0] + mu * o[0, 0]
    full, _ = att.attend_bruteforce(q, [A, B], 0.125, ROPE)
    assert np.allclose(full[0], want, atol=1e-13)


def test_merge_single_chunk_identity_permutation_and_empty():
    ch = _chunks(3, 6, 2, 64)
    q = RNG.standard_normal((2, 64))
    o, l = att.chunk_partials(q, ch, 0.125, ROPE)
    mo, ml = att.lse_merge(o[:1], l[:1])
    assert np.array_equal(mo, o[0]) and np.array_equal(ml, l[0])
    a = att.lse_merge(o, l); b = att.lse_merge(o[[2, 0, 1]], l[[2, 0, 1]])
    assert np.allclose(a[0], b[0], atol=1e-14) and np.allclose(a[1], b[1], atol=1e-14)
    # an empty chunk contributes nothing; all empty => zeros and -inf, no NaN
    empty = {"k": np.zeros((0, 2, 64)), "v": np.zeros((0, 2, 64))}
    c = att.attend_chunks_merge(q, ch + [empty], 0.125, ROPE)
    assert np.allclose(c[0], a[0], atol=1e-14) and np.allclose(c[1], a[1], atol=1e-14)
    z = att.attend_chunks_merge(q, [empty, empty], 0.125, ROPE)
    assert np.all(z[0] == 0) and np.all(np.isneginf(z[1]))


@pytest.mark.parametrize("style", [reuse.HALF, reuse.INTERLEAVED])
def test_on_read_factorisations_equal_the_definition(style):
    rope = dict(ROPE, style=style)
    ch = _chunks(3, 8, 2, 64, m=4, deltas=[17, 0, -1280])
    q = RNG.standard_normal((4, 64))
    o1, l1 = att.attend_bruteforce(q, ch, 0.125, rope)
    o2, l2 = att.attend_on_read_factorized(q, ch, 0.125, rope)
    assert np.max(np.abs(o1 - o2)) < 1e-12 and np.max(np.abs(l1 - l2)) < 1e-12


def test_on_read_equals_materialised_up_to_pool_rounding():
    """Reading a chunk with delta pending == reading the chunk after Eq. 1 was applied in fp64."""
    ch = _chunks(2, 8, 2, 64, m=4, deltas=[55, -7])
    q = RNG.standard_normal((4, 64))
    mat = [{"k": reuse.reuse_k(c["k"], c["delta"], c["Uk"], c["Wk"], **ROPE),
            "v": reuse.reuse_v(c["v"], c["Uv"], c["Wv"]), "delta": 0} for c in ch]
    a = att.attend_bruteforce(q, ch, 0.125, ROPE); b = att.attend_bruteforce(q, mat, 0.125, ROPE)
    assert np.allclose(a[0], b[0], atol=1e-12) and np.allclose(a[1], b[1], atol=1e-12)


def test_mla_absorbed_form_value_is_the_latent():
    rope = dict(theta=1e4, rope_off=512, d_r=64, style=reuse.HALF)
    ch = _chunks(2, 5, 1, 576, m=4, deltas=[9, 1024], with_v=False)
    q = RNG.standard_normal((3, 576))
    o1, l1 = att.attend_bruteforce(q, ch, 0.07, rope, v_dim=512)
    o2, l2 = att.attend_on_read_factorized(q, ch, 0.07, rope, v_dim=512)
    assert o1.shape == (3, 512)
    assert np.max(np.abs(o1 - o2)) < 1e-12 and np.max(np.abs(l1 - l2)) < 1e-12
    # GQA head mapping: with H = 1 every query head reads the same keys; different q => different out
    assert not np.allclose(o1[0], o1[1])


# ---------------------------------------------------------------------------------------- multi-query readout (f4)
def _dense_masked_attention(q, K, V, G, sm_scale, causal):
    """An independent formulation: the full [Tq, N] score matrix per head, a triangular -inf mask, row softmax."""
    Tq, Hq, _ = q.shape
    N = K.shape[0]
    out = np.zeros((Tq, Hq, V.shape[2])); lse = np.zeros((Tq, Hq))
    for hq in range(Hq):
        S = sm_scale * np.einsum("td,nd->tn", q[:, hq], K[:, hq // G])
        if causal:
            S = np.where(np.arange(N)[None, :] <= (N - Tq + np.arange(Tq))[:, None], S, -np.inf)
        m = S.max(axis=1, keepdims=True)
        W = np.exp(S - m)
        out[:, hq] = (W / W.sum(axis=1, keepdims=True)) @ V[:, hq // G]
        lse[:, hq] = m[:, 0] + np.log(W.sum(axis=1))
    return out, lse


@pytest.mark.parametrize("causal", [True, False])
def test_prefill_equals_a_dense_masked_score_matrix(causal):
    """Row-by-row definition vs the matrix formulation with a triangular mask; chunks with pending offsets (applied to the keys
    by hand here, through reuse.relocate) and one empty chunk."""
    H, Hq, D, Tq = 2, 6, 64, 5
    ch = _chunks(3, 4, H, D, deltas=[0, 37, -5])
    ch.insert(1, {"k": np.zeros((0, H, D)), "v": np.zeros((0, H, D)), "delta": 9})
    q = RNG.standard_normal((Tq, Hq, D))
    out, lse = att.attend_prefill_bruteforce(q, ch, 0.11, ROPE, causal=causal)
    K = np.concatenate([reuse.relocate(c["k"], c["delta"], **ROPE) for c in ch]); V = np.concatenate([c["v"] for c in ch])
    want_o, want_l = _dense_masked_attention(q, K, V, Hq // H, 0.11, causal)
    assert np.allclose(out, want_o, atol=1e-12) and np.allclose(lse, want_l, atol=1e-12)


def test_prefill_rows_against_the_single_query_readout_and_closed_forms():
    H, Hq, D = 1, 2, 64
    ch = _chunks(2, 6, H, D)
    N, Tq = 12, 4
    q = RNG.standard_normal((Tq, Hq, D))
    out, lse = att.attend_prefill_bruteforce(q, ch, 0.2, ROPE, causal=True)
    # the LAST row sees every cached token: it is the decode readout
    o_last, l_last = att.attend_bruteforce(q[-1], ch, 0.2, ROPE)
    assert np.allclose(out[-1], o_last, atol=1e-13) and np.allclose(lse[-1], l_last, atol=1e-13)
    # without a mask every row is the decode readout of its own query
    out_nc, lse_nc = att.attend_prefill_bruteforce(q, ch, 0.2, ROPE, causal=False)
    for t in range(Tq):
        o, l = att.attend_bruteforce(q[t], ch, 0.2, ROPE)
        assert np.allclose(out_nc[t], o, atol=1e-13) and np.allclose(lse_nc[t], l, atol=1e-13)
    # pure self-attention (Tq = N): row 0 sees only token 0 -> out = v_0, lse = scale * q_0 . k_0
    qq = RNG.standard_normal((N, Hq, D))
    o_s, l_s = att.attend_prefill_bruteforce(qq, ch, 0.2, ROPE, causal=True)
    assert np.allclose(o_s[0, 0], ch[0]["v"][0, 0], atol=1e-13) and np.isclose(l_s[0, 1], 0.2 * qq[0, 1] @ ch[0]["k"][0, 0], atol=1e-12)
    # uniform keys: row t averages the values it sees; lse = ln(count) + s
    k1 = np.tile(RNG.standard_normal((1, H, D)), (N, 1, 1))
    uni = [{"k": k1[:7], "v": ch[0]["v"][:6].repeat(2, axis=0)[:7], "delta": 0}, {"k": k1[7:], "v": ch[1]["v"][:5], "delta": 0}]
    Vall = np.concatenate([c["v"] for c in uni])
    o_u, l_u = att.attend_prefill_bruteforce(q, uni, 0.2, ROPE, causal=True)
    for t in range(Tq):
        n_vis = N - Tq + t + 1
        assert np.allclose(o_u[t, 0], Vall[:n_vis, 0].mean(axis=0), atol=1e-12)
        assert np.isclose(l_u[t, 0], np.log(n_vis) + 0.2 * q[t, 0] @ k1[0, 0], atol=1e-12)
    # more query rows than cached tokens: the rows before the first cached token see nothing
    o_e, l_e = att.attend_prefill_bruteforce(RNG.standard_normal((N + 2, Hq, D)), ch, 0.2, ROPE, causal=True)
    assert np.all(o_e[:2] == 0) and np.all(np.isneginf(l_e[:2])) and np.all(np.isfinite(l_e[2:]))


def test_prefill_matches_torch_sdpa_for_causal_self_attention():
    """The special case a library routine covers: Tq = N, one chunk, no pending offset -> torch's scaled_dot_product_attention
    with is_causal=True (fp64, CPU); GQA by repeating the KV heads."""
    import torch
    import torch.nn.functional as F
    H, Hq, D, N = 2, 4, 64, 9
    ch = _chunks(1, N, H, D)
    q = RNG.standard_normal((N, Hq, D))
    out, _ = att.attend_prefill_bruteforce(q, ch, D ** -0.5, ROPE, causal=True)
    tq = torch.from_numpy(q).permute(1, 0, 2)[None]                                  # [1, Hq, N, D]
    tk = torch.from_numpy(ch[0]["k"]).permute(1, 0, 2).repeat_interleave(Hq // H, dim=0)[None]
    tv = torch.from_numpy(ch[0]["v"]).permute(1, 0, 2).repeat_interleave(Hq // H, dim=0)[None]
    want = F.scaled_dot_product_attention(tq, tk, tv, is_causal=True)[0].permute(1, 0, 2).numpy()
    assert np.allclose(out, want, atol=1e-12)


def test_prefill_with_patch_on_read_and_mla_value_is_the_latent():
    """The rows carry Eq. 1 like the decode readout does: pending patch factors cut with their chunk; MLA: value = latent."""
    H, Hq, D, Tq = 1, 2, 64, 3
    ch = _chunks(2, 4, H, D, m=2, deltas=[5, 0], with_v=False)
    q = RNG.standard_normal((Tq, Hq, D))
    out, lse = att.attend_prefill_bruteforce(q, ch, 0.3, ROPE, causal=True, v_dim=48)
    K = np.concatenate([reuse.reuse_k(c["k"], c["delta"], c["Uk"], c["Wk"], **ROPE) for c in ch])
    want_o, want_l = _dense_masked_attention(q, K, K[..., :48], Hq // H, 0.3, True)
    assert out.shape == (Tq, Hq, 48) and np.allclose(out, want_o, atol=1e-12) and np.allclose(lse, want_l, atol=1e-12)
