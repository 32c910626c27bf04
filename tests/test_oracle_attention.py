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
