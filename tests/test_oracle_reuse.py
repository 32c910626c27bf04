"""Pins for oracle/reuse.py (Eq. 1: relocate + patch + paged scatter).

Each pin is something the paper or the mathematics fixes, not the oracle's own formula:
closed forms, R(d)R(p)=R(p+d), V untouched, MLA rotates only k_pe,
rank-0 = rotation, exact rank-m reconstruction and Eckart-Young,
an independent textbook RoPE (rotate_half / complex multiply) in torch, brute-force slot loops.
"""
import itertools

import numpy as np
import pytest
import torch

from oracle import reuse
from oracle.bf16 import bf16_bits, bf16_from_bits, ulp_bf16

RNG = np.random.default_rng(123)
GQA = dict(theta=1e6, rope_off=0, d_r=128)
MLA = dict(theta=1e4, rope_off=512, d_r=64)


# ---------------------------------------------------------------- O1 / O2 / O3: rotation
def test_frequencies_closed_form():
    f = reuse.rope_frequencies(1e4, 64)
    assert f[0] == 1.0
    assert f.shape == (32,)
    assert np.allclose(f[16], 1e4 ** -0.5, rtol=1e-15)           # i = d_r/4 -> theta^(-1/2)
    assert np.allclose(f[1:] / f[:-1], 1e4 ** (-2.0 / 64), rtol=1e-13)   # geometric schedule


@pytest.mark.parametrize("style", [reuse.HALF, reuse.INTERLEAVED])
def test_unit_vector_closed_form(style):
    # pair 0 has f_0 = 1: (1, 0) rotated by delta is (cos delta, sin delta)
    d_r = 8
    ia, ib = reuse.rope_pair_columns(style, 0, d_r)
    k = np.zeros((1, 1, d_r)); k[0, 0, ia[0]] = 1.0
    for delta in (1, -3, 1000):
        r = reuse.relocate(k, delta, 1e4, 0, d_r, style)
        assert np.allclose(r[0, 0, ia[0]], np.cos(delta), atol=1e-15)
        assert np.allclose(r[0, 0, ib[0]], np.sin(delta), atol=1e-15)
        rest = np.delete(r[0, 0], [ia[0], ib[0]])
        assert np.all(rest == 0)


def test_pair_columns():
    a, b = reuse.rope_pair_columns(reuse.HALF, 512, 64)
    assert a[0] == 512 and b[0] == 544 and a[-1] == 543 and b[-1] == 575
    a, b = reuse.rope_pair_columns(reuse.INTERLEAVED, 0, 8)
    assert list(a) == [0, 2, 4, 6] and list(b) == [1, 3, 5, 7]


@pytest.mark.parametrize("style", [reuse.HALF, reuse.INTERLEAVED])
def test_delta_zero_is_copy_and_norm_preserved(style):
    k = RNG.standard_normal((5, 2, 128))
    assert np.array_equal(reuse.relocate(k, 0, style=style, **GQA), k)
    r = reuse.relocate(k, 777, style=style, **GQA)
    ia, ib = reuse.rope_pair_columns(style, 0, 128)
    assert np.allclose(r[..., ia] ** 2 + r[..., ib] ** 2, k[..., ia] ** 2 + k[..., ib] ** 2, rtol=1e-12)


@pytest.mark.parametrize("style", [reuse.HALF, reuse.INTERLEAVED])
def test_composition_and_inverse(style):
    """R(delta)R(p) = R(p+delta) 'exactly'; R(-delta)R(delta) = I."""
    k = RNG.standard_normal((7, 4, 128))
    for p, d in itertools.product((0, 5, 31000), (1, -1280, 4096)):
        two = reuse.relocate(reuse.relocate(k, p, style=style, **GQA), d, style=style, **GQA)
        one = reuse.relocate(k, p + d, style=style, **GQA)
        assert np.max(np.abs(two - one)) < 1e-10          # fp64: angle error ~ |p| * 2^-53
    back = reuse.relocate(reuse.relocate(k, 12345, style=style, **GQA), -12345, style=style, **GQA)
    assert np.max(np.abs(back - k)) < 1e-12


def _textbook_rope_half(x, pos, theta):
    """Independent restatement (the rotate_half form used by LLaMA/Qwen-family code), torch fp64."""
    d = x.shape[-1]
    inv = 1.0 / (theta ** (torch.arange(0, d, 2, dtype=torch.float64) / d))
    ang = torch.as_tensor(pos, dtype=torch.float64)[..., None] * inv
    emb = torch.cat([ang, ang], dim=-1)
    x1, x2 = x[..., : d // 2], x[..., d // 2:]
    return x * emb.cos() + torch.cat([-x2, x1], dim=-1) * emb.sin()


def _textbook_rope_interleaved(x, pos, theta):
    """Independent restatement (RoFormer's complex form): (x0 + i x1) * e^{i pos f}."""
    d = x.shape[-1]
    inv = 1.0 / (theta ** (torch.arange(0, d, 2, dtype=torch.float64) / d))
    ang = torch.as_tensor(pos, dtype=torch.float64)[..., None] * inv
    z = torch.view_as_complex(x.reshape(*x.shape[:-1], d // 2, 2).contiguous())
    return torch.view_as_real(z * torch.polar(torch.ones_like(ang), ang)).reshape(x.shape)


def test_equals_textbook_rope_on_unrotated_rows():
    """Special case: p_base = 0 applied to an un-rotated one-token chunk is textbook RoPE at p."""
    x = torch.from_numpy(RNG.standard_normal((3, 2, 64)))
    for p in (0, 1, 17, 4095):
        pos = torch.full((3, 2), p)
        got_h = reuse.relocate(x.numpy(), p, 1e4, 0, 64, reuse.HALF)
        got_i = reuse.relocate(x.numpy(), p, 1e4, 0, 64, reuse.INTERLEAVED)
        assert np.allclose(got_h, _textbook_rope_half(x, pos, 1e4).numpy(), atol=1e-12)
        assert np.allclose(got_i, _textbook_rope_interleaved(x, pos, 1e4).numpy(), atol=1e-12)


def test_relocating_textbook_keys_gives_textbook_keys():
    """Keys stored at positions p0+t, relocated by delta, equal textbook RoPE at p0+delta+t."""
    T, D, theta = 9, 64, 1e4
    raw = torch.from_numpy(RNG.standard_normal((T, 1, D)))
    t = torch.arange(T)[:, None]
    stored = _textbook_rope_half(raw, 0 + t, theta).numpy()          # chunk prefilled alone (p_base = 0)
    want = _textbook_rope_half(raw, 300 + t, theta).numpy()
    got = reuse.relocate(stored, 300, theta, 0, D, reuse.HALF)
    assert np.allclose(got, want, atol=1e-11)


def test_shift_invariance_pins_the_sign_convention():
    """<R(n+d)q, R(m+d)k> = <R(n)q, R(m)k>: fails if sin carries the wrong sign on one side."""
    q = RNG.standard_normal((1, 1, 128)); k = RNG.standard_normal((1, 1, 128))
    for style in (reuse.HALF, reuse.INTERLEAVED):
        base = np.sum(reuse.relocate(q, 40, style=style, **GQA) * reuse.relocate(k, 7, style=style, **GQA))
        moved = np.sum(reuse.relocate(q, 40 + 999, style=style, **GQA) * reuse.relocate(k, 7 + 999, style=style, **GQA))
        assert abs(base - moved) < 1e-9
        # and the query-side identity the fused decode uses: q.(R(d)k) = (R(-d)q).k
        lhs = np.sum(q * reuse.relocate(k, 321, style=style, **GQA))
        rhs = np.sum(reuse.relocate(q, -321, style=style, **GQA) * k)
        assert abs(lhs - rhs) < 1e-10


def test_mla_rotates_only_the_rope_band():
    """'the latent c_KV carries no RoPE, so relocation only re-rotates the 64-dim decoupled k_pe'."""
    k = RNG.standard_normal((6, 1, 576))
    r = reuse.relocate(k, 2048, **MLA)
    assert np.array_equal(r[..., :512], k[..., :512])
    assert not np.any(r[..., 512:] == k[..., 512:])


# ---------------------------------------------------------------- O4: the rank-m patch
def test_rank0_is_pure_rotation_and_v_untouched():
    k = RNG.standard_normal((4, 2, 128)); v = RNG.standard_normal((4, 2, 128))
    assert np.array_equal(reuse.reuse_k(k, 5, None, None, **GQA), reuse.relocate(k, 5, **GQA))
    U0 = np.zeros((4, 2, 0)); W0 = np.zeros((2, 0, 128))
    assert np.array_equal(reuse.reuse_k(k, 5, U0, W0, **GQA), reuse.relocate(k, 5, **GQA))
    assert np.array_equal(reuse.reuse_v(v, None, None), v)


def test_patch_term_against_python_loops():
    T, H, m, D = 3, 2, 4, 8
    U = RNG.standard_normal((T, H, m)); W = RNG.standard_normal((H, m, D))
    want = np.zeros((T, H, D))
    for t in range(T):
        for h in range(H):
            for c in range(D):
                for j in range(m):
                    want[t, h, c] += U[t, h, j] * W[h, j, c]
    assert np.allclose(reuse.patch_term(U, W), want, atol=1e-14)
    # a transposed / head-mixed operand would break these
    assert not np.allclose(reuse.patch_term(U, W[::-1]), want)


@pytest.mark.parametrize("frame", [reuse.TARGET_FRAME, reuse.CANONICAL_FRAME])
def test_exact_rank_m_delta_reconstructs_conditioned_kv(frame):
    """A patch built from an exactly rank-m Delta reconstructs KV(B|A) exactly (BASELINE.json)."""
    T, H, D, m, delta = 40, 2, 128, 4, 1234
    k_solo = RNG.standard_normal((T, H, D)); v_solo = RNG.standard_normal((T, H, D))
    Dk = np.einsum("thj,hjc->thc", RNG.standard_normal((T, H, m)), RNG.standard_normal((H, m, D)))
    Dv = np.einsum("thj,hjc->thc", RNG.standard_normal((T, H, m)), RNG.standard_normal((H, m, D)))
    k_rel = reuse.relocate(k_solo, delta, **GQA)
    k_cond, v_cond = k_rel + Dk, v_solo + Dv                     # KV(B|A) at the target position
    if frame == reuse.TARGET_FRAME:                              # Delta measured against R(delta)KV(B|0)
        Uk, Wk, _ = reuse.form_patch(k_cond, k_rel, m)
    else:                                                        # same Delta carried back to the chunk's own frame
        Uk, Wk, _ = reuse.form_patch(reuse.relocate(k_cond, -delta, **GQA), k_solo, m)
    Uv, Wv, _ = reuse.form_patch(v_cond, v_solo, m)
    assert np.max(np.abs(reuse.reuse_k(k_solo, delta, Uk, Wk, frame=frame, **GQA) - k_cond)) < 1e-10
    assert np.max(np.abs(reuse.reuse_v(v_solo, Uv, Wv) - v_cond)) < 1e-10


def test_eckart_young_residual():
    """General Delta: ||Delta - U W||_F^2 = sum_{i>m} sigma_i^2, per head."""
    T, H, D, m = 50, 2, 32, 5
    kc = RNG.standard_normal((T, H, D)); ks = RNG.standard_normal((T, H, D))
    U, W, S = reuse.form_patch(kc, ks, m)
    res = (kc - ks) - reuse.patch_term(U, W)
    for h in range(H):
        assert np.isclose(np.sum(res[:, h] ** 2), np.sum(S[h, m:] ** 2), rtol=1e-10)
    # S folded into U: rows of W orthonormal, columns of U carry the singular values
    assert np.allclose(W[0] @ W[0].T, np.eye(m), atol=1e-12)
    assert np.allclose(np.linalg.norm(U[:, 0, :], axis=0), S[0, :m], rtol=1e-12)


def test_patch_linearity_and_frames_agree_off_band():
    k = RNG.standard_normal((8, 1, 576))
    U = RNG.standard_normal((8, 1, 3)); W = RNG.standard_normal((1, 3, 576))
    a = reuse.reuse_k(k, 9, U, W, **MLA); b = reuse.reuse_k(k, 9, U, 2 * W, **MLA)
    base = reuse.relocate(k, 9, **MLA)
    assert np.allclose(b - base, 2 * (a - base), atol=1e-12)
    # the latent columns do not rotate, so both frames coincide there ("the same patch transfers unchanged")
    c = reuse.reuse_k(k, 9, U, W, frame=reuse.CANONICAL_FRAME, **MLA)
    assert np.allclose(a[..., :512], c[..., :512], atol=1e-13)
    assert not np.allclose(a[..., 512:], c[..., 512:])


# ---------------------------------------------------------------- O5 / O6: paged scatter
def test_slot_mapping_bruteforce():
    P = 16
    bt = np.array([7, 2, 9, 4], dtype=np.int32)
    page, slot = reuse.slot_mapping(bt, 5, 40, P)               # not page aligned, straddles 3 pages
    for t in range(40):
        g = 5 + t
        assert page[t] == bt[g // P] and slot[t] == g % P


def test_scatter_rounds_once_and_hits_only_its_slots():
    P, H, D = 4, 2, 8
    pool = np.full((6, P, H, D), 0xFFFF, dtype=np.uint16)
    rows = RNG.standard_normal((6, H, D))
    bt = np.array([5, 0, 3], dtype=np.int32)
    reuse.scatter(pool, bt, 2, rows)                            # tokens g = 2..7 -> pages 5 (slots 2,3), 0 (0..3)
    assert np.array_equal(pool[5, 2:4], bf16_bits(rows[0:2]))
    assert np.array_equal(pool[0, 0:4], bf16_bits(rows[2:6]))
    untouched = np.ones(pool.shape, bool); untouched[5, 2:4] = False; untouched[0] = False
    assert np.all(pool[untouched] == 0xFFFF)
    assert np.array_equal(reuse.gather(pool, bt, 2, 6), bf16_from_bits(bf16_bits(rows)))


def test_delta0_rank0_relocate_is_a_bit_exact_copy():
    """'a copy with no arithmetic at all'."""
    T, H, D, P = 32, 2, 128, 16
    kb = bf16_bits(RNG.standard_normal((T, H, D))); vb = bf16_bits(RNG.standard_normal((T, H, D)))
    pk = np.zeros((4, P, H, D), np.uint16); pv = np.zeros_like(pk)
    bt = np.array([3, 1], dtype=np.int32)
    reuse.relocate_patch_layer(pk, pv, bt, 0, bf16_from_bits(kb), bf16_from_bits(vb), 0,
                               None, None, None, None, **GQA)
    assert np.array_equal(pk[bt].reshape(T, H, D), kb) and np.array_equal(pv[bt].reshape(T, H, D), vb)


def test_inplace_rotate_there_and_back_within_one_ulp_and_v_not_needed():
    T, H, D, P = 32, 2, 128, 16
    pk = np.zeros((2, P, H, D), np.uint16)
    bt = np.array([1, 0], dtype=np.int32)
    k0 = bf16_from_bits(bf16_bits(RNG.standard_normal((T, H, D))))
    reuse.scatter(pk, bt, 0, k0)
    reuse.rotate_inplace_layer(pk, bt, 0, T, -1280, **GQA)
    mid = reuse.gather(pk, bt, 0, T)
    assert np.array_equal(bf16_bits(reuse.relocate(k0, -1280, **GQA)), bf16_bits(mid))
    reuse.rotate_inplace_layer(pk, bt, 0, T, +1280, **GQA)
    back = reuse.gather(pk, bt, 0, T)
    # two roundings: each output is a 2-term sum of values carrying <= 1/2 ulp error each
    ia, ib = reuse.rope_pair_columns(reuse.HALF, 0, 128)
    scale = np.zeros_like(k0); mag = np.abs(k0[..., ia]) + np.abs(k0[..., ib])
    scale[..., ia] = mag; scale[..., ib] = mag
    assert np.all(np.abs(back - k0) <= 1.5 * ulp_bf16(scale))
