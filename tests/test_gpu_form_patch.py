"""GPU parity of kam_form_patch (compile side) against oracle/reuse.form_patch (numpy SVD in fp64).

Synthetic conditioning: KV(B|A) = bf16( R(delta) KV(B|0) + Delta_true ), Delta_true of decaying spectrum (the paper's
"functional rank" picture) - no model forward is involved.  Both sides form Delta from the SAME bf16 rows.  Singular
vectors are unique only up to sign, so what is compared is what is unique: sigma and the rank-m product U W; plus the
Eckart-Young residual and the end-to-end statement of Eq. 1: relocate + the formed patch reproduces KV(B|A) up to the
discarded tail.  Tolerances: the factors are stored in bf16 (2^-9 relative each), so ||U_g W_g - U_o W_o||_F <= 2^-7 ||U_o W_o||_F;
sigma is fp32: |sigma_g - sigma_o| <= 1e-3 sigma_o + 1e-4 sigma_1 (the relative part covers the fp32 Gram matrix, errors
~ 2^-24 sigma_1^2 / sigma_m^2; the absolute part is the flat tail left by the bf16 rounding of the rows, ~ 2^-9 of the row
magnitude, inside which singular values are not separated and a subspace method resolves them only to that level).
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import reuse
from synth import CONFIGS, make_block_table
from tests import parity as par

pytestmark = pytest.mark.gpu


def _synthetic(cfg, rng, L, T, delta, n_comp, s_hi, s_lo, style, is_key=True):
    """solo rows, conditioned rows (bf16 tensors [L, T, H, D]) with Delta_true = sum of n_comp rank-one terms per (layer, head)."""
    H, D = cfg.n_kv_heads, cfg.row_dim
    solo = torch.from_numpy(rng.standard_normal((L, T, H, D), dtype=np.float32)).to(torch.bfloat16)
    cond = np.zeros((L, T, H, D))
    sig = np.geomspace(s_hi, s_lo, n_comp)
    for l in range(L):
        base = par.to_f64(solo[l])
        if is_key:
            base = reuse.relocate(base, delta, cfg.theta, cfg.rope_off, cfg.rope_dim, style)
        for h in range(H):
            u, _ = np.linalg.qr(rng.standard_normal((T, n_comp)))
            v, _ = np.linalg.qr(rng.standard_normal((D, n_comp)))
            cond[l, :, h, :] = base[:, h, :] + (u * sig) @ v.T
    return solo, torch.from_numpy(cond).to(torch.bfloat16)


def _check(cfg, L, T, m, delta, n_comp=20, s_hi=30.0, s_lo=1.0, style=reuse.HALF, is_key=True, seed=0):
    rng = np.random.Generator(np.random.PCG64(900 + seed))
    solo, cond = _synthetic(cfg, rng, L, T, delta, n_comp, s_hi, s_lo, style, is_key)
    P = cfg.page_size
    n_pages = T // P + 2
    pool = par.make_pool(cfg, L, n_pages, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L, style), pool)
    sigma = torch.zeros((L, cfg.n_kv_heads, m), dtype=torch.float32, device="cuda")
    cond_d = [cond[l].cuda().contiguous() for l in range(L)]
    solo_d = [solo[l].cuda().contiguous() for l in range(L)]
    U, W = ctx.kam_form_patch(cond_d, solo_d, delta, 1 if is_key else 0, m, sigma=sigma)
    torch.cuda.synchronize()
    sg = par.to_f64(sigma)
    for l in range(L):
        base = par.to_f64(solo[l])
        if is_key:
            base = reuse.relocate(base, delta, cfg.theta, cfg.rope_off, cfg.rope_dim, style)
        Uo, Wo, S = reuse.form_patch(par.to_f64(cond[l]), base, m)                       # the oracle: numpy SVD, fp64
        Dl = par.to_f64(cond[l]) - base
        Ug, Wg = par.to_f64(U[l]), par.to_f64(W[l])
        for h in range(cfg.n_kv_heads):
            assert np.all(np.abs(sg[l, h] - S[h, :m]) <= 1e-3 * S[h, :m] + 1e-4 * S[h, 0]), (l, h, sg[l, h], S[h, :m])
            assert np.all(np.diff(sg[l, h]) <= 1e-6)                                     # descending
            po, pg = Uo[:, h] @ Wo[h], Ug[:, h] @ Wg[h]
            rel = np.linalg.norm(pg - po) / np.linalg.norm(po)
            assert rel <= 2.0 ** -7, (l, h, rel)
            tail = float(np.sum(S[h, m:] ** 2))                                          # Eckart-Young: the best possible residual
            res = float(np.sum((Dl[:, h] - pg) ** 2))
            assert res <= tail + (2.0 ** -7 * np.linalg.norm(po)) ** 2 + 1e-9, (l, h, res, tail)
            assert res >= tail * (1 - 1e-6) - 1e-9                                       # and nothing beats it
    if is_key and cfg.has_v is not None:
        # Eq. 1 end to end: relocate the solo chunk with the formed patch -> the pool holds KV(B|A) up to the discarded tail
        bt_h = make_block_table(rng, T // P, n_pages)
        chunk = kam.Chunk(solo_d, [torch.zeros_like(x) for x in solo_d] if cfg.has_v else None)
        zU = [torch.zeros_like(u) for u in U]; zW = [torch.zeros_like(w) for w in W]
        patch = kam.Patch(U, W, zU if cfg.has_v else None, zW if cfg.has_v else None)
        ctx.kam_relocate_patch(torch.from_numpy(bt_h).cuda(), 0, chunk, delta, patch, m)
        torch.cuda.synchronize()
        for l in range(L):
            got = par.pool_rows(pool.k_layers[l], bt_h, 0, T)
            want = par.to_f64(cond[l])
            Dl = want - reuse.relocate(par.to_f64(solo[l]), delta, cfg.theta, cfg.rope_off, cfg.rope_dim, style)
            _, _, S = reuse.form_patch(want, want - Dl, m)
            tail = np.sqrt(np.sum(S[:, m:] ** 2))
            assert np.linalg.norm(got - want) <= 1.05 * tail + 2.0 ** -7 * np.linalg.norm(want)
    ctx.close()


def test_config2_shape_rank16_keys_and_values():
    _check(CONFIGS[2], 2, 512, 16, 12345, seed=1)
    _check(CONFIGS[2], 1, 512, 16, 0, is_key=False, seed=2)


def test_exactly_low_rank_delta_is_reconstructed():
    """rank(Delta_true) = 8 <= m = 16: U W reproduces Delta up to the bf16 rounding of the rows and factors (BASELINE.json's
    'a patch built from an exactly rank-m Delta reconstructs KV(B|A)')."""
    _check(CONFIGS[2], 1, 256, 16, -777, n_comp=8, s_hi=20.0, s_lo=5.0, seed=3)


def test_rank32_and_rank64_config5_shape_ragged_tokens():
    _check(CONFIGS[5], 1, 400, 32, 99999, n_comp=36, s_hi=40.0, s_lo=2.0, seed=4)
    _check(CONFIGS[4].scaled(n_q_heads=4, n_kv_heads=4), 1, 208, 64, -1280, n_comp=70, s_hi=60.0, s_lo=2.0, seed=5)


def test_mla_latent_plus_rope_rows_and_interleaved_pairs():
    _check(CONFIGS[3], 1, 256, 16, 2048, seed=6)
    _check(CONFIGS[2], 1, 128, 16, 31, style=reuse.INTERLEAVED, seed=7)


def test_invalid_arguments():
    cfg = CONFIGS[3]
    pool = par.make_pool(cfg, 1, 4, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    x = [torch.zeros((64, 1, 576), dtype=torch.bfloat16, device="cuda")]
    with pytest.raises(kam.binding.KameraError) as e:
        ctx.kam_form_patch(x, x, 0, 1, 64)                                                # 576 x 72 does not fit shared memory
    assert e.value.status == kam.binding.KAM_ERR_UNSUPPORTED
    with pytest.raises(kam.binding.KameraError):
        ctx.kam_form_patch(x, x, 0, 1, 0)
    ctx.close()
