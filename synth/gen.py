"""Seeded generators (shapes, seeds, distributions, dtype casts only)."""
import numpy as np
import torch


def torch_dtype(name):
    return {"bf16": torch.bfloat16, "f32": torch.float32}[name]


def _normal(rng, shape, std, dtype):
    x = rng.standard_normal(size=shape, dtype=np.float32) * np.float32(std)
    return torch.from_numpy(x).to(dtype)           # torch's own RNE cast for bf16


def make_chunk(cfg, rng, n_tokens=None, n_layers=None, rank=None):
    """One position-free canonical chunk and its rank-m patch, CPU tensors in storage dtype.

    Draw order is fixed: K, V, U_k, W_k, U_v, W_v.
      K, V   [L, T, H, D]     U [L, T, H, m]     W [L, H, m, D]
    """
    T = cfg.chunk_tokens if n_tokens is None else n_tokens
    L = cfg.n_layers if n_layers is None else n_layers
    m = cfg.rank if rank is None else rank
    H, D = cfg.n_kv_heads, cfg.row_dim
    et, ft = torch_dtype(cfg.elem_dtype), torch_dtype(cfg.factor_dtype)
    out = {"K": _normal(rng, (L, T, H, D), 1.0, et)}
    out["V"] = _normal(rng, (L, T, H, D), 1.0, et) if cfg.has_v else None
    out["Uk"] = _normal(rng, (L, T, H, m), 1.0, ft)
    out["Wk"] = _normal(rng, (L, H, m, D), cfg.w_std, ft)
    out["Uv"] = _normal(rng, (L, T, H, m), 1.0, ft) if cfg.has_v else None
    out["Wv"] = _normal(rng, (L, H, m, D), cfg.w_std, ft) if cfg.has_v else None
    return out


def make_offsets(cfg, rng, n):
    """n target offsets p ~ U{0 .. max_pos-1} (int64)."""
    return rng.integers(0, cfg.max_pos, size=n, dtype=np.int64)


def make_block_table(rng, n_pages_used, num_pages):
    """A random choice of distinct physical pages, in random order (int32)."""
    return rng.permutation(num_pages)[:n_pages_used].astype(np.int32)


def make_query(cfg, rng, batch):
    """Decode queries [B, Hq, D] ~ N(0,1), bf16."""
    return _normal(rng, (batch, cfg.n_q_heads, cfg.row_dim), 1.0, torch.bfloat16)


def randn_device(shape, seed, std, dtype, device):
    """Large tensors generated on the device (configs 4-5): the bits on the device are the ground
    truth - whoever verifies reads them back; nothing regenerates them."""
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    x = torch.empty(shape, dtype=dtype, device=device)
    x.normal_(0.0, float(std), generator=g)
    return x
