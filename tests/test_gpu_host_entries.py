"""GPU parity of the host-buffer entries (the e2e path of bench.py): kam_relocate_patch_host and kam_paged_decode_merge_host.
The chunk and its factors live in HOST memory - as separate pinned tensors, as ONE pinned slab (the library merges copies whose
source and staging destination are contiguous), and as pageable memory - and the result in the pool must match the oracle
exactly as for the device entry; the host decode must return the bits of the device decode."""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from synth import CONFIGS, make_block_table, make_chunk, make_query
from tests import parity as par

pytestmark = pytest.mark.gpu


def _host_lists(ch, mode):
    L = ch["K"].shape[0]
    names = ["K", "V", "Uk", "Wk", "Uv", "Wv"]
    present = [n for n in names if ch[n] is not None]
    if mode == "slab":
        n = sum(ch[x][l].numel() for l in range(L) for x in present)
        buf = torch.empty(n, dtype=ch["K"].dtype).pin_memory()
        out, off = {x: [] for x in names}, 0
        for l in range(L):
            for x in present:
                t = ch[x][l]
                v = buf[off:off + t.numel()].view(t.shape)
                v.copy_(t)
                out[x].append(v)
                off += t.numel()
        out["_keep"] = buf
    else:
        out = {x: [(ch[x][l].contiguous().pin_memory() if mode == "pinned" else ch[x][l].contiguous().clone()) for l in range(L)]
               for x in present}
    return [out.get(x) or None for x in names], out


@pytest.mark.parametrize("mode,overlap", [("pinned", 0), ("pinned", 1), ("slab", 0), ("slab", 1), ("pageable", 0)])
@pytest.mark.parametrize("cfg_id,m", [(2, 16), (3, 16), (2, 0)])
def test_relocate_patch_host_matches_oracle(cfg_id, m, mode, overlap):
    cfg = CONFIGS[cfg_id]
    L, T, P = 3, 272, cfg.page_size
    rng = np.random.Generator(np.random.PCG64(400 + cfg_id + m))
    ch = make_chunk(cfg, rng, n_tokens=T, n_layers=L, rank=max(m, 16))
    dst0 = 2 * P + 5
    n_pages = (dst0 + T + P - 1) // P
    bt_h = make_block_table(rng, n_pages, n_pages + 3)
    pool = par.make_pool(cfg, L, n_pages + 3, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    ctx.kam_set_option("host_copy_overlap", overlap)                # 1: the library's own copy stream + two staging buffers (opt-in)
    (k, v, uk, wk, uv, wv), keep = _host_lists(ch, mode)
    p_target = 31337
    for _ in range(2 + overlap):                                             # twice: the staging buffer and its pointer tables are reused
        ctx.kam_relocate_patch_host(torch.from_numpy(bt_h).cuda(), dst0, T, 0, p_target, k, v, uk, wk, uv, wv, m)
    torch.cuda.synchronize()
    st = par.check_relocated(cfg, pool, ch, bt_h, dst0, p_target, m)
    assert st["fail"] == 0
    assert par.untouched_pages_intact(pool, bt_h, L)
    ctx.close()


def test_relocate_patch_host_reads_stream_ordered_host_data_in_stream_order():
    """The evict-to-host-then-recall pattern of P:88: the pinned host slab is still being FILLED by a device-to-host copy enqueued on
    the caller's stream (held back behind a long kernel) when kam_relocate_patch_host is called.  With the default options the
    library's copies are ordered on that stream, so the recall must see the evicted bits, not the slab's stale contents."""
    cfg = CONFIGS[2]
    L, T, P, m = 2, 256, cfg.page_size, 16
    rng = np.random.Generator(np.random.PCG64(77))
    ch = make_chunk(cfg, rng, n_tokens=T, n_layers=L, rank=m)
    n_pages = T // P
    bt_h = make_block_table(rng, n_pages, n_pages + 2)
    pool = par.make_pool(cfg, L, n_pages + 2, torch.bfloat16)
    ctx = kam.Context(par.layout_of(cfg, L), pool)
    names = ("K", "V", "Uk", "Wk", "Uv", "Wv")
    dev = {x: [ch[x][l].contiguous().cuda() for l in range(L)] for x in names}
    host = {x: [torch.full(ch[x][l].shape, 3.0, dtype=ch[x][l].dtype).pin_memory() for l in range(L)] for x in names}   # stale contents
    bt_d = torch.from_numpy(bt_h).cuda()
    torch.cuda.synchronize()
    torch.cuda._sleep(200_000_000)                                  # ~0.1 s of device time in front of the eviction copies
    for x in names:
        for l in range(L):
            host[x][l].copy_(dev[x][l], non_blocking=True)          # "evict to the host store", stream-ordered
    ctx.kam_relocate_patch_host(bt_d, 0, T, 0, 4242, *[host[x] for x in names], m)
    torch.cuda.synchronize()
    assert par.check_relocated(cfg, pool, ch, bt_h, 0, 4242, m)["fail"] == 0
    ctx.close()


def test_paged_decode_merge_host_returns_the_device_bits():
    cfg = CONFIGS[2]
    rng = np.random.Generator(np.random.PCG64(77))
    P, T = cfg.page_size, 400
    n_pages = (T + P - 1) // P
    pool = kam.Pool([torch.randn((n_pages + 2, P, cfg.n_kv_heads, cfg.row_dim), device="cuda").to(torch.bfloat16)],
                    [torch.randn((n_pages + 2, P, cfg.n_kv_heads, cfg.row_dim), device="cuda").to(torch.bfloat16)])
    ctx = kam.Context(par.layout_of(cfg, 1), pool)
    bt = torch.from_numpy(make_block_table(rng, n_pages, n_pages + 2)).cuda().reshape(1, -1)
    starts = torch.tensor([[0, 150, T]], dtype=torch.int32, device="cuda")
    offs = torch.tensor([[0, -1234]], dtype=torch.int64, device="cuda")
    nc = torch.tensor([2], dtype=torch.int32, device="cuda")
    q = make_query(cfg, rng, 1)
    out_d = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
    lse_d = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32, device="cuda")
    ctx.kam_paged_decode_merge(q.cuda(), bt, starts, offs, nc, 0, 0.09, out_d, lse_d)
    q_h = q.pin_memory()
    out_h = torch.zeros((1, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16).pin_memory()
    lse_h = torch.zeros((1, cfg.n_q_heads), dtype=torch.float32).pin_memory()
    ctx.kam_paged_decode_merge_host(q_h, bt, starts, offs, nc, 0, 0.09, out_h, lse_h)       # synchronises the stream itself
    assert torch.equal(out_h, out_d.cpu()) and torch.equal(lse_h, lse_d.cpu())
    ctx.close()
