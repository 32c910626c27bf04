"""kam_paged_decode_merge_static: the fused decode for hosts that may not allocate device memory (include/kamera.h).

Why the entry exists: every other decode call goes through a kam_ctx, and a context calls cudaMalloc - when it is created and
whenever a call outgrows its plan / partials workspace or names a new pool.  A serving engine that reserved all of HBM for its
own KV allocator at start-up, a plug-in running under somebody else's memory budget, or a loop that cannot pay cudaMalloc's
device-wide synchronisation has no use for such a call.  The static entry keeps its scratch (plan, cos/sin rows, softmax partials)
in a 16 MiB `static __device__` array inside libkamera.so and takes the layout and the pool directly.

What is checked here, on two calls in a row that share that array (different batch sizes and chunk structures, so the second
call runs over the first one's leftovers): the output equals the context path's within the decode tests' bar (max-abs 2e-2,
relative 1e-2, lse 1e-3 - tests/test_gpu_decode.py), the second call leaves the device's free memory untouched, and a problem
that does not fit the array is refused with a message instead of being launched.

This file sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the static call comes FIRST, before any context exists) and after the others.
"""
import numpy as np
import pytest
import torch

import paper_2606_23581_b200 as kam
from oracle import attention as att
from paper_2606_23581_b200 import binding as B
from synth import CONFIGS, make_block_table, make_query, randn_device
from tests import parity as par

pytestmark = pytest.mark.gpu


def _problem(cfg, lens, deltas, seed, L=2):
    """A paged pool of L layers and the CSR metadata of `lens` / `deltas` (one list per request), all on the device."""
    rng = np.random.Generator(np.random.PCG64(seed))
    P = cfg.page_size
    batch = len(lens)
    max_chunks = max(1, max(len(x) for x in lens))
    max_pages = max(1, max((sum(x) + P - 1) // P for x in lens))
    num_pages = batch * max_pages + 5
    shape = (num_pages, P, cfg.n_kv_heads, cfg.row_dim)
    pool = kam.Pool([randn_device(shape, seed + 2 * l, 1.0, torch.bfloat16, "cuda") for l in range(L)],
                    [randn_device(shape, seed + 2 * l + 1, 1.0, torch.bfloat16, "cuda") for l in range(L)])
    perm = make_block_table(rng, batch * max_pages, num_pages).reshape(batch, max_pages)
    starts = np.zeros((batch, max_chunks + 1), np.int32)
    offs = np.zeros((batch, max_chunks), np.int64)
    ncs = np.array([len(x) for x in lens], np.int32)
    for b in range(batch):
        for c, n in enumerate(lens[b]):
            starts[b, c + 1] = starts[b, c] + n
            offs[b, c] = deltas[b][c]
        starts[b, len(lens[b]) + 1:] = starts[b, len(lens[b])]
    q = make_query(cfg, rng, batch)
    meta = (torch.from_numpy(perm).cuda(), torch.from_numpy(starts).cuda(), torch.from_numpy(offs).cuda(), torch.from_numpy(ncs).cuda())
    return dict(cfg=cfg, L=L, pool=pool, perm=perm, lens=lens, deltas=deltas, q=q, qd=q.cuda(), meta=meta, batch=batch,
                scale=cfg.row_dim ** -0.5)


def _outputs(pr, fill):
    cfg = pr["cfg"]
    return (torch.full((pr["batch"], cfg.n_q_heads, cfg.row_dim), fill, dtype=torch.bfloat16, device="cuda"),
            torch.full((pr["batch"], cfg.n_q_heads), fill, dtype=torch.float32, device="cuda"))


def _static(pr, layer, out, lse):
    kam.kam_paged_decode_merge_static(par.layout_of(pr["cfg"], pr["L"]), pr["qd"], pr["pool"], *pr["meta"], layer, pr["scale"], out, lse)


def _context(pr, layer, tma=1):
    ctx = kam.Context(par.layout_of(pr["cfg"], pr["L"]), pr["pool"])
    ctx.kam_set_option("decode_tma", tma)
    out, lse = _outputs(pr, 3.0)
    ctx.kam_paged_decode_merge(pr["qd"], *pr["meta"], layer, pr["scale"], out, lse)
    torch.cuda.synchronize()
    ctx.close()
    return out, lse


def _within_bar(out_a, lse_a, out_b, lse_b, what):
    """The decode tests' bar (tests/test_gpu_decode.py:check_attention), between two device results."""
    oa, ob, la, lb = par.to_f64(out_a), par.to_f64(out_b), par.to_f64(lse_a), par.to_f64(lse_b)
    fin = np.isfinite(lb)
    assert np.array_equal(np.isfinite(la), fin), what
    assert np.all(np.isneginf(la[~fin])) and np.all(oa[~fin] == 0), what
    err = np.abs(oa[fin] - ob[fin])
    assert err.max() <= 2e-2, (what, "max-abs", float(err.max()))
    assert (err.max(axis=1) / np.abs(ob[fin]).max(axis=1)).max() <= 1e-2, (what, "max-rel")
    assert np.abs(la[fin] - lb[fin]).max() <= 1e-3, (what, "lse")
    return bool(torch.equal(out_a, out_b) and torch.equal(lse_a, lse_b))


def test_static_scratch_decode_matches_the_context_path_on_two_calls_in_a_row():
    cfg = CONFIGS[2]                                                # GQA 28 query / 4 KV heads, head_dim 128
    # call 1: three requests, ragged chunks that straddle tiles and pages, offsets pending on read, one request with no tokens
    a = _problem(cfg, [[100, 1024, 37], [], [5, 16, 300, 700]], [[0, 31000, -77], [], [0, 0, -1280, 99999]], seed=41)
    # call 2: another batch size, chunk count and layer - it finds call 1's plan and partials in the array
    b = _problem(cfg, [[640], [33, 2000], [16], [512, 512, 512, 512, 512], [1]], [[-5], [0, 123456], [7], [0, 1, 2, 3, 4], [0]], seed=42)
    out_a, lse_a = _outputs(a, 7.0)
    out_b, lse_b = _outputs(b, 7.0)
    torch.cuda.synchronize()

    _static(a, 1, out_a, lse_a)                                     # in a fresh process: the library's very first CUDA work
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    _static(b, 0, out_b, lse_b)                                     # second call in a row, same stream, nothing in between
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the static entry changed the device's free memory"

    for name, pr, layer, out, lse in (("call 1", a, 1, out_a, lse_a), ("call 2", b, 0, out_b, lse_b)):
        ref_out, ref_lse = _context(pr, layer)                      # the existing path: tensor-map boxes, context workspace
        same = _within_bar(out, lse, ref_out, ref_lse, name + " vs kam_paged_decode_merge")
        alt_out, alt_lse = _context(pr, layer, tma=0)               # the context path on the same per-token copies
        same0 = _within_bar(out, lse, alt_out, alt_lse, name + " vs kam_paged_decode_merge (decode_tma = 0)")
        print("%s: bit-equal to the context path: %s (tensor maps), %s (per-token copies)" % (name, same, same0))

    # and against the paper's definition, for the request with the most chunks of call 2
    r, t0, chunks = 3, 0, []
    for c, n in enumerate(b["lens"][r]):
        chunks.append({"k": par.pool_rows(b["pool"].k_layers[0], b["perm"][r], t0, n),
                       "v": par.pool_rows(b["pool"].v_layers[0], b["perm"][r], t0, n), "delta": int(b["deltas"][r][c])})
        t0 += n
    o, l = att.attend_bruteforce(par.to_f64(b["q"][r]), chunks, b["scale"], par.rope_kw(cfg))
    assert np.abs(par.to_f64(out_b)[r] - o).max() <= 2e-2 and np.abs(par.to_f64(lse_b)[r] - l).max() <= 1e-3

    # a third call repeats call 1 over call 2's leftovers: same bits as the first time
    out_c, lse_c = _outputs(a, 9.0)
    _static(a, 1, out_c, lse_c)
    torch.cuda.synchronize()
    assert torch.equal(out_c, out_a) and torch.equal(lse_c, lse_a)


def test_static_scratch_decode_refuses_what_does_not_fit():
    cfg = CONFIGS[2]
    batch, max_chunks, max_pages = 64, 64, 4                        # 4096 chunk slots: ~65 MB of partials, the array has 16 MiB
    bt = torch.zeros((batch, max_pages), dtype=torch.int32, device="cuda")
    starts = torch.zeros((batch, max_chunks + 1), dtype=torch.int32, device="cuda")
    ncs = torch.zeros(batch, dtype=torch.int32, device="cuda")
    shape = (8, cfg.page_size, cfg.n_kv_heads, cfg.row_dim)
    pool = kam.Pool([torch.zeros(shape, dtype=torch.bfloat16, device="cuda")], [torch.zeros(shape, dtype=torch.bfloat16, device="cuda")])
    q = torch.zeros((batch, cfg.n_q_heads, cfg.row_dim), dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, 5.0)
    lse = torch.full((batch, cfg.n_q_heads), 5.0, dtype=torch.float32, device="cuda")
    with pytest.raises(kam.KameraError) as e:
        kam.kam_paged_decode_merge_static(par.layout_of(cfg, 1), q, pool, bt, starts, None, ncs, 0, 1.0, out, lse)
    assert e.value.status == B.KAM_ERR_INVALID_ARG
    assert "KAM_STATIC_SCRATCH_BYTES" in str(e.value) and str(B.KAM_STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 5.0).all()) and bool((lse == 5.0).all())   # nothing was launched
    # MLA needs tensor maps (device memory of their own): refused by name, not attempted
    with pytest.raises(kam.KameraError) as e:
        kam.kam_paged_decode_merge_static(par.layout_of(CONFIGS[3], 1), q, pool, bt, starts, None, ncs, 0, 1.0, out, lse)
    assert e.value.status == B.KAM_ERR_UNSUPPORTED
