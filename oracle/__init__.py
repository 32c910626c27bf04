"""CPU oracle for the Kamera KV-reuse hot path (arxiv/paper_2606_23581).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.

It is a plain, slow, fp64 numpy restatement of what the paper's serve-time
operator computes, written from `/root/reference/PAPER.md` (cited as `P:NN`)
under the readings listed in DESIGN.md ("Readings of the paper").  It shares no
code with the CUDA path in `paper_2606_23581_b200/` and never imports it.  Only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import it.

Modules
-------
bf16       round-to-nearest-even fp64 -> bf16, bit packing, ulp          ("one bf16 ULP")
reuse      Eq. 1: RoPE re-rotation R(delta), rank-m patch, paged scatter
window     the position-free window store as a deque + page free list
attention  brute-force softmax attention; per-chunk partials + LSE merge; the same readout for a block of
           query rows with a causal mask over the appended tokens
storage    byte accounting of the stored factors

Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function below is pinned to
something other than itself - closed forms, the identities the paper states
(R(d)R(p)=R(p+d), rank-0 = rotation, exact rank-m reconstruction, LSE merge =
softmax over the concatenation), an independent textbook RoPE restatement, torch's
own bf16 cast, Eckart-Young, brute-force list rebuilds, a dense masked score matrix and torch's
scaled_dot_product_attention (multi-query readout), and the storage ratios the
paper prints (tests/golden/).  No function is "parity unpinned".
"""
