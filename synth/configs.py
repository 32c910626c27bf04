"""The five BASELINE.json workloads as plain records (no arithmetic of the method here)."""
from dataclasses import dataclass, replace


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    kind: str                 # "MHA" | "GQA" | "MLA"
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    row_dim: int              # head_dim; 576 for MLA (512 latent + 64 rope)
    rope_off: int
    rope_dim: int
    has_v: bool
    theta: float
    chunk_tokens: int
    rank: int
    page_size: int
    w_std: float
    elem_dtype: str           # "bf16" | "f32"
    factor_dtype: str
    max_pos: int              # p_target ~ U{0 .. max_pos-1}
    chunks_per_step: int      # chunks relocated per window slide / request
    v_dim: int = 0            # MLA absorbed decode: value = first v_dim columns of the row

    def scaled(self, **kw):
        """Same shape family at a test-friendly size (fewer layers / tokens)."""
        return replace(self, **kw)


CONFIGS = {
    # 1. Tiny MHA, seed 0 (BASELINE.json configs[0]); fp32 K/V/factors as written there.
    1: Config("tiny-mha", 0, "MHA", 1, 4, 4, 64, 0, 64, True, 1e4, 256, 4, 16, 0.1,
              "f32", "f32", 4096, 2),
    # 2. GQA vision-video backbone, Qwen2-VL-7B-like (configs[1]) - the bench workload.
    2: Config("gqa-qwen2vl7b", 1, "GQA", 28, 28, 4, 128, 0, 128, True, 1e6, 1024, 16, 16, 0.05,
              "bf16", "bf16", 32768, 8),
    # 3. MLA backbone, DeepSeek-V2-Lite-like (configs[2]); theta not given there: 1e4 (R-2).
    3: Config("mla-dsv2lite", 2, "MLA", 27, 16, 1, 576, 512, 64, False, 1e4, 1024, 16, 64, 0.05,
              "bf16", "bf16", 4096, 4, v_dim=512),
    # 4. MHA backbone with a sliding 3-screenshot window (configs[3]).
    4: Config("mha-slide3", 3, "MHA", 32, 32, 32, 128, 0, 128, True, 1e4, 1280, 16, 16, 0.05,
              "bf16", "bf16", 8192, 1),
    # 5. Large GQA stress (configs[4]).
    5: Config("gqa-stress", 4, "GQA", 80, 64, 8, 128, 0, 128, True, 5e5, 2048, 32, 16, 0.05,
              "bf16", "bf16", 131072 - 2048, 32),
}
