"""The five workloads of BASELINE.json:configs, as plain data."""
from dataclasses import dataclass, field
from typing import Optional, Tuple


@dataclass(frozen=True)
class ModelShape:
    name: str
    n_layers: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    vocab: int
    rms_eps: float
    rope_theta: float

    @property
    def q_dim(self):
        return self.n_q_heads * self.head_dim

    @property
    def kv_dim(self):
        return self.n_kv_heads * self.head_dim

    def weight_bytes_fp8(self):
        """E4M3 bytes streamed per verify step (all linears incl. LM head)."""
        per_layer = (self.q_dim + 2 * self.kv_dim) * self.hidden + self.hidden * self.q_dim \
            + 2 * self.ffn * self.hidden + self.hidden * self.ffn
        return self.n_layers * per_layer + self.vocab * self.hidden

    def kv_bytes_per_token(self):
        return self.n_layers * 2 * self.kv_dim * 2  # bf16

    def linear_flops_per_token(self):
        return 2 * self.weight_bytes_fp8()

    def attn_flops_per_token_pos(self):
        # q.k and p.v : 2 * 2 * q_dim per layer
        return self.n_layers * 4 * self.q_dim


# BASELINE.json:configs[0]
TINY = ModelShape("tiny", 2, 256, 4, 2, 64, 688, 1024, 1e-5, 1e4)
# BASELINE.json:configs[1]; rope theta per DESIGN.md reading A7 (config is silent)
LLAMA8B = ModelShape("llama8b", 32, 4096, 32, 8, 128, 14336, 128256, 1e-5, 5e5)


@dataclass(frozen=True)
class WorkloadSpec:
    name: str
    model: ModelShape
    seed: int
    batch: int
    ctx_len: Optional[int]                 # fixed context length, or None
    ctx_range: Optional[Tuple[int, int]]   # inclusive range when ctx_len is None
    n_nodes: int                           # T, root included (reading A2)
    tree_caps: Optional[Tuple[int, ...]]   # None = chain
    page_size: int = 16
    act_scale_mode: int = 0                # 0 dynamic per-token, 1 static calibrated
    planted_p: float = 0.0                 # config[3]: P(draft == greedy token)
    calib_tokens: int = 0
    notes: str = ""


CONFIGS = {
    0: WorkloadSpec("cfg0_tiny_b1_chain4", TINY, 0, 1, 128, None, 5, None),
    1: WorkloadSpec("cfg1_8b_b1_L2048_T60", LLAMA8B, 1, 1, 2048, None, 60, (4, 3, 2, 2, 1, 1)),
    2: WorkloadSpec("cfg2_8b_b32_L4096_T26", LLAMA8B, 2, 32, 4096, None, 26, (4, 3, 2, 2, 1)),
    3: WorkloadSpec("cfg3_8b_b64_L1024-8192_chain3", LLAMA8B, 3, 64, None, (1024, 8192), 4, None,
                    planted_p=0.7),
    4: WorkloadSpec("cfg4_8b_b8_L16384_T60_static", LLAMA8B, 4, 8, 16384, None, 60,
                    (4, 3, 2, 2, 1, 1), act_scale_mode=1, calib_tokens=512),
}
