"""The five BASELINE.json workloads as named presets, and the fraction -> count rule.

Host-side bookkeeping only (no method arithmetic): used by tests, bench.py and the
input generator.  Shapes follow BASELINE.json `configs`; n_sink / n_recent of configs
3 and 4 are not stated there and inherit the pattern of the others (n_sink=4,
n_recent=P) -- DESIGN.md, reading R7.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace


@dataclass(frozen=True)
class EvictConfig:
    name: str
    config_id: int
    layers: int
    batch: int
    L: int
    Hq: int
    Hkv: int
    d: int
    dtype: str  # "f32" | "bf16"
    P: int
    f_total: float  # kept fraction of L
    f_proxy: float  # share of L kept by Proxy-Tokens Eviction (includes the protected tokens, R7)
    n_sink: int
    n_recent: int
    hh_rate: float  # heavy-hitter rate of the synthetic generator
    hh_alpha: float
    seed: int = 0

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def elem_bytes(self) -> int:
        return 4 if self.dtype == "f32" else 2

    def budgets(self) -> tuple[int, int]:
        return budget_counts(self.L, self.f_total, self.f_proxy)

    @property
    def C(self) -> int:
        bp, br = self.budgets()
        return bp + br

    def alg_bytes_per_layer(self) -> int:
        """K read once for scoring + C rows of K and V read and written (BASELINE.json north star;
        SURVEY.md 8(d)):  B*Hkv*d*e*(L + 4C)."""
        return self.batch * self.Hkv * self.d * self.elem_bytes * (self.L + 4 * self.C)

    def layer_seed(self, layer: int) -> int:
        """Eviction seed of one layer: seed XOR layer (BASELINE.json config 3; R10)."""
        return self.seed ^ layer

    def data_seed(self, layer: int) -> int:
        return 1000 * self.config_id + layer

    def scaled(self, **kw) -> "EvictConfig":
        return replace(self, **kw)


def budget_counts(L: int, f_total: float, f_proxy: float) -> tuple[int, int]:
    """DESIGN.md R8: C = floor(f_total*L), Bp = floor(f_proxy*L), Br = C - Bp (remainder -> random).
    A tiny epsilon keeps exact decimal fractions (0.15*4096 = 614.4, 0.2*512 = 102.4) from
    flooring one short through binary representation error."""
    C = int(math.floor(f_total * L + 1e-9))
    Bp = int(math.floor(f_proxy * L + 1e-9))
    return Bp, C - Bp


CONFIGS = {
    1: EvictConfig("cfg1_tiny", 1, 1, 1, 512, 4, 4, 64, "f32", 16, 0.20, 0.15, 4, 16, 0.01, 4.0),
    2: EvictConfig("cfg2_llama2_7b_1layer", 2, 1, 1, 4096, 32, 32, 128, "bf16", 32, 0.20, 0.15, 4, 32, 0.01, 4.0),
    3: EvictConfig("cfg3_llama2_7b_prefill_16k", 3, 32, 1, 16384, 32, 32, 128, "bf16", 32, 0.20, 0.15, 4, 32, 0.005, 4.0),
    4: EvictConfig("cfg4_mistral_7b_gqa_32k", 4, 32, 4, 32768, 32, 8, 128, "bf16", 64, 0.20, 0.15, 4, 64, 0.005, 4.0),
    5: EvictConfig("cfg5_llama3_8b_128k", 5, 32, 1, 131072, 32, 8, 128, "bf16", 64, 0.10, 0.08, 4, 64, 0.002, 5.0),
}
