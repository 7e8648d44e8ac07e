"""The five BASELINE.json configs as data (binding parametrisation: SURVEY.md §8 table).

Italic entries of that table (readings where BASELINE.json is silent) are listed in
DESIGN.md §3 with their S-numbers.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Tuple

KIND_MLP, KIND_MLP_LN, KIND_GRU, KIND_TRANSH = 0, 1, 2, 3
DTYPE_FP32, DTYPE_BF16 = 0, 1
EMBED_LINEAR, EMBED_BUCKET = 0, 1
PHI_MEAN, PHI_STRUCT, PHI_TYPED = 0, 1, 2     # action features of the ranker: mean action embedding | structured statistics
                                              # pooled per parameter slot (f2, S25) | kept per action type (f2, S28)
RANKER_MLP, RANKER_FOREST = 0, 1   # G: the configs' MLP | a tree ensemble, the paper's own kind of ranker (f4)


@dataclass(frozen=True)
class WMConfig:
    name: str
    number: int                 # 1..5 (BASELINE.json configs[number-1]); 6, 7 = NEXT row f1; 8, 9 = NEXT row f2
    kind: int                   # KIND_*
    dtype: int                  # DTYPE_*
    embed: int                  # EMBED_*
    S: int                      # subgraphs
    per_subgraph: int           # candidates per subgraph
    T_max: int
    len_dist: str               # 'uniform' | 'zipf' | 'const'
    len_lo: int
    len_hi: int
    n_types: int
    P: int
    param_dist: str             # 'uniform' | 'loguniform'
    param_hi: int
    n_buckets: int              # EMBED_BUCKET only, else 0
    d: int
    d_a: int
    hidden: int                 # 0 for GRU
    H: int
    scorer_widths: Tuple[int, ...]   # hidden widths of G; linears = len+1
    k: int
    ln_eps: float = 1e-5
    weight_seed: int = 0
    prefix_children: int = 0    # cfg 4: children per parent (0 = no shared-prefix structure)
    prefix_cut_lo: int = 0
    prefix_cut_hi: int = 0
    phi_kind: int = PHI_MEAN    # PHI_STRUCT: the paper's structured action features (S25)
    ranker_kind: int = RANKER_MLP   # RANKER_FOREST: synthetic complete binary trees (S27)
    n_trees: int = 0
    tree_depth: int = 0

    @property
    def B(self) -> int:
        return self.S * self.per_subgraph

    @property
    def input_seed(self) -> int:
        return 1000 + self.number

    @property
    def phi_dim(self) -> int:
        """Width of phi: d_a for the mean action embedding; per-type counts, length and per-slot sum / mean / max of
        log2 params for the structured form."""
        if self.phi_kind == PHI_TYPED:
            return self.n_types + 1 + 3 * self.n_types * self.P
        return self.d_a if self.phi_kind == PHI_MEAN else self.n_types + 1 + 3 * self.P

    @property
    def scorer_in(self) -> int:
        return self.d + self.phi_dim + self.H

    def scaled(self, S: int | None = None, per_subgraph: int | None = None) -> "WMConfig":
        """Same model, smaller batch (parity-test and cpu-baseline samples)."""
        return replace(self, S=self.S if S is None else S,
                       per_subgraph=self.per_subgraph if per_subgraph is None else per_subgraph)

    def flops_per_step(self) -> int:
        """Literal transition FLOP per rollout step."""
        if self.kind == KIND_GRU:
            return 2 * 3 * self.d * (self.d + self.d_a)
        if self.kind == KIND_TRANSH:   # W_w a, W_d a, then the residual MLP (the projection / norms are O(d))
            return 2 * (2 * self.d * self.d_a + self.hidden * (self.d + self.d_a) + self.d * self.hidden)
        return 2 * (self.hidden * (self.d + self.d_a) + self.d * self.hidden)

    def flops_scorer(self) -> int:
        if self.ranker_kind == RANKER_FOREST:     # comparisons and adds, not a contraction: counted as 0 FLOP
            return 0
        dims = (self.scorer_in,) + tuple(self.scorer_widths) + (1,)
        return 2 * sum(a * b for a, b in zip(dims[:-1], dims[1:]))


CONFIGS = {
    1: WMConfig("cfg1_tiny_fp32", 1, KIND_MLP, DTYPE_FP32, EMBED_LINEAR, S=1, per_subgraph=64, T_max=8,
                len_dist="uniform", len_lo=0, len_hi=8, n_types=16, P=4, param_dist="uniform", param_hi=64,
                n_buckets=0, d=64, d_a=32, hidden=128, H=8, scorer_widths=(128,), k=8),
    2: WMConfig("cfg2_evolution_round", 2, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(512, 512), k=64),
    3: WMConfig("cfg3_throughput_sweep", 3, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=64, per_subgraph=1024,
                T_max=48, len_dist="zipf", len_lo=4, len_hi=48, n_types=48, P=8, param_dist="loguniform",
                param_hi=1024, n_buckets=0, d=512, d_a=256, hidden=1024, H=32, scorer_widths=(1024, 1024),
                k=128),
    4: WMConfig("cfg4_shared_prefix", 4, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=128, per_subgraph=16384,
                T_max=32, len_dist="const", len_lo=32, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=768, H=16, scorer_widths=(512, 512), k=32,
                prefix_children=64, prefix_cut_lo=16, prefix_cut_hi=28),
    5: WMConfig("cfg5_gated", 5, KIND_GRU, DTYPE_BF16, EMBED_BUCKET, S=128, per_subgraph=16384, T_max=64,
                len_dist="uniform", len_lo=16, len_hi=64, n_types=32, P=8, param_dist="loguniform",
                param_hi=1024, n_buckets=40, d=384, d_a=128, hidden=0, H=32, scorer_widths=(768, 768), k=64),
    # NEXT row f1: the paper's TransH-style transition, not a BASELINE.json config.
    # 6 = cfg 1's shapes (fp32, the parity case), 7 = cfg 2's shapes and batch (the measurement case).
    6: WMConfig("f1_transh_tiny_fp32", 6, KIND_TRANSH, DTYPE_FP32, EMBED_LINEAR, S=1, per_subgraph=64, T_max=8,
                len_dist="uniform", len_lo=0, len_hi=8, n_types=16, P=4, param_dist="uniform", param_hi=64,
                n_buckets=0, d=64, d_a=32, hidden=128, H=8, scorer_widths=(128,), k=8),
    7: WMConfig("f1_transh_evolution_round", 7, KIND_TRANSH, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(512, 512), k=64),
    # NEXT row f2: the paper's structured action features phi in place of the mean
    # action embedding.  8 = cfg 1's shapes (fp32, the parity case), 9 = cfg 2's shapes and batch (the measurement case).
    8: WMConfig("f2_structphi_tiny_fp32", 8, KIND_MLP, DTYPE_FP32, EMBED_LINEAR, S=1, per_subgraph=64, T_max=8,
                len_dist="uniform", len_lo=0, len_hi=8, n_types=16, P=4, param_dist="uniform", param_hi=64,
                n_buckets=0, d=64, d_a=32, hidden=128, H=8, scorer_widths=(128,), k=8, phi_kind=PHI_STRUCT),
    9: WMConfig("f2_structphi_evolution_round", 9, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(512, 512), k=64,
                phi_kind=PHI_STRUCT),
    # NEXT row f4: a tree-ensemble ranker (the paper's G is an XGBoost model) on synthetic
    # random trees over [z_T ; structured phi ; h].  10 = cfg 1's shapes (fp32), 11 = cfg 2's shapes and batch.
    10: WMConfig("f4_forest_tiny_fp32", 10, KIND_MLP, DTYPE_FP32, EMBED_LINEAR, S=1, per_subgraph=64, T_max=8,
                 len_dist="uniform", len_lo=0, len_hi=8, n_types=16, P=4, param_dist="uniform", param_hi=64,
                 n_buckets=0, d=64, d_a=32, hidden=128, H=8, scorer_widths=(), k=8, phi_kind=PHI_STRUCT,
                 ranker_kind=RANKER_FOREST, n_trees=32, tree_depth=4),
    11: WMConfig("f4_forest_evolution_round", 11, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                 T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                 param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(), k=64,
                 phi_kind=PHI_STRUCT, ranker_kind=RANKER_FOREST, n_trees=128, tree_depth=6),
    # The paper's own choice for every component at once (not a BASELINE.json config): TransH-style transition (f1),
    # structured phi (f2), tree-ensemble ranker (f4), on cfg 2's shapes and batch.
    12: WMConfig("paper_stack_evolution_round", 12, KIND_TRANSH, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                 T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                 param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(), k=64,
                 phi_kind=PHI_STRUCT, ranker_kind=RANKER_FOREST, n_trees=128, tree_depth=6),
    # NEXT row f2 as SURVEY.md §8(f) words it — PER-TYPE numeric statistics ("action-specific numeric attributes",
    # PAPER.md:186; S28).  13 = cfg 1's shapes (fp32, 209 features), 14 = cfg 2's shapes and batch (609 features).
    13: WMConfig("f2_typedphi_tiny_fp32", 13, KIND_MLP, DTYPE_FP32, EMBED_LINEAR, S=1, per_subgraph=64, T_max=8,
                 len_dist="uniform", len_lo=0, len_hi=8, n_types=16, P=4, param_dist="uniform", param_hi=64,
                 n_buckets=0, d=64, d_a=32, hidden=128, H=8, scorer_widths=(128,), k=8, phi_kind=PHI_TYPED),
    14: WMConfig("f2_typedphi_evolution_round", 14, KIND_MLP_LN, DTYPE_BF16, EMBED_LINEAR, S=16, per_subgraph=2048,
                 T_max=32, len_dist="uniform", len_lo=8, len_hi=32, n_types=32, P=6, param_dist="loguniform",
                 param_hi=1024, n_buckets=0, d=256, d_a=128, hidden=512, H=16, scorer_widths=(512, 512), k=64,
                 phi_kind=PHI_TYPED),
}


def get_config(number: int) -> WMConfig:
    return CONFIGS[number]
