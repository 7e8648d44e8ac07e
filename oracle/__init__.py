"""TEST INFRASTRUCTURE ONLY — the float64 CPU oracle of the candidate evaluator.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It shares no code with the CUDA path (paper_2606_09312_b200/) and never imports it.
"""
from .wm_oracle import (embed_linear, embed_bucket, bucket_index, gelu, layer_norm, step_mlp, step_gru,
                        step_transh, phi_struct, phi_struct_typed, forest_score, scorer, rollout_score_vec, rollout_score_scalar, rollout_latents, rollout_score_from, topk_segments, read_weight_file,
                        score_error, topk_overlap)

__all__ = ["embed_linear", "embed_bucket", "bucket_index", "gelu", "layer_norm", "step_mlp", "step_gru",
           "step_transh", "phi_struct", "phi_struct_typed", "forest_score", "scorer", "rollout_score_vec", "rollout_score_scalar", "rollout_latents", "rollout_score_from", "topk_segments", "read_weight_file",
           "score_error", "topk_overlap"]
