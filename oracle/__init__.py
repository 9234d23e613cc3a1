"""CPU oracle of the grouped MoE-layer forward pass -- TEST INFRASTRUCTURE ONLY (see bm_oracle.c)."""
from .oracle import (build, canon_dot, route, moe_forward, unite_weights, expert_histogram, expert_outputs,
                     cosine_matrix, group_mse, num_threads)

__all__ = ["build", "canon_dot", "route", "moe_forward", "unite_weights", "expert_histogram", "expert_outputs",
           "cosine_matrix", "group_mse", "num_threads"]
