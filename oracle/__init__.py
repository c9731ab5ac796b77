"""fp64 CPU oracle for Sparrow's sparse decode attention -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the CUDA
library in ``paper_2606_08446_b200`` and never imports it.  See ``sparrow_oracle.c``
for the algorithm and its citations.
"""
from .oracle import (  # noqa: F401
    Schedule,
    build,
    budget_tokens,
    k_pages,
    forced_pages,
    summarize,
    scores_unit,
    select_unit,
    attention_unit,
    attention_partial_unit,
    lse_merge,
    sparse_step,
    attention_on_sets,
    dense_step,
    append_step,
    rollout,
    cost_model,
    acceptance_rate,
    binned_quantile,
    summarize_mean,
    mean_landmark_band,
    sparse_step_mean,
    num_threads,
)
