"""Seeded synthetic inputs for the Tropical multiplexed-iteration hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_16264_b200/``).  It holds none of the method's arithmetic: it only
draws lengths, page placements and N(0,1) values, rounds the values to bf16 bit
patterns and lays them out in the paged pool.  numpy only -- no torch, no CUDA.

Recipe: SURVEY.md section 8(d) (restated in DESIGN.md "Input recipe"); it stands in
for the Mooncake trace / InternLM-20B shapes the paper measures on
(PAPER.md:169-171), which are not available here.
"""
from .workloads import (  # noqa: F401
    CONFIG_NAMES,
    POISON_BF16,
    StepInputs,
    bf16_bits_to_f32,
    config_lengths,
    f32_to_bf16_bits,
    make_config,
    make_migration_target,
    make_rope_tables,
    make_step,
    needed_pages,
)
