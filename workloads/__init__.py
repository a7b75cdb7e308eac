"""Seeded synthetic input generators for the paged-KV attention hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_12688_b200/``) and therefore holds none of the method's
arithmetic: it only draws random numbers, rounds them to bf16 bit patterns
and lays out pages / block tables / slot mappings.  It imports neither side.

The five configurations are those of ``BASELINE.json:configs``; the recipe
(seeds, draw order, distributions) is SURVEY.md section 8(d) and is restated
in DESIGN.md ("Input recipe").  They stand in for the paper's VBench /
Seed-TTS / Food101 / DROID workloads: only shapes
and length distributions are taken, no item of those suites is reproduced.
"""
from .generators import (  # noqa: F401
    BF16_NAN,
    PagedBatch,
    bf16_bits_from_f32,
    f64_from_bf16_bits,
    make_batch,
    config1_tiny_decode,
    config2_bagel_cfg_decode,
    config3_prefill,
    config4_thinker,
    config4_talker,
    config5_long_context,
    flow_step_bagel,
    cfg_cascade_decode,
    fp8_page_scales,
    CONFIG_SEED_BASE,
)
from .adversarial import KINDS as ADVERSARIAL_KINDS, logical_kv, make_adversarial, overwrite_k, overwrite_v  # noqa: F401
