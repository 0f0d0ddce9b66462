"""Seeded synthetic input generators for the five BASELINE.json configs.

This package serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench).  It holds
no HDC arithmetic: it only draws random arrays and lays them out in the interface formats
(`include/hdc.h`): fp32 / bf16-representable features, uint8 level indices, packed-bit tables.
"""
from .gen import (  # noqa: F401
    BASE_SEED, rng_for, pack_bits_lsb, to_bf16_bits, from_bf16_bits,
    c1_tiny, c2_isolet_shaped, c3_mnist_shaped, c4_har_shaped, c5_large_batch,
    level_table, id_table, tile_rows,
)
