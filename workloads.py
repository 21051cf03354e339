"""Seeded synthetic workloads shared by tests/ and bench.py (BASELINE.json configs C1..C5).

This module holds configuration data only -- generator names, seeds, stream counts, block lengths,
sizes -- and none of the method's arithmetic.  Every input of the hot path is one of these tuples:
PRAND's workloads are "fill an array with numbers from block-split streams",
so there is no dataset; the recipe is stated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass, replace


@dataclass(frozen=True)
class Workload:
    name: str
    gen: str
    seed: int
    n_streams: int
    block_len: int
    n_per_stream: int
    dtype: str          # "u32" | "f32" | "f64"
    seq: bool = False   # True: PRAND's single-sequence fill (prand_generate_seq_*), out[0..n_per_stream)

    @property
    def numbers(self) -> int:
        return self.n_streams * self.n_per_stream

    @property
    def out_bytes(self) -> int:
        return self.numbers * (8 if self.dtype == "f64" else 4)

    def scaled(self, n_streams: int | None = None, n_per_stream: int | None = None) -> "Workload":
        return replace(self, n_streams=n_streams or self.n_streams,
                       n_per_stream=n_per_stream or self.n_per_stream)


# Block lengths "per the paper": powers of two not above Table 4's maxima that keep
# the ensemble points of 2^20 streams disjoint (reading C5).
BLOCK_LEN = {
    "lfsr113": 2 ** 33, "mrg32k3a": 2 ** 76, "mt19937": 2 ** 64,
    "gm19": 2 ** 12, "gm29": 2 ** 26, "gm31": 2 ** 26, "gm55": 2 ** 33, "gm61": 2 ** 33,
    "gq58.1": 2 ** 26, "gq58.3": 2 ** 26, "gq58.4": 2 ** 26,
}
SEED = {"lfsr113": 12345, "mrg32k3a": 12345, "mt19937": 5489}

C1 = Workload("C1", "lfsr113", 12345, 1024, 2 ** 40, 4096, "u32")
C2 = Workload("C2", "mrg32k3a", 12345, 65536, 2 ** 76, 16384, "f64")
C3 = Workload("C3", "mt19937", 5489, 512, 2 ** 64, 2 ** 20, "u32")
C4 = [Workload("C4-gm61", "gm61", 1, 131072, 2 ** 33, 8192, "f32"),
      Workload("C4-gm31", "gm31", 1, 131072, 2 ** 26, 8192, "f32")]
C5_GENS = ["gm19", "gm29", "gm55", "gq58.1", "gq58.3", "gq58.4", "lfsr113", "mrg32k3a", "mt19937"]
C5 = [Workload(f"C5-{g}", g, SEED.get(g, 1), 2 ** 20, BLOCK_LEN[g], 2048, "u32") for g in C5_GENS]

# The paper's Table 7 task: fill an array of 2^29 doubles in GPU memory with ONE
# sequence (the paper repeats it 100 times); the array layout is PRAND's contiguous sections.
T7 = [Workload("T7-mrg32k3a", "mrg32k3a", 12345, 1, 0, 2 ** 29, "f64", True),
      Workload("T7-mt19937", "mt19937", 5489, 1, 0, 2 ** 29, "f64", True)]

ALL = {w.name: w for w in [C1, C2, C3] + C4 + C5 + T7}
HEADLINE = C2        # BASELINE.json configs[1]: the configuration the bench line is quoted on
