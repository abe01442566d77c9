"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs[0..4]).

This module holds NONE of the method's arithmetic: it only draws random coefficients,
delays and strain, rounds them to the types the library takes (complex64 / int32 /
float32) and counts filter-sample updates (the unit of BASELINE.json's metric,
PAPER.md:88 "12 floating operations" per filter per data point).  Both the CUDA path and
the oracle are fed the arrays produced here (the oracle must promote the
*same rounded* a1, b0).  It imports neither of them.

Recipe: numpy ``default_rng(SeedSequence([1702, 2256, cfg, sub]))``
with sub-streams spawned in the fixed order |a1|, arg a1, Re b0, Im b0, delays, strain.
|a1| ~ U[lo, hi], arg a1 ~ U[0, 2pi), b0 = 1e-3 * CN(0, 1) (re, im iid N(0, 1/2), reading F7),
d ~ U{0..d_max}, x ~ N(0, 1) float32.  These stand in for real SPIIR banks and whitened
LIGO strain, which are not available here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np


@dataclass(frozen=True)
class Bank:
    """One rate's filter group: a1, b0 complex64 [T][L]; delays int32 [T][L]; rate in Hz."""
    a1: np.ndarray
    b0: np.ndarray
    delays: np.ndarray
    rate_hz: int


@dataclass(frozen=True)
class Workload:
    name: str
    banks: Tuple[Bank, ...]          # one entry per rate, highest rate first
    n_streams: int
    block: int                       # samples per streamed block at the base rate
    n_blocks: int
    seed_key: Tuple[int, ...]
    notes: str = ""

    @property
    def n_templates(self) -> int:
        return self.banks[0].a1.shape[0]

    def updates_per_block(self) -> int:
        """Filter-sample updates (Eq. 7 evaluations) in one streamed block: S*T*sum_h L_h*n_h."""
        return updates_per_block([b.a1.shape[1] for b in self.banks], self.n_templates,
                                 self.n_streams, self.block)

    def strain(self, block_index: int) -> np.ndarray:
        """float32 [S][block]: white Gaussian strain for block ``block_index`` (deterministic)."""
        ss = np.random.SeedSequence(list(self.seed_key) + [5, int(block_index)])
        rng = np.random.default_rng(ss)
        return rng.standard_normal((self.n_streams, self.block)).astype(np.float32)


def updates_per_block(filters_per_rate: List[int], n_templates: int, n_streams: int, block: int) -> int:
    """S * T * sum_h L_h * (block / 2^h): the 12*N*M*R cost model of PAPER.md:88 in updates."""
    total = 0
    for h, L in enumerate(filters_per_rate):
        assert block % (1 << h) == 0
        total += L * (block >> h)
    return n_streams * n_templates * total


def make_bank(seed_key, n_templates: int, n_filters: int, rate_hz: int, mag_lo: float, mag_hi: float,
              d_max: int) -> Bank:
    subs = [np.random.default_rng(np.random.SeedSequence(list(seed_key) + [i])) for i in range(5)]
    shape = (n_templates, n_filters)
    mag = subs[0].uniform(mag_lo, mag_hi, shape)
    arg = subs[1].uniform(0.0, 2.0 * np.pi, shape)
    a1 = (mag * np.exp(1j * arg)).astype(np.complex64)
    b0 = (1e-3 * (subs[2].standard_normal(shape) + 1j * subs[3].standard_normal(shape)) / np.sqrt(2.0)
          ).astype(np.complex64)
    delays = subs[4].integers(0, d_max + 1, shape).astype(np.int32)
    return Bank(a1=a1, b0=b0, delays=delays, rate_hz=rate_hz)


MULTIRATE_RATES = (4096, 2048, 1024, 512, 256, 128, 64)
MULTIRATE_FILTERS = (8, 16, 32, 48, 64, 48, 40)
FEW_FILTER_SWEEP = (1, 2, 4, 8, 16, 32)


def config(index: int, *, n_templates: int | None = None, n_blocks: int | None = None,
           n_filters: int | None = None) -> Workload:
    """BASELINE.json configs[index].  Keyword overrides cut a config down for parity tests
    (same distributions, fewer templates / blocks); for index 2 ``n_filters`` picks the sweep point."""
    key = (1702, 2256, index)
    if index == 0:
        T, L = n_templates or 16, n_filters or 128
        bank = make_bank(key, T, L, 4096, 0.9, 0.9999, 2047)
        return Workload("cfg0_single_rate_16x128", (bank,), 1, 4096, n_blocks or 1, key)
    if index == 1:
        T, L = n_templates or 1024, n_filters or 256
        bank = make_bank(key, T, L, 4096, 0.9, 0.9999, 4095)
        return Workload("cfg1_many_filter_1024x256", (bank,), 1, 4096, n_blocks or 16, key)
    if index == 2:
        T, L = n_templates or 4096, n_filters or 8
        bank = make_bank(key + (L,), T, L, 256, 0.5, 0.999, 255)
        return Workload(f"cfg2_few_filter_4096x{L}", (bank,), 1, 256, n_blocks or 64, key + (L,))
    if index == 3:
        T = n_templates or 1024
        banks = tuple(make_bank(key + (h,), T, L, R, 0.9, 0.9999, R - 1)
                      for h, (R, L) in enumerate(zip(MULTIRATE_RATES, MULTIRATE_FILTERS)))
        return Workload("cfg3_multirate_7rates_1024x256", banks, 1, 4096, n_blocks or 32, key)
    if index == 4:
        T, L = n_templates or 16384, n_filters or 256
        bank = make_bank(key, T, L, 2048, 0.9, 0.9999, 2047)
        return Workload("cfg4_full_bank_2x16384x256", (bank,), 2, 2048, n_blocks or 64, key)
    raise ValueError("config index must be 0..4")


def shard_templates(n_templates: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous template range [lo, hi) owned by ``rank`` (templates are independent units,
    PAPER.md:63-67, 112): no data-path collective is needed."""
    base, rem = divmod(n_templates, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
