"""Seeded synthetic SPIIR workloads (BASELINE.json:configs[0..4]; recipe in SURVEY.md §8(d)).

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_1602_05573_b200/``).  It holds none of the method's arithmetic: it draws random
numbers, shapes them into coefficient / delay / strain arrays and rounds them ONCE to the
float32 / complex64 / int32 arrays that both sides consume (SURVEY.md §8(c) finding F1: the
oracle must read the float32-rounded coefficients, widened exactly to double).

The paper's own workload is "real pipeline data" (§3.4) that is not available;
these inputs stand in for it.

Draw order per config, each one array call over all K filters of the bank:
    [K_t if variable] -> r -> omega -> Re b0 -> Im b0 -> d -> x-noise
with ``rng = numpy.random.default_rng(SEED0 + cfg)``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED0 = 160205573          # arXiv id 1602.05573
FS = 4096.0                # sample rate of every config (Hz)


@dataclass
class SpiirInputs:
    """One bank + one strain stream, already rounded to the device dtypes."""
    name: str
    offsets: np.ndarray     # int64 [T+1]   CSR offsets of the templates' filters
    a1: np.ndarray          # complex64 [K] pole of each first-order filter, |a1| < 1
    b0: np.ndarray          # complex64 [K] input gain of each filter
    delays: np.ndarray      # int32 [K]     integer delay d_k >= 0
    x: np.ndarray           # float32 [N]   whitened strain
    chunk: int              # samples per streaming call in the config's run mode
    meta: dict = field(default_factory=dict)

    @property
    def n_templates(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_filters(self) -> int:
        return int(self.offsets[-1])

    @property
    def n_samples(self) -> int:
        return int(self.x.shape[0])

    @property
    def max_delay(self) -> int:
        return int(self.delays.max()) if self.delays.size else 0

    @property
    def filter_samples(self) -> int:
        return self.n_filters * self.n_samples

    def select_templates(self, idx) -> "SpiirInputs":
        """Sub-bank made of the templates ``idx`` (in that order); same strain."""
        idx = np.asarray(idx, dtype=np.int64)
        counts = (self.offsets[idx + 1] - self.offsets[idx]).astype(np.int64)
        offsets = np.zeros(idx.size + 1, dtype=np.int64)
        np.cumsum(counts, out=offsets[1:])
        take = np.concatenate([np.arange(self.offsets[t], self.offsets[t + 1]) for t in idx]) \
            if idx.size else np.zeros(0, dtype=np.int64)
        return SpiirInputs(self.name + f"[{idx.size} templates]", offsets, self.a1[take].copy(),
                           self.b0[take].copy(), self.delays[take].copy(), self.x, self.chunk,
                           dict(self.meta, parent_templates=idx.tolist()))

    def truncate_samples(self, n: int) -> "SpiirInputs":
        return SpiirInputs(self.name + f"[:{n}]", self.offsets, self.a1, self.b0, self.delays,
                           self.x[:n].copy(), min(self.chunk, n), dict(self.meta))


def _uniform_offsets(T: int, K: int) -> np.ndarray:
    return (np.arange(T + 1, dtype=np.int64) * K).astype(np.int64)


def _polar_bank(rng, K_total, r_lo, r_hi, w_lo, w_hi, b_scale, d_max):
    """r -> omega -> Re b0 -> Im b0 -> d, one array call each (float64, rounded once)."""
    r = rng.uniform(r_lo, r_hi, K_total)
    w = rng.uniform(w_lo, w_hi, K_total)
    bre = rng.standard_normal(K_total)
    bim = rng.standard_normal(K_total)
    d = rng.integers(0, d_max + 1, K_total)
    a1 = (r * np.exp(1j * w)).astype(np.complex64)
    b0 = ((bre + 1j * bim) * b_scale).astype(np.complex64)
    return a1, b0, d.astype(np.int32)


def make_random_bank(seed: int, filters_per_template, n_samples: int, *, r_lo=0.95, r_hi=0.9999,
                     w_lo=0.005, w_hi=np.pi / 2, d_max=4095, chunk=None, name="random") -> SpiirInputs:
    """Generic seeded bank with the cfg1-style distributions; used by tests for ragged shapes.

    ``filters_per_template`` is a list of K_t (any positive ints)."""
    rng = np.random.default_rng(seed)
    counts = np.asarray(filters_per_template, dtype=np.int64)
    offsets = np.zeros(counts.size + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    K = int(offsets[-1])
    scale = np.repeat(1.0 / np.sqrt(counts.astype(np.float64)), counts)
    a1, b0, d = _polar_bank(rng, K, r_lo, r_hi, w_lo, w_hi, scale, d_max)
    x = rng.standard_normal(n_samples).astype(np.float32)
    return SpiirInputs(name, offsets, a1, b0, d, x, int(chunk or n_samples), {"seed": seed})


def make_config(cfg: int, *, n_templates: int | None = None, n_samples: int | None = None) -> SpiirInputs:
    """Workload ``BASELINE.json:configs[cfg]``.

    ``n_templates`` / ``n_samples`` shrink the bank / the stream for tests (the draws are then
    those of the smaller arrays, still seeded by ``SEED0 + cfg``); None = the config's full size.
    """
    rng = np.random.default_rng(SEED0 + cfg)
    if cfg == 0:
        T, K, N = n_templates or 1, 128, n_samples or 4096
        a1, b0, d = _polar_bank(rng, T * K, 0.90, 0.999, 0.01, np.pi / 2, 1.0 / np.sqrt(K), 1023)
        x = rng.standard_normal(N).astype(np.float32)
        return SpiirInputs("cfg0", _uniform_offsets(T, K), a1, b0, d, x, N, {"cfg": 0})
    if cfg == 1:
        T, K, N = n_templates or 64, 256, n_samples or 65536
        a1, b0, d = _polar_bank(rng, T * K, 0.95, 0.9999, 0.005, np.pi / 2, 1.0 / np.sqrt(K), 4095)
        x = rng.standard_normal(N).astype(np.float32)
        return SpiirInputs("cfg1", _uniform_offsets(T, K), a1, b0, d, x, min(4096, N), {"cfg": 1})
    if cfg == 2:
        # chirp-structured coefficients: omega_k increasing, d_k decreasing with k (DESIGN.md §4 reading Q13)
        T, K, N = n_templates or 1024, 512, n_samples or 65536
        k = np.arange(K, dtype=np.float64)
        t = np.arange(T, dtype=np.float64)
        u = k / (K - 1)
        r = 0.999 - 0.05 * k / K                                           # |a1| (given)
        f = (30.0 + 370.0 * u)[None, :] * (1.0 + 0.1 * t / 1024.0)[:, None]  # Hz
        w = 2.0 * np.pi * f / FS
        D_t = 2048.0 + 2.0 * t
        d = np.rint((1.0 - u)[None, :] * D_t[:, None]).astype(np.int32)
        bre = rng.standard_normal(T * K)
        bim = rng.standard_normal(T * K)
        a1 = (r[None, :] * np.exp(1j * w)).astype(np.complex64).reshape(-1)
        b0 = ((bre + 1j * bim) / np.sqrt(K)).astype(np.complex64)
        noise = rng.standard_normal(N)
        m = np.arange(N, dtype=np.float64)
        f_inj = 30.0 + 370.0 * m / max(N - 1, 1)
        phi = (2.0 * np.pi / FS) * (np.cumsum(f_inj) - f_inj)             # sum over m < n
        x = (noise + 0.1 * np.sin(phi)).astype(np.float32)
        return SpiirInputs("cfg2", _uniform_offsets(T, K), a1, b0, d.reshape(-1), x, min(4096, N), {"cfg": 2})
    if cfg == 3:
        T, K, N = n_templates or 4096, 1024, n_samples or 262144
        a1, b0, d = _polar_bank(rng, T * K, 0.95, 0.9999, 0.005, np.pi / 2, 1.0 / np.sqrt(K), 16383)
        x = rng.standard_normal(N).astype(np.float32)
        return SpiirInputs("cfg3", _uniform_offsets(T, K), a1, b0, d, x, min(16384, N), {"cfg": 3})
    if cfg == 4:
        T, N = n_templates or 8192, n_samples or 65536
        Kt = np.clip(np.floor(np.exp(rng.uniform(np.log(64.0), np.log(2049.0), T))), 64, 2048).astype(np.int64)
        offsets = np.zeros(T + 1, dtype=np.int64)
        np.cumsum(Kt, out=offsets[1:])
        scale = np.repeat(1.0 / np.sqrt(Kt.astype(np.float64)), Kt)
        a1, b0, d = _polar_bank(rng, int(offsets[-1]), 0.95, 0.9999, 0.005, np.pi / 2, scale, 8191)
        x = rng.standard_normal(N).astype(np.float32)
        return SpiirInputs("cfg4", offsets, a1, b0, d, x, 16, {"cfg": 4})
    raise ValueError(f"unknown config {cfg}")


def parity_subset(n_templates: int, n_pick: int, seed: int) -> np.ndarray:
    """First, last and ``n_pick - 2`` seeded random templates (SURVEY.md §8(c) GPU acceptance)."""
    if n_templates <= n_pick:
        return np.arange(n_templates, dtype=np.int64)
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(1, n_templates - 1), size=n_pick - 2, replace=False)
    return np.concatenate([[0], np.sort(mid), [n_templates - 1]]).astype(np.int64)
