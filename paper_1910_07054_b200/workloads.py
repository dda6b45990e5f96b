"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws geometry and
magnetisation arrays.  It is the one module that tests, bench.py and smoke()
use to feed identical arrays to the CUDA library and to the CPU oracle.

The paper uses no dataset: its workloads are nx = ny = 256 with nz swept
 and the 64 x 64 x 5 SAF stack; the configs take
those shapes.  seed = 191007054*10 + config index.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 191007054 * 10


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: np.ndarray            # [nz] fp64, nm
    Ms: np.ndarray            # [nz] fp64, A/m
    precision: str            # "f32" | "f64"
    B: int = 1
    seed: int = 0
    m_kind: str = "random_unit"
    extra: dict = field(default_factory=dict)

    def m(self, states=None) -> np.ndarray:
        """Magnetisation [B][3][nz][ny][nx] in fp64 (unit vectors), x fastest.
        states: optional list of state indices (batched configs) to generate only those."""
        idx = list(range(self.B)) if states is None else list(states)
        out = np.empty((len(idx), 3, self.nz, self.ny, self.nx), dtype=np.float64)
        for t, b in enumerate(idx):
            out[t] = _draw_m(self, b)
        return out

    def m_rounded(self, states=None) -> np.ndarray:
        """m rounded to the plan precision and promoted back to fp64, so that input rounding
        is not charged to the GPU path ('Inputs')."""
        m = self.m(states)
        if self.precision == "f32":
            return m.astype(np.float32).astype(np.float64)
        return m

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


def _normalise(v, fallback_z=True):
    n = np.sqrt((v ** 2).sum(axis=0))
    bad = n < 1e-3
    if fallback_z and bad.any():
        v = v.copy()
        v[0][bad], v[1][bad], v[2][bad] = 0.0, 0.0, 1.0
        n = np.where(bad, 1.0, n)
    return v / n


def _draw_m(w: Workload, b: int) -> np.ndarray:
    rng = np.random.default_rng([w.seed, 7, b])
    shape = (3, w.nz, w.ny, w.nx)
    if w.m_kind == "random_unit":
        return _normalise(rng.standard_normal(shape))
    if w.m_kind == "pm_z_tilt":
        v = 0.05 * rng.standard_normal(shape)
        sign = np.where(np.arange(w.nz) % 2 == 0, 1.0, -1.0)
        v[2] += sign[:, None, None]
        return _normalise(v)
    if w.m_kind == "smooth":
        x = np.arange(w.nx)[None, None, :] / w.nx
        y = np.arange(w.ny)[None, :, None] / w.ny
        z = np.arange(w.nz)[:, None, None] / w.nz
        v = np.zeros(shape)
        for c in range(3):
            for _ in range(8):
                p, q = rng.integers(-3, 4, size=2)
                r = rng.integers(-1, 2)
                a = rng.uniform(0.5, 1.0)
                ph = rng.uniform(0, 2 * np.pi)
                v[c] += a * np.sin(2 * np.pi * (p * x + q * y + r * z) + ph)
        return _normalise(v)
    raise ValueError(w.m_kind)


def config(k: int, variant: str = "") -> Workload:
    """BASELINE.json configs[k-1], k = 1..5.  variant: 'f64' for C2's fp64 run,
    'equal' for C4's equal-thickness variant."""
    seed = SEED_BASE + k
    rng = np.random.default_rng([seed, 1])
    if k == 1:
        return Workload("C1 16x16x3 f64", 16, 16, 3, 2.0, 2.0, np.array([1.0, 2.0, 0.6]),
                        np.full(3, 8e5), "f64", seed=seed)
    if k == 2:
        Ms = 1.0e6 + 0.4e6 * rng.uniform(size=6)
        prec = "f64" if variant == "f64" else "f32"
        return Workload(f"C2 64x64x6 {prec}", 64, 64, 6, 1.5, 1.5,
                        np.array([1.0, 0.8, 0.9, 1.2, 1.0, 2.5]), Ms, prec, seed=seed, m_kind="pm_z_tilt")
    if k == 3:
        dz = np.exp(rng.uniform(np.log(0.5), np.log(5.0), size=16))
        return Workload("C3 256x256x16 f32", 256, 256, 16, 2.0, 2.0, dz, np.full(16, 8e5), "f32",
                        seed=seed, m_kind="smooth")
    if k == 4:
        if variant == "equal":
            dz = np.full(64, 1.0)
        else:
            dz = np.exp(rng.uniform(np.log(0.3), np.log(3.0), size=64))
        return Workload("C4 256x256x64 f32" + (" equal" if variant == "equal" else ""), 256, 256, 64, 2.0, 2.0,
                        dz, np.full(64, 8e5), "f32", seed=seed)
    if k == 5:
        return Workload("C5 512x512x8 f32 B=32", 512, 512, 8, 2.0, 2.0,
                        np.array([0.6, 1.1, 0.9, 2.0, 0.7, 1.5, 1.0, 3.0]), np.full(8, 8e5), "f32", B=32, seed=seed)
    raise ValueError(k)


def small(nx, ny, nz, precision="f64", B=1, seed=12345, dz=None, m_kind="random_unit") -> Workload:
    """Reduced-size case for parity tests (ragged / tiny / odd layer counts)."""
    rng = np.random.default_rng([seed, 2])
    if dz is None:
        dz = np.exp(rng.uniform(np.log(0.4), np.log(3.0), size=nz))
    Ms = 8e5 * (0.75 + 0.5 * rng.uniform(size=nz))
    return Workload(f"small {nx}x{ny}x{nz} {precision} B={B}", nx, ny, nz, 2.0, 1.5, np.asarray(dz, float), Ms,
                    precision, B=B, seed=seed, m_kind=m_kind)
