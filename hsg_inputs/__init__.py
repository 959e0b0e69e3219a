"""Seeded synthetic input generators — the ONLY code shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic: it only draws the quenched disorder, start configurations
and temperature ladders that both sides are fed.  The paper's inputs are themselves i.i.d. random
numbers ("J_ij ~ N(0,1)", "quenched couplings and fields are generated
off-GPU with the help of another, high-quality RNG"), so these arrays *are* the paper's workload,
not a stand-in for a dataset.  Recipe: DESIGN.md §4.

Every sample is drawn from its own stream keyed by (seed, global sample id), so a rank that owns
samples d0..d1 (multi-GPU sharding) or a test that checks a single sample of a large
configuration generates exactly the same numbers as a run over all samples.
"""
from __future__ import annotations

import numpy as np

_STREAM_J, _STREAM_H, _STREAM_S = 1, 2, 3


def _rng(seed: int, sample: int, stream: int) -> np.random.Generator:
    # numpy's Philox4x64 bit generator; key = (seed, sample<<8 | stream)
    return np.random.Generator(np.random.Philox(key=[int(seed), (int(sample) << 8) | stream]))


def geometric_ladder(t_min: float, t_max: float, n: int) -> np.ndarray:
    """T_i = T_1 f^(i-1), f = (T_n/T_1)^(1/(n-1)), computed in fp64, returned as fp32."""
    if n == 1:
        return np.array([t_min], dtype=np.float32)
    i = np.arange(n, dtype=np.float64)
    return (t_min * (t_max / t_min) ** (i / (n - 1))).astype(np.float32)


def couplings(L: int, n_samples: int, seed: int, sample_offset: int = 0) -> np.ndarray:
    """J[d][dir][z][y][x] ~ N(0,1), bond from site to site+e_dir."""
    out = np.empty((n_samples, 3, L, L, L), dtype=np.float32)
    for d in range(n_samples):
        out[d] = _rng(seed, sample_offset + d, _STREAM_J).standard_normal((3, L, L, L)).astype(np.float32)
    return out


def gaussian_field(L: int, n_samples: int, h_r: float, seed: int, sample_offset: int = 0) -> np.ndarray:
    """H[d][c][z][y][x] ~ N(0, h_r^2) per component (BASELINE.json configs)."""
    out = np.empty((n_samples, 3, L, L, L), dtype=np.float32)
    for d in range(n_samples):
        out[d] = (h_r * _rng(seed, sample_offset + d, _STREAM_H).standard_normal((3, L, L, L))).astype(np.float32)
    return out


def fixed_radius_field(L: int, n_samples: int, radius: float, seed: int, sample_offset: int = 0) -> np.ndarray:
    """H_i uniform on the sphere of radius |H| (the paper's own field distribution)."""
    out = np.empty((n_samples, 3, L, L, L), dtype=np.float32)
    for d in range(n_samples):
        g = _rng(seed, sample_offset + d, _STREAM_H).standard_normal((3, L, L, L))
        out[d] = (radius * g / np.sqrt((g * g).sum(axis=0, keepdims=True))).astype(np.float32)
    return out


def unit_spins(L: int, n_samples: int, n_replicas: int, n_temps: int, seed: int, sample_offset: int = 0) -> np.ndarray:
    """S[d][o][t][c][z][y][x]: unit vectors, uniform on S^2, fp32 (for set_spins tests)."""
    out = np.empty((n_samples, n_replicas, n_temps, 3, L, L, L), dtype=np.float32)
    for d in range(n_samples):
        g = _rng(seed, sample_offset + d, _STREAM_S).standard_normal((n_replicas, n_temps, 3, L, L, L))
        out[d] = (g / np.sqrt((g * g).sum(axis=2, keepdims=True))).astype(np.float32)
    return out


# BASELINE.json configs (c1..c5) and the paper's Table-1 workload (t1: R=256, L=32, T=100).
CONFIGS = {
    "c1": dict(L=8, n_samples=1, n_replicas=2, n_temps=16, t_min=0.08, t_max=0.30, h_r=0.1, n_or=5, n_hb=1, steps=1000, seed=1),
    "c2": dict(L=16, n_samples=256, n_replicas=2, n_temps=24, t_min=0.08, t_max=0.30, h_r=0.0, n_or=5, n_hb=1, steps=10000, seed=2),
    "c3": dict(L=16, n_samples=256, n_replicas=2, n_temps=24, t_min=0.06, t_max=0.25, h_r=0.1, n_or=5, n_hb=1, steps=10000, seed=3,
               h_r_scan=(0.05, 0.1, 0.2), measure_every=1),
    "c4": dict(L=32, n_samples=64, n_replicas=2, n_temps=32, t_min=0.06, t_max=0.25, h_r=0.1, n_or=5, n_hb=1, steps=100, seed=4),
    "c5": dict(L=64, n_samples=8, n_replicas=2, n_temps=32, t_min=0.06, t_max=0.25, h_r=0.05, n_or=10, n_hb=1, steps=20, seed=5),
    "t1": dict(L=32, n_samples=4, n_replicas=2, n_temps=32, t_min=100.0, t_max=100.0, h_r=0.1, n_or=10, n_hb=1, steps=20, seed=6),
}


def make_config(name: str, n_samples: int | None = None, sample_offset: int = 0, h_r: float | None = None):
    """Return (cfg, temps, J, H) for a BASELINE.json config; H is None for zero field.  ``h_r`` overrides the field
    strength (c3's scan {0.05, 0.1, 0.2}: the same couplings and the same unit-variance field draws, scaled)."""
    cfg = dict(CONFIGS[name])
    if n_samples is not None:
        cfg["n_samples"] = n_samples
    if h_r is not None:
        cfg["h_r"] = h_r
    if cfg["t_min"] == cfg["t_max"]:      # Table-1 workload: all systems at one temperature; ladder must ascend
        temps = (cfg["t_min"] * (1.0 + 1e-6 * np.arange(cfg["n_temps"]))).astype(np.float32)
    else:
        temps = geometric_ladder(cfg["t_min"], cfg["t_max"], cfg["n_temps"])
    J = couplings(cfg["L"], cfg["n_samples"], cfg["seed"], sample_offset)
    H = gaussian_field(cfg["L"], cfg["n_samples"], cfg["h_r"], cfg["seed"], sample_offset) if cfg["h_r"] > 0 else None
    return cfg, temps, J, H
