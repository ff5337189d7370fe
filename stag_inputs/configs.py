"""The five synthetic workloads of BASELINE.json:configs (recipes: SURVEY.md §8(d)).

Stand-ins for the paper's own gauge ensembles (not in the container):
lattice shapes follow PAPER.md Table 2 / Fig. 3 (N_t = 4..8 with spatial 16..64, plus a
symmetric volume); shifts are log-spaced stand-ins for rational-approximation poles.
"""
from __future__ import annotations

import numpy as np

from . import gen


def _logspace(lo: float, hi: float, n: int) -> list[float]:
    if n == 1:
        return [lo]
    return [float(lo * (hi / lo) ** (i / (n - 1))) for i in range(n)]


CONFIGS = {
    # name: dict(L, links=(kind, eps), seed, mass, shifts, residues, residue0, stops, nsrc)
    "c1_4x4x4x4": dict(
        L=(4, 4, 4, 4), links=("haar", None), seed=1001, mass=0.1,
        shifts=[0.01, 0.04, 0.16, 0.64], residues=None, residue0=0.0,
        stops=[1e-10], nsrc=1),
    "c2_16x16x16x4": dict(
        L=(16, 16, 16, 4), links=("smooth", 0.3), seed=1002, mass=0.05,
        shifts=[0.0], residues=None, residue0=0.0, stops=[1e-10], nsrc=1),
    "c3_24x24x24x6": dict(
        L=(24, 24, 24, 6), links=("smooth", 0.5), seed=1003, mass=0.02,
        shifts=_logspace(1e-4, 10.0, 12),
        residues=[1.0 / (i + 1) for i in range(12)], residue0=0.0,
        stops=[1e-10, 1e-12], nsrc=1),
    "c4_32x32x32x8": dict(
        L=(32, 32, 32, 8), links=("haar", None), seed=1004, mass=0.01,
        shifts=_logspace(1e-5, 20.0, 16), residues=None, residue0=0.0,
        stops=[1e-10], nsrc=4),
    "c5_64x64x64x64": dict(
        L=(64, 64, 64, 64), links=("haar", None), seed=1005, mass=0.01,
        shifts=_logspace(1e-4, 1.0, 8), residues=None, residue0=0.0,
        stops=[1e-9], nsrc=1),
    # the two other lattices of the paper's Table 2 (4 x 16^3 is config 2's shape): Dslash
    # timing beside the paper's C1060 figures, and a CG at the paper's N_t = 4 shape.  Seeds 1006, 1007.
    "t2_32x32x32x32": dict(
        L=(32, 32, 32, 32), links=("haar", None), seed=1006, mass=0.01,
        shifts=_logspace(1e-4, 1.0, 8), residues=None, residue0=0.0, stops=[1e-9], nsrc=1),
    "t2_48x48x48x4": dict(
        L=(48, 48, 48, 4), links=("haar", None), seed=1007, mass=0.01,
        shifts=_logspace(1e-4, 1.0, 8), residues=None, residue0=0.0, stops=[1e-10], nsrc=1),
}


def get_config(name: str) -> dict:
    return CONFIGS[name]


def make_links(cfg: dict) -> np.ndarray:
    kind, eps = cfg["links"]
    if kind == "haar":
        return gen.links_haar(cfg["L"], cfg["seed"])
    if kind == "smooth":
        return gen.links_smooth(cfg["L"], cfg["seed"], eps)
    if kind == "unit":
        return gen.links_unit(cfg["L"])
    raise ValueError(kind)


def make_source(cfg: dict, k: int = 0) -> np.ndarray:
    """k-th pseudo-fermion source (streams 1..nsrc), even sites."""
    return gen.source_gaussian(cfg["L"], cfg["seed"], stream=1 + k)
