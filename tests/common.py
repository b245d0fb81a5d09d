"""Test helpers: build the operator of a config on both sides (oracle / CUDA library)."""
from __future__ import annotations

import functools

import numpy as np

import synth_inputs as si


def rel_l2(a, b) -> float:
    """||a - b||_2 / ||b||_2 (b = oracle)."""
    a = np.asarray(a)
    b = np.asarray(b)
    den = float(np.linalg.norm(b))
    return float(np.linalg.norm(a - b)) / (den if den > 0 else 1.0)


@functools.lru_cache(maxsize=None)
def oracle_operator(name: str):
    """Oracle route: ladder-operator products into an ordered map (oracle/bs_oracle.cpp)."""
    from oracle import oracle as orc
    cfg = si.CONFIGS[name]
    if cfg.kind == "hubbard":
        return orc.hubbard_h(cfg.n_orb, cfg.hubbard_t, cfg.hubbard_u)
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    return orc.molecular_h(h, g)


def raw_terms(name: str):
    """Harness route: raw 4/16-term expansions (paper_2606_28952_b200/jw_terms.py), unmerged."""
    from paper_2606_28952_b200 import jw_terms as jw
    cfg = si.CONFIGS[name]
    if cfg.kind == "hubbard":
        return jw.hubbard_raw_terms(cfg.n_orb, cfg.hubbard_t, cfg.hubbard_u)
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    return jw.molecular_raw_terms(h, g)


def to_device(psi_np):
    import torch
    return torch.from_numpy(np.ascontiguousarray(psi_np)).cuda()


def to_host(t):
    return t.cpu().numpy()
