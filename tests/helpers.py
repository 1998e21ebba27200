"""Shared test helpers: config recipes and error norms."""
from __future__ import annotations

import numpy as np
import torch

import gen

# BASELINE.json configs (gauge seed = 1000 + cfg, spinor seed = 2000 + cfg + call#)
CONFIGS = {
    1: dict(L=4, T=4, eps=0.3, reunit=False, csw=1.0, m0=-0.1, bc=1, omega=1.0),
    2: dict(L=16, T=16, eps=0.3, reunit=False, csw=1.0, m0=-0.1, bc=1, omega=1.0),
    3: dict(L=32, T=64, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
    4: dict(L=48, T=96, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
    5: dict(L=64, T=128, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
}


def config_gauge(cfg: int, L=None, T=None, device="cpu", dtype=torch.complex128):
    c = CONFIGS[cfg]
    return gen.gauge_field(L or c["L"], T or c["T"], 1000 + cfg, c["eps"], c["reunit"],
                           device=device, dtype=dtype)


def config_spinor(cfg: int, call: int = 0, L=None, T=None, device="cpu", dtype=torch.complex128):
    c = CONFIGS[cfg]
    return gen.spinor_field(L or c["L"], T or c["T"], 2000 + cfg + call, device=device, dtype=dtype)


def rel_l2(a, b) -> float:
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def even_part(psi: np.ndarray, par: np.ndarray) -> np.ndarray:
    return np.where((par == 0)[..., None, None], psi, 0.0)


def odd_part(psi: np.ndarray, par: np.ndarray) -> np.ndarray:
    return np.where((par == 1)[..., None, None], psi, 0.0)
