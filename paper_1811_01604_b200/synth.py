"""Seeded synthetic workloads for the MPR gap-filling path (inputs only).

This module is the ONE piece shared by the CPU oracle's tests and the CUDA
path's tests/bench: it produces inputs (truth field, sample mask, temperature)
and scores outputs (MAE/RMSE).  It holds none of the sweep's arithmetic (`choose_T`, which
manufactures the input temperature, restates Eq. 1, Eq. 4 and the closed form of reading R15 in
float64; tests/test_oracle_inference_pins.py checks it against the oracle's e_s and ladder centre) and it
imports neither `oracle/` nor the CUDA binding.

What the paper measures on: synthetic Gaussian random fields on L x L grids,
simulated by the spectral method, thinned at random by p = 33 % / 66 %
(section 4).  The paper's realisations and seeds cannot be
recovered, so the fields below STAND IN for them ("Input recipe").

Seeds: field 1000+c, mask 2000+c, simulation 3000+c
for configuration c; numpy `default_rng` (PCG64).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field as _field

import numpy as np

__all__ = [
    "grf", "bernoulli_mask", "punch_holes", "choose_T", "n_bonds",
    "validation_measures", "Workload", "make_workload", "WORKLOADS",
]


# --------------------------------------------------------------------------
# Gaussian random fields by circulant embedding (FFT spectral method)
# --------------------------------------------------------------------------
def _torus_side(L: int, ell: float) -> int:
    """Side of the periodic torus the field is drawn on, >= L + 4*ell, rounded
    up to a multiple of 64 so the FFT has small prime factors."""
    need = L + int(math.ceil(4.0 * ell))
    return ((need + 63) // 64) * 64


def grf(rows: int, cols: int, ell: float, kind: str, seed: int,
        mean: float = 0.0, sigma: float = 1.0) -> np.ndarray:
    """Zero-mean stationary Gaussian random field, cropped from a torus.

    kind = "gaussian":    C(h) = sigma^2 exp(-h^2/ell^2)
    kind = "exponential": C(h) = sigma^2 exp(-h/ell)  (Whittle-Matern nu=1/2,
                          kappa = 1/ell; Eq. 7)

    Circulant embedding: eigenvalues of the torus covariance by FFT, negative
    ones (truncation artefacts, tiny) clipped to 0, complex white noise
    coloured by their square roots.  Returns float32 [rows, cols].
    """
    if kind not in ("gaussian", "exponential"):
        raise ValueError(kind)
    n0 = _torus_side(rows, ell)
    n1 = _torus_side(cols, ell)
    d0 = np.minimum(np.arange(n0), n0 - np.arange(n0)).astype(np.float64)
    d1 = np.minimum(np.arange(n1), n1 - np.arange(n1)).astype(np.float64)
    if kind == "gaussian":
        # separable: exp(-(a^2+b^2)/ell^2) = exp(-a^2/ell^2) exp(-b^2/ell^2)
        lam0 = np.fft.fft(np.exp(-(d0 / ell) ** 2)).real
        lam1 = np.fft.fft(np.exp(-(d1 / ell) ** 2)).real
        lam = np.outer(np.clip(lam0, 0.0, None), np.clip(lam1, 0.0, None))
    else:
        h = np.sqrt(d0[:, None] ** 2 + d1[None, :] ** 2)
        lam = np.fft.fft2(np.exp(-h / ell)).real
        np.clip(lam, 0.0, None, out=lam)
    rng = np.random.default_rng(seed)
    amp = np.sqrt(lam / (n0 * n1)).astype(np.float32)
    del lam
    noise = np.empty((n0, n1), dtype=np.complex64)
    noise.real = rng.standard_normal((n0, n1), dtype=np.float32)
    noise.imag = rng.standard_normal((n0, n1), dtype=np.float32)
    noise *= amp
    del amp
    f = np.fft.fft2(noise).real[:rows, :cols]
    out = (mean + sigma * f).astype(np.float32)
    return np.ascontiguousarray(out)


# --------------------------------------------------------------------------
# Sampling masks: 1 = sample (kept, fixed), 0 = prediction site (removed)
# --------------------------------------------------------------------------
def bernoulli_mask(rows: int, cols: int, p_removed: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return (rng.random((rows, cols), dtype=np.float32) >= p_removed).astype(np.uint8)


def punch_holes(mask: np.ndarray, n_holes: int, side: int, seed: int) -> np.ndarray:
    """Remove `n_holes` axis-aligned side x side blocks at seeded uniform
    positions fully inside the grid (cloud-like gaps of configuration 3)."""
    rng = np.random.default_rng(seed)
    rows, cols = mask.shape
    out = mask.copy()
    for _ in range(n_holes):
        r0 = int(rng.integers(0, rows - side + 1))
        c0 = int(rng.integers(0, cols - side + 1))
        out[r0:r0 + side, c0:c0 + side] = 0
    return out


# --------------------------------------------------------------------------
# Temperature input (the paper prints no T; reading R15)
# --------------------------------------------------------------------------
def n_bonds(rows: int, cols: int) -> int:
    """Nearest-neighbour pairs with open boundaries; 2L(L-1) when square
    (PAPER.md L109)."""
    return rows * (cols - 1) + cols * (rows - 1)


def choose_T(values: np.ndarray, mask: np.ndarray, q: float = 0.5) -> float:
    """Input temperature for one grid by specific-energy matching
     with the low-T harmonic closed form for e(T, L).

    e_s = - mean over unordered sample-sample nn pairs of cos[q(phi_i-phi_j)]
    (Eq. 4 read as a mean over pairs), phi from Eq. 1 in float64.
    e(T) = -1 + (N-1) T / (2 N_GP)  (equipartition over N-1 modes), hence
    T = 2 N_GP (1 + e_s) / (N - 1);  = 4 (1+e_s) L/(L+1) on a square grid.
    """
    z = values.astype(np.float64)
    m = mask.astype(bool)
    zs = z[m]
    zmin, zmax = float(zs.min()), float(zs.max())
    phi = 2.0 * math.pi * (z - zmin) / (zmax - zmin)
    one_minus_cos = 0.0
    pairs = 0
    # horizontal pairs
    both = m[:, :-1] & m[:, 1:]
    d = (phi[:, :-1] - phi[:, 1:])[both]
    one_minus_cos += float(np.sum(2.0 * np.sin(0.5 * q * d) ** 2))
    pairs += int(both.sum())
    both = m[:-1, :] & m[1:, :]
    d = (phi[:-1, :] - phi[1:, :])[both]
    one_minus_cos += float(np.sum(2.0 * np.sin(0.5 * q * d) ** 2))
    pairs += int(both.sum())
    if pairs == 0:
        raise ValueError("no sample-sample nearest-neighbour pairs")
    one_plus_es = one_minus_cos / pairs
    rows, cols = mask.shape
    return 2.0 * n_bonds(rows, cols) * one_plus_es / (rows * cols - 1)


# --------------------------------------------------------------------------
# Scores (AAE, ARE, AARE, RASE; reading R18)
# --------------------------------------------------------------------------
def validation_measures(truth: np.ndarray, pred: np.ndarray, mask: np.ndarray) -> dict:
    free = ~mask.astype(bool)
    t = truth.astype(np.float64)[free]
    eps = t - pred.astype(np.float64)[free]
    out = {"mae": float(np.mean(np.abs(eps))), "rmse": float(np.sqrt(np.mean(eps ** 2)))}
    with np.errstate(divide="ignore", invalid="ignore"):
        out["are_pct"] = float(100.0 * np.mean(eps / t))
        out["aare_pct"] = float(100.0 * np.mean(np.abs(eps / t)))
    return out


# --------------------------------------------------------------------------
# The BASELINE.json configurations
# --------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    truth: np.ndarray          # [batch, rows, cols] float32
    mask: np.ndarray           # [batch, rows, cols] uint8, 1 = sample
    T: np.ndarray              # [batch] float32
    seed: int                  # simulation seed
    q: float = 0.5
    equil_cap: int = 1000
    sweeps_per_real: int = 100
    M: int = 100
    meta: dict = _field(default_factory=dict)

    @property
    def batch(self) -> int:
        return self.truth.shape[0]

    @property
    def rows(self) -> int:
        return self.truth.shape[1]

    @property
    def cols(self) -> int:
        return self.truth.shape[2]

    @property
    def n_free(self) -> int:
        return int(self.mask.size - int(self.mask.sum()))


def _single(name, c, L, ell, kind, p, M, noise=0.0, holes=0, s=100, cap=1000):
    truth = grf(L, L, ell, kind, 1000 + c)
    if noise > 0.0:
        rng = np.random.default_rng(1500 + c)
        truth = (truth + noise * float(truth.std()) *
                 rng.standard_normal(truth.shape, dtype=np.float32)).astype(np.float32)
    mask = bernoulli_mask(L, L, p, 2000 + c)
    if holes:
        mask = punch_holes(mask, holes, 64, 2500 + c)
    T = np.array([choose_T(truth, mask)], dtype=np.float32)
    return Workload(name, truth[None], mask[None], T, 3000 + c, M=M,
                    sweeps_per_real=s, equil_cap=cap,
                    meta={"L": L, "ell": ell, "cov": kind, "p_removed": p,
                          "noise": noise, "holes": holes})


def make_workload(name: str, batch: int | None = None, L: int | None = None) -> Workload:
    """BASELINE.json `configs` 1..5 (cfg1..cfg5) and the paper's own workload
    (N(50,10), exponential covariance kappa=0.2, one sweep
    per realization) as `paper33` / `paper66` (`paperNN`: NN % of the nodes removed).  `L`/`batch` override the
    size for tests."""
    if name == "cfg1":
        return _single(name, 1, L or 64, 8.0, "gaussian", 0.33, M=10)
    if name == "cfg2":
        return _single(name, 2, L or 256, 16.0, "gaussian", 0.66, M=100)
    if name == "cfg3":
        return _single(name, 3, L or 1024, 32.0, "exponential", 0.50, M=100,
                       noise=0.05, holes=20)
    if name == "cfg4":
        return _single(name, 4, L or 4096, 64.0, "gaussian", 0.33, M=100)
    if name == "cfg5":
        b = batch or 32
        side = L or 2048
        rng = np.random.default_rng(1005)
        ells = rng.uniform(8.0, 128.0, size=b)
        truth = np.empty((b, side, side), dtype=np.float32)
        mask = np.empty((b, side, side), dtype=np.uint8)
        T = np.empty(b, dtype=np.float32)
        for g in range(b):
            truth[g] = grf(side, side, float(ells[g]), "gaussian", 1005 + 100 * g)
            mask[g] = bernoulli_mask(side, side, 0.66, 2005 + 100 * g)
            T[g] = choose_T(truth[g], mask[g])
        return Workload(name, truth, mask, T, 3005, M=100,
                        meta={"L": side, "ell": [float(x) for x in ells],
                              "cov": "gaussian", "p_removed": 0.66})
    if name.startswith("paper") and name[5:].isdigit() and 1 <= int(name[5:]) <= 99:
        p = int(name[5:]) / 100.0            # paper33 / paper66 are the paper's two cases; any other percentage for sweeps
        side = L or 1024
        truth = grf(side, side, 5.0, "exponential", 1009, mean=50.0, sigma=10.0)
        mask = bernoulli_mask(side, side, p, 2009 + int(p * 100))
        T = np.array([choose_T(truth, mask)], dtype=np.float32)
        return Workload(name, truth[None], mask[None], T, 3009, M=100,
                        sweeps_per_real=1, equil_cap=500,
                        meta={"L": side, "ell": 5.0, "cov": "exponential", "p_removed": p})
    raise ValueError(f"unknown workload {name!r}")


WORKLOADS = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "paper33", "paper66")
