"""Plummer-sphere initial conditions and the five BASELINE.json workload recipes.

Stand-in for the paper's own initial-condition files (Plummer
density Eq. 18, N = 2^k, equal masses, eps = 1e-4), which are not available.
Sampling is the textbook inverse-transform / rejection scheme for the Plummer
model (mass-radius relation inverted; speed fraction q drawn from
g(q) = q^2 (1 - q^2)^(7/2) by rejection).  Everything is a pure function of
(N, seed): numpy Generator(PCG64(seed)).
"""
from __future__ import annotations

import math

import numpy as np

HENON_B = 3.0 * math.pi / 16.0  # Plummer scale length in Henon units (M = G = 1, E = -1/4)


def _isotropic(rng, n):
    z = 1.0 - 2.0 * rng.random(n)
    phi = 2.0 * math.pi * rng.random(n)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def plummer(N: int, seed: int, mass: np.ndarray | None = None, r_cut: float = 20.0):
    """Positions, velocities [N,3] and masses [N] of a Plummer sphere in Henon units.

    Radii beyond r_cut (in units of b) are rejected.  The mass-weighted mean position
    and velocity are subtracted.  No virial rescale: E = -1/4 holds to O(N^-1/2).
    """
    rng = np.random.default_rng(seed)
    # radii: M(<r)/M = X  =>  r = (X^(-2/3) - 1)^(-1/2)
    r = np.empty(0)
    while r.size < N:
        x = rng.random(N)
        x = x[x > 0.0]
        rr = 1.0 / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
        r = np.concatenate([r, rr[rr <= r_cut]])
    r = r[:N]
    pos = r[:, None] * _isotropic(rng, N)
    # speed: q = v / v_esc from g(q) = q^2 (1-q^2)^3.5, accept if 0.1 X5 < g(X4)
    q = np.empty(0)
    while q.size < N:
        x4 = rng.random(N)
        x5 = rng.random(N)
        ok = 0.1 * x5 < x4 * x4 * (1.0 - x4 * x4) ** 3.5
        q = np.concatenate([q, x4[ok]])
    q = q[:N]
    vesc = math.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    vel = (q * vesc)[:, None] * _isotropic(rng, N)
    # model units (b = 1) -> Henon units
    pos *= HENON_B
    vel /= math.sqrt(HENON_B)
    m = np.full(N, 1.0 / N) if mass is None else np.asarray(mass, dtype=np.float64)
    mt = m.sum()
    pos -= (m[:, None] * pos).sum(axis=0) / mt
    vel -= (m[:, None] * vel).sum(axis=0) / mt
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel), m


def power_law_masses(N: int, seed: int, slope: float = 2.35, m_lo: float = 0.1, m_hi: float = 100.0):
    """dN/dm ~ m^-slope on [m_lo, m_hi] by inverse CDF, normalised to total mass 1."""
    rng = np.random.default_rng(seed)
    u = rng.random(N)
    p = 1.0 - slope
    m = (m_lo ** p + u * (m_hi ** p - m_lo ** p)) ** (1.0 / p)
    return m / m.sum()


def mean_field_acc(pos: np.ndarray) -> np.ndarray:
    """Analytic Plummer mean-field acceleration -r/(r^2+b^2)^(3/2), b = 3 pi/16.

    Used only as the INPUT a_j of force-only benchmarks (configs 3, 4): the snap term
    needs predicted accelerations and any smooth field of the right magnitude serves,
    provided both sides receive the same array.
    """
    r2 = (pos * pos).sum(axis=1)
    return -pos / (r2 + HENON_B ** 2)[:, None] ** 1.5


def plummer_with_heavy(N: int, seed: int, heavy_frac: float = 0.05):
    """Plummer sphere of N - 1 equal-mass particles plus ONE heavy particle of mass heavy_frac (total
    mass 1) at rest at the centre: the stand-in for the paper's massive-black-hole runs
    (initial conditions of its ref. [23] are not available), where the stars bound to
    the heavy particle take the smallest steps and small blocks dominate the step count."""
    pos, vel, _ = plummer(N, seed)
    m = np.full(N, (1.0 - heavy_frac) / (N - 1))
    m[0] = heavy_frac
    pos[0] = 0.0
    vel[0] = 0.0
    mt = m.sum()
    pos -= (m[:, None] * pos).sum(axis=0) / mt
    vel -= (m[:, None] * vel).sum(axis=0) / mt
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel), m


def active_subset(N: int, m: int, seed: int = 40) -> np.ndarray:
    """First m entries of a seeded permutation of 0..N-1 (config 4), as int32."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.permutation(N)[:m].astype(np.int32))


def kepler_binary(ecc: float = 0.5, m1: float = 0.5, m2: float = 0.5):
    """Two bodies, G = 1, semi-major axis 1, at apocentre, centre of mass at rest."""
    M = m1 + m2
    ra = 1.0 + ecc
    va = math.sqrt(M * (1.0 - ecc) / (1.0 + ecc))
    pos = np.array([[m2 / M * ra, 0.0, 0.0], [-m1 / M * ra, 0.0, 0.0]])
    vel = np.array([[0.0, m2 / M * va, 0.0], [0.0, -m1 / M * va, 0.0]])
    return pos, vel, np.array([m1, m2])


# The five BASELINE.json configurations (sizes, eps, eta, seeds: DESIGN.md "Input recipe").
CONFIGS = {
    1: dict(name="plummer_1k_t1", N=1 << 10, eps=1e-3, eta=0.45, dt_max=2.0 ** -4, dt_min=2.0 ** -25,
            seed=1, t_end=1.0, kind="integrate"),
    2: dict(name="plummer_64k_t1", N=1 << 16, eps=1e-4, eta=0.45, dt_max=2.0 ** -4, dt_min=2.0 ** -25,
            seed=2, t_end=1.0, kind="integrate"),
    3: dict(name="force_sweep", N=[1 << 14, 1 << 16, 1 << 18, 1 << 20, 1 << 22], eps=1e-3, seed=3,
            kind="force"),
    4: dict(name="small_active", N=1 << 20, eps=1e-4, seed=4, subset_seed=40,
            m=[64, 1024, 16384, 262144, 1 << 20], kind="force"),
    5: dict(name="plummer_8m_8steps", N=1 << 23, eps=1e-4, eta=0.45, dt_max=2.0 ** -4,
            dt_min=2.0 ** -25, seed=5, n_block_steps=8, kind="integrate"),
}


def config_inputs(cfg: int, N: int | None = None):
    """(pos, vel, mass, acc_pred) for a configuration; acc_pred is None for integrations."""
    c = CONFIGS[cfg]
    if cfg == 3:
        assert N is not None
        pos, vel, m = plummer(N, seed=c["seed"] * 1000 + int(math.log2(N)))
        return pos, vel, m, mean_field_acc(pos)
    if cfg == 4:
        n = c["N"] if N is None else N
        m = power_law_masses(n, seed=c["seed"] + 100)
        pos, vel, m = plummer(n, seed=c["seed"], mass=m)
        return pos, vel, m, mean_field_acc(pos)
    n = c["N"] if N is None else N
    pos, vel, m = plummer(n, seed=c["seed"])
    return pos, vel, m, None
