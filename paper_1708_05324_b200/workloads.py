"""Seeded synthetic fibres and pulses: the five BASELINE.json configurations.

This module only *generates inputs* (mode fields, the S tensor by quadrature,
beta tables, Raman response samples, launch fields).  It holds none of the
solver's arithmetic and is the only module shared by the CUDA path's tests /
bench and the fp64 oracle (``oracle/``).  numpy/scipy only; no torch, no CUDA.

The paper's own workloads (Examples 1-3, Fig. 3) need its
released fibre files, which are not available; these configurations stand in
for them with the same shapes (GRIN / step-index silica MMF near 1030 nm, 1-45
modes, 2^10-2^14 samples, sub-ps pulses at 10^2-10^6 W).  Recipe: DESIGN.md §4.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

C_LIGHT = 299792458.0
LAMBDA0 = 1030e-9
OMEGA0 = 2.0 * math.pi * C_LIGHT / LAMBDA0      # 1.828788e15 rad/s
N2 = 2.3e-20                                    # m^2/W
N_CORE = 1.45
F_R = 0.18
TAU1 = 12.2e-15
TAU2 = 32.0e-15
SEED_BASE = 170805324


@dataclass
class Workload:
    name: str
    P: int
    N: int
    M: int
    dt: float
    dz: float
    L: float
    beta: np.ndarray            # [P][n_beta]  (s^k / m)
    S: np.ndarray               # [P][P][P][P] (1/m^2)
    f_R: float
    h_R: np.ndarray | None      # [N] (1/s), sampled at t_j = j dt; None iff f_R == 0
    omega0: float
    n2: float
    shock: bool
    precision: int              # 0 = complex64, 1 = complex128
    tol: float
    A0: np.ndarray              # [P][N] complex128, sqrt(W), t_n = (n - N/2) dt
    meta: dict = field(default_factory=dict)

    @property
    def kappa(self) -> float:
        return self.n2 * self.omega0 / C_LIGHT

    @property
    def n_steps(self) -> int:
        return int(round(self.L / self.dz))


# ----------------------------------------------------------------- Raman input
def raman_response(N: int, dt: float, tau1: float = TAU1, tau2: float = TAU2) -> np.ndarray:
    """Damped-oscillator h_R sampled at t_j = j dt, rescaled so dt*sum(h_R) = 1.

    The paper gives no formula ("phenomenological"); BASELINE.json
    fixes tau1 = 12.2 fs, tau2 = 32 fs (reading S6).
    """
    t = np.arange(N) * dt
    h = (tau1 ** 2 + tau2 ** 2) / (tau1 * tau2 ** 2) * np.exp(-t / tau2) * np.sin(t / tau1)
    return h / (dt * h.sum())


# ------------------------------------------------------------------ mode fields
def _hermite(n: int, x: np.ndarray) -> np.ndarray:
    """Physicists' Hermite polynomial H_n by the three-term recurrence."""
    h0 = np.ones_like(x)
    if n == 0:
        return h0
    h1 = 2.0 * x
    for k in range(1, n):
        h0, h1 = h1, 2.0 * x * h1 - 2.0 * k * h0
    return h1


def grin_mode_list(max_group: int):
    """(a, b) with a + b = g ascending, a descending inside a group (S20)."""
    return [(a, g - a) for g in range(max_group + 1) for a in range(g, -1, -1)]


def grin_spot_size(radius=25e-6, na=0.2, lam=LAMBDA0) -> float:
    return math.sqrt(2.0 * radius / (2.0 * math.pi / lam * na))


def _grid(half_width: float, n_grid: int):
    d = 2.0 * half_width / n_grid
    x = -half_width + (np.arange(n_grid) + 0.5) * d        # midpoint grid
    X, Y = np.meshgrid(x, x, indexing="ij")
    return X, Y, d * d


def grin_modes(max_group: int, radius=25e-6, na=0.2, half_width=40e-6, n_grid=256):
    """Real Hermite-Gaussian fields H_a(sqrt2 x/w) H_b(sqrt2 y/w) exp(-r^2/w^2)."""
    w = grin_spot_size(radius, na)
    X, Y, dA = _grid(half_width, n_grid)
    ab = grin_mode_list(max_group)
    F = np.empty((len(ab), n_grid, n_grid))
    for i, (a, b) in enumerate(ab):
        F[i] = (_hermite(a, math.sqrt(2) * X / w) * _hermite(b, math.sqrt(2) * Y / w)
                * np.exp(-(X ** 2 + Y ** 2) / w ** 2))
    groups = np.array([a + b for a, b in ab])
    return F, dA, groups


def lp_mode_table(V: float, l_max: int | None = None):
    """Roots (l, m, u) of the weakly-guiding characteristic equation, sorted by u.

    u J_{l-1}(u)/J_l(u) = -w K_{l-1}(w)/K_l(w),  u^2 + w^2 = V^2  (reading S21),
    solved in the pole-free form  u J_{l-1}(u) K_l(w) + w K_{l-1}(w) J_l(u) = 0.
    """
    from scipy.special import jv, kve
    from scipy.optimize import brentq

    def f(u, l):
        w = math.sqrt(max(V * V - u * u, 0.0))
        return u * jv(l - 1, u) * kve(l, w) + w * kve(l - 1, w) * jv(l, u)

    roots = []
    us = np.linspace(1e-3, V - 1e-9, 20001)
    if l_max is None:
        l_max = int(V)                      # no guided LP_lm with l > V
    for l in range(l_max + 1):
        vals = np.array([f(u, l) for u in us])
        m = 0
        for i in range(len(us) - 1):
            if vals[i] * vals[i + 1] < 0.0:
                r = brentq(f, us[i], us[i + 1], args=(l,), xtol=1e-14, rtol=1e-14)
                m += 1
                roots.append((l, m, r))
    roots.sort(key=lambda t: t[2])
    return roots


def step_index_modes(n_modes: int, radius=25e-6, na=0.22, half_width=50e-6, n_grid=256,
                     lam=LAMBDA0, n_core=N_CORE):
    """First ``n_modes`` scalar LP modes by decreasing beta, cos then sin (S20)."""
    from scipy.special import jv, kv
    k0 = 2.0 * math.pi / lam
    V = k0 * radius * na
    X, Y, dA = _grid(half_width, n_grid)
    r = np.sqrt(X ** 2 + Y ** 2)
    phi = np.arctan2(Y, X)
    fields, betas, labels = [], [], []
    for (l, m, u) in lp_mode_table(V):
        w = math.sqrt(V * V - u * u)
        rad = np.where(r <= radius, jv(l, u * r / radius) / jv(l, u),
                       kv(l, w * np.maximum(r, radius) / radius) / kv(l, w))
        b = math.sqrt((k0 * n_core) ** 2 - (u / radius) ** 2)
        for orient in ((0,) if l == 0 else (0, 1)):
            ang = np.cos(l * phi) if orient == 0 else np.sin(l * phi)
            fields.append(rad * ang)
            betas.append(b)
            labels.append(f"LP{l}{m}{'' if l == 0 else 'ab'[orient]}")
            if len(fields) == n_modes:
                return np.array(fields), dA, np.array(betas), labels
    raise ValueError("fibre guides fewer modes than requested")


def coupling_tensor(F: np.ndarray, dA: float) -> np.ndarray:
    """S_plmn of Eq. 2 by midpoint quadrature on the mode grid [1/m^2]."""
    P = F.shape[0]
    f = F.reshape(P, -1)
    f = f / np.sqrt((f * f).sum(axis=1, keepdims=True) * dA)
    iu = np.triu_indices(P)
    pp = f[iu[0]] * f[iu[1]]                       # unique pair fields  [Q][grid]
    G = (pp @ pp.T) * dA                           # Gram matrix of pair fields [Q][Q]
    idx = np.zeros((P, P), dtype=np.int64)
    idx[iu] = np.arange(len(iu[0]))
    idx = np.maximum(idx, idx.T)
    flat = idx.reshape(-1)
    return G[np.ix_(flat, flat)].reshape(P, P, P, P)


# ----------------------------------------------------------------------- pulses
def _time_grid(N, dt):
    return (np.arange(N) - N // 2) * dt


def _shape(kind: str, t: np.ndarray, fwhm: float) -> np.ndarray:
    if kind == "gauss":
        T = fwhm / (2.0 * math.sqrt(math.log(2.0)))
        return np.exp(-t ** 2 / (2.0 * T ** 2))
    if kind == "sech":
        T = fwhm / 1.7627471740390859
        return 1.0 / np.cosh(t / T)
    raise ValueError(kind)


def _launch(rng, P, t, kind, fwhm, p_peak, noise):
    c = rng.standard_normal(P) + 1j * rng.standard_normal(P)
    c /= np.sqrt(np.sum(np.abs(c) ** 2))
    A = math.sqrt(p_peak) * c[:, None] * _shape(kind, t, fwhm)[None, :]
    if noise:
        g = rng.standard_normal((2, P, t.size))
        A = A + noise * math.sqrt(p_peak) * (g[0] + 1j * g[1]) / math.sqrt(2.0)
    return A.astype(np.complex128)


# ---------------------------------------------------------------------- configs
_CACHE: dict = {}


def _grin_S(max_group):
    key = ("grin", max_group)
    if key not in _CACHE:
        F, dA, groups = grin_modes(max_group)
        _CACHE[key] = (coupling_tensor(F, dA), groups)
    return _CACHE[key]


def _step_S(n_modes):
    key = ("step", n_modes)
    if key not in _CACHE:
        F, dA, betas, labels = step_index_modes(n_modes)
        _CACHE[key] = (coupling_tensor(F, dA), betas, labels)
    return _CACHE[key]


def make_config(index: int, *, N: int | None = None, L: float | None = None,
                M: int | None = None, max_group: int | None = None,
                n_modes: int | None = None) -> Workload:
    """Build BASELINE.json ``configs[index-1]`` (index 1..5).

    Keyword overrides shrink a configuration for parity tests (fewer samples over
    the same window is NOT what ``N`` does: the window shrinks with N so that dt
    -- and with it the physics per sample -- is unchanged; ``L`` truncates the
    run; ``max_group`` / ``n_modes`` cut the mode set).
    """
    rng = np.random.default_rng(SEED_BASE + index)
    fs_mm = (1e-12, 1e-27, 1e-42)                 # fs/mm, fs^2/mm, fs^3/mm -> SI
    if index == 1:
        Nn = N or 1024
        dt = 20e-12 / 1024
        beta = np.array([[0.0, 0.0, -20.0 * fs_mm[1]]])
        S = np.full((1, 1, 1, 1), 1.0 / 50e-12)
        kappa = N2 * OMEGA0 / C_LIGHT
        T0 = 100e-15
        P0 = abs(beta[0, 2]) / (kappa * S[0, 0, 0, 0] * T0 ** 2)
        t = _time_grid(Nn, dt)
        A0 = (math.sqrt(P0) / np.cosh(t / T0))[None, :].astype(np.complex128)
        L_D = T0 ** 2 / abs(beta[0, 2])
        return Workload("cfg1-soliton-P1", 1, Nn, M or 10, dt, L_D / 200.0, L or 5.0 * L_D,
                        beta, S, 0.0, None, OMEGA0, N2, False, 1, 1e-10, A0,
                        dict(T0=T0, P0=P0, L_D=L_D))
    if index in (2, 3, 5):
        g_max, Nfull, window, fwhm, p_peak, Lfull, dz, Mdef, noise = {
            2: (2, 4096, 10e-12, 200e-15, 50e3, 0.15, 50e-6, 10, 0.0),
            3: (4, 8192, 20e-12, 300e-15, 200e3, 1.0, 100e-6, 10, 1e-4),
            5: (8, 8192, 20e-12, 150e-15, 1e6, 0.5, 25e-6, 20, 1e-4),
        }[index]
        if max_group is not None:
            g_max = max_group
        S, groups = _grin_S(g_max)
        P = len(groups)
        dt = window / Nfull
        Nn = N or Nfull
        b1 = rng.uniform(-1.0, 1.0, P) * fs_mm[0]
        b1[0] = 0.0
        b2 = rng.uniform(18.0, 20.0, P) * fs_mm[1]
        b3 = rng.uniform(35.0, 45.0, P) * fs_mm[2]
        b0 = -groups * (0.2 / (N_CORE * 25e-6))
        beta = np.stack([b0, b1, b2, b3], axis=1)
        A0 = _launch(rng, P, _time_grid(Nn, dt), "gauss", fwhm, p_peak, noise)
        return Workload(f"cfg{index}-grin-P{P}", P, Nn, M or Mdef, dt, dz, L or Lfull, beta, S,
                        F_R, raman_response(Nn, dt), OMEGA0, N2, True, 0, 1e-6, A0,
                        dict(p_peak=p_peak, fwhm=fwhm, groups=groups))
    if index == 4:
        P = n_modes or 20
        S, betas, labels = _step_S(P)
        dt = 40e-12 / 16384
        Nn = N or 16384
        b1 = np.sort(rng.uniform(0.0, 4.0, P)) * fs_mm[0]
        b2 = rng.uniform(17.0, 21.0, P) * fs_mm[1]
        b3 = rng.uniform(30.0, 50.0, P) * fs_mm[2]
        b0 = betas - betas[0]
        beta = np.stack([b0, b1, b2, b3], axis=1)
        A0 = _launch(rng, P, _time_grid(Nn, dt), "sech", 500e-15, 300e3, 0.0)
        return Workload(f"cfg4-step-P{P}", P, Nn, M or 20, dt, 50e-6, L or 0.5, beta, S,
                        F_R, raman_response(Nn, dt), OMEGA0, N2, True, 0, 1e-6, A0,
                        dict(p_peak=300e3, fwhm=500e-15, labels=labels))
    raise ValueError("config index must be 1..5")
