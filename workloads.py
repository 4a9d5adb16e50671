"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NO arithmetic of the method (no LGL nodes, no DG operators, no
Fourier tensor): every generator takes the node coordinates it needs as plain arrays,
produced by whichever side is being exercised (the oracle in the CPU tests, the
library's `dg_get_nodes` in bench.py).  It only evaluates the analytic initial
conditions and the counter-based random numbers that DESIGN.md's input recipe names.

Counter-based generator: u(seed, idx) in [0,1) is the top
53 bits of a SplitMix64-style finaliser applied to `seed*K0 + (idx+1)*K1 (mod 2^64)`;
`idx` is the flat index in the row-major f[g_x][g_u][g_v] layout.
"""
from __future__ import annotations

import math
import numpy as np

_K0 = np.uint64(0xD1B54A32D192ED03)
_K1 = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

SEED_CFG3_NOISE = 0xD60003
SEED_CFG4_F = 0xD60004
SEED_CFG4_E = 0xD61004
SEED_CFG5 = 0xD60005
SEED_CFG6_NOISE = 0xD60006      # 2D2V workload
SEED_CFG6_E = 0xD61006


def counter_uniform(seed: int, start: int, count: int) -> np.ndarray:
    """u(seed, idx) for idx = start .. start+count-1, as float64 in [0, 1)."""
    with np.errstate(over="ignore"):
        idx = np.arange(start + 1, start + 1 + count, dtype=np.uint64)
        z = np.uint64(seed) * _K0 + idx * _K1
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def counter_uniform_chunked(seed: int, count: int, chunk: int = 1 << 24) -> np.ndarray:
    out = np.empty(count, dtype=np.float64)
    for s in range(0, count, chunk):
        m = min(chunk, count - s)
        out[s:s + m] = counter_uniform(seed, s, m)
    return out


def counter_normal(seed: int, start: int, count: int) -> np.ndarray:
    """Standard normals by Box-Muller on u(seed, 2i), u(seed, 2i+1)."""
    u = counter_uniform(seed, 2 * start, 2 * count)
    u1 = 1.0 - u[0::2]            # (0, 1]
    u2 = u[1::2]
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


# ---------------------------------------------------------------------------------------
# Initial conditions (analytic formulas of the configs; coordinates are passed in)
# ---------------------------------------------------------------------------------------

def landau_f0(x: np.ndarray, v: np.ndarray, amp: float = 0.01, k: float = 0.5) -> np.ndarray:
    """Config 1: f0 = (1 + amp cos(k x)) exp(-v^2/2)/sqrt(2 pi), shape [len(x), len(v)]."""
    return (1.0 + amp * np.cos(k * x))[:, None] * (np.exp(-0.5 * v * v) / math.sqrt(2.0 * math.pi))[None, :]


def ring_f0(x: np.ndarray, vx: np.ndarray, vy: np.ndarray, k: float, amp: float = 0.01,
            j: int = 3, alpha: float = 1.0) -> np.ndarray:
    """Configs 2/3: ring distribution of PAPER.md Eq. 31 (ring parameter j, thermal speed
    alpha, analytic unit-density normalisation) times (1 + amp sin(k x))."""
    v2 = (vx * vx)[:, None] + (vy * vy)[None, :]
    s = v2 / (2.0 * alpha * alpha)
    ring = s ** j * np.exp(-s) / (2.0 * math.pi * alpha * alpha * math.factorial(j))
    return (1.0 + amp * np.sin(k * x))[:, None, None] * ring[None, :, :]


def ring2d_f0(x: np.ndarray, y: np.ndarray, vx: np.ndarray, vy: np.ndarray, kx: float, ky: float, amp: float = 0.01,
              j: int = 3, alpha: float = 1.0) -> np.ndarray:
    """2D2V workload: the ring distribution of Eq. 31 times (1 + amp sin(kx x) + amp cos(ky y)), [len(x), len(y), len(vx), len(vy)]."""
    v2 = (vx * vx)[:, None] + (vy * vy)[None, :]
    s = v2 / (2.0 * alpha * alpha)
    ring = s ** j * np.exp(-s) / (2.0 * math.pi * alpha * alpha * math.factorial(j))
    space = 1.0 + amp * np.sin(kx * x)[:, None] + amp * np.cos(ky * y)[None, :]
    return space[:, :, None, None] * ring[None, None, :, :]


def add_uniform_noise(f: np.ndarray, seed: int, amp: float) -> np.ndarray:
    """Config 3: f + amp*(2u(seed, idx) - 1), idx = flat row-major index."""
    flat = f.reshape(-1)
    chunk = 1 << 24
    for s in range(0, flat.size, chunk):
        m = min(chunk, flat.size - s)
        flat[s:s + m] += amp * (2.0 * counter_uniform(seed, s, m) - 1.0)
    return f


def uniform_field(shape, seed: int) -> np.ndarray:
    """Config 4: f ~ U(0,1) from the counter generator."""
    n = int(np.prod(shape))
    return counter_uniform_chunked(seed, n).reshape(shape)


def normal_E(nx_nodes: int, seed: int, sigma: float = 0.1) -> np.ndarray:
    """Config 4: E[g_x] ~ N(0, sigma^2)."""
    return sigma * counter_normal(seed, 0, nx_nodes)


def cosine_sum_density(x: np.ndarray, batch: int, seed: int, nterms: int = 16, mmax: int = 1024,
                       amax: float = 0.1, noise: float = 1e-3, b0: int = 0):
    """Config 5: rho_b(x) = 1 + sum_i A cos(m x + phi) + N(0, noise^2), b = b0..b0+batch-1.
    Returns (rho [batch, len(x)], A [batch, nterms], m [batch, nterms], phi [batch, nterms])."""
    G = x.shape[0]
    rho = np.empty((batch, G))
    A = np.empty((batch, nterms)); M = np.empty((batch, nterms), dtype=np.int64); PH = np.empty((batch, nterms))
    for bi in range(batch):
        b = b0 + bi
        u = counter_uniform(seed, b * 3 * nterms, 3 * nterms)
        a = amax * u[0:nterms]
        m = 1 + np.floor(u[nterms:2 * nterms] * mmax).astype(np.int64)
        ph = 2.0 * math.pi * u[2 * nterms:3 * nterms]
        r = 1.0 + (a[:, None] * np.cos(m[:, None] * x[None, :] + ph[:, None])).sum(axis=0)
        if noise != 0.0:
            r = r + noise * counter_normal(seed ^ 0x5A5A5A, b * G, G)
        rho[bi] = r
        A[bi], M[bi], PH[bi] = a, m, ph
    return rho, A, M, PH


# ---------------------------------------------------------------------------------------------
# Cyclotron-harmonic instability of the paper's Section 4.1 / 6.1 (simulations A and B)
# ---------------------------------------------------------------------------------------------
def ring_distribution(vx: np.ndarray, vy: np.ndarray, j: int, alpha: float = 1.0) -> np.ndarray:
    """Eq. 31: f0 = (v_perp^2 / 2 alpha^2)^j exp(-v_perp^2 / 2 alpha^2) / (2 pi alpha^2 j!), [G_u][G_v]."""
    s = (vx[:, None] ** 2 + vy[None, :] ** 2) / (2.0 * alpha ** 2)
    return s ** j * np.exp(-s) / (2.0 * math.pi * alpha ** 2 * math.factorial(j))


def harris_dispersion(omega: complex, k: float, j: int, ratio: float, alpha: float = 1.0, npts: int = 50) -> complex:
    """Eq. 34: eps(omega, k) = 1 + (omega_p/omega_c)^2 / sin(pi omega) *
    int_0^pi sin(omega th) sin(th) L_j(beta) exp(-beta) dth,  beta = 2 k^2 alpha^2 cos^2(th/2); omega in units of
    omega_c, k in units of 1/r_L; fifty-point Gauss-Legendre as in the paper."""
    from scipy.special import eval_laguerre
    xg, wg = np.polynomial.legendre.leggauss(npts)
    th = 0.5 * math.pi * (xg + 1.0)
    beta = 2.0 * (k * alpha) ** 2 * np.cos(0.5 * th) ** 2
    integ = np.sum(0.5 * math.pi * wg * np.sin(omega * th) * np.sin(th) * eval_laguerre(j, beta) * np.exp(-beta))
    return 1.0 + ratio ** 2 * integ / np.sin(math.pi * omega)


def eigenmode_perturbation(x: np.ndarray, vx: np.ndarray, vy: np.ndarray, k_sim: float, k_larmor: float, omega: complex,
                           j: int, alpha: float = 1.0, nmax: int = 20, sense: int = -1) -> np.ndarray:
    """Eq. 35-36: f1 = (1/v_perp) d f0/d v_perp * Re(psi0),
    psi0 = exp(i (k x + k_L v_perp sin(phi))) sum_{|n| <= nmax} n/(n - omega) J_n(k_L v_perp) exp(-i n phi),
    with (u, v) = v_perp (cos phi, sin phi); k_sim is the wavenumber in the simulation's length unit (x), k_L the same
    wavenumber in units of the Larmor radius (k_L = k_sim * omega_p/omega_c), omega in units of omega_c.
    (1/v) d f0/dv = (j - v^2/2 alpha^2) f0 / v^2 (Eq. 32) is evaluated as (j - s) s^(j-1) e^{-s} / (2 alpha^2 Z), s = v^2/2 alpha^2,
    which is finite at v = 0.  Returns [G_x][G_u][G_v], unnormalised.

    sense: sign of the gyro-angle, (u, v) = v_perp (cos phi, sense * sin phi).  With the force of Eq. 28 as printed
    (du/dt = -B v, dv/dt = +B u: counter-clockwise gyration, x - v/B invariant) integrating the linearised equation along
    the unperturbed orbits gives psi0 = exp(i (k x - k_L v_perp sin phi)) sum n/(n - omega) J_n exp(+i n phi), i.e.
    Eq. 36 with phi -> -phi; sense = -1 (default) is that form, sense = +1 is Eq. 36 literally.  DESIGN.md reading C24:
    only sense = -1 grows at the paper's rate 0.349 omega_c from t = 0 (tests/test_gpu_physics.py)."""
    from scipy.special import jv
    U, V = vx[:, None], vy[None, :]
    vp = np.sqrt(U ** 2 + V ** 2)
    phi = np.arctan2(sense * V, U)
    s = vp ** 2 / (2.0 * alpha ** 2)
    grad = (j - s) * s ** (j - 1) * np.exp(-s) / (2.0 * alpha ** 2) / (2.0 * math.pi * alpha ** 2 * math.factorial(j))
    series = np.zeros(vp.shape, dtype=np.complex128)
    for n in range(-nmax, nmax + 1):
        if n == 0:
            continue
        series += n / (n - omega) * jv(n, k_larmor * vp) * np.exp(-1j * n * phi)
    psi_v = np.exp(1j * k_larmor * vp * np.sin(phi)) * series                     # velocity part of psi0
    psi = np.exp(1j * k_sim * x)[:, None, None] * psi_v[None, :, :]
    return grad[None, :, :] * np.real(psi)
