"""Seeded synthetic workloads (BASELINE.json `configs`).

This module holds NO arithmetic of the method: only the run parameters of the five configs and the
seeded generator of their initial vorticity fields.  It feeds both the CUDA path and the test oracle
(numpy only; importing it never loads the CUDA library).

Generator (reading G15): state s <- seed; per draw
s <- s * 6364136223846793005 + 1442695040888963407 (mod 2^64), u = (s >> 11) * 2^-53 in [0, 1),
value = a * (2u - 1); one draw per interior point in row-major order (j = 1..N-1 outer, i = 1..N-1 inner).
The smooth part of config 5 is 5 sin(2 pi i h) sin(2 pi j h), evaluated in fp64 and added before the noise.
The paper's own runs (Table 1) start from an unstated field (G11); these stand in for them.
"""
from dataclasses import dataclass

import numpy as np

_LCG_A = 6364136223846793005
_LCG_C = 1442695040888963407
_MASK = (1 << 64) - 1


@dataclass(frozen=True)
class Workload:
    name: str
    N: int                 # intervals per side; grid is (N+1) x (N+1)
    Re: float
    dt: float
    sor_omega: float
    sweeps_per_stage: int
    steps: int
    noise: float           # amplitude a of the uniform noise on interior omega
    seed: int
    smooth_amp: float = 0.0     # amplitude of the sin(2 pi x) sin(2 pi y) part (config 5)
    poisson_sweeps: int = 0     # Poisson-only sweeps run before the time steps (config 5, G14)


def _dt(N, Re):
    h = 1.0 / N
    return min(0.5 * h, 0.2 * h * h * Re)


CONFIGS = (
    Workload("cfg1_33_Re100", 32, 100.0, 0.0156, 1.8, 20, 200, 1e-6, 80930981),            # dt literal (G13)
    Workload("cfg2_129_Re1000", 128, 1000.0, _dt(128, 1000.0), 1.95, 50, 2000, 1e-6, 80930982),
    Workload("cfg3_513_Re5000", 512, 5000.0, _dt(512, 5000.0), 1.99, 100, 5000, 1e-6, 80930983),
    Workload("cfg4_1025_Re10000", 1024, 10000.0, _dt(1024, 10000.0), 1.995, 200, 1000, 1e-6, 80930984),
    Workload("cfg5_1025_Re30000", 1024, 30000.0, _dt(1024, 30000.0), 1.995, 200, 1000, 1e-3, 80930985,
             smooth_amp=5.0, poisson_sweeps=10000),
)


def config(k: int) -> Workload:
    """Config k = 1..5 of BASELINE.json."""
    return CONFIGS[k - 1]


def lcg_uniform(seed: int, n: int) -> np.ndarray:
    """n draws u_1..u_n in [0, 1) of the 64-bit LCG above (vectorised with wrap-around uint64 arithmetic)."""
    if n <= 0:
        return np.empty(0, dtype=np.float64)
    with np.errstate(over="ignore"):
        apow = np.full(n, _LCG_A, dtype=np.uint64)
        apow[0] = 1
        apow = np.multiply.accumulate(apow)                 # a^0 .. a^(n-1)  (mod 2^64)
        geo = np.add.accumulate(apow)                       # 1 + a + ... + a^k, k = 0..n-1
        a_n = apow * np.uint64(_LCG_A)                      # a^1 .. a^n
        s = a_n * np.uint64(seed & _MASK) + np.uint64(_LCG_C) * geo
    return (s >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def lcg_uniform_loop(seed: int, n: int) -> np.ndarray:
    """The same draws by the literal recurrence (slow; used by the tests to check lcg_uniform)."""
    out = np.empty(n, dtype=np.float64)
    s = seed & _MASK
    for k in range(n):
        s = (s * _LCG_A + _LCG_C) & _MASK
        out[k] = (s >> 11) * (1.0 / 9007199254740992.0)
    return out


def initial_omega(N: int, noise: float, seed: int, smooth_amp: float = 0.0) -> np.ndarray:
    """(N+1, N+1) array [j, i]; ring = 0; interior = smooth part + uniform noise in [-noise, noise)."""
    w = np.zeros((N + 1, N + 1), dtype=np.float64)
    if smooth_amp != 0.0:
        h = 1.0 / N
        k = np.arange(N + 1, dtype=np.float64)
        sx = np.sin(2.0 * np.pi * (k * h))
        w[1:N, 1:N] = smooth_amp * np.outer(sx, sx)[1:N, 1:N]
    u = lcg_uniform(seed, (N - 1) * (N - 1)).reshape(N - 1, N - 1)
    w[1:N, 1:N] += noise * (2.0 * u - 1.0)
    return w


def initial_fields(wl: Workload):
    """(psi, omega) the config starts from: psi = 0 everywhere (fluid at rest, G11)."""
    psi = np.zeros((wl.N + 1, wl.N + 1), dtype=np.float64)
    return psi, initial_omega(wl.N, wl.noise, wl.seed, wl.smooth_amp)
