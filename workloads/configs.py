"""The five synthetic workloads (BASELINE.json `configs`, recipe of SURVEY.md 8(d)).

Random numbers: splitmix64 counter stream -> 53-bit uniforms -> Box-Muller.
Draw order for a complex field: iy, ix, component, (re, im); one Box-Muller
pair per complex number.  seed = 201015069 + config index (+ a fixed offset per
independent field).  Nothing here evaluates the method (no split step, no
energy): the arrays are inputs only.

Stand-in statement: the paper runs on physical states of its spin-Hall study
(Fig. 5: 1024^2, Omega(y), sweep over the interaction); it
uses no dataset.  Configs 3-4 take that shape with BASELINE.json's tanh profile
for Omega(y) in place of Eq. 13; the vortex-seeded initial
states of PAPER.md L217-L223 are not reproduced (recipe unspecified).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 201015069
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GAMMA = np.uint64(0x9E3779B97F4A7C15)


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """Outputs number start .. start+count-1 of the splitmix64 stream of `seed`.

    Output i (0-based) is mix(seed + (i+1)*GAMMA) with wrap-around uint64
    arithmetic, so any slice of the stream can be produced independently.
    """
    with np.errstate(over="ignore"):
        idx = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + idx * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniforms(seed: int, start: int, count: int) -> np.ndarray:
    """53-bit uniforms in [0, 1)."""
    return (splitmix64(seed, start, count) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normals(seed: int, start_pair: int, n_pairs: int) -> np.ndarray:
    """Box-Muller: pair p uses uniforms 2p, 2p+1 -> (z0, z1); returns shape (n_pairs, 2)."""
    u = uniforms(seed, 2 * start_pair, 2 * n_pairs).reshape(n_pairs, 2)
    r = np.sqrt(-2.0 * np.log1p(-u[:, 0]))  # 1-u in (0, 1]
    ang = 2.0 * np.pi * u[:, 1]
    out = np.empty((n_pairs, 2))
    out[:, 0] = r * np.cos(ang)
    out[:, 1] = r * np.sin(ang)
    return out


def complex_normal_field(seed: int, ny: int, nx: int, ncomp: int) -> np.ndarray:
    """Complex field [ny, nx, ncomp], re and im each N(0,1); generated in row chunks."""
    out = np.empty((ny, nx, ncomp), dtype=np.complex128)
    rows = max(1, (1 << 22) // (nx * ncomp))
    for y0 in range(0, ny, rows):
        y1 = min(ny, y0 + rows)
        n = (y1 - y0) * nx * ncomp
        z = normals(seed, y0 * nx * ncomp, n)
        out[y0:y1] = (z[:, 0] + 1j * z[:, 1]).reshape(y1 - y0, nx, ncomp)
    return out


def real_normal_field(seed: int, ny: int, nx: int, ncomp: int) -> np.ndarray:
    """Real field [ny, nx, ncomp] ~ N(0,1): the first normal of each Box-Muller pair."""
    out = np.empty((ny, nx, ncomp))
    rows = max(1, (1 << 22) // (nx * ncomp))
    for y0 in range(0, ny, rows):
        y1 = min(ny, y0 + rows)
        n = (y1 - y0) * nx * ncomp
        out[y0:y1] = normals(seed, y0 * nx * ncomp, n)[:, 0].reshape(y1 - y0, nx, ncomp)
    return out


def grid(n: int, L: float) -> np.ndarray:
    """x_j = -L/2 + j*L/n, j = 0..n-1 (box [-L/2, L/2))."""
    return -0.5 * L + (L / n) * np.arange(n, dtype=np.float64)


@dataclass
class Workload:
    name: str
    cfg: int
    nx: int
    ny: int
    Lx: float
    Ly: float
    dtype: str  # "c128" | "c64": storage precision of psi and fields on the GPU
    g_uu: float
    g_dd: float
    g_ud: float
    k_L: float
    norm_mode: int  # 0 per component, 1 total
    n_total: float
    V: Optional[np.ndarray]  # float64 [ny, nx] (values fp32-representable when dtype == "c64")
    Omega: Optional[np.ndarray]
    delta: Optional[np.ndarray]
    psi0: np.ndarray  # complex128 [ny, nx, 2]
    schedule: List[Tuple[int, float, int]] = field(default_factory=list)  # (n_steps, dt, imag)

    @property
    def dx(self) -> float:
        return self.Lx / self.nx

    @property
    def dy(self) -> float:
        return self.Ly / self.ny

    @property
    def points(self) -> int:
        return self.nx * self.ny


# grid, box, dtype, (g_uu, g_dd, g_ud), k_L, N_total, schedule; fields/state built below
CONFIGS = {
    1: dict(n=64, L=16.0, dtype="c128", g=(0.0, 0.0, 0.0), k_L=0.0, n_total=1.0,
            schedule=[(200, 1e-3, 1), (200, 1e-3, 0)]),
    2: dict(n=256, L=32.0, dtype="c128", g=(1.0, 1.0, 0.9), k_L=1.0, n_total=1000.0,
            schedule=[(1000, 5e-4, 0)]),
    3: dict(n=1024, L=48.0, dtype="c128", g=(2.0, 2.0, 2.0), k_L=1.0, n_total=1000.0,
            schedule=[(5000, 1e-3, 1)]),
    4: dict(n=2048, L=64.0, dtype="c128", g=(2.0, 2.0, 2.0), k_L=1.0, n_total=1000.0,
            schedule=[(2000, 2.5e-4, 0)]),
    5: dict(n=8192, L=128.0, dtype="c64", g=(1.0, 1.0, 0.5), k_L=1.0, n_total=1000.0,
            schedule=[(500, 1e-4, 0)]),
}


def _tf_state(seed: int, ny: int, nx: int, X: np.ndarray, Y: np.ndarray, g_uu: float, g_ud: float,
              n_total: float, dx: float, dy: float) -> np.ndarray:
    """Thomas-Fermi-shaped amplitude with random phase noise."""
    R2 = 2.0 * np.sqrt((g_uu + g_ud) * n_total / (2.0 * np.pi))
    amp = np.sqrt(np.maximum(0.0, 1.0 - (X * X + Y * Y) / R2))
    phi = real_normal_field(seed, ny, nx, 2)
    psi = amp[:, :, None] * np.exp(1j * 0.05 * phi)
    for c in range(2):
        nc = dx * dy * np.sum(np.abs(psi[:, :, c]) ** 2)
        psi[:, :, c] *= np.sqrt(0.5 * n_total / nc)
    return psi


def _speckle(seed: int, ny: int, nx: int, sigma_pts: float) -> np.ndarray:
    """0.1*|F|^2/<|F|^2>, F = complex white noise blurred by a separable periodic Gaussian."""
    F = complex_normal_field(seed, ny, nx, 1)[:, :, 0]
    for axis, n in ((0, ny), (1, nx)):
        m = np.fft.fftfreq(n) * n  # integer offsets, periodic
        kern = np.exp(-0.5 * (m / sigma_pts) ** 2)
        kern /= kern.sum()
        shape = [1, 1]
        shape[axis] = n
        F = np.fft.ifft(np.fft.fft(F, axis=axis) * np.fft.fft(kern).reshape(shape), axis=axis)
    I = np.abs(F) ** 2
    return 0.1 * I / I.mean()


def make_workload(cfg: int, dtype: Optional[str] = None, g: Optional[float] = None,
                  n: Optional[int] = None, nx: Optional[int] = None, ny: Optional[int] = None) -> Workload:
    """Materialise config `cfg` (1..5).

    dtype overrides the storage precision (config 4 has a c64 variant); g overrides
    the common interaction strength of config 3's sweep; n (or nx, ny) overrides the
    grid size while keeping the box (a "proxy" of the same recipe for parity tests the
    oracle can finish in seconds).
    """
    c = CONFIGS[cfg]
    nx = int(nx or n or c["n"])
    ny = int(ny or n or c["n"])
    L = c["L"]
    dt_ = dtype or c["dtype"]
    g_uu, g_dd, g_ud = c["g"]
    if g is not None:
        if cfg not in (3, 4):
            raise ValueError("g override is config 3/4's sweep parameter")
        g_uu = g_dd = g_ud = float(g)
    seed = SEED_BASE + cfg
    x = grid(nx, L)
    y = grid(ny, L)
    X, Y = np.meshgrid(x, y)  # [ny, nx]
    dx, dy = L / nx, L / ny
    V = 0.5 * (X * X + Y * Y)
    Omega = None
    delta = None
    if cfg == 1:
        noise = complex_normal_field(seed, ny, nx, 2) * (1e-3 / np.sqrt(2.0))
        psi = np.exp(-0.5 * (X * X + Y * Y))[:, :, None] + noise
        for k in range(2):
            nc = dx * dy * np.sum(np.abs(psi[:, :, k]) ** 2)
            psi[:, :, k] *= np.sqrt(0.5 * c["n_total"] / nc)
    else:
        psi = _tf_state(seed, ny, nx, X, Y, g_uu, g_ud, c["n_total"], dx, dy)
        if cfg == 2:
            Omega = np.full((ny, nx), 2.0)
            delta = np.full((ny, nx), 0.5)
        elif cfg in (3, 4):
            Omega = 4.0 * np.tanh(Y / 2.0)
            delta = 0.2 * X
        elif cfg == 5:
            Omega = 4.0 * np.tanh(Y / 2.0)
            delta = None
            # correlation length 0.5 at dx = 128/8192 = 1/64 -> sigma = 32 grid points
            V = V + _speckle(seed + 1000, ny, nx, 0.5 / dx)
    if dt_ == "c64":
        # inputs are rounded to fp32 first and THOSE values go to both sides
        psi = psi.astype(np.complex64).astype(np.complex128)
        V = V.astype(np.float32).astype(np.float64)
        Omega = None if Omega is None else Omega.astype(np.float32).astype(np.float64)
        delta = None if delta is None else delta.astype(np.float32).astype(np.float64)
    return Workload(
        name=f"config{cfg}_{nx}x{ny}_{dt_}" + (f"_g{g_uu:g}" if cfg == 3 else ""),
        cfg=cfg, nx=nx, ny=ny, Lx=L, Ly=L, dtype=dt_, g_uu=g_uu, g_dd=g_dd, g_ud=g_ud, k_L=c["k_L"],
        norm_mode=0, n_total=c["n_total"], V=np.ascontiguousarray(V),
        Omega=None if Omega is None else np.ascontiguousarray(Omega),
        delta=None if delta is None else np.ascontiguousarray(delta),
        psi0=np.ascontiguousarray(psi), schedule=list(c["schedule"]),
    )
