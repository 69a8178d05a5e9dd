"""Seeded synthetic input generators for the five BASELINE.json configs (+ 4b).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and it holds
NONE of the radiation method's arithmetic: it only produces particle state (r, beta,
betadot, w), observation directions and frequency grids.  numpy only (no torch, no CUDA).

The paper's workload is a live PIConGPU Kelvin-Helmholtz run; it is
not a dataset and PIConGPU is not available, so these generators stand in for it, taking
its structure (two counter-streaming beta = +-0.2 populations in a shear layer).  Recipe:
BASELINE.json `configs`, readings Q14-Q19 of SURVEY.md section 8(c), restated in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Iterator, Optional

import numpy as np

C_LIGHT = 299792458.0            # m/s
E_CHARGE = 1.602176634e-19       # C
M_ELECTRON = 9.1093837015e-31    # kg
BASE_SEED = 250103383

STATE_NAMES = ("rx", "ry", "rz", "bx", "by", "bz", "bdx", "bdy", "bdz", "w")


# ----------------------------------------------------------------------------- RNG (Q19)
def _splitmix64(x: np.ndarray) -> np.ndarray:
    """Counter-based splitmix64 finaliser on uint64 arrays (wraps mod 2^64)."""
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles in (0,1): value i depends only on (seed, stream, offset+i)."""
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0x100000001B3) + np.uint64(stream))
        bits = _splitmix64(idx * np.uint64(0x9E3779B97F4A7C15) ^ key)
    return ((bits >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """Box-Muller Gaussians from two uniform streams (2*stream, 2*stream+1)."""
    u1 = uniform01(seed, 2 * stream, n, offset)
    u2 = uniform01(seed, 2 * stream + 1, n, offset)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ------------------------------------------------------------------- grids (Q15, Q16)
def dirs_seeded_uniform(n_dir: int, seed: int) -> np.ndarray:
    z = 2.0 * uniform01(seed, 100, n_dir) - 1.0
    phi = 2.0 * np.pi * uniform01(seed, 101, n_dir)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def dirs_fibonacci(n_dir: int) -> np.ndarray:
    """Golden-spiral lattice: z_i = 1-(2i+1)/D, phi_i = 2 pi i / golden (Q15)."""
    i = np.arange(n_dir, dtype=np.float64)
    z = 1.0 - (2.0 * i + 1.0) / n_dir
    phi = 2.0 * np.pi * i / ((1.0 + np.sqrt(5.0)) / 2.0)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def omega_log(n: int, lo: float = 1e14, hi: float = 1e18) -> np.ndarray:
    if n == 1:
        return np.array([lo])
    return lo * (hi / lo) ** (np.arange(n, dtype=np.float64) / (n - 1))


def omega_dyadic(n: int, bins_per_octave: int, hi: float = 1e18) -> np.ndarray:
    """Log grid with an integer number of bins per octave, top bin = hi: w_(j+b) = 2 w_j EXACTLY
    (one octave of b values times exact powers of two)."""
    b = int(bins_per_octave)
    j = np.arange(n, dtype=np.int64) - (n - 1)              # <= 0: octaves below the top bin
    base = hi * 2.0 ** (-(np.arange(b, dtype=np.float64)) / b)   # one octave, descending from hi
    return np.ldexp(base[(-j) % b], -((-j) // b).astype(np.int64))


def omega_linear(n: int, hi: float) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 1.0) * (hi / n)


# ------------------------------------------------------------------------- trajectories
class HelixSource:
    """Analytic helical electron orbits in uniform B_z (config 0, Q18)."""

    def __init__(self, n: int, seed: int, omega_c=1e14, beta_perp=0.1, beta_z=0.05, box=1e-6):
        self.n, self.omega_c, self.bp, self.bz = n, omega_c, beta_perp, beta_z
        self.r0 = np.stack([box * uniform01(seed, s, n) for s in (0, 1, 2)], axis=0)
        self.phi0 = 2.0 * np.pi * uniform01(seed, 3, n)
        self.w = np.ones(n)

    def state(self, t: float):
        wc, bp, bz = self.omega_c, self.bp, self.bz
        ph = wc * t + self.phi0
        rho = C_LIGHT * bp / wc
        rx = self.r0[0] + rho * (np.sin(ph) - np.sin(self.phi0))
        ry = self.r0[1] + rho * (-np.cos(ph) + np.cos(self.phi0))
        rz = self.r0[2] + C_LIGHT * bz * t
        bx, by = bp * np.cos(ph), bp * np.sin(ph)
        bzv = np.full(self.n, bz)
        bdx, bdy = -wc * bp * np.sin(ph), wc * bp * np.cos(ph)
        return [rx, ry, rz, bx, by, bzv, bdx, bdy, np.zeros(self.n), self.w]


class KHISource:
    """KHI-like shear flow pushed with a Boris rotation (configs 1-4, Q17).

    r ~ U[0,L)^3; beta_x = +0.2 (y<L/2) / -0.2 (y>=L/2) + N(0, 0.01^2) per axis;
    B_z(x,y) = B0 tanh((y-L/2)/0.5um) (1 + 0.1 sin(2 pi x/L)), E = 0, no boundaries.
    State handed out at step t is (r^t, beta^t, betadot^t = q/(gamma m) beta^t x B(r^t)).
    """

    def __init__(self, n: int, seed: int, dt: float, L=10e-6, B0=50.0, stream=0.2,
                 sigma=0.01, shear=0.5e-6, regions=None, weights=None):
        self.n, self.dt, self.L, self.B0, self.shear = n, dt, L, B0, shear
        self.r = np.stack([L * uniform01(seed, s, n) for s in (0, 1, 2)], axis=0)
        self.b = np.stack([sigma * normal01(seed, 10 + s, n) for s in (0, 1, 2)], axis=0)
        self.b[0] += np.where(self.r[1] < 0.5 * L, stream, -stream)
        self.region_offsets = None
        if regions is not None:
            # sub-volumes: an (Rx, Ry) grid of boxes in the x-y plane; particles are stored
            # sorted by the box their INITIAL position lies in (region id = ix*Ry + iy), as a
            # PIC code stores them cell by cell.  Membership is kept for the run: over the few
            # hundred steps of 1e-17 s used here a particle moves < 1 nm.
            rx_n, ry_n = regions
            ix = np.minimum((self.r[0] / L * rx_n).astype(np.int64), rx_n - 1)
            iy = np.minimum((self.r[1] / L * ry_n).astype(np.int64), ry_n - 1)
            rid = ix * ry_n + iy
            order = np.argsort(rid, kind="stable")
            self.r, self.b = self.r[:, order], self.b[:, order]
            counts = np.bincount(rid, minlength=rx_n * ry_n)
            self.region_offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
        g = 1.0 / np.sqrt(1.0 - np.sum(self.b * self.b, axis=0))
        self.qm = (-E_CHARGE / M_ELECTRON) / g      # q/(gamma m); gamma is conserved (E=0)
        # macro weights: 1 (BASELINE.json configs), or seeded log-uniform in [1, wmax) for the
        # form-factor workloads (a PIC run with density gradients has weights spanning decades)
        self.w = np.ones(n) if weights is None else float(weights) ** uniform01(seed, 20, n)
        if weights is not None and regions is not None:
            self.w = self.w[order]

    def _Bz(self):
        x, y = self.r[0], self.r[1]
        return self.B0 * np.tanh((y - 0.5 * self.L) / self.shear) * (
            1.0 + 0.1 * np.sin(2.0 * np.pi * x / self.L))

    def state(self):
        k = self.qm * self._Bz()                    # betadot = k * (beta x z_hat)
        return [self.r[0], self.r[1], self.r[2], self.b[0], self.b[1], self.b[2],
                k * self.b[1], -k * self.b[0], np.zeros(self.n), self.w]

    def advance(self):
        t = self.qm * self._Bz() * (0.5 * self.dt)  # rotation vector t*z_hat
        s = 2.0 * t / (1.0 + t * t)
        bx, by = self.b[0], self.b[1]
        px, py = bx + by * t, by - bx * t           # b' = b + b x t
        self.b[0], self.b[1] = bx + py * s, by - px * s
        self.r = self.r + (C_LIGHT * self.dt) * self.b


# ------------------------------------------------------------------------------ configs
@dataclass
class Workload:
    name: str
    n_particles: int
    n_steps: int
    dt: float
    dirs: np.ndarray
    omega: np.ndarray
    state_dtype: type
    seed: int
    kind: str                      # "helix" | "khi"
    t0: float = 0.0
    extra: dict = field(default_factory=dict)
    form_factor: Optional[tuple] = None     # (type name, size[3] in metres) for rad_config / the oracle
    nyquist: float = 0.0                    # rad_config.nyquist_factor (0: limiter off)
    precise: bool = False                   # RAD_FLAG_PRECISE (all-polynomial sincos)

    @property
    def n_dir(self) -> int:
        return self.dirs.shape[0]

    @property
    def n_omega(self) -> int:
        return self.omega.shape[0]

    @property
    def updates_per_step(self) -> int:
        return self.n_particles * self.n_dir * self.n_omega

    @property
    def n_regions(self) -> int:
        rg = self.extra.get("regions")
        return 1 if rg is None else int(rg[0] * rg[1])

    def region_offsets(self, n_particles: Optional[int] = None) -> np.ndarray:
        """[n_regions+1] int64 offsets of the region-sorted particle arrays steps() yields."""
        N = self.n_particles if n_particles is None else n_particles
        if self.kind != "khi" or self.extra.get("regions") is None:
            return np.array([0, N], dtype=np.int64)
        return KHISource(N, self.seed, self.dt, **self.extra).region_offsets

    def steps(self, n_steps: Optional[int] = None, n_particles: Optional[int] = None
              ) -> Iterator[tuple]:
        """Yield (step_index, [10 arrays of state_dtype]); optionally only the first
        n_steps steps / first n_particles particles (particle i is the same in both)."""
        T = self.n_steps if n_steps is None else n_steps
        N = self.n_particles if n_particles is None else n_particles
        if self.kind == "helix":
            src = HelixSource(N, self.seed, **self.extra)
            for t in range(T):
                yield t, [np.ascontiguousarray(a, dtype=self.state_dtype)
                          for a in src.state(self.t0 + t * self.dt)]
        else:
            src = KHISource(N, self.seed, self.dt, **self.extra)
            for t in range(T):
                yield t, [np.ascontiguousarray(a, dtype=self.state_dtype) for a in src.state()]
                if t + 1 < T:
                    src.advance()


SWEEP_SHAPES = ((16, 4096), (64, 1024), (256, 256), (1024, 64))


def make_workload(cfg: str) -> Workload:
    """cfg in {"0","1","2","3a","3b","3c","3d","4","4b"} (BASELINE.json configs, 0-based),
    or "5r": the per-region (sub-volume) detector workload of SURVEY.md section 8(f) NEXT-2."""
    if cfg == "0":
        wc = 1e14
        return Workload("cfg0_tiny_helical", 256, 128, 1.0 / (20.0 * wc),
                        dirs_seeded_uniform(8, BASE_SEED), omega_linear(64, 4.0 * wc),
                        np.float64, BASE_SEED, "helix")
    if cfg == "1":
        return Workload("cfg1_khi_like", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_log(512), np.float32, BASE_SEED + 1, "khi")
    if cfg == "2":
        return Workload("cfg2_production_like", 1048576, 2000, 1e-17, dirs_fibonacci(256),
                        omega_log(1024), np.float32, BASE_SEED + 2, "khi")
    if cfg in ("3a", "3b", "3c", "3d"):
        D, W = SWEEP_SHAPES["abcd".index(cfg[1])]
        return Workload(f"cfg3_sweep_{D}x{W}", 262144, 200, 1e-17, dirs_fibonacci(D),
                        omega_log(W), np.float32, BASE_SEED + 3, "khi")
    if cfg == "4":
        return Workload("cfg4_streaming", 16777216, 4, 1e-17, dirs_fibonacci(16),
                        omega_log(128), np.float32, BASE_SEED + 4, "khi")
    if cfg == "4b":
        return Workload("cfg4b_streaming_1x8", 16777216, 4, 1e-17, dirs_fibonacci(1),
                        omega_log(8), np.float32, BASE_SEED + 4, "khi")
    if cfg == "1u":
        # config 1 on a LINEAR frequency grid (not a BASELINE.json config): the shape on which the
        # uniform-grid rotation-recurrence kernel (a2') is measured
        return Workload("cfg1u_khi_linear_grid", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_linear(512, 1e17), np.float32, BASE_SEED + 1, "khi")
    if cfg == "1f":
        # config 1 with macro weights log-uniform in [1, 1e4) and a Gaussian macro-particle shape of
        # 30 nm (the form factor passes from coherent to incoherent around w = c / 30 nm = 1e16 rad/s,
        # the middle of the grid): the form-factor leg of bench.py (not a BASELINE.json config)
        return Workload("cfg1f_khi_form_factor", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_log(512), np.float32, BASE_SEED + 1, "khi", extra={"weights": 1e4},
                        form_factor=("gaussian", (3e-8, 3e-8, 3e-8)))
    if cfg == "1d":
        # config 1 on a DYADIC log grid: 32 bins per octave, 512 bins = 16 octaves below 1e18 rad/s
        # ([1.56e13, 1e18]): the shape on which the squaring-chain variant of the general kernel is
        # measured (not a BASELINE.json config, whose log grids have
        # 38.46 / 76.99 bins per octave)
        return Workload("cfg1d_khi_dyadic_grid", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_dyadic(512, 32), np.float32, BASE_SEED + 1, "khi")
    if cfg == "1p":
        # config 1 with RAD_FLAG_PRECISE (every sincos by the fp32 polynomial): the precise-mode leg of bench.py
        return Workload("cfg1p_khi_precise", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_log(512), np.float32, BASE_SEED + 1, "khi", precise=True)
    if cfg == "1n":
        # config 1 with the Nyquist limiter at nu = 1 (w dt (1 - beta.n) >= pi dropped: at dt = 1e-17 s the
        # top ~1/8 of the log grid, the cut-off Doppler-shifted per particle and direction): the limiter
        # leg of bench.py (not a BASELINE.json config)
        return Workload("cfg1n_khi_nyquist", 65536, 1000, 1e-17, dirs_fibonacci(128),
                        omega_log(512), np.float32, BASE_SEED + 1, "khi", nyquist=1.0)
    if cfg == "5r":
        # smallest KHI run = 192 x 256 x 12 cells x 9 particles per cell on 16
        # GPUs -> 331 776 particles per GPU; line 196: one ML sample = the ~3e4 particles of a
        # sub-volume -> 12 sub-volumes; line 184: "spectrum observed in one direction".
        return Workload("cfg5r_regions_12x1x512", 331776, 200, 1e-17, np.array([[1.0, 0.0, 0.0]]),
                        omega_log(512), np.float32, BASE_SEED + 5, "khi", extra={"regions": (2, 6)})
    if cfg == "5s":
        # config 5r with a COARSER spectrum per sub-volume, 1 direction x 128 frequencies: a few-direction detector whose
        # frequency tile (16 lanes x 8 bins) would leave half of every warp idle; the lane groups then split the
        # particles of a batch ("particle split").  Not a BASELINE.json config.
        return Workload("cfg5s_regions_12x1x128", 331776, 200, 1e-17, np.array([[1.0, 0.0, 0.0]]),
                        omega_log(128), np.float32, BASE_SEED + 5, "khi", extra={"regions": (2, 6)})
    raise KeyError(cfg)


ALL_CONFIGS = ("0", "1", "1u", "1f", "1n", "1d", "1p", "2", "3a", "3b", "3c", "3d", "4", "4b", "5r", "5s")
