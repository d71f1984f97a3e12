"""Seeded synthetic sky catalogs standing in for the MICE mocks.

Everything here produces *inputs*: RA/Dec rows in degrees, explicit theta-edge arrays and seeded
row subsets.  None of the method's arithmetic (unit vectors, dot products, binning, estimator)
lives here, so the module can feed both the oracle and the CUDA library without coupling them.

Random numbers come from a counter-based SplitMix64 stream implemented below (numpy is only the
array engine), so the catalogs do not depend on numpy's Generator bit streams.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_MASK = (1 << 64) - 1


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


class SplitMix:
    """Counter-based SplitMix64: output n of stream (seed, stream) is mix(base + (n+1)*GAMMA)."""

    def __init__(self, seed: int, stream: int = 0):
        s = (int(seed) * 0x9E3779B97F4A7C15 + int(stream) * 0xD1B54A32D192ED03 + 0x2545F4914F6CDD1D) & _MASK
        # one scalar mix so that nearby seeds give unrelated bases
        self._base = int(_mix(np.array([s], dtype=np.uint64))[0])
        self._n = 0

    def u64(self, n: int) -> np.ndarray:
        idx = np.arange(self._n + 1, self._n + n + 1, dtype=np.uint64)
        self._n += n
        return _mix(np.uint64(self._base) + idx * _GAMMA)

    def uniform(self, n: int) -> np.ndarray:
        """n doubles uniform in [0, 1) with 53 random bits."""
        return (self.u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)

    def normal(self, n: int) -> np.ndarray:
        """n standard normals by Box-Muller (two uniforms per pair of outputs)."""
        m = (n + 1) // 2
        u1 = 1.0 - self.uniform(m)  # (0, 1]
        u2 = self.uniform(m)
        r = np.sqrt(-2.0 * np.log(u1))
        out = np.empty(2 * m, dtype=np.float64)
        out[0::2] = r * np.cos(2.0 * np.pi * u2)
        out[1::2] = r * np.sin(2.0 * np.pi * u2)
        return out[:n]

    def integers(self, n: int, hi: int) -> np.ndarray:
        return np.minimum((self.uniform(n) * hi).astype(np.int64), hi - 1)


Patch = Tuple[float, float, float, float]  # ra0, ra1, dec0, dec1 (degrees)


def uniform_patch(n: int, patch: Patch, rng: SplitMix) -> np.ndarray:
    """Uniform in area on an RA/Dec rectangle: uniform RA, uniform sin(Dec)."""
    ra0, ra1, dec0, dec1 = patch
    s0, s1 = np.sin(np.radians(dec0)), np.sin(np.radians(dec1))
    ra = ra0 + (ra1 - ra0) * rng.uniform(n)
    dec = np.degrees(np.arcsin(np.clip(s0 + (s1 - s0) * rng.uniform(n), -1.0, 1.0)))
    return np.stack([ra, dec], axis=1)


def uniform_sphere(n: int, rng: SplitMix) -> np.ndarray:
    return uniform_patch(n, (0.0, 360.0, -90.0, 90.0), rng)


def _inside(radec: np.ndarray, patch: Patch) -> np.ndarray:
    ra0, ra1, dec0, dec1 = patch
    return (radec[:, 0] >= ra0) & (radec[:, 0] < ra1) & (radec[:, 1] >= dec0) & (radec[:, 1] < dec1)


def _scatter(centres: np.ndarray, pick: np.ndarray, sigma_deg: float, patch: Patch, rng: SplitMix) -> np.ndarray:
    """Gaussian offsets (dRA*cos(Dec_c), dDec) ~ N(0, sigma)^2 around centres[pick]; redraw outside rows."""
    n = pick.shape[0]
    out = np.empty((n, 2), dtype=np.float64)
    todo = np.arange(n)
    while todo.size:
        c = centres[pick[todo]]
        g = rng.normal(2 * todo.size).reshape(-1, 2)
        cand = np.empty((todo.size, 2))
        cand[:, 0] = c[:, 0] + sigma_deg * g[:, 0] / np.maximum(np.cos(np.radians(c[:, 1])), 1e-6)
        cand[:, 1] = c[:, 1] + sigma_deg * g[:, 1]
        ok = _inside(cand, patch)
        out[todo[ok]] = cand[ok]
        todo = todo[~ok]
    return out


def gaussian_clumps(n: int, n_clumps: int, sigma_deg: float, patch: Patch, rng: SplitMix,
                    clump_major: bool = False) -> np.ndarray:
    """Clump centres uniform on the patch; each point belongs to one clump (configs 1 and 5).

    clump_major=False: each point picks a clump uniformly at random (generation order).
    clump_major=True : equal counts per clump, emitted clump after clump (config 5).
    """
    centres = uniform_patch(n_clumps, patch, rng)
    if clump_major:
        pick = (np.arange(n, dtype=np.int64) * n_clumps) // n
    else:
        pick = rng.integers(n, n_clumps)
    return _scatter(centres, pick, sigma_deg, patch, rng)


def neyman_scott(n: int, patch: Patch, parents_inside: int, sigma_deg: float, rng: SplitMix) -> np.ndarray:
    """Neyman-Scott process conditioned on n points inside the patch (config 2).

    Parents are uniform on the patch padded by 5 sigma, with a density that puts about
    `parents_inside` of them inside the patch; every point picks a parent uniformly (Poisson
    children conditioned on the total) and is kept only if it falls inside.
    """
    ra0, ra1, dec0, dec1 = patch
    pad = 5.0 * sigma_deg
    padded = (ra0 - pad, ra1 + pad, max(dec0 - pad, -90.0), min(dec1 + pad, 90.0))

    def area(p):
        return (p[1] - p[0]) * (np.sin(np.radians(p[3])) - np.sin(np.radians(p[2])))

    n_par = int(round(parents_inside * area(padded) / area(patch)))
    parents = uniform_patch(n_par, padded, rng)
    out = np.empty((0, 2))
    while out.shape[0] < n:
        m = int((n - out.shape[0]) * 1.15) + 64
        pick = rng.integers(m, n_par)
        c = parents[pick]
        g = rng.normal(2 * m).reshape(-1, 2)
        cand = np.empty((m, 2))
        cand[:, 0] = c[:, 0] + sigma_deg * g[:, 0] / np.maximum(np.cos(np.radians(c[:, 1])), 1e-6)
        cand[:, 1] = c[:, 1] + sigma_deg * g[:, 1]
        out = np.concatenate([out, cand[_inside(cand, patch)]], axis=0)
    return out[:n]


def lognormal_mock(n: int, patch: Patch, grid: Tuple[int, int], slope: float, rng: SplitMix) -> np.ndarray:
    """Lognormal density mock (configs 3 and 4).

    Equal-area grid in (RA, sin Dec) of grid=(n_ra, n_sd) cells; Gaussian field by FFT with flat-sky
    P(k) ~ k^slope (stand-in for C_l ~ l^slope), scaled to unit variance; rho = exp(g - 1/2);
    exactly n points drawn over cells with probability ~ rho, uniform inside the cell.
    """
    ra0, ra1, dec0, dec1 = patch
    n_ra, n_sd = grid
    white = rng.normal(n_ra * n_sd).reshape(n_sd, n_ra)
    fk = np.fft.rfft2(white)
    ky = np.fft.fftfreq(n_sd)[:, None] * n_sd
    kx = np.fft.rfftfreq(n_ra)[None, :] * n_ra
    k = np.sqrt(kx * kx + ky * ky)
    k[0, 0] = 1.0
    amp = k ** (0.5 * slope)
    amp[0, 0] = 0.0
    g = np.fft.irfft2(fk * amp, s=(n_sd, n_ra))
    g /= g.std()
    rho = np.exp(g - 0.5).ravel()
    cdf = np.cumsum(rho)
    cdf /= cdf[-1]
    cell = np.minimum(np.searchsorted(cdf, rng.uniform(n), side="right"), n_ra * n_sd - 1)
    iy, ix = np.divmod(cell, n_ra)
    s0, s1 = np.sin(np.radians(dec0)), np.sin(np.radians(dec1))
    ra = ra0 + (ra1 - ra0) * (ix + rng.uniform(n)) / n_ra
    sd = s0 + (s1 - s0) * (iy + rng.uniform(n)) / n_sd
    dec = np.degrees(np.arcsin(np.clip(sd, -1.0, 1.0)))
    return np.stack([ra, dec], axis=1)


def great_circle_ring(n: int, tilt_deg: float = 33.0, node_deg: float = 21.0, phase_deg: float = 0.0) -> np.ndarray:
    """n points equally spaced by 360/n degrees on a great circle tilted by tilt_deg.

    Only emits positions; the separations m*360/n and their multiplicities are a property of the
    ring that the tests state independently.
    """
    t = np.radians(phase_deg + 360.0 * np.arange(n) / n)
    i, o = np.radians(tilt_deg), np.radians(node_deg)
    # circle in the plane spanned by a=(cos o, sin o, 0) and b=(-sin o cos i, cos o cos i, sin i)
    x = np.cos(t) * np.cos(o) - np.sin(t) * np.sin(o) * np.cos(i)
    y = np.cos(t) * np.sin(o) + np.sin(t) * np.cos(o) * np.cos(i)
    z = np.sin(t) * np.sin(i)
    ra = np.degrees(np.arctan2(y, x)) % 360.0
    dec = np.degrees(np.arcsin(np.clip(z, -1.0, 1.0)))
    return np.stack([ra, dec], axis=1)


# --------------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# --------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class Config:
    name: str
    n_d: int
    n_r: int
    nbins: int
    theta_min: float
    theta_max: float
    mode: str            # "log" | "linear"
    dtype: str           # "f64" | "f32": dtype of the RA/Dec rows handed to the library
    note: str = ""
    extra: Dict = field(default_factory=dict)


CONFIGS: Dict[int, Config] = {
    1: Config("cfg1_tiny_clumps", 4096, 4096, 20, 0.01, 10.0, "log", "f64",
              "64 Gaussian clumps sigma 0.5 deg on a 10x10 deg patch; R uniform"),
    2: Config("cfg2_neyman_scott", 100_000, 100_000, 30, 0.01, 30.0, "log", "f32",
              "Neyman-Scott, ~2000 parents, sigma 0.2 deg, 30x30 deg patch; float32 rows"),
    3: Config("cfg3_paper_scale_octant", 430_000, 430_000, 40, 0.01, 60.0, "log", "f64",
              "lognormal mock on one octant, P(k)~k^-1.2; Table 2 row 1 size (PAPER.md:61)"),
    4: Config("cfg4_fullsky_large", 1_000_000, 2_000_000, 50, 0.005, 90.0, "log", "f64",
              "lognormal mock full sky; 4.5e12 pairs"),
    5: Config("cfg5_contention", 500_000, 500_000, 512, 0.0, 7.1, "linear", "f64",
              "200 clumps sigma 0.05 deg on a 5x5 deg patch, clump-major rows; 512 linear bins"),
}


def edges(nbins: int, theta_min: float, theta_max: float, mode: str) -> np.ndarray:
    """Explicit theta edges in degrees for a (nbins, min, max, mode) specification.

    This is input preparation: parity tests hand the *same array* to the oracle and (in EXPLICIT
    mode) to the library, so neither side's edge generator is trusted by the other.
    """
    k = np.arange(nbins + 1, dtype=np.float64)
    if mode == "linear":
        e = theta_min + k * ((theta_max - theta_min) / nbins)
    elif mode == "log":
        e = theta_min * np.power(theta_max / theta_min, k / nbins)
    else:
        raise ValueError(mode)
    e[0], e[-1] = theta_min, theta_max
    return e


def config_edges(cfg: Config) -> np.ndarray:
    return edges(cfg.nbins, cfg.theta_min, cfg.theta_max, cfg.mode)


def make_config(idx: int, n_d: int | None = None, n_r: int | None = None, shuffle_d: bool = False):
    """Return (D, R, edges, cfg) for BASELINE config idx; n_d/n_r override the sizes (same recipe).

    D, R are (n, 2) RA/Dec degree arrays in cfg.dtype (float32 rows are the float64 draw rounded once).
    """
    cfg = CONFIGS[idx]
    nd = cfg.n_d if n_d is None else n_d
    nr = cfg.n_r if n_r is None else n_r
    rd, rr = SplitMix(1, idx), SplitMix(2, idx)
    if idx == 1:
        patch = (0.0, 10.0, -5.0, 5.0)
        D = gaussian_clumps(nd, 64, 0.5, patch, rd)
        R = uniform_patch(nr, patch, rr)
    elif idx == 2:
        patch = (0.0, 30.0, -15.0, 15.0)
        D = neyman_scott(nd, patch, 2000, 0.2, rd)
        R = uniform_patch(nr, patch, rr)
    elif idx == 3:
        patch = (0.0, 90.0, 0.0, 90.0)
        D = lognormal_mock(nd, patch, (2048, 2048), -1.2, rd)
        R = uniform_patch(nr, patch, rr)
    elif idx == 4:
        patch = (0.0, 360.0, -90.0, 90.0)
        D = lognormal_mock(nd, patch, (4096, 2048), -1.2, rd)
        R = uniform_patch(nr, patch, rr)
    elif idx == 5:
        patch = (0.0, 5.0, -2.5, 2.5)
        D = gaussian_clumps(nd, 200, 0.05, patch, rd, clump_major=True)
        R = uniform_patch(nr, patch, rr)
    else:
        raise KeyError(idx)
    if shuffle_d:
        D = D[np.argsort(SplitMix(3, idx).u64(nd), kind="stable")]
    dt = np.float32 if cfg.dtype == "f32" else np.float64
    return np.ascontiguousarray(D, dtype=dt), np.ascontiguousarray(R, dtype=dt), config_edges(cfg), cfg


def subset_rows(n: int, k: int = 2000, seed: int = 12345) -> np.ndarray:
    """k distinct row indices out of n, seeded (2,000-row validation subset)."""
    k = min(k, n)
    order = np.argsort(SplitMix(seed, 7).u64(n), kind="stable")
    return np.sort(order[:k]).astype(np.int64)


# ---- 3-D boxes for the xi(r) variant; positions only, no distances are formed here ---------------
def uniform_box(n: int, side: float, rng: SplitMix) -> np.ndarray:
    """n rows (x, y, z) uniform in the cube [0, side)^3."""
    return (rng.uniform(3 * n) * side).reshape(n, 3)


def clustered_box(n: int, side: float, n_clumps: int, sigma: float, rng: SplitMix) -> np.ndarray:
    """n rows in [0, side)^3: Gaussian clumps of width sigma around n_clumps uniform centres, emitted clump-major;
    points that fall outside the cube are reflected back in (a stand-in for a clustered 3-D galaxy mock)."""
    centres = rng.uniform(3 * n_clumps).reshape(n_clumps, 3) * side
    pick = np.sort(rng.integers(n, n_clumps))
    x = centres[pick] + sigma * rng.normal(3 * n).reshape(n, 3)
    x = np.abs(x)
    x = np.where(x >= side, 2.0 * side - x, x)
    return np.clip(x, 0.0, np.nextafter(side, 0.0))


def cubic_lattice(m: int) -> np.ndarray:
    """The m^3 points of the integer lattice {0..m-1}^3 (hand-checkable pair multiplicities)."""
    g = np.arange(m, dtype=np.float64)
    return np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)


def make_box_config(n_d: int = 430_000, n_r: int = 430_000, side: float = 1000.0, nbins: int = 40,
                    r_min: float = 1.0, r_max: float = 200.0, mode: str = "log", seed: int = 31):
    """3-D stand-in at paper scale: D clustered (n_d / 400 clumps of width side / 200), R uniform, in a cube of `side`
    (think Mpc/h); `nbins` bins in r from r_min to r_max.  Returns (D, R, r_edges)."""
    D = clustered_box(n_d, side, max(1, n_d // 400), side / 200.0, SplitMix(seed, 0))
    R = uniform_box(n_r, side, SplitMix(seed, 1))
    return D, R, edges(nbins, r_min, r_max, mode)
