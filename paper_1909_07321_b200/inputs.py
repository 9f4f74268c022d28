"""Seeded synthetic inputs shaped like PSTGF's R-matrix formation workloads.

This module only draws random numbers and lays out energy meshes.  It holds
none of the method's arithmetic (no 1/(E_k - E), no contraction) and imports
neither the CUDA binding nor ``oracle/``: tests and ``bench.py`` hand the
arrays it returns to both sides.

The five configurations are the ones ``BASELINE.json`` lists.  Their shapes
stand in for the paper's workloads, whose ``H.DATXXX`` inputs are not
available: n_poles = 20 * n_chan follows MNP2 ~ NCHAN x NRANG
(and 106661/7261 ~ 14.7 at PAPER.md:168), tens of partial
waves of unequal channel count follow PAPER.md:676, and the linear energy
meshes follow IMESH=1, ``E0 + i*EINCR``.

Readings: R10 deterministic meshes, R11 pole
clearance rule, R12 generator and draw order.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

CLEARANCE_RYD = 1.0e-3  # BASELINE.json: every energy >= 1e-3 Ryd from any pole


@dataclass
class Wave:
    """One partial wave's inputs for eq. 4.

    W        [n_chan, n_poles] float64, row-major: surface amplitudes w_nk
             (record WMAT)
    E_k      [n_poles] float64: R-matrix poles (record VALUE)
    energies [n_E] float64: impact energies, same units and origin as E_k
    a        R-matrix radius r0 in a.u. (record RA)
    """

    W: np.ndarray
    E_k: np.ndarray
    energies: np.ndarray
    a: float

    @property
    def n_chan(self) -> int:
        return int(self.W.shape[0])

    @property
    def n_poles(self) -> int:
        return int(self.W.shape[1])

    @property
    def n_E(self) -> int:
        return int(self.energies.shape[0])

    def counted_flop(self) -> float:
        """north_star's count: 2 * n_chan^2 * n_poles / 2 per energy."""
        return float(self.n_E) * float(self.n_chan) ** 2 * float(self.n_poles)

    def r_bytes(self) -> float:
        return 8.0 * self.n_E * self.n_chan * self.n_chan


@dataclass
class Workload:
    name: str
    seed: int
    waves: list[Wave] = field(default_factory=list)

    def counted_flop(self) -> float:
        return sum(w.counted_flop() for w in self.waves)

    def r_bytes(self) -> float:
        return sum(w.r_bytes() for w in self.waves)

    def n_energies(self) -> int:
        return sum(w.n_E for w in self.waves)

    def sha256(self) -> str:
        h = hashlib.sha256()
        for w in self.waves:
            for arr in (w.W, w.E_k, w.energies):
                h.update(memoryview(np.ascontiguousarray(arr)).cast("B"))   # no 6 GB copy at paper scale
            h.update(np.float64(w.a).tobytes())
        return h.hexdigest()


def linear_mesh(lo: float, hi: float, n: int) -> np.ndarray:
    """lo + i*(hi-lo)/(n-1): the paper's IMESH=1 grid."""
    if n == 1:
        return np.array([lo], dtype=np.float64)
    i = np.arange(n, dtype=np.float64)
    return lo + i * ((hi - lo) / (n - 1))


def geometric_mesh(lo: float, hi: float, n: int) -> np.ndarray:
    """lo * (hi/lo)^(i/(n-1)): config 4's log-spaced mesh."""
    if n == 1:
        return np.array([lo], dtype=np.float64)
    i = np.arange(n, dtype=np.float64)
    return lo * (hi / lo) ** (i / (n - 1))


def min_pole_distance(energies: np.ndarray, poles_sorted: np.ndarray) -> np.ndarray:
    """Distance from each energy to its nearest pole (poles sorted ascending)."""
    if poles_sorted.size == 0:
        return np.full(energies.shape, np.inf)
    idx = np.searchsorted(poles_sorted, energies)
    left = np.where(idx > 0, np.abs(energies - poles_sorted[np.maximum(idx - 1, 0)]), np.inf)
    right = np.where(idx < poles_sorted.size,
                     np.abs(poles_sorted[np.minimum(idx, poles_sorted.size - 1)] - energies), np.inf)
    return np.minimum(left, right)


def nudge_off_poles(energies: np.ndarray, poles: np.ndarray, clearance: float = CLEARANCE_RYD) -> np.ndarray:
    """Move every energy closer than ``clearance`` to a pole out of the way.

    Forbidden intervals [E_k - c, E_k + c] are merged where they overlap; a
    point strictly inside a merged interval (lo, hi) moves to the nearer end
    (tie -> hi), then steps away ulp by ulp until the clearance holds in
    floating point.  The clearance is asserted on the result.
    """
    e = np.array(energies, dtype=np.float64, copy=True)
    p = np.sort(np.asarray(poles, dtype=np.float64))
    if p.size == 0 or e.size == 0:
        return e
    lo = p - clearance
    hi = p + clearance
    # merge overlapping intervals
    m_lo = [lo[0]]
    m_hi = [hi[0]]
    for a, b in zip(lo[1:], hi[1:]):
        if a <= m_hi[-1]:
            if b > m_hi[-1]:
                m_hi[-1] = b
        else:
            m_lo.append(a)
            m_hi.append(b)
    m_lo = np.array(m_lo)
    m_hi = np.array(m_hi)
    j = np.searchsorted(m_lo, e, side="left") - 1  # last interval with m_lo < e
    for i in range(e.size):
        k = j[i]
        if k < 0 or not (m_lo[k] < e[i] < m_hi[k]):
            continue
        go_up = (m_hi[k] - e[i]) <= (e[i] - m_lo[k])
        x = m_hi[k] if go_up else m_lo[k]
        away = np.inf if go_up else -np.inf
        while min_pole_distance(np.array([x]), p)[0] < clearance:
            x = np.nextafter(x, away)
        e[i] = x
    # points that sat exactly on an interval end may still be an ulp short
    d = min_pole_distance(e, p)
    for i in np.nonzero(d < clearance)[0]:
        x = e[i]
        k = np.searchsorted(p, x)
        nearest_below = k > 0 and (k == p.size or (x - p[k - 1]) <= (p[k] - x))
        away = np.inf if nearest_below else -np.inf
        while min_pole_distance(np.array([x]), p)[0] < clearance:
            x = np.nextafter(x, away)
        e[i] = x
    assert np.all(min_pole_distance(e, p) >= clearance)
    return e


def _draw_wave(rng: np.random.Generator, n_chan: int, n_poles: int, sigma: float,
               pole_lo: float, pole_hi: float):
    W = rng.normal(0.0, sigma, (n_chan, n_poles))
    E_k = np.sort(rng.uniform(pole_lo, pole_hi, n_poles))
    return np.ascontiguousarray(W, dtype=np.float64), E_k.astype(np.float64)


# (P, n_chan, n_E, a, sigma, pole range, mesh range, mesh kind) per BASELINE.json config
_CONFIGS = {
    1: dict(seed=0, P=1, C=8, N=1000, a=20.0, sigma=0.1, poles=(-5.0, 50.0), mesh=(0.1, 10.0), kind="linear"),
    2: dict(seed=1, P=1, C=64, N=4096, a=20.0, sigma=0.1, poles=(-10.0, 100.0), mesh=(0.05, 20.0), kind="linear"),
    3: dict(seed=2, P=8, C=256, N=2048, a=25.0, sigma=0.05, poles=(-20.0, 200.0), mesh=(0.05, 30.0), kind="linear"),
    4: dict(seed=3, P=32, C=None, N=512, a=25.0, sigma=0.05, poles=(-20.0, 300.0), mesh=(0.01, 50.0), kind="geometric"),
    5: dict(seed=4, P=1, C=512, N=256, a=30.0, sigma=0.03, poles=(-30.0, 400.0), mesh=(0.01, 60.0), kind="linear"),
    # Not in BASELINE.json: the one workload the paper times for this path, "7261 channels and a
    # Hamiltonian size of 106 661" (neutral Fe).  W is 6.2 GB, R 422 MB per energy.
    6: dict(seed=5, P=1, C=7261, K=106661, N=16, a=30.0, sigma=0.03, poles=(-30.0, 2000.0), mesh=(0.01, 10.0),
            kind="linear"),
    # Not in BASELINE.json: many small partial waves in one call (PAPER.md:676 runs 42 partial waves of at most
    # 1818 channels, the low-L ones with few channels): 256 waves, n_chan uniform in [8, 32], config 4's recipe.
    7: dict(seed=6, P=256, C=None, C_range=(8, 33), N=512, a=25.0, sigma=0.05, poles=(-20.0, 300.0), mesh=(0.01, 50.0),
            kind="geometric"),
}
POLES_PER_CHANNEL = 20
PAPER_SCALE_CONFIG = 6


def _n_poles(c: dict, n_chan: int) -> int:
    return int(c["K"]) if "K" in c else POLES_PER_CHANNEL * n_chan


def _draw_channels(c: dict, rng: np.random.Generator) -> list[int]:
    """n_chan of every wave: fixed, or drawn first (reading R12) from integers(lo, hi)."""
    if c["C"] is None:
        lo, hi = c.get("C_range", (16, 401))
        return [int(x) for x in rng.integers(lo, hi, size=c["P"])]
    return [c["C"]] * c["P"]


def config_shapes(cfg: int, seed: int | None = None) -> list[tuple[int, int, int]]:
    """(n_chan, n_poles, n_E) per wave without drawing W (cheap; for planning)."""
    c = _CONFIGS[cfg]
    rng = np.random.default_rng(c["seed"] if seed is None else seed)
    chans = _draw_channels(c, rng)
    return [(n, _n_poles(c, n), c["N"]) for n in chans]


def make_config(cfg: int, seed: int | None = None, n_E: int | None = None) -> Workload:
    """Build BASELINE.json config ``cfg`` (1..5), or 6: the paper-scale wave of PAPER.md:168.

    Draw order (reading R12): config 4 first draws all n_chan; then per wave,
    in order, W (row-major fill) and then E_k.  ``n_E`` overrides the mesh
    size (the mesh keeps its range), for bounded samples.
    """
    c = _CONFIGS[cfg]
    s = c["seed"] if seed is None else seed
    rng = np.random.default_rng(s)
    N = c["N"] if n_E is None else int(n_E)
    chans = _draw_channels(c, rng)
    drawn = [_draw_wave(rng, n, _n_poles(c, n), c["sigma"], *c["poles"]) for n in chans]
    mesh_fn = linear_mesh if c["kind"] == "linear" else geometric_mesh
    mesh = mesh_fn(c["mesh"][0], c["mesh"][1], N)
    wl = Workload(name=f"config{cfg}", seed=s)
    if cfg == 3:
        # one shared mesh, nudged against the union of all waves' poles
        union = np.concatenate([ek for _, ek in drawn])
        shared = nudge_off_poles(mesh, union)
        for W, ek in drawn:
            wl.waves.append(Wave(W, ek, shared, c["a"]))
    else:
        for W, ek in drawn:
            wl.waves.append(Wave(W, ek, nudge_off_poles(mesh, ek), c["a"]))
    return wl


def make_wave(seed: int, n_chan: int, n_poles: int, n_E: int, a: float = 20.0, sigma: float = 0.1,
              poles: tuple[float, float] = (-5.0, 50.0), mesh: tuple[float, float] = (0.1, 10.0)) -> Wave:
    """A free-form wave for edge-shape tests (same recipe as the configs)."""
    rng = np.random.default_rng(seed)
    W, ek = _draw_wave(rng, n_chan, n_poles, sigma, *poles)
    e = nudge_off_poles(linear_mesh(mesh[0], mesh[1], n_E), ek) if n_E > 0 else np.zeros(0)
    return Wave(W, ek, e, float(a))


def sample_energy_indices(wave: Wave, n_random: int = 5, seed: int = 12345) -> np.ndarray:
    """Energies the oracle checks at full size: first, last, the one nearest a
    pole, and ``n_random`` seeded picks (sorted, unique)."""
    n = wave.n_E
    if n == 0:
        return np.zeros(0, dtype=np.int64)
    picks = {0, n - 1, int(np.argmin(min_pole_distance(wave.energies, wave.E_k)))}
    rng = np.random.default_rng(seed)
    picks.update(int(i) for i in rng.integers(0, n, size=n_random))
    return np.array(sorted(picks), dtype=np.int64)
