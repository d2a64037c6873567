"""Seeded synthetic calibration intervals (stations, uvw, sky model, Jones, noise).

Recipe: SURVEY.md §8(d) "Synthetic inputs", shapes from BASELINE.json:7-11
(configs[0..4]); readings Q3, Q6, Q19-Q22 of SURVEY.md §8(c).  The paper's
own artificial datasets are not available; these arrays
stand in for them.

Nothing here evaluates the method: visibilities are NOT produced in this
module.  Each side (oracle, CUDA) builds V = sum_k J C J^H + noise with its
own arithmetic from the arrays returned here.

Every random component has its own child stream of
SeedSequence([seed, component]) so that e.g. the (large) noise array can be
skipped or regenerated without disturbing the other draws.
"""
from __future__ import annotations

import dataclasses
import hashlib
from typing import Optional

import numpy as np

C0 = 299792458.0  # m/s
SEED_BASE = 191013908  # arXiv number 1910.13908; seed = SEED_BASE + config index
OMEGA_E = 7.2921150e-5  # rad/s, earth rotation
LATITUDE_DEG = 52.9  # Q22
DECLINATION_DEG = 52.0  # BASELINE.json:7
DT_S = 10.0  # s per time slot, BASELINE.json:7-8

_STREAM_STATIONS, _STREAM_SOURCES, _STREAM_JONES, _STREAM_NOISE, _STREAM_POL = range(5)


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(np.random.SeedSequence([int(seed), int(stream)])))


def baseline_pairs(nstations: int):
    """(p, q) station indices, p < q, row-major over the upper triangle
    (canonical order of SURVEY.md §8(b)): b(p,q) = p*N - p(p+1)/2 + (q-p-1)."""
    p, q = np.triu_indices(nstations, 1)
    return p.astype(np.int32), q.astype(np.int32)


def baseline_index(nstations: int, p: int, q: int) -> int:
    assert 0 <= p < q < nstations
    return p * nstations - p * (p + 1) // 2 + (q - p - 1)


@dataclasses.dataclass
class Problem:
    """One calibration interval's inputs.  Plain numpy arrays, C-contiguous."""

    name: str
    seed: int
    N: int  # stations
    T: int  # time slots
    F: int  # channels
    K: int  # clusters
    freqs: np.ndarray  # [F] Hz
    f0: float  # Hz
    stations_en: np.ndarray  # [N, 2] east, north (m)
    uvw: np.ndarray  # [T*B, 3] metres, row r = t*B + b
    cluster_offset: np.ndarray  # [K+1] int32
    src_l: np.ndarray  # [S_tot]
    src_m: np.ndarray
    src_I: np.ndarray  # Jy at f0
    src_Q: Optional[np.ndarray]  # None = unpolarised
    src_U: Optional[np.ndarray]
    src_V: Optional[np.ndarray]
    src_alpha: np.ndarray
    jones_true: np.ndarray  # [K, N, 2, 2] complex128
    sigma: float  # Jy, per real and per imaginary part (Q19)
    n_em: int = 3
    n_lm: int = 10
    tau: float = 1e-3

    @property
    def B(self) -> int:
        return self.N * (self.N - 1) // 2

    @property
    def rows(self) -> int:
        return self.T * self.B

    @property
    def samples(self) -> int:
        return self.rows * self.F

    @property
    def S_tot(self) -> int:
        return int(self.cluster_offset[-1])

    @property
    def vis_src(self) -> int:
        """vis*src work units of the predict step (SURVEY.md §8 size table)."""
        return self.samples * self.S_tot

    @property
    def polarised(self) -> bool:
        return self.src_Q is not None

    def jones_init(self) -> np.ndarray:
        """Start values: identity for every station and cluster (Q8)."""
        j = np.zeros((self.K, self.N, 2, 2), dtype=np.complex128)
        j[..., 0, 0] = 1.0
        j[..., 1, 1] = 1.0
        return j

    def noise(self, out: Optional[np.ndarray] = None) -> np.ndarray:
        """[T*B, F, 4] complex128 Gaussian noise, sigma per real/imag part.

        Drawn one time slot at a time from the slot's own stream, so a slot can
        be regenerated alone (noise_rows) and memory stays bounded."""
        if out is None:
            out = np.empty((self.rows, self.F, 4), dtype=np.complex128)
        view = out.view(np.float64).reshape(self.T, self.B * self.F * 8)
        for t in range(self.T):
            view[t] = _noise_slot(self.seed, t, self.B * self.F * 8, self.sigma)
        return out

    def sha256(self) -> dict:
        """Digest of every generated array (logged by the harness)."""
        out = {}
        for f in dataclasses.fields(self):
            v = getattr(self, f.name)
            if isinstance(v, np.ndarray):
                out[f.name] = hashlib.sha256(np.ascontiguousarray(v).tobytes()).hexdigest()[:16]
        return out


def _noise_slot(seed: int, t: int, n: int, sigma: float) -> np.ndarray:
    g = np.random.Generator(np.random.Philox(np.random.SeedSequence([int(seed), _STREAM_NOISE, int(t)])))
    x = g.standard_normal(n)
    x *= sigma
    return x


def noise_rows(prob: Problem, rows: np.ndarray) -> np.ndarray:
    """Noise for a subset of rows, identical to prob.noise()[rows]."""
    rows = np.asarray(rows, dtype=np.int64)
    out = np.empty((rows.size, prob.F, 4), dtype=np.complex128)
    ts = rows // prob.B
    for t in np.unique(ts):
        slot = _noise_slot(prob.seed, int(t), prob.B * prob.F * 8, prob.sigma)
        slot = slot.view(np.complex128).reshape(prob.B, prob.F, 4)
        sel = np.nonzero(ts == t)[0]
        out[sel] = slot[rows[sel] - int(t) * prob.B]
    return out


# ----------------------------------------------------------------------------
# geometry (input generation only)
# ----------------------------------------------------------------------------
def _uvw_tracks(east: np.ndarray, north: np.ndarray, T: int) -> np.ndarray:
    """Earth-rotation synthesis, SURVEY.md §8(d).2.  Returns [T*B, 3] metres for
    baseline vector position(p) - position(q) (Q3)."""
    lat = np.deg2rad(LATITUDE_DEG)
    dec = np.deg2rad(DECLINATION_DEG)
    X = -np.sin(lat) * north
    Y = east
    Z = np.cos(lat) * north
    p, q = baseline_pairs(east.size)
    Lx, Ly, Lz = X[p] - X[q], Y[p] - Y[q], Z[p] - Z[q]
    H = OMEGA_E * DT_S * (np.arange(T) + 0.5 - T / 2.0)
    sH, cH = np.sin(H)[:, None], np.cos(H)[:, None]
    u = sH * Lx + cH * Ly
    v = -np.sin(dec) * cH * Lx + np.sin(dec) * sH * Ly + np.cos(dec) * Lz
    w = np.cos(dec) * cH * Lx - np.cos(dec) * sH * Ly + np.sin(dec) * Lz
    return np.ascontiguousarray(np.stack([u, v, w], axis=-1).reshape(-1, 3))


def _disc(rng, n, radius):
    r = radius * np.sqrt(rng.random(n))
    a = 2 * np.pi * rng.random(n)
    return r * np.cos(a), r * np.sin(a)


def _stations(layout: str, N: int, rng) -> np.ndarray:
    if layout.startswith("disc:"):
        e, n = _disc(rng, N, float(layout.split(":")[1]))
    elif layout == "core+halo":  # cfg3: 50% within 1 km, rest log-uniform to 20 km
        nc = N // 2
        e1, n1 = _disc(rng, nc, 1000.0)
        r = np.exp(rng.uniform(np.log(1000.0), np.log(20000.0), N - nc))
        a = 2 * np.pi * rng.random(N - nc)
        e, n = np.concatenate([e1, r * np.cos(a)]), np.concatenate([n1, r * np.sin(a)])
    elif layout == "core+spiral":  # cfg4: SKA1-LOW-like, 65 km
        nc = N // 2
        e1, n1 = _disc(rng, nc, 500.0)
        no = N - nc
        r = np.exp(rng.uniform(np.log(500.0), np.log(32500.0), no))
        arm = np.arange(no) % 3
        az = 2 * np.pi * arm / 3.0 + 1.2 * np.log(r / 500.0)
        jit = rng.standard_normal((2, no)) * 0.05 * r
        e = np.concatenate([e1, r * np.cos(az) + jit[0]])
        n = np.concatenate([n1, r * np.sin(az) + jit[1]])
    else:
        raise ValueError(layout)
    return np.ascontiguousarray(np.stack([e, n], axis=-1))


def _power_law_flux(rng, n, lo=0.1, hi=50.0, slope=1.6):
    """Inverse CDF of dN/dS ~ S^-slope on [lo, hi]."""
    g = 1.0 - slope
    return (lo**g + rng.random(n) * (hi**g - lo**g)) ** (1.0 / g)


def _sources(K, S, field_deg, patch_deg, flux_law, rng):
    """K clusters x S sources.  patch_deg None: one cluster filling the field."""
    l, m = [], []
    for _ in range(K):
        if patch_deg is None:
            lc = mc = 0.0
            rad = np.sin(np.deg2rad(field_deg))
        else:
            rho = np.sin(np.deg2rad(field_deg)) * np.sqrt(rng.random())
            psi = 2 * np.pi * rng.random()
            lc, mc = rho * np.cos(psi), rho * np.sin(psi)
            rad = np.sin(np.deg2rad(patch_deg))
        dl, dm = _disc(rng, S, rad)
        l.append(lc + dl)
        m.append(mc + dm)
    l, m = np.concatenate(l), np.concatenate(m)
    if flux_law == "uniform":
        flux = rng.uniform(1.0, 10.0, K * S)
    else:
        flux = _power_law_flux(rng, K * S)
    return l, m, flux


def _channel_centres(F: int, lo=140e6, hi=160e6) -> np.ndarray:
    if F == 1:
        return np.array([150e6])
    return lo + (np.arange(F) + 0.5) * (hi - lo) / F  # Q6


def make_problem(
    N: int,
    T: int,
    F: int,
    K: int,
    S: int,
    *,
    seed: int,
    layout: str = "disc:1000",
    field_deg: float = 2.0,
    patch_deg: Optional[float] = None,
    flux_law: str = "uniform",
    sigma: float = 0.01,
    jones_std: float = 0.1,
    polarised: bool = False,
    alpha: float = -0.7,
    freqs: Optional[np.ndarray] = None,
    n_em: int = 3,
    n_lm: int = 10,
    name: str = "custom",
) -> Problem:
    st = _stations(layout, N, _rng(seed, _STREAM_STATIONS))
    uvw = _uvw_tracks(st[:, 0], st[:, 1], T)
    l, m, flux = _sources(K, S, field_deg, patch_deg, flux_law, _rng(seed, _STREAM_SOURCES))
    rj = _rng(seed, _STREAM_JONES)
    z = (rj.standard_normal((K, N, 2, 2)) + 1j * rj.standard_normal((K, N, 2, 2))) / np.sqrt(2.0)  # Q20
    jones = np.eye(2, dtype=np.complex128) + jones_std * z
    q = u = v = None
    if polarised:  # not used by the configs; exercises the general 2x2 brightness
        rp = _rng(seed, _STREAM_POL)
        q, u, v = (flux * rp.uniform(-0.3, 0.3, flux.size) for _ in range(3))
    fr = _channel_centres(F) if freqs is None else np.asarray(freqs, dtype=np.float64)
    assert fr.size == F
    return Problem(
        name=name, seed=seed, N=N, T=T, F=F, K=K,
        freqs=np.ascontiguousarray(fr, dtype=np.float64), f0=150e6,
        stations_en=st, uvw=uvw,
        cluster_offset=(np.arange(K + 1) * S).astype(np.int32),
        src_l=np.ascontiguousarray(l), src_m=np.ascontiguousarray(m),
        src_I=np.ascontiguousarray(flux),
        src_Q=None if q is None else np.ascontiguousarray(q),
        src_U=None if u is None else np.ascontiguousarray(u),
        src_V=None if v is None else np.ascontiguousarray(v),
        src_alpha=np.full(K * S, alpha),
        jones_true=np.ascontiguousarray(jones), sigma=float(sigma),
        n_em=n_em, n_lm=n_lm,
    )


# BASELINE.json:7-11, made concrete per SURVEY.md §8(d)
CONFIGS = {
    0: dict(N=8, T=10, F=1, K=1, S=3, layout="disc:1000", field_deg=2.0, patch_deg=None,
            flux_law="uniform", sigma=0.01),
    1: dict(N=64, T=20, F=1, K=1, S=20, layout="disc:15000", field_deg=3.0, patch_deg=None,
            flux_law="power", sigma=0.1),
    2: dict(N=64, T=20, F=4, K=50, S=20, layout="disc:15000", field_deg=5.0, patch_deg=0.5,
            flux_law="power", sigma=0.1),
    3: dict(N=256, T=20, F=4, K=50, S=20, layout="core+halo", field_deg=5.0, patch_deg=0.5,
            flux_law="power", sigma=0.1),
    4: dict(N=512, T=20, F=8, K=50, S=40, layout="core+spiral", field_deg=5.0, patch_deg=0.5,
            flux_law="power", sigma=0.1),
}


def make_config(index: int, **overrides) -> Problem:
    """configs[index] of BASELINE.json, seed = SEED_BASE + index.

    overrides (e.g. N=, K=, sigma=) derive the paper's scaling-grid variants
    (64..512 stations x 1..50 clusters) from a config."""
    kw = dict(CONFIGS[index])
    kw.update(overrides)
    seed = kw.pop("seed", SEED_BASE + index)
    return make_problem(seed=seed, name=f"cfg{index}", n_em=3, n_lm=10, **kw)


# ----------------------------------------------------------------------------
# measurement-set style row lists (second part)
# ----------------------------------------------------------------------------
@dataclasses.dataclass
class RowList:
    """The rows of one interval as a measurement set would hand them over: arbitrary order, either station
    orientation, some (time slot, baseline) pairs absent, per-sample flags.  Index and flag arrays only -- the
    visibilities of these rows are formed by whoever consumes them."""

    ant1: np.ndarray  # [n] int32
    ant2: np.ndarray  # [n] int32 (ant1 != ant2, either order)
    tslot: np.ndarray  # [n] int32 in [0, T)
    uvw: np.ndarray  # [n, 3] metres for the baseline as ordered (ant1, ant2)
    flags: np.ndarray  # [n, F] uint8, non-zero = sample excluded
    canonical_row: np.ndarray  # [n] int64: t*B + b(min, max) -- bookkeeping for tests
    noise: np.ndarray  # [n, F, 4] complex128, sigma per real/imag part


def make_rowlist(prob: Problem, *, seed: int, drop_frac: float = 0.1, swap_frac: float = 0.3,
                 flag_frac: float = 0.05, shuffle: bool = True) -> RowList:
    """Derive a row list from a Problem: drop `drop_frac` of the canonical rows, list the rest in random order,
    give `swap_frac` of them as (q, p) with uvw negated, flag `flag_frac` of the samples."""
    g = _rng(seed, 17)
    rows = np.arange(prob.rows, dtype=np.int64)
    keep = g.random(prob.rows) >= drop_frac
    rows = rows[keep]
    if shuffle:
        rows = g.permutation(rows)
    p, q = baseline_pairs(prob.N)
    b = rows % prob.B
    swap = g.random(rows.size) < swap_frac
    a1 = np.where(swap, q[b], p[b]).astype(np.int32)
    a2 = np.where(swap, p[b], q[b]).astype(np.int32)
    uvw = prob.uvw[rows] * np.where(swap, -1.0, 1.0)[:, None]
    flags = (g.random((rows.size, prob.F)) < flag_frac).astype(np.uint8)
    noise = (g.standard_normal((rows.size, prob.F, 4)) + 1j * g.standard_normal((rows.size, prob.F, 4))) * prob.sigma
    return RowList(ant1=a1, ant2=a2, tslot=(rows // prob.B).astype(np.int32), uvw=np.ascontiguousarray(uvw),
                   flags=np.ascontiguousarray(flags), canonical_row=rows, noise=noise)
