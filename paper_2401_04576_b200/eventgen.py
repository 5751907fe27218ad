"""Seeded synthetic-input generator: chambers, helix tracks, drift-distance hits, noise.

This module serves BOTH the oracle (`oracle/`) and the CUDA path: it builds the inputs and
nothing else.  It holds none of the method's arithmetic (no interval code, no residual, no
vote); it only knows the geometry needed to *make* hits:

* the wire parametrisation of PAPER.md L147-152, eq. (A.1a,b),
* the helix parametrisation of PAPER.md L41-51, eq. (1a-d),
* "the drift distance is defined as the smallest distance between the wire and the helix"
  (PAPER.md L88), found here by a 1-D safeguarded Newton solve on the closed-form
  point-to-line distance,
* the orientation of the drift line `u_d = w x t` that makes (A.2)/(A.4) hold.

The chambers, track distributions and the parameter box are BASELINE.json `configs[0..4]`
(they stand in for the paper's unpublished COMET-like toy Monte Carlo, L86-88).  Units: cm, rad.

RNG: splitmix64 -> 53-bit uniforms; normals by Box-Muller (cosine branch, two
uniforms per normal).  Draw order per event: R, phi, z0, lambda, then one smear per layer,
then per noise hit (layer, wire, drift).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MASK64 = (1 << 64) - 1

#: parameter box shared by every BASELINE config: xc, yc, R, z0, lambda
BOX_LO = (-450.0, -450.0, 50.0, -10.0, -0.6)
BOX_HI = (450.0, 450.0, 450.0, 10.0, 0.6)
TOL = 0.045          # vote tolerance on the drift distance, cm (+/-450 um)
SMEAR = 0.015        # drift-distance resolution, cm (150 um)
DRIFT_MAX = 1.5      # clip, cm


class SplitMix64:
    """splitmix64 counter generator (public-domain algorithm, Steele/Lea/Flood 2014)."""

    def __init__(self, seed: int):
        self.state = seed & MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        """U[0,1) with 53 random bits."""
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)

    def normal(self) -> float:
        u1 = 1.0 - self.uniform()          # (0,1]
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def randint(self, n: int) -> int:
        return min(int(self.uniform() * n), n - 1)


@dataclass
class Chamber:
    """Full-stereo cylindrical drift chamber, SoA over wires (eq. (A.1a,b))."""
    n_layers: int
    wires_per_layer: int
    x0: np.ndarray          # wire point in the plane z=0
    y0: np.ndarray
    sin_phi_s: np.ndarray   # projection angle phi_s
    cos_phi_s: np.ndarray
    tan_tau: np.ndarray     # signed tan(stereo angle)
    half_len: np.ndarray
    layer: np.ndarray
    radius: np.ndarray      # per layer

    @property
    def n_wires(self) -> int:
        return int(self.x0.shape[0])


def make_chamber(n_layers: int, r0: float, dr: float, wires_per_layer: int, tau0: float,
                 half_len: float = 100.0) -> Chamber:
    """Layer l: radius r0+dr*l, wires at azimuth 2*pi*(j+0.5*[l odd])/n_w, stereo +tau0 (l even) /
    -tau0 (l odd); wire j of layer l has global id l*n_w+j (BASELINE.json configs[0])."""
    lay = np.repeat(np.arange(n_layers), wires_per_layer)
    j = np.tile(np.arange(wires_per_layer), n_layers)
    radius = r0 + dr * np.arange(n_layers, dtype=np.float64)
    alpha = 2.0 * np.pi * (j + 0.5 * (lay % 2)) / wires_per_layer
    r = radius[lay]
    tau = np.where(lay % 2 == 0, tau0, -tau0)
    return Chamber(
        n_layers=n_layers, wires_per_layer=wires_per_layer,
        x0=r * np.cos(alpha), y0=r * np.sin(alpha),
        sin_phi_s=np.sin(alpha), cos_phi_s=np.cos(alpha),
        tan_tau=np.tan(tau), half_len=np.full(lay.shape, half_len),
        layer=lay.astype(np.int32), radius=radius)


def chamber_c0() -> Chamber:      # configs[0]: 8 layers r=20+4l, 64 wires/layer, tau=+/-0.1
    return make_chamber(8, 20.0, 4.0, 64, 0.1)


def chamber_c1() -> Chamber:      # configs[1..3]: 20 layers r=20+2.5l, 128 wires/layer
    return make_chamber(20, 20.0, 2.5, 128, 0.1)


def chamber_c4() -> Chamber:      # configs[4]: 40 layers r=20+1.25l, 256 wires/layer, tau=+/-0.08
    return make_chamber(40, 20.0, 1.25, 256, 0.08)


@dataclass
class Track:
    """Helix of eq. (1a-d): counter-clockwise, R>0, emitted at (xv, yv, z0) with direction phi in the
    transverse plane; the emission point is the reference point (0,0) unless stated (PAPER.md L123 also emits at
    (5 cm, 0) and (0, 5 cm))."""
    R: float
    phi: float
    z0: float
    lam: float
    xv: float = 0.0
    yv: float = 0.0

    @property
    def xc(self) -> float:
        return self.xv - self.R * math.sin(self.phi)

    @property
    def yc(self) -> float:
        return self.yv + self.R * math.cos(self.phi)

    @property
    def params(self):
        """(xc, yc, R, z0, lambda) - the order of the vote's five axes; z0 = z at the emission point."""
        return (self.xc, self.yc, self.R, self.z0, self.lam)

    def z0_at(self, x_ref: float, y_ref: float, unwrap: bool = False) -> float:
        """z where the helix is closest (in the transverse plane) to the reference point (x_ref, y_ref): the z0 of eq. (1)
        for that reference point (phi0 = atan2(x_ref - xc, yc - y_ref), L49), on the turn that contains the emission."""
        phi0 = math.atan2(x_ref - self.xc, self.yc - y_ref)
        if unwrap:
            # turning angles counted from the point of the circle closest to the z axis, in [-0.3, 2 pi - 0.3): the
            # convention of the paper-mode vote for tracks of up to one turn (reading M6)
            phi00 = math.atan2(-self.xc, self.yc)
            th_ref = (phi0 - phi00 + 0.3) % (2.0 * math.pi) - 0.3
            th_v = (self.phi - phi00 + math.pi) % (2.0 * math.pi) - math.pi
            dphi = th_ref - th_v
        else:
            dphi = (phi0 - self.phi + math.pi) % (2.0 * math.pi) - math.pi
        return self.z0 + self.lam * self.R * dphi

    def params_at(self, x_ref: float, y_ref: float, unwrap: bool = False):
        return (self.xc, self.yc, self.R, self.z0_at(x_ref, y_ref, unwrap), self.lam)


def helix_wire_dca(trk: Track, ch: Chamber, wire_ids: np.ndarray, s_init: np.ndarray,
                   window: float = 15.0, iters: int = 60):
    """Closest approach of the helix to each listed wire line near abscissa `s_init`.

    g(s) = |p(s)|^2 with p the component of M(s)-W0 perpendicular to the wire; Newton on
    g'(s)=0 with the step clamped to 5 cm and s kept inside s_init +/- window.
    Returns (signed d_St, s_perp, z on the wire, |g'|/2 stationarity residual, |p|).
    Sign convention: d_St = p . (w x t)/|w x t|, w=(sin phi_s T, -cos phi_s T, 1),
    t=(cos theta, sin theta, lambda), theta = s/R + phi0.
    """
    R, phi0, z0, lam = trk.R, trk.phi, trk.z0, trk.lam
    xc, yc = trk.xc, trk.yc
    T = ch.tan_tau[wire_ids]
    wx, wy, wz = ch.sin_phi_s[wire_ids] * T, -ch.cos_phi_s[wire_ids] * T, np.ones_like(T)
    wn = np.sqrt(wx * wx + wy * wy + wz * wz)
    ux, uy, uz = wx / wn, wy / wn, wz / wn
    X0, Y0 = ch.x0[wire_ids], ch.y0[wire_ids]
    s = np.array(s_init, dtype=np.float64, copy=True)
    s_lo, s_hi = s - window, s + window

    def geom(s):
        th = s / R + phi0
        st, ct = np.sin(th), np.cos(th)
        qx, qy, qz = xc + R * st - X0, yc - R * ct - Y0, z0 + lam * s
        a = qx * ux + qy * uy + qz * uz
        px, py, pz = qx - a * ux, qy - a * uy, qz - a * uz
        return st, ct, a, px, py, pz

    for _ in range(iters):
        st, ct, a, px, py, pz = geom(s)
        tx, ty, tz = ct, st, lam
        g1 = px * tx + py * ty + pz * tz
        tu = tx * ux + ty * uy + tz * uz
        g2 = (tx * tx + ty * ty + tz * tz) - tu * tu + (px * (-st) + py * ct) / R
        step = np.where(g2 > 0, g1 / np.where(g2 > 0, g2, 1.0), np.sign(g1) * 1.0)
        step = np.clip(step, -5.0, 5.0)
        s = np.clip(s - step, s_lo, s_hi)
    st, ct, a, px, py, pz = geom(s)
    tx, ty, tz = ct, st, np.full_like(s, lam)
    g1 = px * tx + py * ty + pz * tz
    # u_d = w x t (unnormalised w; only the direction matters)
    cxv = wy * tz - wz * ty
    cyv = wz * tx - wx * tz
    czv = wx * ty - wy * tx
    cn = np.sqrt(cxv * cxv + cyv * cyv + czv * czv)
    d = (px * cxv + py * cyv + pz * czv) / cn
    z_wire = a * uz
    dist = np.sqrt(px * px + py * py + pz * pz)
    return d, s, z_wire, np.abs(g1), dist


@dataclass
class Event:
    chamber: Chamber
    track: Track
    wire: np.ndarray            # int32 [n_hits] global wire id
    drift: np.ndarray           # float64 [n_hits] measured |d_St| (smeared, clipped), cm
    is_noise: np.ndarray        # bool
    clipped: np.ndarray         # bool: true DCA or smeared value hit the [0,1.5] clip
    d_true: np.ndarray          # signed noise-free d_St (nan for noise hits)
    s_perp: np.ndarray          # transverse abscissa of the closest helix point (nan for noise)
    z_wire: np.ndarray          # z of the closest wire point (nan for noise)
    seed: int = 0

    @property
    def n_hits(self) -> int:
        return int(self.wire.shape[0])


def make_track(rng: SplitMix64) -> Track:
    R = 80.0 + 320.0 * rng.uniform()
    phi = 2.0 * math.pi * rng.uniform()
    z0 = 2.0 * rng.normal()
    lam = -0.5 + rng.uniform()
    return Track(R, phi, z0, lam)


def track_hits(trk: Track, ch: Chamber, n_cand: int = 8):
    """One noise-free hit per layer: the wire of that layer nearest the helix (outgoing branch).

    Candidates: the `n_cand` wires of the layer closest to the helix point at the layer crossing
    (distance evaluated once for every wire); the DCA is then solved for the candidates only."""
    nw = ch.wires_per_layer
    n_cand = min(n_cand, nw)
    all_ids = np.arange(ch.n_wires)
    # layer crossing of a circle through the origin: r = 2R sin(s/2R)
    s_cross = 2.0 * trk.R * np.arcsin(ch.radius / (2.0 * trk.R))
    _, _, _, _, dist0 = helix_wire_dca(trk, ch, all_ids, np.repeat(s_cross, nw), iters=0)
    cand = np.argsort(dist0.reshape(ch.n_layers, nw), axis=1, kind="stable")[:, :n_cand]
    cand_ids = (cand + nw * np.arange(ch.n_layers)[:, None]).reshape(-1)
    d, s, zw, res, dist = helix_wire_dca(trk, ch, cand_ids, np.repeat(s_cross, n_cand))
    wires, ds, ss, zs = [], [], [], []
    for l in range(ch.n_layers):
        sl = slice(l * n_cand, (l + 1) * n_cand)
        k = l * n_cand + int(np.argmin(dist[sl]))
        if not res[k] < 1e-9:
            raise RuntimeError(f"DCA solve did not converge for wire {cand_ids[k]}: residual {res[k]}")
        wires.append(int(cand_ids[k]))
        ds.append(float(d[k]))
        ss.append(float(s[k]))
        zs.append(float(zw[k]))
    return np.array(wires, np.int32), np.array(ds), np.array(ss), np.array(zs)


def make_event(ch: Chamber, seed: int, n_noise: int = 0, smear: float = SMEAR,
               track: Track | None = None) -> Event:
    rng = SplitMix64(seed)
    trk = track if track is not None else make_track(rng)
    wires, d_true, s_perp, z_wire = track_hits(trk, ch)
    drift = np.empty(len(wires))
    clipped = np.zeros(len(wires), bool)
    for i in range(len(wires)):
        raw = abs(d_true[i])
        meas = raw + (smear * rng.normal() if smear > 0 else 0.0)
        clipped[i] = raw > DRIFT_MAX or meas < 0.0 or meas > DRIFT_MAX
        drift[i] = min(max(meas, 0.0), DRIFT_MAX)
    nz_w, nz_d = [], []
    for _ in range(n_noise):
        lay = rng.randint(ch.n_layers)
        j = rng.randint(ch.wires_per_layer)
        nz_w.append(lay * ch.wires_per_layer + j)
        nz_d.append(DRIFT_MAX * rng.uniform())
    nan = np.full(n_noise, np.nan)
    return Event(
        chamber=ch, track=trk,
        wire=np.concatenate([wires, np.array(nz_w, np.int32)]).astype(np.int32),
        drift=np.concatenate([drift, np.array(nz_d, np.float64)]),
        is_noise=np.concatenate([np.zeros(len(wires), bool), np.ones(n_noise, bool)]),
        clipped=np.concatenate([clipped, np.zeros(n_noise, bool)]),
        d_true=np.concatenate([d_true, nan]), s_perp=np.concatenate([s_perp, nan]),
        z_wire=np.concatenate([z_wire, nan]), seed=seed)


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs (seeds per SURVEY G23)
# ---------------------------------------------------------------------------------------------
@dataclass
class Config:
    name: str
    chamber: Chamber
    events: list
    grid: tuple                      # start grid dims (xc, yc, R, z0, lambda)
    levels: int = 1                  # number of vote passes incl. the start grid
    k: int = 0                       # top-K kept (0: no selection)
    box_lo: tuple = BOX_LO
    box_hi: tuple = BOX_HI
    tol: float = TOL
    extra: dict = field(default_factory=dict)

    @property
    def n_cells(self) -> int:
        return int(np.prod(self.grid))


def config(idx: int, n_events: int | None = None) -> Config:
    if idx == 0:
        ch = chamber_c0()
        return Config("C0", ch, [make_event(ch, 0)], (16,) * 5)
    if idx == 1:
        ch = chamber_c1()
        return Config("C1", ch, [make_event(ch, 1, n_noise=20)], (32,) * 5, k=10)
    if idx == 2:
        ch = chamber_c1()
        return Config("C2", ch, [make_event(ch, 2, n_noise=20)], (8,) * 5, levels=10, k=16)
    if idx == 3:
        ch = chamber_c1()
        n = 1024 if n_events is None else n_events
        return Config("C3", ch, [make_event(ch, 1000 + e, n_noise=10) for e in range(n)],
                      (8,) * 5, levels=8, k=8)
    if idx == 4:
        ch = chamber_c4()
        return Config("C4", ch, [make_event(ch, 4, n_noise=20)], (64,) * 5, k=10)
    raise ValueError(f"no config {idx}")


def cell_edges(lo: float, hi: float, n: int) -> np.ndarray:
    """Dense-grid cell edges e_k = lo + k*((hi-lo)/n), e_n = hi, round-to-nearest, unfused
    (SURVEY S9/G14).  Input plumbing shared by both sides: a cell is [e_k, e_{k+1}]."""
    w = (hi - lo) / n
    e = lo + np.arange(n + 1, dtype=np.float64) * w
    e[n] = hi
    return e


def truth_cell(params, lo, hi, dims) -> int:
    """Linear index (row-major, lambda fastest) of the dense cell containing `params`."""
    idx = 0
    for p, a, b, n in zip(params, lo, hi, dims):
        e = cell_edges(a, b, n)
        k = int(np.searchsorted(e, p, side="right") - 1)
        k = min(max(k, 0), n - 1)
        idx = idx * n + k
    return idx


# ---------------------------------------------------------------------------------------------
# Paper-shaped workload.  The paper's COMET-like toy chamber is
# not published; this one has its stated shape: 20 layers between r = 49.6 and 83.7 cm, |tau| = 0.1 rad
# alternating, length 153.6 cm, 250 wires per layer (5,000 against the paper's 4,986), 1 T.
# Electrons of 105 MeV/c from the origin: momentum radius P = p/(0.3 B) = 35 cm, R = P/sqrt(1+lambda^2);
# |lambda| ~ U[0.45, 0.85], random sign (reaches the first three layers, leaves the chamber before one
# turn: L88), phi ~ U[0, 2 pi), z0 = 0.  A hit = every wire whose 3-D distance of closest approach to
# the helix, over the arc inside the chamber, is <= 0.8 cm (L88); drift = that distance (+ optional smear).
# ---------------------------------------------------------------------------------------------
PAPER_P = 35.0                      # cm: 105 MeV/c in 1 T
PAPER_DRIFT_MAX = 0.8               # cm
PAPER_BOX_LO = (-45.0, -45.0, 22.5, -75.0)      # Table 1 (L100-106) in cm: xc, yc, R, z0
PAPER_BOX_HI = (45.0, 45.0, 37.5, 75.0)
PAPER_HALF_LEN = 76.8


def chamber_paper() -> Chamber:
    return make_chamber(20, 49.6, (83.7 - 49.6) / 19.0, 250, 0.1, half_len=PAPER_HALF_LEN)


def make_track_paper(rng: SplitMix64, vertex=(0.0, 0.0)) -> Track:
    lam = 0.45 + 0.40 * rng.uniform()
    if rng.uniform() < 0.5:
        lam = -lam
    phi = 2.0 * math.pi * rng.uniform()
    R = PAPER_P / math.sqrt(1.0 + lam * lam)
    return Track(R, phi, 0.0, lam, float(vertex[0]), float(vertex[1]))


def track_hits_all_wires(trk: Track, ch: Chamber, d_max: float = PAPER_DRIFT_MAX, ds: float = 0.25):
    """Every wire whose distance of closest approach to the helix, over the arc from the origin to the end
    plate (or one full turn), is <= d_max.  Coarse scan of the arc in steps of `ds`, then the exact
    stationarity solve of helix_wire_dca around the best sample of each candidate wire; a wire approached
    on both the outgoing and the returning arc keeps the smaller distance (the first drift electrons)."""
    half = float(ch.half_len[0])
    s_end = 2.0 * math.pi * trk.R
    if abs(trk.lam) > 0:
        s_end = min(s_end, (half - math.copysign(trk.z0, trk.lam)) / abs(trk.lam))
    s = np.arange(0.0, s_end + ds, ds)
    th = s / trk.R + trk.phi
    hx, hy, hz = trk.xc + trk.R * np.sin(th), trk.yc - trk.R * np.cos(th), trk.z0 + trk.lam * s
    T = ch.tan_tau
    wx, wy = ch.sin_phi_s * T, -ch.cos_phi_s * T
    wn = np.sqrt(wx * wx + wy * wy + 1.0)
    ux, uy, uz = wx / wn, wy / wn, 1.0 / wn
    best_d = np.full(ch.n_wires, np.inf)
    best_s = np.zeros(ch.n_wires)
    for i0 in range(0, len(s), 128):                      # chunks keep the temporary at n_wires x 128
        sl = slice(i0, i0 + 128)
        qx = hx[None, sl] - ch.x0[:, None]
        qy = hy[None, sl] - ch.y0[:, None]
        qz = np.broadcast_to(hz[None, sl], qx.shape)
        a = qx * ux[:, None] + qy * uy[:, None] + qz * uz[:, None]
        d2 = qx * qx + qy * qy + qz * qz - a * a
        k = np.argmin(d2, axis=1)
        dmin = np.sqrt(np.maximum(d2[np.arange(ch.n_wires), k], 0.0))
        upd = dmin < best_d
        best_d[upd] = dmin[upd]
        best_s[upd] = s[i0 + k[upd]]
    cand = np.nonzero(best_d < d_max + 2.0 * ds)[0]
    if len(cand) == 0:
        return (np.zeros(0, np.int32),) + (np.zeros(0),) * 3
    d, sp, zw, res, dist = helix_wire_dca(trk, ch, cand, best_s[cand], window=2.0 * ds + 1.0)
    ok = (dist <= d_max) & (res < 1e-9) & (np.abs(zw) <= half) & (sp >= 0.0) & (sp <= s_end)
    order = np.argsort(sp[ok], kind="stable")
    return cand[ok][order].astype(np.int32), d[ok][order], sp[ok][order], zw[ok][order]


def make_event_paper(ch: Chamber, seed: int, n_noise: int = 0, smear: float = 0.0, track: Track | None = None,
                     vertex=(0.0, 0.0)) -> Event:
    """Paper-shaped event: the paper simulates no measurement error (L88: smear = 0 by default) and no noise.
    vertex: emission point in the transverse plane (L123: the origin, (5, 0) cm, (0, 5) cm)."""
    rng = SplitMix64(seed)
    trk = track if track is not None else make_track_paper(rng, vertex)
    wires, d_true, s_perp, z_wire = track_hits_all_wires(trk, ch)
    drift = np.empty(len(wires))
    clipped = np.zeros(len(wires), bool)
    for i in range(len(wires)):
        meas = abs(d_true[i]) + (smear * rng.normal() if smear > 0 else 0.0)
        clipped[i] = meas < 0.0
        drift[i] = max(meas, 0.0)
    nz_w, nz_d = [], []
    for _ in range(n_noise):
        lay = rng.randint(ch.n_layers)
        j = rng.randint(ch.wires_per_layer)
        nz_w.append(lay * ch.wires_per_layer + j)
        nz_d.append(PAPER_DRIFT_MAX * rng.uniform())
    nan = np.full(n_noise, np.nan)
    return Event(
        chamber=ch, track=trk,
        wire=np.concatenate([wires, np.array(nz_w, np.int32)]).astype(np.int32),
        drift=np.concatenate([drift, np.array(nz_d, np.float64)]),
        is_noise=np.concatenate([np.zeros(len(wires), bool), np.ones(n_noise, bool)]),
        clipped=np.concatenate([clipped, np.zeros(n_noise, bool)]),
        d_true=np.concatenate([d_true, nan]), s_perp=np.concatenate([s_perp, nan]),
        z_wire=np.concatenate([z_wire, nan]), seed=seed)
