"""Seeded synthetic events and grid definitions for the five BASELINE.json workloads.

This module only *generates inputs* (toy-detector hits) and names the grids.  It holds
none of the Hough method's arithmetic (no kappa closed form, no binning, no peak rule),
so that both the CPU oracle (``oracle/``) and the CUDA path can be fed from it without
sharing any code of the method (SURVEY.md §8(c), §8(d) "Synthetic inputs").

Recipe (BASELINE.json ``configs``; readings B10-B13 of SURVEY.md §8(c)):

* 10 barrel layers at r = 4.4 ... 78.0 cm, B = 3.8 T, transverse plane only
  (the paper's toy detector is also transverse-only, §8).
* track: 1/pT ~ U[a, b] GeV^-1, kappa = 0.003*B/pT cm^-1 with a random sign,
  phi0 ~ U[-pi, pi); displaced tracks add d0 ~ U[-10, 10] cm and only leave hits on
  layers with r > |d0| + 2 cm.
* hit on a layer of radius r: s = (kappa*(r^2 + d0^2) + 2*d0) / (2*(1 + kappa*d0))
  (= kappa*r^2/2 for d0 = 0), phi = phi0 + asin(s/r), smeared by N(0, 20 um)/r;
  x = r*cos(phi), y = r*sin(phi) in fp64, stored as fp32.
* noise hits: uniform layer, uniform phi.
* draw order: tracks (1/pT, sign, phi0, [d0]) prompt first then displaced; smear per
  hit in ascending layer order; then noise; then one seeded permutation of all hits.
"""
from __future__ import annotations

import dataclasses
import hashlib
import math

import numpy as np

LAYER_RADII_CM = (4.4, 7.3, 10.2, 25.5, 34.0, 42.0, 50.0, 60.8, 69.2, 78.0)
B_TESLA = 3.8
SIGMA_RPHI_CM = 0.002  # 20 um
KAPPA_PER_INV_PT = 0.003 * B_TESLA  # cm^-1 per GeV^-1


@dataclasses.dataclass(frozen=True)
class Grid:
    """Accumulator grid: ranges, bin counts, L_min (BASELINE.json configs)."""

    n_phi: int
    n_d0: int
    n_kappa: int
    L_min: int
    phi_min: float = -math.pi
    phi_max: float = math.pi
    d0_min: float = -10.0
    d0_max: float = 10.0
    kappa_min: float = -0.012
    kappa_max: float = 0.012
    phi_wrap: int = 1
    layer_radii: tuple = LAYER_RADII_CM

    @property
    def n_layers(self) -> int:
        return len(self.layer_radii)

    @property
    def n_bins(self) -> int:
        return self.n_phi * self.n_d0 * self.n_kappa


@dataclasses.dataclass(frozen=True)
class EventSpec:
    n_prompt: int
    n_displaced: int
    n_noise: int
    inv_pt_lo: float
    inv_pt_hi: float


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    grid: Grid
    event: EventSpec
    seeds: tuple
    cap_peaks: int
    cap_hits: int


def _grid2d(L_min):
    return Grid(n_phi=256, n_d0=1, n_kappa=128, L_min=L_min, d0_min=0.0, d0_max=0.0)


WORKLOADS = {
    # BASELINE.json configs[0]
    "prompt2d": Workload("prompt2d", _grid2d(8), EventSpec(20, 0, 50, 1 / 20, 1 / 2), (0,),
                         1 << 12, 1 << 16),
    # configs[1]
    "displaced3d": Workload("displaced3d", Grid(1024, 64, 256, 6),
                            EventSpec(100, 10, 500, 1 / 20, 1 / 2), (0,), 1 << 16, 1 << 20),
    # configs[2]
    "pileup": Workload("pileup", Grid(1024, 64, 256, 7),
                       EventSpec(1000, 50, 5000, 1 / 50, 1 / 1), (0,), 1 << 20, 1 << 24),
    # configs[3]: 100 events shaped like "pileup", seeds 0..99
    "batch100": Workload("batch100", Grid(1024, 64, 256, 7),
                         EventSpec(1000, 50, 5000, 1 / 50, 1 / 1), tuple(range(100)),
                         1 << 20, 1 << 24),
    # configs[4] (pT range: reading B10 = same as "pileup")
    "finegrid": Workload("finegrid", Grid(2048, 128, 512, 7),
                         EventSpec(4000, 200, 20000, 1 / 50, 1 / 1), (0,), 1 << 23, 1 << 27),
}


def _track_hits(rng, radii, kappa, phi0, d0, displaced):
    """Noise-free azimuths of one track on the layers it crosses, then smear."""
    out_layer, out_phi, out_r = [], [], []
    for layer, r in enumerate(radii):
        if displaced and not (r > abs(d0) + 2.0):
            continue
        s = (kappa * (r * r + d0 * d0) + 2.0 * d0) / (2.0 * (1.0 + kappa * d0))
        if abs(s) > r:
            continue  # the circle does not reach this layer
        phi = phi0 + math.asin(s / r)
        phi += rng.normal(0.0, SIGMA_RPHI_CM) / r
        out_layer.append(layer)
        out_phi.append(phi)
        out_r.append(r)
    return out_layer, out_phi, out_r


def generate_event(spec: EventSpec, seed: int, radii=LAYER_RADII_CM):
    """Return (x fp32[n], y fp32[n], layer int32[n], truth dict) for one event."""
    rng = np.random.default_rng(seed)
    layers, phis, rs = [], [], []
    truth = []
    for t in range(spec.n_prompt + spec.n_displaced):
        displaced = t >= spec.n_prompt
        inv_pt = rng.uniform(spec.inv_pt_lo, spec.inv_pt_hi)
        sign = 1.0 if rng.random() < 0.5 else -1.0
        phi0 = rng.uniform(-math.pi, math.pi)
        d0 = rng.uniform(-10.0, 10.0) if displaced else 0.0
        kappa = sign * KAPPA_PER_INV_PT * inv_pt
        la, ph, rr = _track_hits(rng, radii, kappa, phi0, d0, displaced)
        layers += la
        phis += ph
        rs += rr
        truth.append((phi0, d0, kappa, len(la)))
    if spec.n_noise:
        nl = rng.integers(0, len(radii), size=spec.n_noise)
        nphi = rng.uniform(-math.pi, math.pi, size=spec.n_noise)
        layers += [int(v) for v in nl]
        phis += [float(v) for v in nphi]
        rs += [radii[int(v)] for v in nl]
    layer = np.asarray(layers, dtype=np.int32)
    phi = np.asarray(phis, dtype=np.float64)
    r = np.asarray(rs, dtype=np.float64)
    perm = rng.permutation(layer.shape[0])
    layer, phi, r = layer[perm], phi[perm], r[perm]
    x = (r * np.cos(phi)).astype(np.float32)
    y = (r * np.sin(phi)).astype(np.float32)
    return x, y, layer, {"tracks": truth}


def single_track_event(grid: Grid, i: int, j: int, kappa: float):
    """Noise-free, unsmeared hits of ONE track whose (phi0, d0) are the centres of
    bins (i, j) -- the generator side of the SURVEY.md §8(c) C "single track" pin (B9)."""
    phi0 = grid.phi_min + (i + 0.5) * (grid.phi_max - grid.phi_min) / grid.n_phi
    d0 = grid.d0_min + (j + 0.5) * (grid.d0_max - grid.d0_min) / grid.n_d0
    xs, ys, ls = [], [], []
    for layer, r in enumerate(grid.layer_radii):
        s = (kappa * (r * r + d0 * d0) + 2.0 * d0) / (2.0 * (1.0 + kappa * d0))
        if abs(s) > r:
            continue
        phi = phi0 + math.asin(s / r)
        xs.append(r * math.cos(phi))
        ys.append(r * math.sin(phi))
        ls.append(layer)
    return (np.asarray(xs, dtype=np.float32), np.asarray(ys, dtype=np.float32),
            np.asarray(ls, dtype=np.int32))


def event_sha256(x, y, layer) -> str:
    h = hashlib.sha256()
    for a in (x, y, layer):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


# ---------------------------------------------------------------------------------------
# Inputs for the rows SURVEY.md 8(f) marks "next".  Geometry of the
# generated tracks only, as above: nothing here bins, votes, finds peaks or fits.

@dataclasses.dataclass(frozen=True)
class VertexGrid:
    """(x_v, y_v) accumulator of the second transform (section 9), V_min = its peak threshold."""

    n_x: int
    n_y: int
    V_min: int
    x_min: float = -8.0
    x_max: float = 8.0
    y_min: float = -8.0
    y_max: float = 8.0


def track_from_vertex(xv: float, yv: float, psi: float, kappa: float):
    """(phi0, d0) of the circle of curvature kappa that passes through (xv, yv) with direction
    psi there (conventions of SURVEY.md section 8: n = (-sin phi0, cos phi0), centre
    C = (d0 + 1/kappa) n); kappa = 0 is the straight line."""
    if kappa == 0.0:
        return psi, -xv * math.sin(psi) + yv * math.cos(psi)
    cx = xv - math.sin(psi) / kappa
    cy = yv + math.cos(psi) / kappa
    rho = math.hypot(cx, cy)
    sgn = 1.0 if kappa > 0 else -1.0  # d0 + 1/kappa has the sign of kappa while |d0| < 1/|kappa|
    nx, ny = sgn * cx / rho, sgn * cy / rho
    return math.atan2(-nx, ny), sgn * rho - 1.0 / kappa


@dataclasses.dataclass(frozen=True)
class JetSpec:
    """Displaced jets (PAPER.md:154 Fig. 7, :168 Fig. 8): n_jets vertices at radius U[r_lo, r_hi] and
    uniform azimuth, each with tracks_per_jet tracks whose direction at the vertex is the
    vertex's azimuth + U[-cone, cone]; plus prompt tracks and noise as in EventSpec."""

    n_jets: int
    tracks_per_jet: int
    n_prompt: int
    n_noise: int
    inv_pt_lo: float = 1 / 20
    inv_pt_hi: float = 1 / 2
    r_lo: float = 1.0
    r_hi: float = 6.0
    cone: float = 0.5


def generate_jet_event(spec: JetSpec, seed: int, radii=LAYER_RADII_CM):
    """(x, y, layer, truth) with truth["vertices"] = [(xv, yv)], truth["tracks"] as generate_event."""
    rng = np.random.default_rng(seed)
    layers, phis, rs, truth, vertices = [], [], [], [], []

    def add_track(kappa, phi0, d0, r_from):
        n0 = len(layers)
        for layer, r in enumerate(radii):
            if not (r > r_from):
                continue
            s = (kappa * (r * r + d0 * d0) + 2.0 * d0) / (2.0 * (1.0 + kappa * d0))
            if abs(s) > r:
                continue
            layers.append(layer)
            phis.append(phi0 + math.asin(s / r) + rng.normal(0.0, SIGMA_RPHI_CM) / r)
            rs.append(r)
        truth.append((phi0, d0, kappa, len(layers) - n0))

    for _ in range(spec.n_jets):
        rv = rng.uniform(spec.r_lo, spec.r_hi)
        av = rng.uniform(-math.pi, math.pi)
        xv, yv = rv * math.cos(av), rv * math.sin(av)
        vertices.append((xv, yv))
        for _ in range(spec.tracks_per_jet):
            inv_pt = rng.uniform(spec.inv_pt_lo, spec.inv_pt_hi)
            sign = 1.0 if rng.random() < 0.5 else -1.0
            psi = av + rng.uniform(-spec.cone, spec.cone)
            kappa = sign * KAPPA_PER_INV_PT * inv_pt
            phi0, d0 = track_from_vertex(xv, yv, psi, kappa)
            add_track(kappa, phi0, d0, rv + 1.0)
    for _ in range(spec.n_prompt):
        inv_pt = rng.uniform(spec.inv_pt_lo, spec.inv_pt_hi)
        sign = 1.0 if rng.random() < 0.5 else -1.0
        phi0 = rng.uniform(-math.pi, math.pi)
        add_track(sign * KAPPA_PER_INV_PT * inv_pt, phi0, 0.0, 0.0)
    if spec.n_noise:
        nl = rng.integers(0, len(radii), size=spec.n_noise)
        nphi = rng.uniform(-math.pi, math.pi, size=spec.n_noise)
        layers += [int(v) for v in nl]
        phis += [float(v) for v in nphi]
        rs += [radii[int(v)] for v in nl]
    layer = np.asarray(layers, dtype=np.int32)
    phi = np.asarray(phis, dtype=np.float64)
    r = np.asarray(rs, dtype=np.float64)
    perm = rng.permutation(layer.shape[0])
    layer, phi, r = layer[perm], phi[perm], r[perm]
    x = (r * np.cos(phi)).astype(np.float32)
    y = (r * np.sin(phi)).astype(np.float32)
    return x, y, layer, {"tracks": truth, "vertices": vertices}


# The paper's own toy detector: beampipe of radius 3.0 cm, ten concentric evenly
# spaced layers, the last at 110.0 cm (reading X1: spacing (110 - 3)/10 from the beampipe), hit
# resolution 0.4 mm in each direction; Fig. 3: straight-line tracks with 10 hits each.
TOY_LAYER_RADII_CM = tuple(3.0 + (110.0 - 3.0) * (l + 1) / 10.0 for l in range(10))
TOY_SIGMA_CM = 0.04


@dataclasses.dataclass(frozen=True)
class LineSpec:
    n_tracks: int
    n_noise: int
    rho_max: float = 3.0  # lines start inside the beampipe


def generate_line_event(spec: LineSpec, seed: int, radii=TOY_LAYER_RADII_CM):
    """Straight tracks of direction theta ~ U[-pi, pi) and signed offset rho ~ U[-rho_max, rho_max]
    from the origin; one hit where the outward half-line meets each layer, each coordinate smeared
    by N(0, 0.4 mm); uniform noise; a seeded permutation.  truth["tracks"] = [(theta, rho)]."""
    rng = np.random.default_rng(seed)
    xs, ys, ls, truth = [], [], [], []
    for _ in range(spec.n_tracks):
        theta = rng.uniform(-math.pi, math.pi)
        rho = rng.uniform(-spec.rho_max, spec.rho_max)
        truth.append((theta, rho))
        for layer, r in enumerate(radii):
            t = math.sqrt(r * r - rho * rho)
            xs.append(-rho * math.sin(theta) + t * math.cos(theta) + rng.normal(0.0, TOY_SIGMA_CM))
            ys.append(rho * math.cos(theta) + t * math.sin(theta) + rng.normal(0.0, TOY_SIGMA_CM))
            ls.append(layer)
    if spec.n_noise:
        nl = rng.integers(0, len(radii), size=spec.n_noise)
        nphi = rng.uniform(-math.pi, math.pi, size=spec.n_noise)
        for l, a in zip(nl, nphi):
            xs.append(radii[int(l)] * math.cos(a))
            ys.append(radii[int(l)] * math.sin(a))
            ls.append(int(l))
    perm = rng.permutation(len(ls))
    x = np.asarray(xs, dtype=np.float64)[perm].astype(np.float32)
    y = np.asarray(ys, dtype=np.float64)[perm].astype(np.float32)
    layer = np.asarray(ls, dtype=np.int32)[perm]
    return x, y, layer, {"tracks": truth}


# grids of the extension workloads (kappa axis of a line grid = rho in cm)
JETS_GRID = Grid(1024, 64, 256, 6)
JETS_VGRID = VertexGrid(32, 32, 8)
JETS_SPEC = JetSpec(n_jets=3, tracks_per_jet=12, n_prompt=40, n_noise=400)
TOY_LINE_GRID = Grid(n_phi=2048, n_d0=1, n_kappa=256, L_min=8, d0_min=0.0, d0_max=0.0, kappa_min=-4.0,
                     kappa_max=4.0, layer_radii=TOY_LAYER_RADII_CM)
TOY_LINE_SPEC = LineSpec(n_tracks=50, n_noise=100)        # Fig. 3: 50 tracks x 10 hits
TOY_LINE_SPEC_5000 = LineSpec(n_tracks=450, n_noise=500)  # "up to 5000 hits"
