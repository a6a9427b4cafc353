"""Seeded synthetic input generators (geometries, coercive fields, spins, field protocols).

This module serves BOTH the CPU oracle (tests, ``bench.py --impl reference``) and the CUDA path.
It holds none of the method's arithmetic: no dipolar field, no astroid, no relaxation, no thermal
draw.  It only produces the *inputs* the paper's model takes ("each magnetic dipole is
modelled with a position r_i and rotation theta_i ... each magnet is assigned a coercive field"),
in the shapes of BASELINE.json's five configs.  numpy only.

Recipes:

* geometries, PAPER.md:140-148 (section II.I, Fig. 3): square closed/open, kagome, pinwheel diamond,
  ising, plus "rotated square" (BASELINE.json config 3).
* coercive-field disorder, PAPER.md:118 (section II.G): h_k^(i) ~ N(h_k, (k_disorder h_k)^2), kept
  positive by redrawing.
* field protocols, PAPER.md:63 / :124: a discrete series of global fields, relaxed at each value.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SQRT3 = math.sqrt(3.0)


# --------------------------------------------------------------------------- geometries
def square_closed(n: int):
    """Square ASI, closed edges, n x n cells -> N = 2 n (n+1)   (Fig. 3a).

    Horizontals (i+1/2, j), i<n, j<=n, theta=0, index j*n+i; then verticals (i, j+1/2), i<=n, j<n,
    theta=pi/2, index Nh + j*(n+1)+i.  Lattice spacing 1.
    """
    j, i = np.meshgrid(np.arange(n + 1), np.arange(n), indexing="ij")
    hpos = np.stack([i.ravel() + 0.5, j.ravel().astype(np.float64)], axis=1)
    j, i = np.meshgrid(np.arange(n), np.arange(n + 1), indexing="ij")
    vpos = np.stack([i.ravel().astype(np.float64), j.ravel() + 0.5], axis=1)
    pos = np.concatenate([hpos, vpos]).astype(np.float64)
    angle = np.concatenate([np.zeros(len(hpos)), np.full(len(vpos), math.pi / 2)])
    return np.ascontiguousarray(pos), np.ascontiguousarray(angle)


def square_open(n: int):
    """Square ASI, open edges: n x n vertices, magnets on the edges between them -> N = 2 n (n-1)
    (Fig. 3b; the geometry of the paper's Fig. 9 throughput test)."""
    j, i = np.meshgrid(np.arange(n), np.arange(n - 1), indexing="ij")
    hpos = np.stack([i.ravel() + 0.5, j.ravel().astype(np.float64)], axis=1)
    j, i = np.meshgrid(np.arange(n - 1), np.arange(n), indexing="ij")
    vpos = np.stack([i.ravel().astype(np.float64), j.ravel() + 0.5], axis=1)
    pos = np.concatenate([hpos, vpos]).astype(np.float64)
    angle = np.concatenate([np.zeros(len(hpos)), np.full(len(vpos), math.pi / 2)])
    return np.ascontiguousarray(pos), np.ascontiguousarray(angle)


def rotated_square(n: int, rot: float = math.pi / 4):
    """BASELINE.json config 3: closed-square positions, every magnet rotated `rot` about its centre."""
    pos, angle = square_closed(n)
    return pos, angle + rot


def pinwheel_lucky_knot(n: int, rot: float = math.pi / 4):
    """Pinwheel "lucky-knot" edges (Fig. 3e): the closed-square lattice with every magnet rotated
    45 degrees -> N = 2 n (n+1).  Same construction as BASELINE.json config 3 (`rotated_square`)."""
    return rotated_square(n, rot)


def pinwheel_diamond(n: int, rot: float = math.pi / 4):
    """Pinwheel "diamond" with 2 n^2 magnets (PAPER.md:286: 25x25 -> 1250; :288: 708x708 -> >1e6).

    One horizontal (i+1/2, j) and one vertical (i, j+1/2) magnet per cell i,j<n, each rotated `rot`.
    """
    j, i = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    hpos = np.stack([i.ravel() + 0.5, j.ravel().astype(np.float64)], axis=1)
    vpos = np.stack([i.ravel().astype(np.float64), j.ravel() + 0.5], axis=1)
    pos = np.concatenate([hpos, vpos]).astype(np.float64)
    angle = np.concatenate([np.zeros(len(hpos)), np.full(len(vpos), math.pi / 2)]) + rot
    return np.ascontiguousarray(pos), np.ascontiguousarray(angle)


def ising(nx: int, ny: int):
    """Ising geometry (Fig. 3f): nx x ny collinear magnets on a unit square grid, theta=0."""
    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    pos = np.stack([i.ravel().astype(np.float64), j.ravel().astype(np.float64)], axis=1)
    return np.ascontiguousarray(pos), np.zeros(nx * ny)


def kagome(n: int):
    """Kagome ASI: honeycomb of n x n flat-top hexagons, edge length 1, one magnet per unique edge at
    its midpoint along the edge direction (0, 60, 120 degrees)  -> N = 3 n^2 + 4 n - 1
    (29 x 29 hexagons = 2638 magnets; Fig. 3c).

    Hexagon centres (1.5 c, sqrt3 r + (sqrt3/2 if c odd)), c,r in [0,n).  Index order = first
    occurrence iterating c (outer), r (inner), then the six edges counter-clockwise from the edge
    whose midpoint lies at 30 degrees.  Midpoints are stored on the exact lattice
    (x = q/4, y = p*sqrt3/4 with integers q,p) so equal edges coincide bit-exactly.
    """
    seen = {}
    qs, ps, ths = [], [], []
    # edge midpoints of a unit flat-top hexagon in units (1/4, sqrt3/4): angle 30+60k at radius sqrt3/2
    mids = [(3, 1), (0, 2), (-3, 1), (-3, -1), (0, -2), (3, -1)]
    dirs = [2, 0, 1, 2, 0, 1]  # edge direction = multiples of 60 degrees: 120, 0, 60, 120, 0, 60
    for c in range(n):
        for r in range(n):
            cq = 6 * c                      # 1.5 c  in units of 1/4
            cp = 4 * r + (2 if c % 2 else 0)  # sqrt3 r + sqrt3/2 in units of sqrt3/4
            for (dq, dp), d in zip(mids, dirs):
                key = (cq + dq, cp + dp)
                if key in seen:
                    continue
                seen[key] = len(qs)
                qs.append(key[0]); ps.append(key[1]); ths.append(d)
    pos = np.stack([np.array(qs) * 0.25, np.array(ps) * (SQRT3 / 4.0)], axis=1).astype(np.float64)
    angle = np.array(ths, dtype=np.float64) * (math.pi / 3.0)
    return np.ascontiguousarray(pos), np.ascontiguousarray(angle)


def square_vertices(n: int):
    """Interior vertices of `square_closed(n)`: the lattice points (x, y), 0 < x, y < n, where four magnets meet
    (Fig. 6a "ASI vertices").  Returns [V,4] spin indices (left, right, below, above), V = (n-1)^2."""
    y, x = np.meshgrid(np.arange(1, n), np.arange(1, n), indexing="ij")
    x = x.ravel(); y = y.ravel()
    nh = n * (n + 1)
    left = y * n + (x - 1); right = y * n + x
    below = nh + (y - 1) * (n + 1) + x; above = nh + y * (n + 1) + x
    return np.ascontiguousarray(np.stack([left, right, below, above], axis=1).astype(np.int32))


def square_ground_state(n: int):
    """The antiferromagnetic ground state of `square_closed(n)` (every vertex Type I): horizontal
    spins alternate with (i + j), vertical spins with (i + j + 1)."""
    j, i = np.meshgrid(np.arange(n + 1), np.arange(n), indexing="ij")
    sh = np.where((i + j) % 2 == 0, 1, -1).ravel()
    j, i = np.meshgrid(np.arange(n), np.arange(n + 1), indexing="ij")
    sv = np.where((i + j) % 2 == 0, -1, 1).ravel()
    return np.concatenate([sh, sv]).astype(np.int8)


# --------------------------------------------------------------------------- per-magnet inputs
def coercive_fields(N: int, hk: float = 0.2, k_disorder: float = 0.05, seed: int = 0, replicas: int = 0):
    """h_k^(i) ~ N(h_k, (k_disorder h_k)^2), redrawn until positive.

    Uses numpy's counter-based Philox bit generator keyed by `seed` (an input recipe, not the
    method's thermal stream).  `replicas` > 0 returns [replicas, N] with seeds seed, seed+1, ...
    """
    def one(sd):
        rng = np.random.Generator(np.random.Philox(key=sd))
        hc = hk * (1.0 + k_disorder * rng.standard_normal(N))
        bad = hc <= 0
        while bad.any():
            hc[bad] = hk * (1.0 + k_disorder * rng.standard_normal(int(bad.sum())))
            bad = hc <= 0
        return hc
    if replicas > 0:
        return np.ascontiguousarray(np.stack([one(seed + r) for r in range(replicas)]))
    return np.ascontiguousarray(one(seed))


def random_spins(N: int, seed: int = 1):
    rng = np.random.Generator(np.random.Philox(key=seed))
    return (2 * rng.integers(0, 2, size=N, dtype=np.int8) - 1).astype(np.int8)


# --------------------------------------------------------------------------- field protocols
def ramp(A: float, B: float, K: int, phi_deg: float, legs: int = 1):
    """K+1 global field vectors t=0..K at angle phi (reading C-13).

    one leg : H_t = A + (B-A) t/K;   two legs: H_t = A + (B-A) (1 - |1 - 2t/K|)   (A -> B -> A).
    Returns [K+1, 2] (hx, hy).
    """
    t = np.arange(K + 1, dtype=np.float64)
    if legs == 1:
        H = A + (B - A) * t / K
    else:
        H = A + (B - A) * (1.0 - np.abs(1.0 - 2.0 * t / K))
    phi = math.radians(phi_deg)
    return np.ascontiguousarray(np.stack([H * math.cos(phi), H * math.sin(phi)], axis=1))


def sinusoidal(amplitude: float, periods: float, steps_per_period: int, phi_deg: float, offset: float = 0.0):
    """Input encoder "sinusoidal field": H_t = offset + A sin(2 pi t / steps_per_period) along
    the fixed direction phi, t = 0 .. periods * steps_per_period.  Returns [T,2]."""
    T = int(round(periods * steps_per_period)) + 1
    t = np.arange(T, dtype=np.float64)
    H = offset + amplitude * np.sin(2.0 * math.pi * t / steps_per_period)
    phi = math.radians(phi_deg)
    return np.ascontiguousarray(np.stack([H * math.cos(phi), H * math.sin(phi)], axis=1))


def sawtooth(amplitude: float, periods: float, steps_per_period: int, phi_deg: float):
    """Input encoder "sawtooth field": H_t rises linearly from -A to +A over one period, then jumps
    back.  Returns [T,2]."""
    T = int(round(periods * steps_per_period)) + 1
    t = np.arange(T, dtype=np.float64)
    H = amplitude * (2.0 * ((t / steps_per_period) % 1.0) - 1.0)
    phi = math.radians(phi_deg)
    return np.ascontiguousarray(np.stack([H * math.cos(phi), H * math.sin(phi)], axis=1))


def rotating(amplitude: float, periods: float, steps_per_period: int, phi0_deg: float = 0.0):
    """Input encoder "rotational field": constant magnitude A, direction phi0 + 2 pi t /
    steps_per_period.  Returns [T,2]."""
    T = int(round(periods * steps_per_period)) + 1
    phi = math.radians(phi0_deg) + 2.0 * math.pi * np.arange(T, dtype=np.float64) / steps_per_period
    return np.ascontiguousarray(np.stack([amplitude * np.cos(phi), amplitude * np.sin(phi)], axis=1))


# --------------------------------------------------------------------------- geometries that are NOT lattices
# The library takes any pos[N,2] / angle[N] ("each magnet has a position and a rotation"); flatspin's stock
# geometries are lattices, user-defined ones need not be.  These two exercise the general path: cell-grid neighbour
# lists with ragged rows, the ELL gather, relax / batched flips / sweeps without the lattice's cell index.
def jittered_square(n: int, sigma_pos: float = 0.03, sigma_angle: float = 0.08, seed: int = 0):
    """Closed square ASI n x n with every magnet displaced by N(0, sigma_pos) per coordinate and rotated by
    N(0, sigma_angle) radians: fabrication disorder in the geometry itself.  2n(n+1) magnets."""
    pos, ang = square_closed(n)
    rng = np.random.default_rng(seed)
    return (np.ascontiguousarray(pos + sigma_pos * rng.standard_normal(pos.shape)),
            np.ascontiguousarray(ang + sigma_angle * rng.standard_normal(ang.shape)))


def point_cloud(n_target: int, r_min: float = 0.7, seed: int = 0, rounds: int = 40):
    """Random point cloud with a minimum distance (Poisson-disc sampling by vectorised dart throwing) and uniformly
    random angles in [0, pi).  The box is sized for about n_target points at ~0.62 / r_min^2 points per unit area.
    A background grid of cell side r_min / sqrt(2) holds at most one accepted point per cell; each round throws
    darts, drops those in occupied cells or within r_min of an accepted point (5 x 5 cells around the dart), and
    among the darts of one round drops every dart that has an earlier dart of the round within r_min.
    Returns (pos [N,2], angle [N]) with N close to n_target (deterministic for a given seed)."""
    rng = np.random.default_rng(seed)
    side = math.sqrt(n_target * r_min * r_min / 0.62)
    cell = r_min / math.sqrt(2.0)
    G = int(math.ceil(side / cell))
    grid = np.full((G + 4, G + 4), -1, np.int64)            # 2 cells of border: no bounds checks on the 5 x 5 window
    pts = np.zeros((0, 2))
    offs = [(a, b) for a in range(-2, 3) for b in range(-2, 3)]
    for _ in range(rounds):
        m = max(4 * n_target // 3, 64)
        d = rng.random((m, 2)) * side
        cx = (d[:, 0] / cell).astype(np.int64) + 2; cy = (d[:, 1] / cell).astype(np.int64) + 2
        ok = np.ones(m, bool)
        for a, b in offs:                                    # against the accepted points
            j = grid[cx + a, cy + b]
            has = j >= 0
            if has.any():
                dd = d[has] - pts[j[has]]
                ok[np.flatnonzero(has)[(dd * dd).sum(1) < r_min * r_min]] = False
        d, cx, cy = d[ok], cx[ok], cy[ok]
        # among this round's darts: keep a dart only if no EARLIER dart of the round lies within r_min
        tmp = np.full_like(grid, -1)
        keep = np.ones(len(d), bool)
        order = np.arange(len(d))
        first = np.full_like(grid, len(d))
        np.minimum.at(first, (cx, cy), order)
        keep &= first[cx, cy] == order                       # one dart per cell: the earliest
        d, cx, cy = d[keep], cx[keep], cy[keep]
        tmp[cx, cy] = np.arange(len(d))
        keep = np.ones(len(d), bool)
        for a, b in offs:
            if (a, b) == (0, 0):
                continue
            j = tmp[cx + a, cy + b]
            has = (j >= 0) & (j < np.arange(len(d)))
            if has.any():
                dd = d[has] - d[j[has]]
                keep[np.flatnonzero(has)[(dd * dd).sum(1) < r_min * r_min]] = False
        d, cx, cy = d[keep], cx[keep], cy[keep]
        grid[cx, cy] = len(pts) + np.arange(len(d))
        pts = np.concatenate([pts, d])
    ang = rng.random(len(pts)) * math.pi
    return np.ascontiguousarray(pts), np.ascontiguousarray(ang)


def off_lattice(kind: str, n: int, seed: int = 0, K_steps: int = 40, sigma_th: float = 0.005) -> "Workload":
    """A whole workload on a non-lattice geometry: `kind` = "jittered_square" (n x n cells) or "point_cloud" (about n
    magnets), 5 % h_k disorder, all spins +1, thermal ramp 0.2 -> -0.2 at 45 degrees in K_steps steps (the config-4
    protocol, shortened)."""
    if kind == "jittered_square":
        pos, ang = jittered_square(n, seed=seed)
        nd = 1.6
    elif kind == "point_cloud":
        pos, ang = point_cloud(n, seed=seed)
        nd = 1.5
    else:
        raise ValueError(kind)
    N = len(ang)
    return Workload(f"{kind}_{n}_seed{seed}", pos, ang, coercive_fields(N, seed=seed), np.ones(N, np.int8),
                    _params(0.001, 1, 1, 3, 3, nd), ramp(0.2, -0.2, K_steps, 45.0, legs=1), sigma_th=sigma_th,
                    thermal_seed=seed)


# --------------------------------------------------------------------------- the five configs
@dataclass
class Workload:
    name: str
    pos: np.ndarray
    angle: np.ndarray
    hc: np.ndarray
    spins: np.ndarray
    params: dict           # alpha, b, c, beta, gamma, neighbor_distance
    fields: np.ndarray     # [T, 2] global field per step (step key = row index)
    sigma_th: float = 0.0
    thermal_seed: int = 0
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def N(self):
        return int(self.pos.shape[0])


def _params(alpha, b, c, beta, gamma, nd):
    return dict(alpha=float(alpha), b=float(b), c=float(c), beta=float(beta), gamma=float(gamma),
                neighbor_distance=float(nd))


def config(which, scale: int | None = None) -> Workload:
    """BASELINE.json configs 1..5 (and '2b').  `scale` overrides the lattice size n (parity tests
    at reduced size use the same recipe)."""
    which = str(which)
    if which == "1":
        n = scale or 10
        pos, ang = square_closed(n)
        return Workload(f"cfg1_square_closed_{n}x{n}", pos, ang, coercive_fields(len(ang)),
                        np.ones(len(ang), np.int8), _params(0.001, 1, 1, 3, 3, 1.0),
                        ramp(0.2, -0.2, 500, 45.0, legs=2))
    if which in ("2", "2b"):
        n = scale or (50 if which == "2" else 70)
        pos, ang = kagome(n)
        return Workload(f"cfg{which}_kagome_{n}x{n}", pos, ang, coercive_fields(len(ang)),
                        np.ones(len(ang), np.int8), _params(0.001, 1, 1, 3, 3, SQRT3),
                        ramp(-0.15, 0.15, 1000, 5.0, legs=2))
    if which == "3":
        n = scale or 200
        pos, ang = rotated_square(n)
        return Workload(f"cfg3_rotated_square_{n}x{n}", pos, ang, coercive_fields(len(ang)),
                        np.ones(len(ang), np.int8), _params(0.0013, 0.38, 1, 1.7, 3, 3.0),
                        ramp(0.12, -0.12, 2000, -40.0, legs=2))
    if which == "4":
        n = scale or 1000
        pos, ang = square_closed(n)
        return Workload(f"cfg4_square_closed_{n}x{n}_thermal", pos, ang, coercive_fields(len(ang)),
                        np.ones(len(ang), np.int8), _params(0.001, 1, 1, 3, 3, 1.0),
                        ramp(0.2, -0.2, 200, 45.0, legs=1), sigma_th=0.01, thermal_seed=0)
    if which == "5":
        n = scale or 500
        pos, ang = square_closed(n)
        phi = math.radians(45.0)
        return Workload(f"cfg5_square_closed_{n}x{n}_nd10", pos, ang, coercive_fields(len(ang)),
                        random_spins(len(ang), seed=1), _params(0.001, 1, 1, 3, 3, 10.0),
                        np.array([[0.10 * math.cos(phi), 0.10 * math.sin(phi)]]),
                        note="field + scan only, spins not flipped")
    raise ValueError(f"unknown config {which!r}")


# --------------------------------------------------------------------------- the paper's own parameter sets
def paper_pinwheel_reversal(n: int = 25, theta_deg: float = 0.0, K: int = 2500, amplitude: float = 0.08) -> Workload:
    """PAPER.md:220-240 (section IV.C) and :286-288: pinwheel "diamond" ASI of n x n units (25 -> 1250 magnets,
    708 -> 1,002,528), b = 0.28, c = 1, beta = 4.8, gamma = 3, alpha = 0.00033, h_k = 0.098, k_disorder = 0.05,
    neighbor distance 10, one reversal in K = 2500 field values at angle theta (0, -6, 30 degrees in Fig. 7).
    The paper does not print the field range: `amplitude` (+A -> -A, enough to reverse the array) is this
    recipe's choice; the array starts polarised along +x."""
    pos, ang = pinwheel_diamond(n)
    spins = np.where(np.cos(ang) > 0, 1, -1).astype(np.int8)
    return Workload(f"paperIVC_pinwheel_diamond_{n}x{n}_theta{theta_deg:g}", pos, ang,
                    coercive_fields(len(ang), hk=0.098, k_disorder=0.05, seed=0), spins,
                    _params(0.00033, 0.28, 1.0, 4.8, 3.0, 10.0), ramp(amplitude, -amplitude, K, theta_deg, legs=1),
                    note="PAPER.md:230 parameters; field range not given in the paper")


def paper_kagome_dirac_strings(n: int = 29, K: int = 400, amplitude: float = 0.12) -> Workload:
    """PAPER.md:174-188 (section IV.A): kagome ASI of 29 x 29 hexagons (2638 magnets) polarised to the left,
    reversal field to the right with a downward offset of 3.6 degrees; alpha = 0.00103, h_k = 0.216, beta = 2.5,
    gamma = 3, b = 0.212, c = 1, sigma_th = 0.002, k_disorder = 0.05.  Neighbourhood and field range are not
    printed: neighbor distance sqrt(3) (as BASELINE.json config 2) and 0 -> +A in K steps are this recipe's."""
    pos, ang = kagome(n)
    spins = np.where(np.cos(ang) > 1e-9, -1, np.where(np.cos(ang) < -1e-9, 1, -1)).astype(np.int8)   # m_x <= 0
    return Workload(f"paperIVA_kagome_{n}x{n}", pos, ang, coercive_fields(len(ang), hk=0.216, k_disorder=0.05, seed=0),
                    spins, _params(0.00103, 0.212, 1.0, 2.5, 3.0, SQRT3), ramp(0.0, amplitude, K, -3.6, legs=1),
                    sigma_th=0.002, thermal_seed=0, note="PAPER.md:182 parameters; neighbourhood and field range not given")


def paper_square_anneal(n: int = 50, alpha: float = 0.0015, T: int = 200, sigma0: float = 0.1, decay: float = 40.0,
                        replicas: int = 0, seed: int = 0) -> Workload:
    """PAPER.md:196-206 (section IV.B): 50 x 50 square ASI (closed edges), annealed by a thermal protocol of
    exponentially decreasing sigma_th; b = 0.4, c = 1, beta = gamma = 3, h_k = 0.186, k_disorder = 0.05, neighbor
    distance 10; no external field.  The paper gives neither the map from the lattice constant a to alpha nor the
    protocol constants: alpha, sigma0 and the decay (sigma_t = sigma0 exp(-t / decay), T steps) are this recipe's.
    Spins start random.  `extra` carries sigma[T] and the interior vertices [V,4]; `replicas` > 0 draws that many
    h_c disorder realisations [R,N] (an ensemble, "across the ensembles")."""
    pos, ang = square_closed(n)
    N = len(ang)
    hc = coercive_fields(N, hk=0.186, k_disorder=0.05, seed=seed, replicas=replicas)
    sigma = sigma0 * np.exp(-np.arange(T, dtype=np.float64) / decay)
    return Workload(f"paperIVB_square_anneal_{n}x{n}", pos, ang, hc, random_spins(N, seed=seed + 1),
                    _params(alpha, 0.4, 1.0, 3.0, 3.0, 10.0), np.zeros((T, 2)), sigma_th=float(sigma[0]), thermal_seed=seed,
                    note="PAPER.md:202 parameters; alpha and the annealing schedule are not given in the paper",
                    extra={"sigma": sigma, "vertices": square_vertices(n)})
