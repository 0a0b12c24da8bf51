"""Seeded synthetic vesicle suspensions (host, numpy, fp64).

This module serves both the tests' oracle side and the CUDA side and therefore holds
NONE of the method's arithmetic: no Stokeslet, no quadrature weights, no spectral
derivative.  It only draws shapes, places them and draws densities.  (The reduced-area
rescaling needs an area and a perimeter of the *analytic* shape; they are taken from a
1024-gon of r(theta), which is input recipe, not the path's arclength quadrature.)

The suspensions stand in for the paper's runs, whose actual configurations are not
available: sizes, area fractions and box shapes follow PAPER.md:25, 554 (2,000 vesicles,
Poiseuille channel, 30 %), PAPER.md:89, 540, 552 (Taylor-Green, free space, 25-30 %) and
BASELINE.json `configs`; the recipe is written out in DESIGN.md ("Input recipe").

Draw order (numpy Generator(PCG64(seed)), seed = 260625569 + config index):
shapes (a_k, phi_k)  ->  placement trials (psi, cx, cy)  ->  forces (x: a, b; y: a, b)
->  config 4's position perturbations.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
from scipy.spatial import cKDTree

BASE_SEED = 260625569
MIN_GAP = 0.05            # minimum point-to-point distance between different vesicles
REDUCED_AREA = 0.65


@dataclass
class Suspension:
    X: np.ndarray                 # [nves, npts, 2] float64 membrane points
    F: np.ndarray                 # [nves, npts, 2] float64 density (traction jump)
    mu: float = 1.0
    box: tuple = (0.0, 0.0)       # (Lx, Ly); (0, 0) = free-space grid (config 0)
    trials: int = 0               # placement trials used
    name: str = ""
    X_sequence: list = field(default_factory=list)   # config 4: ten position arrays

    @property
    def nves(self):
        return self.X.shape[0]

    @property
    def npts(self):
        return self.X.shape[1]

    @property
    def pairs(self):
        """Interactions of one evaluation: P (P - npts); own-vesicle pairs are not counted."""
        P = self.nves * self.npts
        return P * (P - self.npts)


def _rot(psi):
    c, s = np.cos(psi), np.sin(psi)
    return np.stack([np.stack([c, -s], -1), np.stack([s, c], -1)], -2)     # [..., 2, 2]


def fourier_density(rng, nves, npts, nmodes):
    """F = sum_{k=1..nmodes} (a_k cos k alpha + b_k sin k alpha) / k^2, a, b ~ N(0,1); x then y."""
    al = 2 * np.pi * np.arange(npts) / npts
    k = np.arange(1, nmodes + 1)
    C = np.cos(k[:, None] * al[None, :]) / (k[:, None] ** 2)               # [K, npts]
    S = np.sin(k[:, None] * al[None, :]) / (k[:, None] ** 2)
    comps = []
    for _ in range(2):
        a = rng.standard_normal((nves, nmodes))
        b = rng.standard_normal((nves, nmodes))
        comps.append(a @ C + b @ S)
    return np.stack(comps, -1)


def _polygon_area_perimeter(x, y):
    xn, yn = np.roll(x, -1, -1), np.roll(y, -1, -1)
    area = 0.5 * np.abs((x * yn - xn * y).sum(-1))
    per = np.hypot(xn - x, yn - y).sum(-1)
    return area, per


def random_shapes(rng, nves, npts):
    """Body-frame shapes r(theta) = 1 + sum_{k=2..6} a_k cos(k theta + phi_k), a_k ~ U(0, 0.15/k),
    stretched y -> s y (bisection, 60 steps on [0.05, 1]) to reduced area 4 pi A / L^2 = 0.65.
    Returns body points [nves, npts, 2] (theta_j = 2 pi j / npts) and areas [nves]."""
    ks = np.arange(2, 7)
    a = rng.uniform(0.0, 0.15 / ks, size=(nves, 5))
    phi = rng.uniform(0.0, 2 * np.pi, size=(nves, 5))

    def radius(theta):
        return 1.0 + (a[:, :, None] * np.cos(ks[None, :, None] * theta[None, None, :] + phi[:, :, None])).sum(1)

    fine = 2 * np.pi * np.arange(1024) / 1024
    rf = radius(fine)
    xf, yf = rf * np.cos(fine), rf * np.sin(fine)
    area1, _ = _polygon_area_perimeter(xf, yf)                  # polygon area is linear in the stretch s
    ex2 = (np.roll(xf, -1, -1) - xf) ** 2
    ey2 = (np.roll(yf, -1, -1) - yf) ** 2
    lo = np.full(nves, 0.05)
    hi = np.ones(nves)
    for _ in range(60):
        s = 0.5 * (lo + hi)
        L = np.sqrt(ex2 + (s * s)[:, None] * ey2).sum(-1)       # polygon perimeter after y -> s y
        too_round = 4 * np.pi * (s * area1) / L ** 2 > REDUCED_AREA
        hi = np.where(too_round, s, hi)
        lo = np.where(too_round, lo, s)
    s = 0.5 * (lo + hi)
    area = s * area1
    th = 2 * np.pi * np.arange(npts) / npts
    r = radius(th)
    body = np.stack([r * np.cos(th), s[:, None] * r * np.sin(th)], -1)
    return body, area


def place(rng, body, area, phi_area, aspect):
    """Random sequential insertion in a box of area sum(A_v)/phi with Lx = aspect * Ly.
    A trial is accepted when every point is >= MIN_GAP from every point of every vesicle
    already placed.  Returns X [nves, npts, 2], (Lx, Ly), trials."""
    nves, npts, _ = body.shape
    box_area = area.sum() / phi_area
    Ly = float(np.sqrt(box_area / aspect))
    Lx = aspect * Ly
    rad = np.sqrt((body ** 2).sum(-1)).max(1)                                # bounding radius per shape
    cell = 2.0 * rad.max() + MIN_GAP
    ncx, ncy = int(Lx / cell) + 1, int(Ly / cell) + 1
    cells = {}
    trees = [None] * nves                                                    # one k-d tree per placed vesicle
    X = np.empty_like(body)
    centre = np.empty((nves, 2))
    trials = 0
    for v in range(nves):
        while True:
            trials += 1
            psi = rng.uniform(0.0, 2 * np.pi)
            cx = rng.uniform(1.2, Lx - 1.2)
            cy = rng.uniform(1.2, Ly - 1.2)
            cs, sn = np.cos(psi), np.sin(psi)
            pts = np.empty((npts, 2))
            pts[:, 0] = cs * body[v, :, 0] - sn * body[v, :, 1] + cx
            pts[:, 1] = sn * body[v, :, 0] + cs * body[v, :, 1] + cy
            ix, iy = int(cx / cell), int(cy / cell)
            cand = []
            for jx in range(max(ix - 1, 0), min(ix + 2, ncx)):
                for jy in range(max(iy - 1, 0), min(iy + 2, ncy)):
                    cand += cells.get((jx, jy), ())
            ok = True
            if cand:
                cand = np.asarray(cand)
                dc = np.hypot(cx - centre[cand, 0], cy - centre[cand, 1])
                for u in cand[dc <= rad[v] + rad[cand] + MIN_GAP]:
                    # nearest placed point of vesicle u strictly closer than MIN_GAP?
                    d, _ = trees[u].query(pts, k=1, distance_upper_bound=MIN_GAP)
                    if np.isfinite(d).any():
                        ok = False
                        break
            if ok:
                X[v] = pts
                centre[v] = (cx, cy)
                trees[v] = cKDTree(pts)
                cells.setdefault((ix, iy), []).append(v)
                break
    return X, (Lx, Ly), trials


def suspension(nves, npts, phi_area, aspect, seed, nmodes=16, name="", perturb_calls=0):
    """Dense suspension of reduced-area-0.65 vesicles (configs 1-4 and any size like them)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    body, area = random_shapes(rng, nves, npts)
    X, box, trials = place(rng, body, area, phi_area, aspect)
    F = fourier_density(rng, nves, npts, nmodes)
    seq = []
    if perturb_calls:
        seq = [X]
        for _ in range(perturb_calls - 1):
            seq.append(seq[-1] + 1e-3 * rng.standard_normal(X.shape))
    return Suspension(X=X, F=F, mu=1.0, box=box, trials=trials, name=name, X_sequence=seq)


def config0():
    """16 ellipses (1, 0.4) on a 4x4 grid of spacing 3, random angles, 32 points, K = 8 force modes."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 0))
    nves, npts = 16, 32
    psi = rng.uniform(0.0, 2 * np.pi, size=nves)
    al = 2 * np.pi * np.arange(npts) / npts
    body = np.stack([np.cos(al), 0.4 * np.sin(al)], -1)                      # [npts, 2]
    p, q = np.divmod(np.arange(nves), 4)
    centres = np.stack([3.0 * p, 3.0 * q], -1).astype(np.float64)
    X = np.einsum("vab,jb->vja", _rot(psi), body) + centres[:, None, :]
    F = fourier_density(rng, nves, npts, 8)
    return Suspension(X=X, F=F, mu=1.0, name="config0: 16x32 free-space grid")


_CONFIGS = {
    1: dict(nves=256, npts=128, phi_area=0.20, aspect=1.0, name="config1: 256x128, 20% square box"),
    2: dict(nves=1000, npts=128, phi_area=0.30, aspect=1.0, name="config2: 1000x128, 30% square box"),
    3: dict(nves=2000, npts=128, phi_area=0.30, aspect=4.0, name="config3: 2000x128, 30% 4:1 channel"),
    4: dict(nves=8000, npts=128, phi_area=0.30, aspect=1.0, name="config4: 8000x128, 30% square box, 10 calls",
            perturb_calls=10),
}


def config(index: int) -> Suspension:
    """BASELINE.json configs[index]."""
    if index == 0:
        return config0()
    return suspension(seed=BASE_SEED + index, **_CONFIGS[index])


def config_shape(index: int):
    """(nves, npts) without generating anything."""
    if index == 0:
        return 16, 32
    return _CONFIGS[index]["nves"], _CONFIGS[index]["npts"]
