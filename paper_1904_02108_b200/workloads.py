"""Seeded synthetic workloads W1..W5 (BASELINE.json configs[0..4]).

This module is the ONLY code shared by the fp64 oracle side and the CUDA side of the tests:
it produces plain numpy input arrays (lattice parameters, rest-pose marker positions, marker
areas, per-body kinematics, initial fields).  It contains none of the method's arithmetic
(no delta kernel, no collision, no interpolation) -- only geometry of the synthetic stand-in
for the paper's Blender propeller mesh (not in the container).

Propeller template (body frame, rotation axis = e3): blade j at azimuth psi0 + 2*pi*j/n_b with
radial unit r, chord c = cos(beta) t + sin(beta) e3 (pitch beta = 30 deg), normal n = r x c;
markers at the centres of an h = 0.5 grid,
    p = (a + 1/2) h r + ((b + 1/2) h - w/2) c + (l - (L-1)/2) h n,   a < R/h, b < w/h, l < L,
then rotated so e3 -> the body's axis and translated to its centre.  Marker area s = h*h / L.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

H_SPACING = 0.5
PITCH_DEG = 30.0


@dataclass
class Body:
    """One rigid body: rest-pose markers (float32, as they cross the C ABI) + kinematics."""
    pos: np.ndarray        # [n,3] float32 rest positions (lattice units)
    area: np.ndarray       # [n]   float32 marker areas s(k)
    omega: float           # rad / step
    axis: np.ndarray       # [3] float64 unit vector
    center: np.ndarray     # [3] float64
    vel: np.ndarray | None = None   # [n,3] float32 extra (unrotated) velocity, None = 0


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    tau: float
    wall: tuple            # (wx, wy, wz): 0 periodic, 1 half-way bounce-back on both faces
    g: tuple               # uniform body acceleration
    bodies: list = field(default_factory=list)
    steps: int = 100
    mdf_iters: int = 0
    rho0: np.ndarray | None = None   # [nz,ny,nx] float32 or None (=1)
    u0: np.ndarray | None = None     # [3,nz,ny,nx] float32 or None (=0)
    note: str = ""

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_markers(self) -> int:
        return int(sum(b.pos.shape[0] for b in self.bodies))


def _frame_from_axis(axis: np.ndarray) -> np.ndarray:
    """Orthonormal matrix Q (columns q1,q2,q3) with q3 = axis: maps the body frame to the lab."""
    a = np.asarray(axis, dtype=np.float64)
    a = a / np.linalg.norm(a)
    helper = np.array([1.0, 0.0, 0.0]) if abs(a[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    q1 = np.cross(helper, a)
    q1 /= np.linalg.norm(q1)
    q2 = np.cross(a, q1)
    return np.stack([q1, q2, a], axis=1)


def propeller(n_blades: int, radius: float, width: float, layers: int, psi0: float,
              axis, center, omega: float, h: float = H_SPACING) -> Body:
    """Flat-plate propeller markers in the lab frame (see module docstring); h = marker spacing."""
    beta = np.deg2rad(PITCH_DEG)
    na = int(round(radius / h))
    nb = int(round(width / h))
    a = (np.arange(na) + 0.5) * h
    b = (np.arange(nb) + 0.5) * h - width / 2.0
    l = (np.arange(layers) - (layers - 1) / 2.0) * h
    A, B, Lr = np.meshgrid(a, b, l, indexing="ij")
    pts = []
    e3 = np.array([0.0, 0.0, 1.0])
    for j in range(n_blades):
        psi = psi0 + 2.0 * np.pi * j / n_blades
        r = np.array([np.cos(psi), np.sin(psi), 0.0])
        t = np.array([-np.sin(psi), np.cos(psi), 0.0])
        c = np.cos(beta) * t + np.sin(beta) * e3
        n = np.cross(r, c)
        p = A[..., None] * r + B[..., None] * c + Lr[..., None] * n
        pts.append(p.reshape(-1, 3))
    body = np.concatenate(pts, axis=0)
    Q = _frame_from_axis(np.asarray(axis, dtype=np.float64))
    lab = body @ Q.T + np.asarray(center, dtype=np.float64)
    n_m = lab.shape[0]
    area = np.full(n_m, h * h / layers, dtype=np.float32)
    ax = np.asarray(axis, dtype=np.float64)
    return Body(pos=lab.astype(np.float32), area=area, omega=float(omega),
                axis=ax / np.linalg.norm(ax), center=np.asarray(center, dtype=np.float64))


def _random_unit(rng) -> np.ndarray:
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def poiseuille_profile(nz: int, tau: float, g: float) -> np.ndarray:
    """Initial velocity profile of config 2 (a parabola between walls half a link outside the
    first / last node; this is the *input recipe*, the oracle's steady state is checked against
    its own closed form in tests/)."""
    nu = (tau - 0.5) / 3.0
    z = np.arange(nz, dtype=np.float64)
    return g / (2.0 * nu) * (z + 0.5) * (nz - 0.5 - z)


def w1(seed: int = 0) -> Workload:
    rng = np.random.default_rng(seed)
    psi0 = float(rng.uniform(0.0, 2.0 * np.pi))
    b = propeller(2, 10.0, 3.0, 1, psi0, [0.0, 0.0, 1.0], [16.0, 16.0, 16.0], 0.005)
    return Workload("W1", 32, 32, 32, 0.8, (0, 0, 0), (0.0, 0.0, 0.0), [b], steps=100,
                    mdf_iters=3, note="configs[0]: oracle-sized, 1x2-blade propeller")


def w2(seed: int = 0, n: int = 256) -> Workload:
    rng = np.random.default_rng(seed)
    tau, g = 0.6, 1e-6
    # keep the centre-line Mach number of the 256^3 case when n is reduced for parity tests
    g_eff = g * (256.0 / n) ** 2
    prof = poiseuille_profile(n, tau, g_eff)
    u0 = np.zeros((3, n, n, n), dtype=np.float32)
    u0[0] = prof[:, None, None].astype(np.float32)
    u0 += rng.uniform(-1e-4, 1e-4, size=u0.shape).astype(np.float32)
    return Workload("W2" if n == 256 else f"W2-{n}", n, n, n, tau, (0, 0, 1), (g_eff, 0.0, 0.0), [],
                    steps=1000, mdf_iters=0, u0=u0,
                    note="configs[1]: pure-LBM channel, Poiseuille + noise")


def w3(seed: int = 0, layers: int = 2) -> Workload:
    rng = np.random.default_rng(seed)
    axis = _random_unit(rng)
    psi0 = float(rng.uniform(0.0, 2.0 * np.pi))
    b = propeller(4, 40.0, 12.0, layers, psi0, axis, [64.0, 64.0, 64.0], 0.002)
    return Workload("W3" if layers == 2 else f"W3-L{layers}", 128, 128, 128, 0.7, (1, 1, 1),
                    (0.0, 0.0, 0.0), [b], steps=500, mdf_iters=5,
                    note="configs[2]: single dense propeller, walls on all faces")


def w4(seed: int = 0, layers: int = 8, n: int = 256) -> Workload:
    """configs[3]; n < 256 keeps the 64-cell pitch and shrinks the grid of propellers (n/64)^3."""
    rng = np.random.default_rng(seed)
    per = n // 64
    bodies = []
    for i in range(per):
        for j in range(per):
            for k in range(per):
                c = np.array([32.0 + 64 * i, 32.0 + 64 * j, 32.0 + 64 * k]) + rng.uniform(-2.0, 2.0, size=3)
                axis = _random_unit(rng)
                omega = float(rng.uniform(0.001, 0.004))
                psi0 = float(rng.uniform(0.0, 2.0 * np.pi))
                bodies.append(propeller(3, 24.0, 8.0, layers, psi0, axis, c, omega))
    name = "W4" if (layers == 8 and n == 256) else f"W4-L{layers}-{n}"
    return Workload(name, n, n, n, 0.7, (0, 0, 0), (0.0, 0.0, 0.0), bodies, steps=200, mdf_iters=5,
                    note="configs[3]: lattice of propellers, periodic")


def w5(seed: int = 0, layers: int = 12, n: int = 512, n_bodies: int | None = None) -> Workload:
    """configs[4]; n < 512 keeps the body number density (512 bodies per 512^3)."""
    rng = np.random.default_rng(seed)
    if n_bodies is None:
        n_bodies = max(1, int(round(512 * (n / 512.0) ** 3)))
    centers = []
    box = float(n)
    guard = 0
    while len(centers) < n_bodies:
        guard += 1
        if guard > 200000:
            raise RuntimeError("rejection sampling did not converge")
        c = rng.uniform(0.0, box, size=3)
        ok = True
        for d in centers:
            diff = np.abs(c - d)
            diff = np.minimum(diff, box - diff)
            if np.dot(diff, diff) < 30.0 * 30.0:
                ok = False
                break
        if ok:
            centers.append(c)
    bodies = []
    for c in centers:
        axis = _random_unit(rng)
        omega = float(rng.uniform(0.001, 0.004))
        psi0 = float(rng.uniform(0.0, 2.0 * np.pi))
        bodies.append(propeller(3, 20.0, 8.0, layers, psi0, axis, c, omega))
    name = "W5" if (layers == 12 and n == 512) else f"W5-L{layers}-{n}"
    return Workload(name, n, n, n, 0.65, (0, 0, 0), (0.0, 0.0, 0.0), bodies, steps=100, mdf_iters=5,
                    note="configs[4]: extreme density, periodic")


def paper_case(n_bodies: int, seed: int = 0) -> Workload:
    """the shape of the paper's own test cases: a 160 x 160 x 320 lattice
    with 1, 6 or 18 rotating propellers of about 3930 Lagrangian points each whose area is about one
    cell face (spacing 1, s = 1), 5 MDF iterations.  The paper's Blender mesh is not in the
    container: a three-blade flat-plate propeller (R = 41, w = 32: 3936 points) stands in for it; the
    bodies sit on the long axis of the box at equal distances, as in the paper's Fig. 4.  The paper
    states neither tau, omega nor the boundary: tau = 0.7, omega = 0.002, periodic (R15)."""
    rng = np.random.default_rng(seed)
    bodies = []
    for i in range(n_bodies):
        c = np.array([80.0, 80.0, 320.0 * (i + 0.5) / n_bodies])
        psi0 = float(rng.uniform(0.0, 2.0 * np.pi))
        bodies.append(propeller(3, 41.0, 32.0, 1, psi0, [0.0, 0.0, 1.0], c, 0.002 * (1 if i % 2 == 0 else -1), h=1.0))
    return Workload(f"P{n_bodies}", 160, 160, 320, 0.7, (0, 0, 0), (0.0, 0.0, 0.0), bodies, steps=1000, mdf_iters=5,
                    note="SURVEY 8(f3): paper-shaped case, 160x160x320, %d propellers x 3936 points" % n_bodies)


def get(name: str, seed: int = 0) -> Workload:
    """Named workloads: W1, W2, W3, W3lit, W3x4, W4, W4lit, W5, W5lit (lit = single layer, 'literal'; x4 = 8 layers);
    P1, P6, P18 = the paper-shaped cases of SURVEY 8(f3)."""
    table = {
        "W1": lambda: w1(seed),
        "W2": lambda: w2(seed),
        "W3": lambda: w3(seed, 2),
        "W3lit": lambda: w3(seed, 1),
        "W3x4": lambda: w3(seed, 8),        # the same propeller with four times the marker density (61,440 markers)
        "W4": lambda: w4(seed, 8),
        "W4lit": lambda: w4(seed, 1),
        "W5": lambda: w5(seed, 12),
        "W5lit": lambda: w5(seed, 1),
        "P1": lambda: paper_case(1, seed),
        "P6": lambda: paper_case(6, seed),
        "P18": lambda: paper_case(18, seed),
    }
    if name not in table:
        raise KeyError(f"unknown workload {name!r}; choose from {sorted(table)}")
    return table[name]()
