"""Seeded synthetic workloads (BASELINE.json configs 1-5) for BOTH the CUDA path and the CPU oracle.

This module holds none of the method's arithmetic: no dispersion function, no ray equations, no spline
fitting.  It draws launch positions and unit directions from ``numpy.random.default_rng`` and writes down
the equilibrium descriptors (numbers and, for config 5, nodal arrays).  Turning a direction into an
on-shell wave vector k0 is the method's job: ``rt_launch`` in the library, ``oracle.launch``
in the oracle.  numpy only; imports neither the binding nor the oracle.

The workloads stand in for the paper's "1e6 rays in a realistic tokamak equilibrium", whose
equilibrium file is not available; recipe and draw order are stated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# CODATA-2022 numerals (reading A6) -- a table of values, used here only to express the
# config texts' "wpe^2/w^2 = 0.5 ..." as a reference density.
C_LIGHT = 299792458.0
Q_E = 1.602176634e-19
M_E = 9.1093837139e-31
M_D = 3.3435837768e-27
EPS0 = 8.8541878188e-12

GHZ = 2.0 * np.pi * 1e9


@dataclass
class Workload:
    name: str
    eq: dict                    # equilibrium descriptor: plain numbers (+ nodal arrays for grid_rz)
    disp: str                   # 'omode' | 'xmode' | 'cold_full'
    branch: int                 # root selector for the launch solve (0 = "O", 1 = "X"); reading A11
    omega: float                # rad/s
    x0: np.ndarray              # [3, n_rays] launch positions, m
    dirs: np.ndarray            # [3, n_rays] unit launch directions
    dt: float                   # step in tau = c t, metres (reading A3)
    n_steps: int
    save_stride: int            # 0 = final state only
    precisions: tuple = ("f64",)
    seed: int = 0
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_rays(self) -> int:
        return int(self.x0.shape[1])


def _deg(a):
    return np.deg2rad(a)


def parabolic_slab(n_rays: int, n_steps: int, seed: int, save_stride: int, precisions, name: str) -> Workload:
    """Configs 1-2: unmagnetised O-mode, X_e = 0.5 (1 + (x^2+y^2)/L^2), L = 1 m, 110 GHz (reading A13)."""
    rng = np.random.default_rng(seed)
    y0 = rng.uniform(-0.2, 0.2, n_rays)                    # all y0 first,
    th = _deg(rng.uniform(-20.0, 20.0, n_rays))            # then all angles
    x0 = np.stack([np.full(n_rays, -0.5), y0, np.zeros(n_rays)])
    dirs = np.stack([np.cos(th), np.sin(th), np.zeros(n_rays)])
    omega = 110.0 * GHZ
    n_ref = 0.5 * EPS0 * M_E * omega**2 / Q_E**2           # density at which wpe^2/w^2 = 0.5
    eq = dict(kind="slab_parabolic", n_ref=n_ref, L=1.0, ion_mass=0.0, ion_charge=0.0)
    return Workload(name, eq, "omode", 0, omega, x0, dirs, 1e-3, n_steps, save_stride, tuple(precisions), seed)


def linear_slab(n_rays: int, n_steps: int, seed: int) -> Workload:
    """Config 3: X-mode, e + D, B = B0 R0 / x z^, density ramp 0 -> 5e19 over 0.5 m; launched at the foot (A8)."""
    rng = np.random.default_rng(seed)
    y0 = rng.uniform(-0.2, 0.2, n_rays)
    th = _deg(rng.uniform(-20.0, 20.0, n_rays))
    x0 = np.stack([np.full(n_rays, 2.3), y0, np.zeros(n_rays)])
    dirs = np.stack([-np.cos(th), np.sin(th), np.zeros(n_rays)])
    eq = dict(kind="slab_linear_br", n_ref=5e19, x_foot=2.3, L_ramp=0.5, B0=2.0, R0=1.7,
              ion_mass=M_D, ion_charge=1.0)
    return Workload("cfg3_xmode_linear_slab", eq, "xmode", 0, 60.0 * GHZ, x0, dirs, 2.5e-4, n_steps, 0,
                    ("f64",), seed)


TOKAMAK = dict(R0=1.7, a=0.6, B0=2.0, q0=1.0, q1=2.0, n_ref=5e19, p_exp=1.5, rho_max=0.98,
               ion_mass=M_D, ion_charge=1.0)


def tokamak_launch(rng, n_rays: int, R0: float, a: float, rho0: float = 0.95):
    """Reading A11: points on the outboard side at rho0, directions steered about the inward minor-radius
    normal.  Draw order: theta_p, phi, alpha, beta (each a full array)."""
    thp = _deg(rng.uniform(-30.0, 30.0, n_rays))
    phi = rng.uniform(0.0, 2.0 * np.pi, n_rays)
    al = _deg(rng.uniform(-20.0, 20.0, n_rays))
    be = _deg(rng.uniform(-20.0, 20.0, n_rays))
    R = R0 + rho0 * a * np.cos(thp)
    Z = rho0 * a * np.sin(thp)
    x0 = np.stack([R * np.cos(phi), R * np.sin(phi), Z])
    dR = -np.cos(thp + al) * np.cos(be)
    dphi = np.sin(be)
    dZ = -np.sin(thp + al) * np.cos(be)
    dirs = np.stack([dR * np.cos(phi) - dphi * np.sin(phi), dR * np.sin(phi) + dphi * np.cos(phi), dZ])
    return x0, dirs


def tokamak_analytic(n_rays: int, n_steps: int, seed: int, save_stride: int = 10) -> Workload:
    """Config 4: full Stix determinant, analytic circular tokamak, 110 GHz, O-mode launch."""
    rng = np.random.default_rng(seed)
    x0, dirs = tokamak_launch(rng, n_rays, TOKAMAK["R0"], TOKAMAK["a"])
    eq = dict(kind="tokamak_circular", **TOKAMAK)
    return Workload("cfg4_cold_full_tokamak", eq, "cold_full", 0, 110.0 * GHZ, x0, dirs, 1e-3, n_steps,
                    save_stride, ("f64",), seed)


def synth_grid(seed: int, eps: float = 1e-3, nR: int = 257, nZ: int = 257, nPsi: int = 257) -> dict:
    """Config 5's nodal data: the analytic case of config 4 sampled on an R-Z grid, times (1 + eps * a
    seed-drawn low-order Fourier perturbation).  Draw order: a_pq, b_pq (15 each, row-major (p,q) without
    (0,0)), then a,b (3 each) for F, then a,b (3 each) for n_e."""
    t = TOKAMAK
    R0, a, B0 = t["R0"], t["a"], t["B0"]
    rng = np.random.default_rng(seed)
    apq, bpq = rng.uniform(-1, 1, 15), rng.uniform(-1, 1, 15)
    aF, bF = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
    an, bn = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
    Rmin, Rmax, Zmin, Zmax = R0 - 1.25 * a, R0 + 1.25 * a, -1.25 * a, 1.25 * a
    R = Rmin + np.arange(nR) * ((Rmax - Rmin) / (nR - 1))
    Z = Zmin + np.arange(nZ) * ((Zmax - Zmin) / (nZ - 1))
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    rho2 = ((RR - R0) ** 2 + ZZ**2) / a**2
    psi = 0.25 * B0 * a**2 * np.log1p(2.0 * rho2)
    u = (RR - Rmin) / (Rmax - Rmin)
    v = (ZZ - Zmin) / (Zmax - Zmin)
    P = np.zeros_like(psi)
    m = 0
    for p in range(4):
        for q in range(4):
            if p == 0 and q == 0:
                continue
            ph = 2.0 * np.pi * (p * u + q * v)
            P += apq[m] * np.cos(ph) + bpq[m] * np.sin(ph)
            m += 1
    psi = psi * (1.0 + eps * P / 15.0)
    psi_edge = 0.25 * B0 * a**2 * np.log(3.0)
    s = np.arange(nPsi) / (nPsi - 1)
    pF = sum(aF[j] * np.cos(2 * np.pi * (j + 1) * s) + bF[j] * np.sin(2 * np.pi * (j + 1) * s) for j in range(3)) / 3.0
    pn = sum(an[j] * np.cos(2 * np.pi * (j + 1) * s) + bn[j] * np.sin(2 * np.pi * (j + 1) * s) for j in range(3)) / 3.0
    F = B0 * R0 * (1.0 + eps * pF)
    rho2_s = np.clip(0.5 * np.expm1(4.0 * s * psi_edge / (B0 * a**2)), 0.0, 1.0)
    ne = t["n_ref"] * (1.0 - rho2_s) ** t["p_exp"] * (1.0 + eps * pn)
    return dict(kind="grid_rz", nR=nR, nZ=nZ, nPsi=nPsi, Rmin=Rmin, Rmax=Rmax, Zmin=Zmin, Zmax=Zmax,
                psi_min=0.0, psi_max=psi_edge, psi_RZ=np.ascontiguousarray(psi), F_psi=np.ascontiguousarray(F),
                ne_psi=np.ascontiguousarray(ne), R0=R0, a=a, B0=B0, ion_mass=t["ion_mass"],
                ion_charge=t["ion_charge"])


def tokamak_grid(n_rays: int, n_steps: int, seed: int, eps: float = 1e-3, precisions=("f64", "f32")) -> Workload:
    """Config 5: as config 4 but psi(R,Z), F(psi), n_e(psi) come from bicubic / cubic splines of nodal data."""
    eq = synth_grid(seed, eps)
    rng = np.random.default_rng(seed + 500000)             # launch stream separate from the grid's
    x0, dirs = tokamak_launch(rng, n_rays, TOKAMAK["R0"], TOKAMAK["a"])
    return Workload("cfg5_cold_full_grid", eq, "cold_full", 0, 110.0 * GHZ, x0, dirs, 1e-3, n_steps, 0,
                    tuple(precisions), seed, extra=dict(eps=eps))


def frequency_scan(n_rays: int, omega0: float, seed: int, spread: float = 0.1) -> np.ndarray:
    """One wave frequency per ray, w_i = omega0 (1 + spread u_i), u_i ~ U[-1, 1] (frequency scans;
    PAPER.md L147: w is a per-ray kernel input).  Drawn from its own stream ``default_rng(seed + 900000)``."""
    rng = np.random.default_rng(seed + 900000)
    return omega0 * (1.0 + spread * rng.uniform(-1.0, 1.0, n_rays))


@dataclass
class OrbitWorkload:
    name: str
    eq: dict
    charge_over_mass: float     # C/kg
    x0: np.ndarray              # [3, n] launch positions, m
    v0: np.ndarray              # [3, n] launch velocities, m/s
    dt: float                   # s
    n_steps: int
    save_stride: int            # 0 = final state only
    seed: int = 0

    @property
    def n(self) -> int:
        return int(self.x0.shape[1])


ORBIT_FULL_SIZE = (2**20, 1000)


def orbit_config(eq_cfg: int = 4, n: int | None = None, n_steps: int | None = None, seed: int | None = None,
                 energy_keV: float = 10.0) -> OrbitWorkload:
    """The second ensemble workload (PAPER.md L121 / L213): deuterons of `energy_keV` on full orbits in
    the equilibrium of config `eq_cfg` (3: the B0 R0/x slab, 4: analytic tokamak, 5: spline grid).  2^20 particles x
    1000 steps of dt = 1 ns (about 66 steps per gyration at 2 T), trajectories every 10 steps like config 4.
    Draw order (``default_rng(2000 + eq_cfg)``), whole arrays: rho, theta_p, phi (positions: rho ~ U[0.1, 0.8] a;
    slab: x ~ U[1.9, 2.2], y ~ U[-0.2, 0.2], z ~ U[-0.2, 0.2] in the same three draws), then cos(pitch) ~ U[-1, 1] and
    gyro-angle ~ U[0, 2 pi) (isotropic directions about z^)."""
    nn, ns = ORBIT_FULL_SIZE
    n = nn if n is None else int(n)
    n_steps = ns if n_steps is None else int(n_steps)
    seed = 2000 + eq_cfg if seed is None else int(seed)
    rng = np.random.default_rng(seed)
    a1, a2, a3 = rng.uniform(0.0, 1.0, n), rng.uniform(0.0, 1.0, n), rng.uniform(0.0, 1.0, n)
    cp = rng.uniform(-1.0, 1.0, n)
    ga = rng.uniform(0.0, 2.0 * np.pi, n)
    if eq_cfg == 3:
        eq = linear_slab(1, 1, 0).eq
        x0 = np.stack([1.9 + 0.3 * a1, -0.2 + 0.4 * a2, -0.2 + 0.4 * a3])
    elif eq_cfg in (4, 5):
        t = TOKAMAK
        eq = dict(kind="tokamak_circular", **t) if eq_cfg == 4 else synth_grid(1005)
        rho, thp, phi = (0.1 + 0.7 * a1) * t["a"], 2.0 * np.pi * a2, 2.0 * np.pi * a3
        R, Z = t["R0"] + rho * np.cos(thp), rho * np.sin(thp)
        x0 = np.stack([R * np.cos(phi), R * np.sin(phi), Z])
    else:
        raise ValueError("orbit workloads exist on the equilibria of configs 3, 4 and 5")
    speed = np.sqrt(2.0 * energy_keV * 1e3 * Q_E / M_D)
    sp = np.sqrt(1.0 - cp * cp)
    v0 = speed * np.stack([sp * np.cos(ga), sp * np.sin(ga), cp])
    return OrbitWorkload(f"orbits_D_{energy_keV:g}keV_on_cfg{eq_cfg}", eq, Q_E / M_D, x0, v0, 1e-9, n_steps, 10, seed)


# (n_rays, n_steps) of BASELINE.json's configs 1..5
FULL_SIZES = {1: (1024, 1000), 2: (2**20, 2000), 3: (2**18, 3000), 4: (2**20, 1000), 5: (2**24, 500)}


def config(k: int, n_rays: int | None = None, n_steps: int | None = None, seed: int | None = None) -> Workload:
    """BASELINE.json config k (1..5); n_rays / n_steps override the full size (tests use small slices);
    seed defaults to 1000 + k (reading A17)."""
    nr, ns = FULL_SIZES[k]
    n_rays = nr if n_rays is None else int(n_rays)
    n_steps = ns if n_steps is None else int(n_steps)
    seed = 1000 + k if seed is None else int(seed)
    if k == 1:
        return parabolic_slab(n_rays, n_steps, seed, 1, ("f64",), "cfg1_omode_parabolic_traj")
    if k == 2:
        return parabolic_slab(n_rays, n_steps, seed, 0, ("f64", "f32"), "cfg2_omode_parabolic_final")
    if k == 3:
        return linear_slab(n_rays, n_steps, seed)
    if k == 4:
        return tokamak_analytic(n_rays, n_steps, seed)
    if k == 5:
        return tokamak_grid(n_rays, n_steps, seed)
    raise ValueError(f"no config {k}")
