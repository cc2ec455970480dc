"""Seeded synthetic workloads (host, NumPy only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic (no force law, no Runge-Kutta, no observables): it only turns
uniform random numbers into initial conditions ``y0[12][N]`` and carries the physical
parameters of the five BASELINE.json configs.  It imports neither the CUDA binding
nor anything under ``oracle/``.

State layout (section 2.1): rows 0-2 ion position, 3-5 ion velocity,
6-8 atom position, 9-11 atom velocity; element (k, i) at offset k*N + i (SoA).

Generator recipe:
``U = Generator(PCG64(seed)).random((N, 10))``, row i <-> trajectory i, so any
prefix or slice of a larger run is reproducible (``offset`` uses PCG64.advance).
Only uniform doubles are drawn; every transform is explicit below.

Unit literals are the ones printed in the paper's Fig. 10 (PAPER.md:295-297, :322,
:341-342).
"""
from __future__ import annotations

import copy
import math
from dataclasses import dataclass, field

import numpy as np

# PAPER.md:295-297 (amu -> electron masses), :322 (k_B in Hartree/K), :341 (a.u. of time in s)
AMU = 1822.88848628276014097
KB = 3.16681156345647751469e-06
AU_TIME_S = 2.4188843265864e-17

DRAWS_PER_TRAJECTORY = 10


@dataclass
class Workload:
    """One BASELINE.json config: physical parameters + sampling recipe."""

    name: str
    N: int
    seed: int
    kind: str  # "thermal" (configs 0, 2-4) or "two_body" (config 1)
    # aig_params fields (paper's per-axis trap convention, eq. (4)-(6))
    m_ion: float
    m_atom: float
    C4: float
    C8: float
    a: tuple
    q: tuple
    omega_rf: float
    t0: float = 0.0
    r_exit: float = 5050.0
    r_turn: float = math.inf
    max_steps: int = 1_000_000
    # integration controls
    t_max: float = 2e11
    rtol: float = 1e-10
    atol: float = 1e-12
    # sampling
    T_ion: float = 0.5e-3
    T_atom: float = 1e-3
    R0: float = 5000.0
    b_max: float = 600.0
    E_coll: float = 0.0  # two_body only: fixed collision energy (Hartree)
    notes: dict = field(default_factory=dict)

    def params(self) -> dict:
        """Fields of ``aig_params`` / the oracle's parameter struct, as plain Python values."""
        return dict(m_ion=self.m_ion, m_atom=self.m_atom, C4=self.C4, C8=self.C8,
                    a=tuple(self.a), q=tuple(self.q), omega_rf=self.omega_rf, t0=self.t0,
                    r_exit=self.r_exit, r_turn=self.r_turn, max_steps=self.max_steps)

    def replace(self, **kw) -> "Workload":
        w = copy.deepcopy(self)
        for k, v in kw.items():
            if not hasattr(w, k):
                raise AttributeError(k)
            setattr(w, k, v)
        return w


def trap_axes(a: float, q: float):
    """BASELINE.json trap (x'' = -(W^2/4)(a - 2q cos Wt) x, same for y,
    z'' = +(W^2/2)(a - 2q cos Wt) z) in the paper's per-axis convention
    acc_k = -(a_k + 2 q_k cos Wt) W^2/4 x_k (eq. (4)-(6)):
    a[] = (a, a, -2a), q[] = (-q, -q, +2q)   (reading S2)."""
    return (a, a, -2.0 * a), (-q, -q, 2.0 * q)


def omega_from_mhz(f_mhz: float) -> float:
    """2*pi*f in atomic units of 1/time (OmegaRF = 2*pi*f*2.4188843265864e-17)."""
    return 2.0 * math.pi * f_mhz * 1e6 * AU_TIME_S


def potential_CnDe(n: int, m: int, Cn: float, De: float):
    """'CnDe' front-end of PAPER.md:428: given V = -Cn/r^n + Cm/r^m with well depth De,
    return (Cm, Re).  From V'(Re) = 0 and V(Re) = -De:
    Re^(m-n) = m Cm / (n Cn),  De = Cn (1 - n/m) / Re^n."""
    Re = (Cn * (1.0 - n / m) / De) ** (1.0 / n)
    Cm = n * Cn * Re ** (m - n) / m
    return Cm, Re


def potential_DeRe(n: int, m: int, De: float, Re: float):
    """'DeRe' front-end of PAPER.md:428: given the well depth De and the equilibrium distance Re of
    V = -Cn/r^n + Cm/r^m, return (Cn, Cm).  From V'(Re) = 0 and V(Re) = -De:
    Cn = De m Re^n / (m - n),  Cm = De n Re^m / (m - n)."""
    return De * m * Re ** n / (m - n), De * n * Re ** m / (m - n)


def config(i: int, **overrides) -> Workload:
    """The five BASELINE.json configs (index 0..4).  Config 4's sweep point is chosen with
    ``q=...``/``rtol=...`` overrides (atol follows as rtol*1e-2 unless given)."""
    omega = omega_from_mhz(2.0)
    if i in (0, 2, 4):
        a, q = trap_axes(0.0, 0.1)
        w = Workload(name=f"cfg{i}", N=256, seed=0, kind="thermal",
                     m_ion=138.0 * AMU, m_atom=87.0 * AMU, C4=159.5, C8=5.23e5,
                     a=a, q=q, omega_rf=omega)
        if i == 2:
            a, q = trap_axes(0.0, 0.2)
            w = w.replace(name="cfg2", N=65536, seed=2, a=a, q=q, T_atom=0.5e-3, rtol=1e-9)
        if i == 4:
            w = w.replace(name="cfg4", N=4194304, seed=4)
    elif i == 1:
        m_ion, m_atom = 138.0 * AMU, 87.0 * AMU
        E = KB * 1e-3
        C4 = 159.5
        w = Workload(name="cfg1", N=65536, seed=1, kind="two_body",
                     m_ion=m_ion, m_atom=m_atom, C4=C4, C8=5.23e5,
                     a=(0.0, 0.0, 0.0), q=(0.0, 0.0, 0.0), omega_rf=0.0,
                     T_ion=0.0, T_atom=0.0, E_coll=E,
                     b_max=1.5 * (2.0 * C4 / E) ** 0.25)  # DESIGN.md reading S13
    elif i == 3:
        a, q = trap_axes(0.001, 0.3)
        w = Workload(name="cfg3", N=1048576, seed=3, kind="thermal",
                     m_ion=174.0 * AMU, m_atom=7.0 * AMU, C4=82.0, C8=2.7e5,
                     a=a, q=q, omega_rf=omega, T_ion=0.1e-3, T_atom=0.1e-3,
                     b_max=400.0, t_max=1e12)
    else:
        raise ValueError("config index must be 0..4")
    if "q_trap" in overrides:  # scalar BASELINE-style q (config 4 sweep)
        qq = overrides.pop("q_trap")
        aa = overrides.pop("a_trap", 0.0 if i != 3 else 0.001)
        a, q = trap_axes(aa, qq)
        w = w.replace(a=a, q=q)
    if "rtol" in overrides and "atol" not in overrides and i == 4:
        overrides["atol"] = overrides["rtol"] * 1e-2
    return w.replace(**overrides) if overrides else w


def paper_workload(ntheta: int = 50, nphi: int = 50, theta=(0.0, math.pi / 2), phi=(0.0, math.pi / 2),
                   positions: str = "uniform", collisiontype: str = "head-on", **overrides) -> Workload:
    """NEXT-2: the paper's OWN workload (not a BASELINE.json config): Yb+ + Rb, the atom launched head-on
    at fixed speed v0 = sqrt(3 k_B T / m_a) from an equal-solid-angle (theta, phi) grid on the sphere
    r0 = 5000 a0 towards an ion at rest at the centre of a linear Paul trap, integrated for 1 ms with no
    exit radius (parameter listing Fig. 10 at :291-345).  Default grid: the
    50 x 50 first-octant benchmark of :102, :116.  The listing is partly garbled in the text
    (reading S28): taken here are
      m_ion 170.936323 amu, m_atom 86.9091805310 amu, T_atom 1 uK; potential 'CnDe' n = 4, m = 8,
      C4 = 159.5455, De = 1 K k_B  =>  C8 = 2.00949488627505e9, Re = 70.84 a0 (both printed);
      ax = ay = -2.982e-4, az = -2 ax, qx = 0.219, qy = -qx, qz = 0, Omega = 2 pi 2.5 MHz;
      tmax = 1000 us, maxsteps 1e6, rtol 1e-10, atol 1e-20.
    A radial minimum counts as a bounce inside r_turn = 500 a0 (the paper gives no formula).
    positions = "random": ntheta * nphi directions drawn uniformly in solid angle inside the
    (theta, phi) window instead of the grid.  collisiontype = "thermal": normal velocity
    components for atom (T_atom) and ion (T_ion = 10 uK, the listing's other temperature; reading S30) and a
    normal ion position of standard deviation sqrt(k_B T_ion / m_ion) / omega, omega = (Omega/2) sqrt(ax + qx^2/2)."""
    if positions not in ("uniform", "random") or collisiontype not in ("head-on", "thermal"):
        raise ValueError("positions: 'uniform' | 'random'; collisiontype: 'head-on' | 'thermal'")
    Cm, _Re = potential_CnDe(4, 8, 159.5455, 1.0 * KB)
    ax = -2.982e-4
    w = Workload(name="paper", N=int(ntheta) * int(nphi), seed=0, kind="grid",
                 m_ion=170.936323 * AMU, m_atom=86.9091805310 * AMU, C4=159.5455, C8=Cm,
                 a=(ax, ax, -2.0 * ax), q=(0.219, -0.219, 0.0), omega_rf=omega_from_mhz(2.5),
                 r_exit=0.0, r_turn=500.0, max_steps=1_000_000,
                 t_max=1000e-6 / AU_TIME_S, rtol=1e-10, atol=1e-20,
                 T_ion=10.0e-6 if collisiontype == "thermal" else 0.0, T_atom=1.0e-6, R0=5000.0, b_max=0.0,
                 notes=dict(ntheta=int(ntheta), nphi=int(nphi), theta=tuple(theta), phi=tuple(phi),
                            positions=positions, collisiontype=collisiontype))
    return w.replace(**overrides) if overrides else w


def uniforms(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """Rows [offset, offset+n) of the (N, 10) uniform matrix of stream ``seed``."""
    bg = np.random.PCG64(seed)
    if offset:
        bg.advance(offset * DRAWS_PER_TRAJECTORY)  # one 64-bit output per double
    return np.random.Generator(bg).random((n, DRAWS_PER_TRAJECTORY))


def generate_y0(w: Workload, n: int | None = None, offset: int = 0) -> np.ndarray:
    """Initial conditions ``y0[12][n]`` (float64, C-contiguous) for trajectories
    offset .. offset+n-1 of workload ``w`` (default: all ``w.N``)."""
    n = w.N if n is None else int(n)
    if w.kind == "grid":
        return _grid_y0(w, n, offset)
    U = uniforms(w.seed, n, offset)
    y0 = np.zeros((12, n), dtype=np.float64)
    two_pi = 2.0 * math.pi

    # isotropic approach direction and the two unit vectors spanning the impact plane
    ct = 1.0 - 2.0 * U[:, 4]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = two_pi * U[:, 5]
    cp, sp = np.cos(ph), np.sin(ph)
    nhat = np.stack([st * cp, st * sp, ct])
    e1 = np.stack([ct * cp, ct * sp, -st])
    e2 = np.stack([-sp, cp, np.zeros(n)])
    b = w.b_max * np.sqrt(U[:, 6])
    psi = two_pi * U[:, 7]
    rel = np.sqrt(w.R0 * w.R0 - b * b) * nhat + b * (np.cos(psi) * e1 + np.sin(psi) * e2)

    if w.kind == "thermal":
        # ion at the trap centre, Maxwell-Boltzmann velocity (Box-Muller on explicit uniforms)
        s_i = math.sqrt(KB * w.T_ion / w.m_ion)
        r01 = s_i * np.sqrt(-2.0 * np.log1p(-U[:, 0]))
        y0[3] = r01 * np.cos(two_pi * U[:, 1])
        y0[4] = r01 * np.sin(two_pi * U[:, 1])
        y0[5] = s_i * np.sqrt(-2.0 * np.log1p(-U[:, 2])) * np.cos(two_pi * U[:, 3])
        # atom on the sphere of radius R0 about the ion, flux-weighted speed pdf ~ v^3 exp(-m v^2/2kT)
        s_a = math.sqrt(KB * w.T_atom / w.m_atom)
        v = s_a * np.sqrt(-2.0 * (np.log1p(-U[:, 8]) + np.log1p(-U[:, 9])))
        y0[6:9] = rel
        y0[9:12] = -v * nhat
    elif w.kind == "two_body":
        # fixed collision energy E = mu v^2 / 2 (v = relative speed), centre-of-mass frame:
        # total momentum and centre of mass are both zero (reading S16).
        M = w.m_ion + w.m_atom
        mu = w.m_ion * w.m_atom / M
        v = math.sqrt(2.0 * w.E_coll / mu)
        vrel = -v * nhat  # atom velocity minus ion velocity
        y0[0:3] = -(w.m_atom / M) * rel
        y0[3:6] = -(w.m_atom / M) * vrel
        y0[6:9] = (w.m_ion / M) * rel
        y0[9:12] = (w.m_ion / M) * vrel
    else:
        raise ValueError(w.kind)
    return np.ascontiguousarray(y0)


def grid_angles(w: Workload):
    """(theta[ntheta], phi[nphi]) of a "grid" workload (positions = "uniform"): nphi evenly
    spaced phi between phimin and phimax; theta = arccos(1 - 2u) with ntheta evenly spaced u between
    (1 - cos thetamin)/2 and (1 - cos thetamax)/2, so that every (theta, phi) occupies the same solid angle."""
    nt, nph = w.notes["ntheta"], w.notes["nphi"]
    (t0, t1), (p0, p1) = w.notes["theta"], w.notes["phi"]
    u = np.linspace((1.0 - math.cos(t0)) / 2.0, (1.0 - math.cos(t1)) / 2.0, nt)
    return np.arccos(1.0 - 2.0 * u), np.linspace(p0, p1, nph)


def map_edges(w: Workload, n_u: int | None = None, n_phi: int | None = None):
    """Cell edges (u_edges, phi_edges) for a map of an observable against the launch direction (aig_map2d) over the
    (theta, phi) window of a "grid" workload, u = (1 - cos theta)/2.  Defaults: one cell per grid direction, edges
    half-way between neighbouring directions (the outer ones half a spacing beyond the window), so that on a
    "uniform" grid the map is the value array reshaped; for random directions pass the cell counts: equal steps of u
    (equal solid angles) and of phi inside the window."""
    (t0, t1), (p0, p1) = w.notes["theta"], w.notes["phi"]
    u0, u1 = (1.0 - math.cos(t0)) / 2.0, (1.0 - math.cos(t1)) / 2.0
    if n_u is None and n_phi is None:
        nt, nph = w.notes["ntheta"], w.notes["nphi"]
        du = (u1 - u0) / max(nt - 1, 1)
        dp = (p1 - p0) / max(nph - 1, 1)
        return (u0 - du / 2 + du * np.arange(nt + 1), p0 - dp / 2 + dp * np.arange(nph + 1))
    return np.linspace(u0, u1, int(n_u) + 1), np.linspace(p0, p1, int(n_phi) + 1)


PAPER_DRAWS = 16  # uniforms per trajectory of a "grid" workload: 0-1 direction, 2-15 seven Box-Muller pairs


def secular_frequency(w: Workload) -> float:
    """omega = (Omega_rf / 2) sqrt(a_x + q_x^2 / 2): "the trap's secular frequency in the x direction"."""
    return 0.5 * w.omega_rf * math.sqrt(w.a[0] + 0.5 * w.q[0] ** 2)


def _paper_uniforms(seed: int, n: int, offset: int) -> np.ndarray:
    bg = np.random.PCG64(seed)
    if offset:
        bg.advance(offset * PAPER_DRAWS)
    return np.random.Generator(bg).random((n, PAPER_DRAWS))


def _grid_y0(w: Workload, n: int, offset: int) -> np.ndarray:
    """eq. (12)-(13): atom at r0 (sin th cos ph, sin th sin ph, cos th) with velocity
    -v0 times the same unit vector, v0 = sqrt(3 k_B T / m_a); ion at rest at the origin.  Trajectory
    i <-> (theta index i // nphi, phi index i % nphi).  notes["positions"] = "random" draws the directions
    (PAPER.md:483), notes["collisiontype"] = "thermal" the velocities and the ion position."""
    positions = w.notes.get("positions", "uniform")
    thermal = w.notes.get("collisiontype", "head-on") == "thermal"
    U = _paper_uniforms(w.seed, n, offset) if (thermal or positions == "random") else None
    if positions == "random":
        (t0, t1), (p0, p1) = w.notes["theta"], w.notes["phi"]
        u0, u1 = (1.0 - math.cos(t0)) / 2.0, (1.0 - math.cos(t1)) / 2.0
        t = np.arccos(1.0 - 2.0 * (u0 + (u1 - u0) * U[:, 0]))
        f = p0 + (p1 - p0) * U[:, 1]
    else:
        th, ph = grid_angles(w)
        idx = np.arange(offset, offset + n)
        t, f = th[idx // len(ph)], ph[idx % len(ph)]
    nhat = np.stack([np.sin(t) * np.cos(f), np.sin(t) * np.sin(f), np.cos(t)])
    y0 = np.zeros((12, n), dtype=np.float64)
    y0[6:9] = w.R0 * nhat
    if not thermal:
        v0 = math.sqrt(3.0 * KB * w.T_atom / w.m_atom)
        y0[9:12] = -v0 * nhat
        return np.ascontiguousarray(y0)
    # nine standard normals per trajectory: Box-Muller on explicit uniforms (pairs (2+2j, 3+2j))
    two_pi = 2.0 * math.pi
    rad = np.sqrt(-2.0 * np.log1p(-U[:, 2::2]))      # [n, 7]
    ang = two_pi * U[:, 3::2]
    z = np.concatenate([rad * np.cos(ang), rad * np.sin(ang)], axis=1)   # [n, 14] independent N(0, 1)
    s_a = math.sqrt(KB * w.T_atom / w.m_atom)
    s_i = math.sqrt(KB * w.T_ion / w.m_ion)
    y0[9:12] = s_a * z[:, 0:3].T
    y0[3:6] = s_i * z[:, 3:6].T
    y0[0:3] = (s_i / secular_frequency(w)) * z[:, 6:9].T
    return np.ascontiguousarray(y0)


def impact_parameters(w: Workload, n: int | None = None, offset: int = 0) -> np.ndarray:
    """The impact parameters b_i the generator used (for the Langevin / quadrature checks)."""
    n = w.N if n is None else int(n)
    return w.b_max * np.sqrt(uniforms(w.seed, n, offset)[:, 6])


def shard_range(N: int, rank: int, world: int):
    """Contiguous index range [lo, hi) of trajectories owned by ``rank`` (paper: trajectories
    'distributed evenly across the ncores cores')."""
    base, rem = divmod(int(N), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def histogram_edges(n_angle: int = 180, n_life: int = 120, life_lo: float = 1e6, life_hi: float = 1e12):
    """Default bin edges (SURVEY.md 8(d) 'Histogram spec'): angle uniform on [0, pi],
    lifetime log-uniform on [life_lo, life_hi] atomic units of time."""
    angle_edges = np.linspace(0.0, math.pi, n_angle + 1)
    life_edges = np.logspace(math.log10(life_lo), math.log10(life_hi), n_life + 1)
    return np.ascontiguousarray(angle_edges), np.ascontiguousarray(life_edges)
