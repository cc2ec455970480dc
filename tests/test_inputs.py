"""Seeded input generator: structure of the synthetic workloads (no GPU)."""
import math

import numpy as np
import pytest

from paper_2509_12381_b200 import inputs


def test_configs_match_baseline_json():
    Ns = [256, 65536, 65536, 1048576, 4194304]
    for i in range(5):
        w = inputs.config(i)
        assert w.N == Ns[i] and w.seed == i
    w0 = inputs.config(0)
    assert w0.m_ion == 138 * inputs.AMU and w0.m_atom == 87 * inputs.AMU
    assert (w0.C4, w0.C8, w0.t_max, w0.rtol, w0.atol) == (159.5, 5.23e5, 2e11, 1e-10, 1e-12)
    assert w0.r_exit == 1.01 * w0.R0
    # BASELINE trap -> paper's per-axis convention; Laplace: sum a = sum q = 0
    assert w0.a == (0.0, 0.0, -0.0) and w0.q == (-0.1, -0.1, 0.2)
    w3 = inputs.config(3)
    assert abs(sum(w3.a)) < 1e-18 and abs(sum(w3.q)) < 1e-18 and w3.q[2] == 0.6 and w3.a[2] == -0.002
    assert abs(w0.omega_rf - 2 * math.pi * 2e6 * 2.4188843265864e-17) < 1e-25
    w1 = inputs.config(1)
    assert w1.omega_rf == 0 and abs(w1.b_max - 845.05) < 0.01
    w4 = inputs.config(4, q_trap=0.4, rtol=1e-12)
    assert w4.q == (-0.4, -0.4, 0.8) and w4.atol == 1e-14 and w4.N == 4194304
    assert inputs.config(2).rtol == 1e-9 and inputs.config(2).T_atom == 0.5e-3


def test_thermal_generator_geometry_and_statistics():
    w = inputs.config(0)
    n = 20000
    y0 = inputs.generate_y0(w, n=n)
    assert y0.shape == (12, n) and y0.flags.c_contiguous and y0.dtype == np.float64
    assert np.all(y0[0:3] == 0)
    rel = y0[6:9]
    assert np.allclose(np.linalg.norm(rel, axis=0), w.R0, rtol=1e-14)
    v = y0[9:12]
    speed = np.linalg.norm(v, axis=0)
    nhat = -v / speed
    # impact parameter = |rel - (rel.n) n| and equals the generator's b; uniform in area
    b = np.linalg.norm(rel - (rel * nhat).sum(0) * nhat, axis=0)
    assert np.allclose(b, inputs.impact_parameters(w, n=n), rtol=1e-9, atol=1e-9)
    assert abs((b**2).mean() / (w.b_max**2 / 2) - 1) < 0.02 and b.max() <= w.b_max
    # isotropic directions
    assert np.all(np.abs(nhat.mean(axis=1)) < 0.02) and abs((nhat[2] ** 2).mean() - 1 / 3) < 0.01
    # flux-weighted speed: <v^2> = 4 kT/m ; ion Maxwell-Boltzmann: <v_k^2> = kT/m
    assert abs((speed**2).mean() / (4 * inputs.KB * w.T_atom / w.m_atom) - 1) < 0.03
    for k in range(3):
        assert abs((y0[3 + k] ** 2).mean() / (inputs.KB * w.T_ion / w.m_ion) - 1) < 0.04
    # atom moves toward the ion: radial velocity negative
    assert np.all((rel * v).sum(0) < 0)


def test_two_body_generator_cm_frame():
    w = inputs.config(1)
    y0 = inputs.generate_y0(w, n=1000)
    P = w.m_ion * y0[3:6] + w.m_atom * y0[9:12]
    R = w.m_ion * y0[0:3] + w.m_atom * y0[6:9]
    mu = w.m_ion * w.m_atom / (w.m_ion + w.m_atom)
    vrel = y0[9:12] - y0[3:6]
    assert np.max(np.abs(P)) < 1e-12 * mu * 2.6e-7 * 100 and np.max(np.abs(R)) < 1e-9 * w.m_ion
    assert np.allclose(0.5 * mu * (vrel**2).sum(0), inputs.KB * 1e-3, rtol=1e-13)
    assert np.allclose(np.linalg.norm(y0[6:9] - y0[0:3], axis=0), w.R0, rtol=1e-14)
    assert abs(math.sqrt(2 * w.E_coll / mu) - 2.5518e-7) < 1e-10


def test_prefix_and_offset_reproducibility_and_sharding():
    w = inputs.config(4)
    full = inputs.generate_y0(w, n=300)
    assert np.array_equal(inputs.generate_y0(w, n=100), full[:, :100])
    assert np.array_equal(inputs.generate_y0(w, n=120, offset=57), full[:, 57:177])
    for N, world in ((10, 3), (4194304, 8), (7, 8)):
        spans = [inputs.shard_range(N, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == N
        assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
        sizes = [hi - lo for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1


def test_potential_front_ends_are_consistent():
    """'CnCm', 'CnDe', 'DeRe' describe the same V = -Cn/r^n + Cm/r^m."""
    for n, m, De, Re in ((4, 8, 0.012, 9.0), (6, 12, 3e-4, 12.0), (3, 9, 0.5, 2.5)):
        Cn, Cm = inputs.potential_DeRe(n, m, De, Re)
        V = lambda r: -Cn / r ** n + Cm / r ** m
        assert abs(V(Re) + De) <= 1e-14 * De                       # depth
        h = 1e-5 * Re
        assert abs(V(Re + h) - V(Re - h)) <= 1e-9 * De             # minimum at Re
        Cm2, Re2 = inputs.potential_CnDe(n, m, Cn, De)             # and back through 'CnDe'
        assert abs(Cm2 / Cm - 1) <= 1e-13 and abs(Re2 / Re - 1) <= 1e-13


def test_paper_grid_workload():
    """NEXT-2: head-on launch from an equal-solid-angle grid."""
    w = inputs.paper_workload(ntheta=40, nphi=30)
    y0 = inputs.generate_y0(w)
    assert y0.shape == (12, 1200) and np.all(y0[0:6] == 0)                  # ion at rest at the origin
    r = np.linalg.norm(y0[6:9], axis=0)
    v = np.linalg.norm(y0[9:12], axis=0)
    assert np.allclose(r, 5000.0, rtol=1e-15)
    assert np.allclose(v, math.sqrt(3 * inputs.KB * 1e-6 / w.m_atom), rtol=1e-15)
    assert np.allclose(y0[9:12] / v, -y0[6:9] / r, atol=1e-15)              # head-on
    th, ph = inputs.grid_angles(w)
    assert np.allclose(np.diff(np.cos(th)), np.diff(np.cos(th))[0])         # equal steps in cos(theta): equal solid angle
    assert np.allclose(np.diff(ph), np.diff(ph)[0]) and th[0] == 0 and abs(th[-1] - math.pi / 2) < 1e-12
    assert np.array_equal(inputs.generate_y0(w, n=7, offset=95), y0[:, 95:102])   # slices reproduce
    # the paper's printed derived constants (Fig. 10): Cm and tmax
    assert abs(w.C8 / 2.00949488627505397797e+09 - 1) < 1e-13
    assert abs(w.t_max * inputs.AU_TIME_S - 1e-3) < 1e-15


def test_paper_random_positions_and_thermal_mode():
    """NEXT-2, PAPER.md:483 ("random" positions: uniform in solid angle inside the window) and :282
    ("thermal": normal velocity components of standard deviation sqrt(k_B T / m), normal ion position of
    standard deviation sqrt(k_B T_ion / m_ion) / omega, omega = (Omega/2) sqrt(ax + qx^2/2))."""
    n_t, n_p = 200, 200
    w = inputs.paper_workload(n_t, n_p, theta=(0.3, 2.0), phi=(0.5, 4.0), positions="random", collisiontype="thermal")
    y0 = inputs.generate_y0(w)
    n = n_t * n_p
    assert y0.shape == (12, n)
    r = np.linalg.norm(y0[6:9], axis=0)
    assert np.allclose(r, 5000.0, rtol=1e-14)
    cth = y0[8] / r
    phi = np.mod(np.arctan2(y0[7], y0[6]), 2 * math.pi)
    assert cth.min() >= math.cos(2.0) - 1e-12 and cth.max() <= math.cos(0.3) + 1e-12
    assert phi.min() >= 0.5 - 1e-12 and phi.max() <= 4.0 + 1e-12
    # uniform in solid angle: cos(theta) and phi uniform on their windows (Kolmogorov-Smirnov)
    from scipy import stats
    assert stats.kstest(cth, stats.uniform(math.cos(2.0), math.cos(0.3) - math.cos(2.0)).cdf).pvalue > 1e-3
    assert stats.kstest(phi, stats.uniform(0.5, 3.5).cdf).pvalue > 1e-3
    # the nine normal components: zero mean, the stated standard deviations, uncorrelated
    s_a = math.sqrt(inputs.KB * 1.0e-6 / w.m_atom)
    s_i = math.sqrt(inputs.KB * 10.0e-6 / w.m_ion)
    om = 0.5 * (2 * math.pi * 2.5e6 * inputs.AU_TIME_S) * math.sqrt(-2.982e-4 + 0.5 * 0.219 ** 2)
    assert abs(inputs.secular_frequency(w) / om - 1) < 1e-12
    assert abs(om / inputs.AU_TIME_S / (2 * math.pi) / 192.36e3 - 1) < 1e-3      # ~192 kHz for the listing's trap
    Z = np.vstack([y0[9:12] / s_a, y0[3:6] / s_i, y0[0:3] / (s_i / om)])
    tol = 5.0 / math.sqrt(n)
    assert np.max(np.abs(Z.mean(axis=1))) < tol
    assert np.max(np.abs(Z.std(axis=1) - 1)) < tol
    Cc = np.corrcoef(Z)
    assert np.max(np.abs(Cc - np.eye(9))) < tol
    for k in range(9):
        assert stats.kstest(Z[k], "norm").pvalue > 1e-4, k
    # slices of the stream reproduce (sharding), head-on grid unchanged by the new arguments
    assert np.array_equal(inputs.generate_y0(w, n=9, offset=1234), y0[:, 1234:1243])
    g0 = inputs.generate_y0(inputs.paper_workload(12, 7))
    g1 = inputs.generate_y0(inputs.paper_workload(12, 7, positions="uniform", collisiontype="head-on"))
    assert np.array_equal(g0, g1) and np.all(g0[0:6] == 0)
    # mixed modes: grid directions with thermal velocities; random directions head-on
    gt = inputs.generate_y0(inputs.paper_workload(12, 7, collisiontype="thermal"))
    assert np.array_equal(gt[6:9], g0[6:9]) and np.all(gt[0:6] != 0)
    rh = inputs.generate_y0(inputs.paper_workload(12, 7, positions="random"))
    v = np.linalg.norm(rh[9:12], axis=0)
    assert np.all(rh[0:6] == 0) and np.allclose(rh[9:12] / v, -rh[6:9] / 5000.0, atol=1e-15)
    with pytest.raises(ValueError):
        inputs.paper_workload(4, 4, positions="grid")
