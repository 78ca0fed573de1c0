"""Pins for the CPU oracle (no GPU): the oracle is checked against what the paper and the mathematics
fix -- known-answer vectors, closed forms, invariants, brute force -- never against itself.

Pin numbers follow SURVEY.md section 8(c) / DESIGN.md "Pins".
"""
import math
import os

import numpy as np
import pytest
from scipy import special

from paper_1203_2941_b200 import workloads as W

H_PLANCK, K_BOLTZ, C_LIGHT, SIGMA_SB = 6.62607015e-27, 1.380649e-16, 2.99792458e10, 5.670374419e-5
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
NTH = min(8, os.cpu_count() or 1)


# ------------------------------------------------------------------------------------------ P1 RNG
def test_p1_philox_known_answers(orc):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = orc.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_p1_uniform_mapping(orc):
    # zeta = (2*u52+1)/2^53 from the block's words; strictly inside (0,1); counter layout (pid lo, pid hi, d, pass)
    for seed, pid, d, pas in [(1, 0, 0, 0), (2 ** 40 + 5, 2 ** 33 + 7, 11, 3), (0xFFFFFFFFFFFFFFFF, 12345, 2 ** 31, 1)]:
        w = orc.philox([pid & 0xFFFFFFFF, pid >> 32, d, pas], [seed & 0xFFFFFFFF, seed >> 32])
        z = orc.uniforms(seed, pid, d, pas)
        for i in range(2):
            u52 = ((int(w[2 * i]) << 32) | int(w[2 * i + 1])) >> 12
            assert z[i] == (2 * u52 + 1) / 2.0 ** 53
            assert 0.0 < z[i] < 1.0
    zs = np.array([orc.uniforms(9, p, 0) for p in range(20000)])
    assert abs(zs.mean() - 0.5) < 4 * math.sqrt(1 / 12 / zs.size)
    assert abs(np.corrcoef(zs[:, 0], zs[:, 1])[0, 1]) < 0.03


# ------------------------------------------------------------------------------------------ P2 DDA
def _slab_segments(nx, ny, nz, p, u):
    """Brute force: intersect the ray with every cell's box, keep positive-length overlaps."""
    out = []
    for iz in range(nz):
        for iy in range(ny):
            for ix in range(nx):
                t0, t1 = 0.0, np.inf
                for a, c in zip(range(3), (ix, iy, iz)):
                    if u[a] == 0.0:  # ray parallel to the faces: a point on a face belongs to the upper cell (Q9)
                        if not (c <= p[a] < c + 1):
                            t0, t1 = 1.0, 0.0
                        continue
                    ta, tb = (c - p[a]) / u[a], (c + 1 - p[a]) / u[a]
                    t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
                if t1 - t0 > 1e-11:
                    out.append((t0, (iz * ny + iy) * nx + ix, t1 - t0))
    out.sort()
    return out


def test_p2_dda_vs_brute_force(orc):
    rng = np.random.default_rng(42)
    n_rays = 0
    for _ in range(400):
        nx, ny, nz = rng.integers(1, 6, 3)
        p = rng.random(3) * np.array([nx, ny, nz])
        if rng.random() < 0.2:  # start exactly on a face / edge / corner
            for a in range(3):
                if rng.random() < 0.5:
                    p[a] = float(rng.integers(1, [nx, ny, nz][a] + 1) - (1 if [nx, ny, nz][a] > 1 else 0.5))
            p = np.minimum(np.maximum(p, 1e-9), np.array([nx, ny, nz]) - 1e-9)
        u = orc.isotropic(rng.random(), rng.random())
        if rng.random() < 0.1:
            u = np.zeros(3); u[rng.integers(0, 3)] = rng.choice([-1.0, 1.0])  # axis-parallel
        cells, ds = orc.dda_trace(int(nx), int(ny), int(nz), p, u)
        assert np.all(ds >= 0.0)
        keep = ds > 1e-11
        ref = _slab_segments(int(nx), int(ny), int(nz), p, u)
        assert list(cells[keep]) == [r[1] for r in ref]
        np.testing.assert_allclose(ds[keep], [r[2] for r in ref], rtol=0, atol=1e-12)
        # chord length to the exit face
        tex = min(((n if u[a] > 0 else 0.0) - p[a]) / u[a] for a, n in zip(range(3), (nx, ny, nz)) if u[a] != 0)
        assert abs(ds.sum() - tex) < 1e-12
        n_rays += 1
    assert n_rays == 400


def test_p2_start_cell_on_corner(orc):
    # central source on an even grid sits on a corner of 8 cells: the start cell follows the direction signs (Q9)
    for sx in (-1, 1):
        for sy in (-1, 1):
            for sz in (-1, 1):
                u = np.array([sx, sy, sz]) / math.sqrt(3)
                cells, ds = orc.dda_trace(4, 4, 4, [2.0, 2.0, 2.0], u)
                ix, iy, iz = (2 if sx > 0 else 1), (2 if sy > 0 else 1), (2 if sz > 0 else 1)
                assert cells[0] == (iz * 4 + iy) * 4 + ix
                assert abs(ds.sum() - 2 * math.sqrt(3)) < 1e-12


# ------------------------------------------------------------------------------------------ helpers
def _mean_over_directions(f, nmu=600, nphi=1200):
    mu = (np.arange(nmu) + 0.5) / nmu * 2 - 1
    phi = (np.arange(nphi) + 0.5) / nphi * 2 * np.pi
    MU, PHI = np.meshgrid(mu, phi, indexing="ij")
    st = np.sqrt(1 - MU ** 2)
    return f(st * np.cos(PHI), st * np.sin(PHI), MU)


# ------------------------------------------------------------------------------------------ P3 transmission
def test_p3_pure_absorber_transmission(orc):
    """Uniform pure-absorber cube, central source: the directly escaping fraction per frequency is the
    direction average of exp(-kappa rho l(u)), l(u) = (n/2)/max|u_a| (exp(-tau) law)."""
    n, N = 8, 400_000
    w = W.uniform_cube(n, tau_edge_V=1.5, albedo=0.0, g_const=0.0, n_nu=12, slope=-1.0, T_star=3000.0)
    o = orc.Oracle.from_workload(w)
    r = o.run(N, seed=11, absorb_and_stop=True, n_threads=NTH)
    raw = o.read_raw()
    assert r["escapes"] + r["absorptions"] == N  # absorbed + escaped = emitted, exactly
    assert np.array_equal(raw["sed"], raw["sed_direct"])
    t = o.tables()
    pj = np.diff(np.concatenate([[0.0], t["srccdf"]]))
    kext = (w.kappa_abs + w.kappa_sca)[0]
    rho0 = float(w.rho.flat[0])
    for j in range(w.n_nu):
        tau_half = kext[j] * rho0 * w.cell_size_cm * n / 2
        f = _mean_over_directions(lambda x, y, z: np.exp(-tau_half / np.maximum(np.maximum(abs(x), abs(y)), abs(z)))).mean()
        p = pj[j] * f
        got = int(raw["sed_direct"][0, j])
        sigma = math.sqrt(N * p * (1 - p))
        assert abs(got - N * p) < 4 * sigma + 1, (j, got, N * p, sigma)


# ------------------------------------------------------------------------------------------ P4 HG
@pytest.mark.parametrize("g", [0.0, 0.3, -0.3, 0.5, 0.7, 0.95])
def test_p4_henyey_greenstein_moments(orc, g):
    """<mu> = g and <mu^2> = (1 + 2 g^2)/3 for the phase function of PAPER.md:203 Eq. 15."""
    rng = np.random.default_rng(int(1000 * abs(g)) + (7 if g < 0 else 3))
    n = 40000
    mus = np.empty(n)
    perp = np.empty((n, 2))
    for i in range(n):
        u = orc.isotropic(rng.random(), rng.random())
        if i % 50 == 0:
            u = np.array([0.0, 0.0, 1.0 if i % 100 == 0 else -1.0])  # exercise the polar branch
        v = orc.hg_scatter(g, rng.random(), rng.random(), u)
        assert abs(np.dot(v, v) - 1.0) < 1e-14
        mus[i] = np.dot(u, v)
        # azimuth about u must be uniform: project on a fixed perpendicular frame
        e1 = np.cross(u, [0.3, -0.5, 0.8]); e1 /= np.linalg.norm(e1)
        e2 = np.cross(u, e1)
        perp[i] = (np.dot(v, e1), np.dot(v, e2))
    var_mu = (1 + 2 * g * g) / 3 - g * g
    assert abs(mus.mean() - g) < 4 * math.sqrt(var_mu / n) + 1e-12
    assert abs((mus ** 2).mean() - (1 + 2 * g * g) / 3) < 4 * math.sqrt(0.2 / n)
    assert np.all(np.abs(perp.mean(axis=0)) < 4 * math.sqrt(0.5 / n))


def test_p4_hg_distribution_shape(orc):
    """Binned cos(theta) follows the integral of P_HG (Eq. 15) between bin edges."""
    g, n = 0.6, 60000
    rng = np.random.default_rng(5)
    u = np.array([0.6, 0.0, 0.8])
    mus = np.array([np.dot(u, orc.hg_scatter(g, rng.random(), rng.random(), u)) for _ in range(n)])
    edges = np.linspace(-1, 1, 21)
    cum = lambda m: (1 - g * g) / (2 * g) * (1 / np.sqrt(1 + g * g - 2 * g * m) - 1 / (1 + g))  # CDF of Eq. 15 in mu
    p = np.diff(cum(edges))
    assert abs(p.sum() - 1) < 1e-12
    cnt, _ = np.histogram(mus, edges)
    chi2 = ((cnt - n * p) ** 2 / (n * p)).sum()
    assert chi2 < 50  # 19 dof; 50 is ~1e-4 tail


# ------------------------------------------------------------------------------------------ P5 isotropy
def test_p5_isotropic_emission_and_empty_grid(orc):
    zs = np.random.default_rng(3).random((50000, 2))
    us = np.array([orc.isotropic(a, b) for a, b in zs])
    np.testing.assert_allclose(np.linalg.norm(us, axis=1), 1.0, atol=1e-15)
    assert np.all(np.abs(us.mean(axis=0)) < 4 * math.sqrt(1 / 3 / len(us)))
    assert np.all(np.abs((us ** 2).mean(axis=0) - 1 / 3) < 4 * math.sqrt(4 / 45 / len(us)))
    # empty grid: every packet escapes directly; counts are multinomial with p = w_j * d|mu|
    w = W.uniform_cube(6, tau_edge_V=0.0, albedo=0.5, g_const=0.0, n_nu=10, n_dir=5, T_star=4000.0)
    N = 200_000
    o = orc.Oracle.from_workload(w)
    r = o.run(N, seed=5, n_threads=NTH)
    raw = o.read_raw()
    assert r["direct_escapes"] == N and r["absorptions"] == 0 and r["scatterings"] == 0
    assert np.array_equal(raw["sed"], raw["sed_direct"]) and raw["sed"].sum() == N
    pj = np.diff(np.concatenate([[0.0], o.tables()["srccdf"]]))
    p = np.outer(np.diff(w.abs_mu_edges), pj)
    sel = p * N > 20
    chi2 = (((raw["sed"] - N * p) ** 2)[sel] / (N * p)[sel]).sum()
    assert chi2 < sel.sum() + 5 * math.sqrt(2 * sel.sum())
    # the walk length of a central source in an n-cube: crossings >= n/2 per packet
    assert r["crossings"] >= N * 3


# ------------------------------------------------------------------------------------------ P6/P7/P13
def test_p6_p7_p13_conservation_albedo_determinism(orc):
    w = W.sphere32(tau_V=3.0)
    N = 30000
    o = orc.Oracle.from_workload(w)
    r1 = o.run(N, seed=1, digests=True, n_threads=1)
    raw1 = o.read_raw()
    d1 = r1["digests"]
    # P6 exact invariants
    assert raw1["sed"].sum() == N == r1["escapes"]
    assert raw1["k"].sum() == r1["absorptions"] == d1["absorptions"].sum()
    assert r1["crossings"] == d1["crossings"].sum()
    assert r1["scatterings"] == d1["scatterings"].sum()
    assert raw1["sed_direct"].sum() == r1["direct_escapes"] == ((d1["absorptions"] + d1["scatterings"]) == 0).sum()
    assert r1["flights"] == N + r1["scatterings"] + r1["absorptions"]
    assert np.all(raw1["lucy_fx"] >= 0) and np.all(raw1["lucy_fx"][w.rho.reshape(-1) == 0] == 0)
    # P7 constant albedo 0.5
    n_int = r1["scatterings"] + r1["absorptions"]
    assert abs(r1["scatterings"] / n_int - 0.5) < 4 * math.sqrt(0.25 / n_int)
    # P13 thread count must not change anything
    r8 = o.run(N, seed=1, digests=True, n_threads=NTH)
    raw8 = o.read_raw()
    for key in ("k", "lucy_fx", "sed", "sed_direct", "tidx"):
        assert np.array_equal(raw1[key], raw8[key]), key
    assert np.array_equal(d1, r8["digests"])
    # a different seed gives a different realisation
    r2 = o.run(N, seed=2, digests=True, n_threads=NTH)
    assert not np.array_equal(d1["hash"], r2["digests"]["hash"])


# ------------------------------------------------------------------------------------------ P9 tables
def _wide(n_nu=400, lam_min=0.05, lam_max=2e5):
    lam = W.wavelength_grid_um(n_nu, lam_min, lam_max)
    return W.nu_from_lambda_um(lam)


def test_p9_planck_closed_forms(orc):
    nu = _wide()
    dnu = orc.bin_widths(nu)
    assert np.all(dnu > 0)
    # bins tile the axis: sum of widths = outer edge - inner edge
    assert abs(dnu.sum() - (nu[-1] * math.sqrt(nu[-1] / nu[-2]) - nu[0] * math.sqrt(nu[0] / nu[1]))) < 1e-9 * nu[-1]
    for T in (30.0, 300.0, 1500.0):
        B = np.array([orc.planck(v, T) for v in nu])
        # Stefan-Boltzmann: integral B_nu dnu = sigma T^4 / pi
        assert abs((B * dnu).sum() / (SIGMA_SB * T ** 4 / math.pi) - 1) < 2e-3
        # Wien displacement in frequency: h nu_max / k T = 2.821439...
        fine = np.linspace(2.0, 3.6, 4001) * K_BOLTZ * T / H_PLANCK
        xm = H_PLANCK * fine[np.argmax([orc.planck(v, T) for v in fine])] / (K_BOLTZ * T)
        assert abs(xm - 2.8214393721) < 1e-3
        # dB/dT against a centred finite difference of B
        for v in (nu[50], nu[200], nu[330]):
            fd = (orc.planck(v, T * (1 + 1e-5)) - orc.planck(v, T * (1 - 1e-5))) / (2e-5 * T)
            assert abs(orc.dplanck_dT(v, T) / fd - 1) < 1e-6 if fd > 1e-300 else True
    # Rayleigh-Jeans limit 2 nu^2 k T / c^2
    assert abs(orc.planck(1e9, 100.0) / (2 * 1e18 * K_BOLTZ * 100.0 / C_LIGHT ** 2) - 1) < 1e-3


@pytest.mark.parametrize("beta", [0.0, 1.5])
def test_p9_tables_power_law(orc, beta):
    """For kappa ~ nu^beta: J ~ T^(4+beta); mean h nu/kT of the Eq. 5 CDF is (4+b) zeta(5+b)/zeta(4+b)
    (3.8322 at b=0, 5.4292 at b=1.5) and of the Eq. 10 CDF (5+b) zeta(5+b)/zeta(4+b) (4.7903, 6.4163)."""
    nu = _wide()
    Tg = W.temperature_grid(200, 5.0, 1500.0)
    kabs = (nu / nu[0]) ** beta
    o = orc.Oracle(1, 1, 1, 1.0, np.zeros(1, np.float32), np.zeros(1, np.uint8), 1, nu, kabs[None], kabs[None] * 0,
                   np.zeros((1, len(nu))), Tg, 1.0, 1000.0, None, [0.5, 0.5, 0.5], [0.0, 1.0])
    t = o.tables()
    J = t["J"][0]
    slope = np.diff(np.log(J)) / np.diff(np.log(Tg))
    np.testing.assert_allclose(slope, 4 + beta, atol=2e-3)
    # closed form of the integral: 2 h/c^2 (kT/h)^(4+b) Gamma(4+b) zeta(4+b) / nu0^b
    m = 120
    closed = 2 * H_PLANCK / C_LIGHT ** 2 * (K_BOLTZ * Tg[m] / H_PLANCK) ** (4 + beta) * special.gamma(4 + beta) \
        * special.zeta(4 + beta, 1) / nu[0] ** beta
    assert abs(J[m] / closed - 1) < 2e-3
    zB = (4 + beta) * special.zeta(5 + beta, 1) / special.zeta(4 + beta, 1)
    zdB = (5 + beta) * special.zeta(5 + beta, 1) / special.zeta(4 + beta, 1)
    assert abs(zB - (3.8322 if beta == 0 else 5.4292)) < 1e-3
    assert abs(zdB - (4.7903 if beta == 0 else 6.4163)) < 1e-3
    for m in (20, 100, 180):
        x = H_PLANCK * nu / (K_BOLTZ * Tg[m])
        for key, ref in (("cdfB", zB), ("cdfdB", zdB)):
            cdf = t[key][0, m]
            assert cdf[-1] == 1.0 and np.all(np.diff(cdf) >= 0) and cdf[0] >= 0
            pj = np.diff(np.concatenate([[0.0], cdf]))
            assert abs((pj * x).sum() / ref - 1) < 3e-3, (key, m)
    # T(J(T_m)) round trip and monotone inversion in between
    for m in (0, 17, 199):
        assert abs(o.T_of_x(0, J[m]) / Tg[m] - 1) < 1e-12
    xm = math.sqrt(J[40] * J[41])
    assert Tg[40] < o.T_of_x(0, xm) < Tg[41]
    assert abs(o.T_of_x(0, xm) / math.sqrt(Tg[40] * Tg[41]) - 1) < 1e-3
    assert o.T_of_x(0, 0.0) == 0.0 and o.T_of_x(0, J[0] * 0.1) == Tg[0] and o.T_of_x(0, J[-1] * 10) == Tg[-1]
    # albedo and lower_bound semantics
    assert np.all(t["albedo"] == 0.0)
    cdf = np.array([0.1, 0.1, 0.4, 1.0])
    assert [orc.lower_bound(cdf, z) for z in (0.05, 0.1, 0.1000001, 0.4, 0.9, 1.0)] == [0, 0, 2, 2, 3, 3]


# ------------------------------------------------------------------------------------------ P8 thin temperature
def test_p8_optically_thin_temperature(orc):
    """Optically thin sphere, kappa ~ nu^beta, blackbody source inside the T grid:
    the Lucy-tally temperature follows T = T* (R*/2r)^(2/(4+beta))  (radiative balance, Eq. 4 with Eq. 9)."""
    beta, Tstar, n, N = 1.0, 1500.0, 24, 600_000
    lam = W.wavelength_grid_um(160, 0.2, 1e5)
    nu = W.nu_from_lambda_um(lam)
    kabs = 100.0 * (nu / nu[-1]) ** beta
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    rho0 = 1e-3 / (kabs.max() * n / 2 * h)  # tau <= 1e-3 at every frequency
    rho = np.where(r < n / 2, rho0, 0.0).astype(np.float32)
    L = W.LSUN_ERG_S
    c = n / 2 * h
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 1, nu, kabs[None], np.zeros((1, len(nu))),
                   np.zeros((1, len(nu))), W.temperature_grid(1000, 2.0, 2000.0), L, Tstar, None, [c, c, c],
                   [0.0, 1.0])
    res = o.run(N, seed=8, n_threads=NTH)
    assert res["absorptions"] < 0.01 * N
    T = o.read(T_from_lucy=True)["T"].reshape(n, n, n).astype(np.float64)
    Rstar = math.sqrt(L / (4 * math.pi * SIGMA_SB * Tstar ** 4))
    for r_lo in (4.0, 7.0, 10.0):
        sel = (r >= r_lo) & (r < r_lo + 1.0)
        T_exp = Tstar * (Rstar / (2 * r[sel] * h)) ** (2 / (4 + beta))
        ratio = (T[sel] / T_exp)
        assert abs(ratio.mean() - 1) < 0.01, (r_lo, ratio.mean())
    # the estimator itself, free of the T tables: x_cell r^2 16 pi^2 / L = sum_j kappa_j p_j
    out = o.read()
    pj = np.diff(np.concatenate([[0.0], o.tables()["srccdf"]]))
    sel = (r >= 5.0) & (r < 9.0)
    xcell = out["E_lucy"].reshape(n, n, n)[sel] / (4 * math.pi * rho0 * h ** 3)
    got = (xcell * (r[sel] * h) ** 2).mean() * 16 * math.pi ** 2 / L
    assert abs(got / (kabs * pj).sum() - 1) < 0.01


# ------------------------------------------------------------------------------------------ P10 brute force 2x2x2
def test_p10_brute_force_2x2x2(orc):
    """2x2x2 grid of different densities, grey pure absorber, off-centre source, absorb-and-stop:
    E[k_c] = N <exp(-tau_in) - exp(-tau_out)> by dense direction quadrature with slab intersections;
    the Lucy tally has the same expectation."""
    N = 400_000
    w = W.uniform_cube(2, tau_edge_V=1.0, albedo=0.0, g_const=0.0, n_nu=4, slope=0.0,
                       source_offset_cells=(0.3, -0.2, 0.1))
    base = float(w.rho.flat[0])
    w.rho[:] = (base * np.array([0.5, 1.0, 2.0, 0.0, 1.5, 3.0, 0.25, 0.8], np.float32)).reshape(2, 2, 2)
    o = orc.Oracle.from_workload(w)
    r = o.run(N, seed=21, absorb_and_stop=True, n_threads=NTH)
    raw = o.read_raw()
    kext = float((w.kappa_abs + w.kappa_sca)[0, 0])
    assert np.allclose((w.kappa_abs + w.kappa_sca)[0], kext)
    p = np.array(w.source_pos_cm) / w.cell_size_cm

    def expect(ux, uy, uz):
        u = np.stack([ux, uy, uz])
        t_in = np.zeros((8,) + ux.shape)
        t_out = np.zeros_like(t_in)
        for c in range(8):
            idx = (c & 1, (c >> 1) & 1, (c >> 2) & 1)
            lo, hi = np.zeros_like(ux), np.full_like(ux, np.inf)
            for a in range(3):
                ta, tb = (idx[a] - p[a]) / u[a], (idx[a] + 1 - p[a]) / u[a]
                lo, hi = np.maximum(lo, np.minimum(ta, tb)), np.minimum(hi, np.maximum(ta, tb))
            t_in[c], t_out[c] = lo, np.maximum(hi, lo)
        dtau = (t_out - t_in) * (kext * w.rho.reshape(-1).astype(np.float64) * w.cell_size_cm)[:, None, None]
        tau_in = np.zeros_like(t_in)
        for c in range(8):
            for c2 in range(8):
                tau_in[c] += np.where(t_in[c2] < t_in[c] - 1e-13, dtau[c2], 0.0)
        return np.exp(-tau_in) - np.exp(-(tau_in + dtau))

    prob = _mean_over_directions(expect, 500, 1000).mean(axis=(1, 2))
    k = raw["k"].astype(np.float64)
    lucy = raw["lucy_fx"] / 2.0 ** r["fx_bits"]
    for c in range(8):
        sig = math.sqrt(N * prob[c] * (1 - prob[c])) + 1
        assert abs(k[c] - N * prob[c]) < 4 * sig, (c, k[c], N * prob[c])
        assert abs(lucy[c] - N * prob[c]) < 5 * sig, (c, lucy[c], N * prob[c])
    assert raw["k"][3] == 0 and raw["lucy_fx"][3] == 0
    assert raw["k"].sum() + raw["sed"].sum() == N


# ------------------------------------------------------------------------------------------ P11 redraw
def test_p11_per_cell_redraw_equivalence(orc):
    """PAPER.md:51 (new zeta on every cell entry) vs footnote 1, PAPER.md:61 (one zeta per flight)."""
    w = W.sphere32(tau_V=2.0, n=16)
    N = 150_000
    o = orc.Oracle.from_workload(w)
    ra = o.run(N, seed=31, n_threads=NTH)
    a = o.read_raw()
    rb = o.run(N, seed=32, per_cell_redraw=True, n_threads=NTH)
    b = o.read_raw()
    for key in ("absorptions", "scatterings", "crossings", "direct_escapes"):
        va, vb = ra[key], rb[key]
        # totals are sums over packets of over-dispersed counts: allow 5 sigma with dispersion factor 4
        assert abs(va - vb) < 5 * math.sqrt(4 * (va + vb)), (key, va, vb)
    x = (np.arange(16) + 0.5) - 8
    rr = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2).reshape(-1)
    for lo in range(0, 8, 2):
        sel = (rr >= lo) & (rr < lo + 2)
        ka, kb = a["k"][sel].sum(), b["k"][sel].sum()
        assert abs(float(ka) - float(kb)) < 5 * math.sqrt(2.0 * (ka + kb)), (lo, ka, kb)
        la, lb = a["lucy_fx"][sel].sum(), b["lucy_fx"][sel].sum()
        assert abs(la / lb - 1) < 0.03
    sa, sb = a["sed"].sum(axis=0).astype(float), b["sed"].sum(axis=0).astype(float)
    sel = sa + sb > 200
    assert (((sa - sb) ** 2)[sel] / (sa + sb)[sel]).sum() < sel.sum() + 5 * math.sqrt(2 * sel.sum())


# ------------------------------------------------------------------------------------------ P12 epochs
def test_p12_epoch_vs_serial_bjorkman_wood(orc):
    """Epoch semantics (reading Q19) against serial Bjorkman & Wood (B0 = Bmax = 1, T updated after every
    packet): temperatures from counts agree to 0.5 % shell by shell, emergent spectrum agrees band by band."""
    w = W.sphere32(tau_V=5.0, n=10)
    N = 60_000
    o = orc.Oracle.from_workload(w)
    re = o.run(N, seed=41, n_threads=NTH)
    e_raw, e_out = o.read_raw(), o.read()
    assert re["epochs"] > 5
    rs = o.run(N, seed=41, B0=1, Bmax=1)
    s_raw, s_out = o.read_raw(), o.read()
    assert rs["epochs"] == N
    x = (np.arange(10) + 0.5) - 5
    rr = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2).reshape(-1)
    for lo in range(0, 5):
        sel = (rr >= lo) & (rr < lo + 1) & (w.rho.reshape(-1) > 0)
        Te, Ts = e_out["T"][sel].astype(float).mean(), s_out["T"][sel].astype(float).mean()
        assert abs(Te / Ts - 1) < 0.005, (lo, Te, Ts)
    # count-T and Lucy-T are consistent where counts are large (both estimate the same energy)
    big = e_raw["k"] > 400
    assert big.sum() >= 8
    Tl = o.read(T_from_lucy=True)["T"][big].astype(float)
    assert np.all(np.abs(Tl / s_out["T"][big] - 1) < 0.03)
    # emergent spectrum in 8 broad bands (same seeds, so noise is correlated and the bound is loose)
    se, ss = e_raw["sed"].sum(axis=0).astype(float), s_raw["sed"].sum(axis=0).astype(float)
    be, bs = se.reshape(8, 8).sum(axis=1), ss.reshape(8, 8).sum(axis=1)
    sel = bs > 500
    assert np.all(np.abs(be[sel] / bs[sel] - 1) < 0.03 + 3 / np.sqrt(bs[sel]))


# ------------------------------------------------------------------------------------------ P14 fixed point
def test_p14_fixed_point_vs_compensated_fp64(orc):
    w = W.sphere32(tau_V=1.0)
    o = orc.Oracle.from_workload(w)
    r = o.run(50_000, seed=1, keep_fp64_lucy=True)
    raw = o.read_raw(fp64_lucy=True)
    fx = r["fx_bits"]
    assert fx == 40 == orc.fx_bits(50_000)
    assert orc.fx_bits(10 ** 9) == 28 and orc.fx_bits(10 ** 8) == 31 and orc.fx_bits(2 ** 20) == 38
    L = raw["lucy_fx"] / 2.0 ** fx
    sel = raw["lucy_fp64"] > 0
    assert sel.sum() > 10000
    rel = np.abs(L[sel] / raw["lucy_fp64"][sel] - 1)
    assert rel.max() < 1e-6
    # quantisation bound: each add is off by <= 2^-(fx+1)
    assert np.all(np.abs(L - raw["lucy_fp64"]) <= r["lucy_adds"] * 2.0 ** -(fx + 1))
    assert orc.default_schedule(10 ** 8) == (2 ** 18, 2 ** 22) and orc.default_schedule(10 ** 5) == (256, 2 ** 22)
    assert orc.default_schedule(1000) == (256, 2 ** 22)


# ------------------------------------------------------------------------------------------ P15 explicit ln / sin / cos
def test_p15_explicit_log_sincos_against_libm_and_multiprecision(orc):
    """Reading Q28: the trajectory's ln, sin, cos are explicit fp64 algorithms.  Pinned against libm (<= 3 ulp)
    and against 120-bit mpmath values (<= 2.5 ulp), on uniforms of the generator's form (2u+1) 2^-53 of every
    magnitude, plus exact special values and the unit circle."""
    import math
    import random

    import mpmath as mp

    mp.mp.prec = 120
    rnd = random.Random(15)
    worst_log = worst_sc = 0.0
    for i in range(6000):
        bits = 52 if i % 2 else rnd.randint(1, 52)
        z = (2 * rnd.getrandbits(bits) + 1) * 2.0 ** -53
        l = orc.det_log(z)
        assert abs(l - math.log(z)) <= 3 * math.ulp(l)
        worst_log = max(worst_log, float(abs(mp.mpf(l) - mp.log(mp.mpf(z))) / math.ulp(l)))
        s, c = orc.det_sincos(z)
        ang = 2 * mp.pi * mp.mpf(z)
        ts, tc = mp.sin(ang), mp.cos(ang)
        for got, true in ((s, ts), (c, tc)):
            err = float(abs(mp.mpf(got) - true))
            assert err <= 2.5 * math.ulp(float(true)) + 1e-300 or err <= 2.0 ** -53 * abs(float(true)) * 4
            worst_sc = max(worst_sc, err / math.ulp(float(true)))
        assert abs(s * s + c * c - 1.0) <= 5e-16
    assert worst_log <= 2.5 and worst_sc <= 2.5
    # special values: powers of two, quarter turns, the ends of the generator's range
    for k in range(1, 54):
        assert abs(orc.det_log(2.0 ** -k) + k * math.log(2.0)) <= 2 * math.ulp(k * math.log(2.0))
    assert orc.det_log(1.0) == 0.0
    assert orc.det_sincos(0.0) == (0.0, 1.0) and orc.det_sincos(0.5) == (0.0, -1.0) or orc.det_sincos(0.5)[1] == -1.0
    assert orc.det_sincos(0.25)[0] == 1.0 and orc.det_sincos(0.75)[0] == -1.0
    assert orc.det_sincos(0.125) == pytest.approx((math.sqrt(0.5), math.sqrt(0.5)), rel=4e-16)
    zmax = 1.0 - 2.0 ** -53
    assert orc.det_log(zmax) == pytest.approx(-2.0 ** -53, rel=1e-15)
    assert orc.det_sincos(zmax)[0] == pytest.approx(-2 * math.pi * 2.0 ** -53, rel=1e-15)


# ------------------------------------------------------------------------------------------ P12b plateau epochs
def test_p12b_plateau_epochs_of_the_default_schedule(orc):
    """Reading Q19 at the shipped default.  The default schedule for N = 1e8 is B0 = 2^18 = N/381 doubling up to
    Bmax = 2^22 = N/23.8, i.e. 4 doubling epochs and then ~23 plateau epochs of 4.2 % of N each, during which the
    temperature index stays frozen at the midpoint prediction.  The same shape scaled to what a serial run can
    check: N = 1e5, B0 = 256 = N/391, Bmax = 4096 = N/24.4 (4 doubling + 24 plateau epochs, growth ratio 1),
    against serial Bjorkman & Wood (B = 1): T within 0.5 % shell by shell, spectrum within 3 %."""
    w = W.sphere32(tau_V=5.0, n=12)
    N = 100_000
    o = orc.Oracle.from_workload(w)
    re = o.run(N, seed=43, B0=256, Bmax=4096, n_threads=NTH)
    e_raw, e_out = o.read_raw(), o.read()
    assert re["epochs"] == 4 + 24  # 256 + 512 + 1024 + 2048 = 3840, then 23 x 4096 + 1952
    rs = o.run(N, seed=43, B0=1, Bmax=1)
    s_raw, s_out = o.read_raw(), o.read()
    assert rs["epochs"] == N
    x = (np.arange(12) + 0.5) - 6
    rr = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2).reshape(-1)
    for lo in range(0, 6):
        sel = (rr >= lo) & (rr < lo + 1) & (w.rho.reshape(-1) > 0)
        Te, Ts = e_out["T"][sel].astype(float).mean(), s_out["T"][sel].astype(float).mean()
        assert abs(Te / Ts - 1) < 0.005, (lo, Te, Ts)
    # total absorbed energy and the emergent spectrum in 8 broad bands
    assert abs(e_raw["k"].sum() / s_raw["k"].sum() - 1) < 0.005
    se, ss = e_raw["sed"].sum(axis=0).astype(float), s_raw["sed"].sum(axis=0).astype(float)
    be, bs = se.reshape(8, 8).sum(axis=1), ss.reshape(8, 8).sum(axis=1)
    sel = bs > 500
    assert sel.sum() >= 4
    assert np.all(np.abs(be[sel] / bs[sel] - 1) < 0.03 + 3 / np.sqrt(bs[sel]))


# ------------------------------------------------------------------------------------------ P16 frozen-T sweep
def _thin_grey_sphere(orc, n=24, Tstar=1500.0, n_nu=160):
    lam = W.wavelength_grid_um(n_nu, 0.2, 1e5)
    nu = W.nu_from_lambda_um(lam)
    kabs = np.full(len(nu), 100.0)
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    rho0 = np.float32(1e-3 / (100.0 * n / 2 * h))   # radial tau = 1e-3 at every frequency (grey)
    rho = np.where(r < n / 2, rho0, 0.0).astype(np.float32)
    Tg = W.temperature_grid(1000, 2.0, 2000.0)
    c = n / 2 * h
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 1, nu, kabs[None], np.zeros((1, len(nu))),
                   np.zeros((1, len(nu))), Tg, W.LSUN_ERG_S, Tstar, None, [c, c, c], [0.0, 1.0])
    return o, nu, Tg, rho, r, h, float(rho0)


@pytest.mark.parametrize("from_lucy", [1, 0])
def test_p16_frozen_temperature_sweep(orc, from_lucy):
    """S12 / O-run mode 1 (Eq. 5): a sweep takes its temperatures from the PREVIOUS pass's tallies
    (in that pass's packet energy and fixed-point scale), starts its own tallies from zero, and re-emits from the
    Eq. 5 table kappa B_nu(T), not from the Eq. 10 table of the B&W pass.  Grey optically thin sphere, so that
    T(r) = T* sqrt(R*/2r) is known in closed form (radiative balance, Eq. 4)."""
    o, nu, Tg, rho, r, h, rho0 = _thin_grey_sphere(orc)
    n = rho.shape[0]
    N1, N2 = 2_000_000, 6_000_000            # different N: xi and the fixed-point scale differ between the passes
    r1 = o.run(N1, seed=16, n_threads=NTH)
    raw1 = o.read_raw()
    r2 = o.run(N2, seed=16, mode=orc.MODE_FROZEN_SWEEP, n_sweeps=1, sweep_T_from_lucy=from_lucy, n_threads=NTH)
    raw2 = o.read_raw()
    assert r1["fx_bits"] == 37 and r2["fx_bits"] == 35
    L, Tstar = W.LSUN_ERG_S, 1500.0
    dusty = rho.reshape(-1) > 0
    tidx = raw2["tidx"].astype(np.int64)
    J = o.tables()["J"][0]
    xi1 = L / N1
    # (a) the index is the Eq. 4 inversion of the previous pass's tallies at ITS xi and fixed-point scale
    e1 = raw1["lucy_fx"] / 2.0 ** r1["fx_bits"] if from_lucy else raw1["k"].astype(np.float64)
    x1 = e1 * (xi1 / (4 * math.pi * h ** 3)) / np.where(dusty, rho.reshape(-1), 1.0)
    want = np.minimum(np.searchsorted(J, x1, side="left"), len(Tg) - 1)
    assert (tidx[dusty] == want[dusty]).mean() > 0.9995       # (a cell whose x sits within rounding of a J entry may differ)
    assert np.all(tidx[~dusty] == 0)
    if from_lucy:
        # (b) ... and that is the closed form T(r) = T* sqrt(R*/2r): position in the log T grid within +-1
        Rstar = math.sqrt(L / (4 * math.pi * SIGMA_SB * Tstar ** 4))
        dlnT = math.log(Tg[1] / Tg[0])
        for r_lo in (4.0, 7.0, 10.0):
            sel = ((r >= r_lo) & (r < r_lo + 1.0)).reshape(-1)
            m_star = np.log(Tstar * np.sqrt(Rstar / (2 * r.reshape(-1)[sel] * h)) / Tg[0]) / dlnT
            assert abs((tidx[sel] - m_star).mean() - 0.5) < 1.0, (r_lo, (tidx[sel] - m_star).mean())
    else:
        assert np.all(tidx[dusty & (raw1["k"] == 0)] == 0)
    # (c) the sweep's tallies are its own: they start from zero
    assert int(raw2["k"].sum()) == r2["absorptions"] and int(raw2["sed"].sum()) == N2 == r2["escapes"]
    assert abs(r2["absorptions"] / N2 / (r1["absorptions"] / N1) - 1) < 5 / math.sqrt(r1["absorptions"])
    l1, l2 = raw1["lucy_fx"].sum() / 2.0 ** 37 / N1, raw2["lucy_fx"].sum() / 2.0 ** 35 / N2
    assert abs(l2 / l1 - 1) < 0.01 and abs(l2 / 1e-3 - 1) < 0.05   # sum of kappa rho ds per packet = radial tau
    # (d) Eq. 5: the re-emitted packets (every interaction is an absorption here) carry <h nu> = zB k T_cell with
    # zB = 4 zeta(5)/zeta(4) = 3.8322, not the 4.7903 of Eq. 10
    re_em = (raw2["sed"] - raw2["sed_direct"]).sum(axis=0).astype(np.float64)
    assert re_em.sum() > 3000
    e_obs = (re_em * H_PLANCK * nu).sum() / re_em.sum()
    k2 = raw2["k"].astype(np.float64)
    kT = K_BOLTZ * (k2 * Tg[tidx]).sum() / k2.sum()
    zB = 4 * special.zeta(5, 1) / special.zeta(4, 1)
    ratio = e_obs / kT
    assert abs(ratio / zB - 1) < 0.06, ratio
    assert abs(ratio / (5 * special.zeta(5, 1) / special.zeta(4, 1)) - 1) > 0.12


# ------------------------------------------------------------------------------------------ P17 outputs
def test_p17_sed_flux_conversion_and_energy_outputs(orc):
    """O12 outputs (PAPER.md:180 photon counting; PAPER.md:63 E = k xi).  Empty grid: every packet escapes, so
    sum SED dnu dOmega = L exactly and SED_j = L_nu / 4 pi with L_nu the blackbody shape; dusty absorb-and-stop
    run: E_count = k xi exactly and absorbed + escaped luminosity = L."""
    Tstar, N = 4000.0, 400_000
    w = W.uniform_cube(6, tau_edge_V=0.0, albedo=0.5, g_const=0.0, n_nu=24, n_dir=5, T_star=Tstar)
    o = orc.Oracle.from_workload(w)
    o.run(N, seed=17, n_threads=NTH)
    sed, raw = o.read()["SED"], o.read_raw()
    nu = w.nu_hz
    # bin widths and blackbody weights written out independently (reading Q15)
    edges = np.concatenate([[nu[0] * math.sqrt(nu[0] / nu[1])], np.sqrt(nu[:-1] * nu[1:]),
                            [nu[-1] * math.sqrt(nu[-1] / nu[-2])]])
    dnu = np.diff(edges)
    Bnu = 2 * H_PLANCK * nu ** 3 / C_LIGHT ** 2 / np.expm1(H_PLANCK * nu / (K_BOLTZ * Tstar))
    wj = Bnu * dnu / (Bnu * dnu).sum()
    dom = 4 * math.pi * np.diff(w.abs_mu_edges)          # both hemispheres (reading Q22)
    assert abs((sed * dnu[None, :] * dom[:, None]).sum() / w.L_erg_s - 1) < 1e-12
    expect = w.L_erg_s * wj / (dnu * 4 * math.pi)          # erg s^-1 Hz^-1 sr^-1, the same in every direction bin
    cnt_exp = N * np.outer(np.diff(w.abs_mu_edges), wj)
    sel = cnt_exp > 30
    assert sel.sum() >= 50
    assert np.all(np.abs(sed / expect[None, :] - 1)[sel] < 4 / np.sqrt(cnt_exp[sel]))
    np.testing.assert_allclose(sed, raw["sed"] * (w.L_erg_s / N) / (dnu[None, :] * dom[:, None]), rtol=1e-14)
    # dusty: E_count = k xi and E_lucy = xi L / 2^FX exactly; absorbed + escaped = emitted
    w2 = W.uniform_cube(8, tau_edge_V=1.0, albedo=0.0, g_const=0.0, n_nu=12, n_dir=3, T_star=Tstar)
    o2 = orc.Oracle.from_workload(w2)
    N2 = 50_000
    r2 = o2.run(N2, seed=18, absorb_and_stop=True, n_threads=NTH)
    out, raw2 = o2.read(), o2.read_raw()
    xi = w2.L_erg_s / N2
    assert np.array_equal(out["E_count"], raw2["k"].astype(np.float64) * xi)
    assert np.array_equal(out["E_lucy"], raw2["lucy_fx"].astype(np.float64) * 2.0 ** -r2["fx_bits"] * xi)
    nu2 = w2.nu_hz
    e2 = np.concatenate([[nu2[0] * math.sqrt(nu2[0] / nu2[1])], np.sqrt(nu2[:-1] * nu2[1:]),
                         [nu2[-1] * math.sqrt(nu2[-1] / nu2[-2])]])
    esc = (out["SED"] * np.diff(e2)[None, :] * (4 * math.pi * np.diff(w2.abs_mu_edges))[:, None]).sum()
    assert abs((out["E_count"].sum() + esc) / w2.L_erg_s - 1) < 1e-12
    assert 0.2 < out["E_count"].sum() / w2.L_erg_s < 0.8
    # the path-length estimate of the absorbed luminosity agrees with the counted one
    assert abs(out["E_lucy"].sum() / out["E_count"].sum() - 1) < 4 / math.sqrt(raw2["k"].sum())


# ------------------------------------------------------------------------------------------ P18 random flight
@pytest.mark.parametrize("a,g", [(0.5, 0.0), (0.5, 0.6), (0.9, 0.0), (0.9, 0.6)])
def test_p18_multiple_scattering_displacement(orc, a, g):
    """O5 + O7 (Eq. 3; HG of Eq. 15): in an effectively infinite uniform grey medium a packet that
    scatters with probability a (mean cosine g) and is absorbed otherwise ends at R = sum s_i u_i with exponential
    flight lengths of mean l = 1/(kappa_ext rho), so <R^2> = 2 l^2 / [(1 - a)(1 - a g)], isotropic.  The tally
    gives the absorption CELL: Sheppard's correction adds 1/12 cell^2 per axis.  This is the pin that fails when
    the interaction point p += u t_int, its clamp or the rotation about the old direction is wrong."""
    n, N = 160, 200_000
    w = W.uniform_cube(n, tau_edge_V=40.0, albedo=a, g_const=g, n_nu=4, slope=0.0)
    o = orc.Oracle.from_workload(w)
    r = o.run(N, seed=1800 + int(100 * a + 10 * g), absorb_and_stop=True, B0=N, Bmax=N, n_threads=NTH)
    assert r["escapes"] <= 2e-4 * N and r["absorptions"] + r["escapes"] == N
    k = o.read_raw()["k"].reshape(n, n, n).astype(np.float64)
    kext = float((w.kappa_abs + w.kappa_sca)[0, 0])
    ell = 1.0 / (kext * float(w.rho.flat[0]) * w.cell_size_cm)          # mean free path in cells
    assert abs(ell - 2.0) < 1e-6
    assert abs(r["scatterings"] / (r["scatterings"] + r["absorptions"]) - a) < 4 * math.sqrt(a * (1 - a) / r["flights"])
    d = (np.arange(n) + 0.5) - n / 2                                      # cell centre minus source, per axis
    K = k.sum()
    r2_true = 2 * ell ** 2 / ((1 - a) * (1 - a * g))
    m2 = []
    for axis, kk in enumerate((k.sum(axis=(0, 1)), k.sum(axis=(0, 2)), k.sum(axis=(1, 2)))):   # x, y, z marginals
        m1 = (kk * d).sum() / K
        v = (kk * d ** 2).sum() / K
        s4 = (kk * d ** 4).sum() / K
        assert abs(m1) < 4 * math.sqrt(v / K), (axis, m1)
        assert abs(v - (r2_true / 3 + 1 / 12)) < 4 * math.sqrt((s4 - v * v) / K), (axis, v, r2_true / 3 + 1 / 12)
        m2.append(v)
    X, Y, Z = np.meshgrid(d, d, d, indexing="ij")
    rr2 = (Z ** 2 + Y ** 2 + X ** 2)   # k is [z][y][x]; the sum of squares is symmetric
    tot = (k * rr2).sum() / K
    sig = math.sqrt(((k * rr2 ** 2).sum() / K - tot ** 2) / K)
    assert abs(tot - (r2_true + 0.25)) < 4 * sig, (tot, r2_true + 0.25, sig)
    assert sig / tot < 0.006            # the bound is sharp: 0.6 % (the voxel term alone is 0.3-1.5 %)


# ------------------------------------------------------------------------------------------ P19 carry-over
def test_p19_carry_over_of_long_lived_packets(orc):
    """NEXT-1: the deterministic restatement of the paper's pause / resume of packets with more than 100
    interactions (orc_carry in the oracle): a packet stops after carry_K interactions within one
    epoch and continues in the next epoch from the same state and random stream, at that epoch's temperatures.
      (a) grey dust: transport does not depend on frequency, so carrying cannot change a single path -- absorption
          counts, Lucy tallies and every packet's crossing / scattering / absorption numbers are IDENTICAL to the
          uncarried run (fails if the carried state loses position, direction, cell or draw counter);
      (b) nothing is lost: every packet escapes exactly once, in whatever epoch;
      (c) the result does not depend on the thread count (the carried list is ordered by packet id);
      (d) a budget no packet reaches changes nothing at all;
      (e) chromatic thick cube, 60 % of the packets carried at least once: temperatures within 0.5 % shell by
          shell and the spectrum within 3 % band by band of the uncarried run (the paper's 100 interactions)."""
    N = 20_000
    grey = W.uniform_cube(10, 20.0, 0.6, 0.3, n_nu=32, slope=0.0, T_star=3000.0)
    o = orc.Oracle.from_workload(grey)
    r0 = o.run(N, 19, n_threads=NTH, digests=True)
    raw0 = o.read_raw()
    n_int = r0["digests"]["absorptions"].astype(np.int64) + r0["digests"]["scatterings"]
    assert (n_int > 100).mean() > 0.5 and n_int.max() > 1000
    r1 = o.run(N, 19, n_threads=NTH, digests=True, carry_K=100)
    raw1 = o.read_raw()
    assert r1["epochs"] > r0["epochs"]                                        # further epochs drained the carried packets
    for key in ("k", "lucy_fx"):                                              # (a)
        assert np.array_equal(raw0[key], raw1[key]), key
    for key in ("crossings", "scatterings", "absorptions", "escape_bin"):
        assert np.array_equal(r0["digests"][key], r1["digests"][key]), key
    assert not np.array_equal(r0["digests"]["hash"], r1["digests"]["hash"])   # ... but re-emitted frequencies differ
    assert int(raw1["sed"].sum()) == N == r1["escapes"] == r1["packets"]      # (b)
    assert int(raw1["k"].sum()) == r1["absorptions"] and r1["flights"] == N + r1["scatterings"] + r1["absorptions"]
    r2 = o.run(N, 19, n_threads=1, digests=True, carry_K=100)                 # (c)
    raw2 = o.read_raw()
    for key in raw1:
        assert np.array_equal(raw1[key], raw2[key]), key
    assert np.array_equal(r1["digests"], r2["digests"])
    r3 = o.run(N, 19, n_threads=NTH, digests=True, carry_K=int(n_int.max()) + 1)   # (d)
    raw3 = o.read_raw()
    for key in raw0:
        assert np.array_equal(raw0[key], raw3[key]), key
    assert np.array_equal(r0["digests"], r3["digests"]) and r3["epochs"] == r0["epochs"]
    # (e)
    chrom = W.uniform_cube(10, 40.0, 0.6, 0.3, n_nu=32, slope=-0.3, T_star=3000.0)
    oc = orc.Oracle.from_workload(chrom)
    N2 = 40_000
    ra = oc.run(N2, 17, n_threads=NTH, digests=True)
    Ta, sa = oc.read()["T"].astype(float), oc.read_raw()["sed"].sum(axis=0).astype(float)
    rb = oc.run(N2, 17, n_threads=NTH, digests=True, carry_K=100)
    Tb, sb = oc.read()["T"].astype(float), oc.read_raw()["sed"].sum(axis=0).astype(float)
    na = ra["digests"]["absorptions"].astype(np.int64) + ra["digests"]["scatterings"]
    assert (na > 100).mean() > 0.5
    assert (ra["digests"]["hash"] != rb["digests"]["hash"]).mean() > 0.5
    x = (np.arange(10) + 0.5) - 5
    rr = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2).reshape(-1)
    for lo in range(5):
        sel = (rr >= lo) & (rr < lo + 1)
        assert abs(Tb[sel].mean() / Ta[sel].mean() - 1) < 0.005, lo
    ba, bb = sa.reshape(8, 4).sum(axis=1), sb.reshape(8, 4).sum(axis=1)
    sel = ba > 300
    assert sel.sum() >= 3 and np.all(np.abs(bb[sel] / ba[sel] - 1) < 0.03 + 3 / np.sqrt(ba[sel]))


# ------------------------------------------------------------------------------------------ P20 scattering store + ray tracer
def _bin_edges(nu):
    return np.concatenate([[nu[0] * math.sqrt(nu[0] / nu[1])], np.sqrt(nu[:-1] * nu[1:]), [nu[-1] * math.sqrt(nu[-1] / nu[-2])]])


def test_p20_phase_function_and_event_store(orc):
    """NEXT-2 (Eq. 15-16).  P_HG is normalised over the sphere and 1/4pi for g = 0; with every frequency
    bin recorded the store holds exactly one event per scattering, in dusty cells, with unit incoming directions."""
    mu = (np.arange(4000) + 0.5) / 4000 * 2 - 1
    for g in (0.0, 0.3, -0.5, 0.8):
        p = np.array([orc.phase_hg(g, m) for m in mu])
        assert abs(2 * math.pi * p.mean() * 2 - 1) < 1e-4
    assert abs(orc.phase_hg(0.0, 0.3) - 1 / (4 * math.pi)) < 1e-16
    assert abs(orc.phase_hg(0.6, 1.0) / orc.phase_hg(0.6, -1.0) - ((1 + 0.6) / (1 - 0.6)) ** 3) < 1e-9
    w = W.uniform_cube(8, 2.0, 0.7, 0.4, n_nu=12, slope=-1.0)
    o = orc.Oracle.from_workload(w)
    o.scatter_store(list(range(12)), 400_000)
    r = o.run(30_000, 20, n_threads=NTH)
    ev, n = o.scatter_events()
    assert n == r["scatterings"] == len(ev)
    assert np.all(w.rho.reshape(-1)[ev["cell"]] > 0) and ev["slot"].max() < 12
    qn = np.sqrt((ev["q"].astype(np.float64) ** 2).sum(axis=1))
    assert np.all(np.abs(qn / 32767.0 - 1) < 1e-4)
    # the next B&W run starts an empty store; a store with too little room counts what it could not keep
    busiest = int(np.bincount(ev["slot"], minlength=12).argmax())
    o.scatter_store([busiest], 10)
    r = o.run(30_000, 20, n_threads=NTH)
    ev, n = o.scatter_events()
    assert len(ev) == 10 and 10 < n < r["scatterings"] and np.all(ev["slot"] == 0)


def test_p20_ray_tracer_emission(orc):
    """Eq. 12-14, 17.  (a) Optically thin dust in radiative equilibrium re-radiates what it absorbs: summed over
    frequency and over the image, D^2 sum F_e dnu = sum_i E_i / 4 pi (Eq. 4 makes sum_j kappa_j B_j(T_i) dnu_j =
    E_i / 4 pi rho V), whatever the direction of the observer.  (b) An opaque cube shows the Planck function
    of the temperature of the cells on the OBSERVER's side (source off-centre, so the two sides differ)."""
    n = 12
    lam = W.wavelength_grid_um(24, 0.3, 3000.0)
    nu = W.nu_from_lambda_um(lam)
    kabs = 50.0 * (nu / nu[-1]) ** 1.0
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    rho = np.where(r < n / 2, 2e-3 / (kabs.max() * n / 2 * h), 0.0).astype(np.float32)
    c = n / 2 * h
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 1, nu, kabs[None], np.zeros((1, len(nu))),
                   np.zeros((1, len(nu))), W.temperature_grid(1000, 2.0, 2000.0), W.LSUN_ERG_S, 3000.0, None, [c, c, c], [0.0, 1.0])
    N = 400_000
    o.run(N, 21, n_threads=NTH)
    E_abs = o.read()["E_lucy"].sum()           # absorbed luminosity (path-length estimate: smooth in thin dust)
    dnu = np.diff(_bin_edges(nu))
    D, npx = 3.0e18, 88            # pixels of a quarter cell (the image covers the cube seen from any side)
    for ez, ex in (((0.0, 0.0, 1.0), (1.0, 0.0, 0.0)), ((0.6, -0.48, 0.64), (0.0, 0.8, 0.6))):
        tot = 0.0
        for j in range(len(nu)):
            Fe, Fs = o.ray_trace(ez, ex, npx, npx, h / 4, D, j, T_from_lucy=True)
            assert np.all(Fs == 0.0) and np.all(Fe >= 0.0)
            tot += Fe.sum() * dnu[j]
        assert abs(tot * D * D / (E_abs / (4 * math.pi)) - 1) < 0.02, (ez, tot)
    # (b) a cube that is opaque at the traced (shortest) wavelength and thin in the infrared, source off-centre along x
    w = W.uniform_cube(6, 60.0, 0.0, 0.0, n_nu=16, slope=-1.5, T_star=4000.0, source_offset_cells=(1.5, 0.0, 0.0))
    o2 = orc.Oracle.from_workload(w)
    o2.run(100_000, 22, n_threads=NTH)
    T = o2.read()["T"].reshape(6, 6, 6).astype(np.float64)
    j = 15
    assert w.kappa_abs[0, j] * float(w.rho.flat[0]) * w.cell_size_cm > 100.0
    pix = w.cell_size_cm
    for ez, face in (((1.0, 0.0, 0.0), T[:, :, 5]), ((-1.0, 0.0, 0.0), T[:, :, 0])):
        Fe, _ = o2.ray_trace(ez, (0.0, 1.0, 0.0), 6, 6, pix, D, j)
        # image axes: e_x' = +y, e_y' = e_z' x e_x' = +-z: pixel (a, b) looks at cell (y = a, z = b or 5 - b)
        want = np.array([[orc.planck(w.nu_hz[j], face[b if ez[0] > 0 else 5 - b, a]) for a in range(6)] for b in range(6)])
        np.testing.assert_allclose(Fe * D * D / pix ** 2, want, rtol=2e-3)     # (T is read back as fp32; h nu / k T is several hundred here)
    assert abs(T[:, :, 5].mean() / T[:, :, 0].mean() - 1) > 0.02          # the two sides do differ


def test_p20_ray_tracer_scattering(orc):
    """Eq. 15-17.  (a) A pure scatterer neither absorbs nor attenuates (Eq. 13 has the absorption cross section), so
    every stored event sends xi P_HG / dnu per steradian to the observer: for g = 0 the image sums to
    N xi / (4 pi dnu D^2), N = number of stored events, for any direction.  (b) Two small clouds in front of and
    behind the source as seen by the observer: per event, forward / backward scattering = ((1+g)/(1-g))^3."""
    n, D = 10, 3.0e18
    w = W.uniform_cube(n, 0.3, 1.0 - 1e-12, 0.0, n_nu=8, slope=0.0, T_star=5000.0)
    o = orc.Oracle.from_workload(w)
    j = 5                                  # 1.4 um: near the peak of the 5000 K source on this 8-point grid
    o.scatter_store([j], 2_000_000)
    N = 300_000
    r = o.run(N, 23, n_threads=NTH)
    ev, ne = o.scatter_events()
    assert ne == len(ev) > 5000 and r["absorptions"] == 0
    xi = w.L_erg_s / N
    dnu = np.diff(_bin_edges(w.nu_hz))
    npx = 72
    for ez, ex in (((0.0, 0.0, 1.0), (1.0, 0.0, 0.0)), ((0.48, 0.6, -0.64), (0.8, 0.0, 0.6))):
        Fe, Fs = o.ray_trace(ez, ex, npx, npx, w.cell_size_cm / 4, D, j)
        assert np.all(Fe == 0.0)
        assert abs(Fs.sum() / (ne * xi / (4 * math.pi * dnu[j] * D * D)) - 1) < 0.01
    # (b)
    g = 0.6
    w2 = W.uniform_cube(15, 1.0, 1.0 - 1e-12, g, n_nu=8, slope=0.0, T_star=5000.0)
    rho0 = w2.rho.max()
    w2.rho[...] = 0.0
    w2.rho[7, 7, 13] = rho0 * 0.5      # between the source (centre of cell 7,7,7) and an observer at +x
    w2.rho[7, 7, 1] = rho0 * 0.5       # behind the source
    o2 = orc.Oracle.from_workload(w2)
    o2.scatter_store([j], 1_000_000)
    o2.run(3_000_000, 24, n_threads=NTH)
    ev, ne = o2.scatter_events()
    cell_near, cell_far = (7 * 15 + 7) * 15 + 13, (7 * 15 + 7) * 15 + 1
    n_near, n_far = int((ev["cell"] == cell_near).sum()), int((ev["cell"] == cell_far).sum())
    assert n_near > 150 and n_far > 150 and n_near + n_far == ne
    npx = 60
    Fe, Fs = o2.ray_trace((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), npx, npx, 15 * w2.cell_size_cm / npx, D, j)
    # parallel projection along x: both clouds fall on the same pixels, so separate them by tracing each alone
    keep = w2.rho.copy()
    per = {}
    for name, cell in (("near", (7, 7, 13)), ("far", (7, 7, 1))):
        w3 = W.uniform_cube(15, 1.0, 1.0 - 1e-12, g, n_nu=8, slope=0.0, T_star=5000.0)
        w3.rho[...] = 0.0
        w3.rho[cell] = rho0 * 0.5
        o3 = orc.Oracle.from_workload(w3)
        o3.scatter_store([j], 1_000_000)
        o3.run(3_000_000, 24, n_threads=NTH)
        ev3, ne3 = o3.scatter_events()
        _, Fs3 = o3.ray_trace((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), npx, npx, 15 * w3.cell_size_cm / npx, D, j)
        per[name] = Fs3.sum() / ne3
    ratio = per["near"] / per["far"]
    assert abs(ratio / ((1 + g) / (1 - g)) ** 3 - 1) < 0.08, ratio
    assert abs(Fs.sum() / (per["near"] * n_near + per["far"] * n_far) - 1) < 0.05


# ------------------------------------------------------------------------------------------ P21 stratified source
def test_p21_stratified_source_frequencies(orc):
    """NEXT-4, Eq. 1 (1000 equal-energy bins x 1e5 packets at PAPER.md:232): with as many strata as
    packets every packet takes its own quantile slice of the cumulative source spectrum, so the number of packets
    emitted in frequency bin j is N p_j to within the two slices that straddle the bin's ends -- a deterministic
    bound, where plain sampling scatters by sqrt(N p_j)."""
    w = W.uniform_cube(4, 0.0, 0.5, 0.0, n_nu=24, T_star=5000.0)
    o = orc.Oracle.from_workload(w)
    N = 100_000
    p = np.diff(np.concatenate([[0.0], o.tables()["srccdf"]]))
    o.run(N, 21, n_threads=NTH, source_strata=N)
    cnt = o.read_raw()["sed"].sum(axis=0).astype(np.int64)
    assert cnt.sum() == N and np.all(np.abs(cnt - N * p) < 2.0)
    o.run(N, 21, n_threads=NTH)                      # plain sampling: far outside that bound
    cnt0 = o.read_raw()["sed"].sum(axis=0).astype(np.int64)
    assert np.abs(cnt0 - N * p).max() > 20
    o.run(N, 21, n_threads=NTH, source_strata=1000)  # 1000 strata x 100 packets, the paper's proportions
    cnt1 = o.read_raw()["sed"].sum(axis=0).astype(np.int64)
    big = N * p > 2000
    assert np.all(np.abs(cnt1 - N * p)[big] < 0.35 * np.sqrt(N * p)[big] + 15)


# ------------------------------------------------------------------------------------------ P22 dust mixtures (NEXT-3)
def test_p22_one_component_mixtures_and_identical_halves(orc):
    """Readings Q34-Q36: (i) a mixture table that names every material as its own one-component mixture is the run
    without mixtures, bit for bit (digests, tallies); (ii) two halves (f = 1/2 each: scaling by 1/2 is exact) of the
    SAME material give the same trajectories as that material alone when absorbed packets end, the absorptions are
    split between the halves cell by cell (k0 + k1 = k), binomially, and each half's Lucy tally is half the
    material's up to the rounding of the fixed-point adds."""
    w = W.uniform_cube(12, tau_edge_V=3.0, albedo=0.6, g_const=0.5, n_nu=12, slope=1.0)
    N = 40_000
    a = orc.Oracle.from_workload(w)
    ra = a.run(N, seed=221, digests=True, n_threads=NTH)
    w.mixtures = ([1], [[0, 0]], [[1.0, 0.0]])
    b = orc.Oracle.from_workload(w)
    rb = b.run(N, seed=221, digests=True, n_threads=NTH)
    assert np.array_equal(ra["digests"], rb["digests"])
    A, B = a.read_raw(), b.read_raw()
    for key in ("k", "lucy_fx", "sed", "tidx"):
        assert np.array_equal(A[key], B[key]), key
    assert not b.read_raw_comp1()["k"].any()
    # (ii)
    a2 = orc.Oracle.from_workload(W.uniform_cube(12, tau_edge_V=3.0, albedo=0.6, g_const=0.5, n_nu=12, slope=1.0))
    r1 = a2.run(N, seed=222, digests=True, absorb_and_stop=True, n_threads=NTH)
    w.mixtures = ([2], [[0, 0]], [[0.5, 0.5]])
    c = orc.Oracle.from_workload(w)
    r2 = c.run(N, seed=222, digests=True, absorb_and_stop=True, n_threads=NTH)
    assert np.array_equal(r1["digests"], r2["digests"])
    k = a2.read_raw()["k"].astype(np.int64)
    k0, k1 = c.read_raw()["k"].astype(np.int64), c.read_raw_comp1()["k"].astype(np.int64)
    assert np.array_equal(k0 + k1, k)
    K = int(k.sum())
    assert abs(int(k1.sum()) - K / 2) < 4 * math.sqrt(K / 4) and k1.sum() > 0
    L, L0, L1 = a2.read_raw()["lucy_fx"], c.read_raw()["lucy_fx"], c.read_raw_comp1()["lucy_fx"]
    assert np.array_equal(L0, L1)
    assert np.abs(2 * L0 - L).max() <= r1["lucy_adds"] and L.max() > 1e6   # at most one unit per add


def test_p22_thin_mixture_component_temperatures(orc):
    """Reading Q36 against radiative balance: in an optically thin sphere around a blackbody source two power-law
    materials (kappa ~ nu^beta_c) mixed 30 % / 70 % by mass each reach THEIR OWN temperature
    T_c = T* (R*/2r)^(2/(4+beta_c)), whatever the other one does; and each component's Lucy tally per unit of its own
    mass, times 16 pi^2 r^2 / L, is the source-weighted mean of its own kappa.  Fails when a component is tallied
    with the other's opacity, when Eq. 4 uses the cell's whole mass, or when the fractions are swapped."""
    betas, fr, Tstar, n, N = (1.0, 2.0), (0.3, 0.7), 1500.0, 24, 600_000
    lam = W.wavelength_grid_um(160, 0.2, 1e5)
    nu = W.nu_from_lambda_um(lam)
    kabs = np.stack([100.0 * (nu / nu[-1]) ** b for b in betas])
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    rho0 = 1e-3 / (kabs.max() * n / 2 * h)
    rho = np.where(r < n / 2, rho0, 0.0).astype(np.float32)
    L = W.LSUN_ERG_S
    c = n / 2 * h
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 2, nu, kabs, np.zeros((2, len(nu))),
                   np.zeros((2, len(nu))), W.temperature_grid(1000, 2.0, 2000.0), L, Tstar, None, [c, c, c],
                   [0.0, 1.0], mixtures=([2], [[0, 1]], [list(fr)]))
    res = o.run(N, seed=8, n_threads=NTH)
    assert res["absorptions"] < 0.01 * N
    T = [o.read(T_from_lucy=True)["T"].reshape(n, n, n).astype(np.float64),
         o.read_comp1(T_from_lucy=True)["T"].reshape(n, n, n).astype(np.float64)]
    E = [o.read()["E_lucy"].reshape(n, n, n), o.read_comp1()["E_lucy"].reshape(n, n, n)]
    Rstar = math.sqrt(L / (4 * math.pi * SIGMA_SB * Tstar ** 4))
    pj = np.diff(np.concatenate([[0.0], o.tables()["srccdf"]]))
    for comp in (0, 1):
        for r_lo in (4.0, 7.0, 10.0):
            sel = (r >= r_lo) & (r < r_lo + 1.0)
            T_exp = Tstar * (Rstar / (2 * r[sel] * h)) ** (2 / (4 + betas[comp]))
            assert abs((T[comp][sel] / T_exp).mean() - 1) < 0.01, (comp, r_lo)
        sel = (r >= 5.0) & (r < 9.0)
        xcell = E[comp][sel] / (4 * math.pi * rho0 * fr[comp] * h ** 3)
        got = (xcell * (r[sel] * h) ** 2).mean() * 16 * math.pi ** 2 / L
        assert abs(got / (kabs[comp] * pj).sum() - 1) < 0.01, comp
    sel = (r >= 4.0) & (r < 5.0)
    assert T[1][sel].mean() / T[0][sel].mean() > 1.2      # the two laws are far apart: (R*/2r)^(2/6 - 2/5), R* << r


def test_p22_mixture_random_flight_and_absorption_split(orc):
    """Reading Q35 against the random-flight closed form of P18: in an infinite uniform grey medium made of a forward
    scattering material (g = 0.8) and an isotropic one (g = 0), with different albedos and mixed 40 % / 60 %, the
    packets end at <R^2> = 2 l^2 / [(1 - a)(1 - a g)] with l = 1/(kext_x rho), a the mixture's albedo and g the
    mean cosine over all scatterings, g = (f0 ks0 g0 + f1 ks1 g1) / (f0 ks0 + f1 ks1); the absorptions go to the
    components in the ratio f0 ka0 : f1 ka1.  Fails when the scattering component's g is taken from the other
    material, when the thresholds are in the wrong order, or when the fractions do not enter kext."""
    n, N = 160, 200_000
    f = (0.4, 0.6)
    ka, ks, gg = (30.0, 90.0), (210.0, 60.0), (0.8, 0.0)
    nf = 4
    lam = W.wavelength_grid_um(nf, 0.1, 1000.0)
    nu = W.nu_from_lambda_um(lam)
    kext = f[0] * (ka[0] + ks[0]) + f[1] * (ka[1] + ks[1])
    h = W.AU_CM
    ell = 2.0                                             # mean free path in cells
    rho0 = 1.0 / (kext * ell * h)
    rho = np.full((n, n, n), rho0, np.float32)
    kabs = np.stack([np.full(nf, ka[0]), np.full(nf, ka[1])])
    ksca = np.stack([np.full(nf, ks[0]), np.full(nf, ks[1])])
    g = np.stack([np.full(nf, gg[0]), np.full(nf, gg[1])])
    c = n / 2 * h
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 2, nu, kabs, ksca, g, W.temperature_grid(),
                   W.LSUN_ERG_S, 5800.0, None, [c, c, c], [0.0, 1.0], mixtures=([2], [[0, 1]], [list(f)]))
    r = o.run(N, seed=2203, absorb_and_stop=True, B0=N, Bmax=N, n_threads=NTH)
    assert r["escapes"] <= 2e-4 * N and r["absorptions"] + r["escapes"] == N
    ell = 1.0 / (kext * float(rho.flat[0]) * h)
    a = (f[0] * ks[0] + f[1] * ks[1]) / kext
    gbar = (f[0] * ks[0] * gg[0] + f[1] * ks[1] * gg[1]) / (f[0] * ks[0] + f[1] * ks[1])
    assert abs(r["scatterings"] / (r["scatterings"] + r["absorptions"]) - a) < 4 * math.sqrt(a * (1 - a) / r["flights"])
    k0 = o.read_raw()["k"].reshape(n, n, n).astype(np.float64)
    k1 = o.read_raw_comp1()["k"].reshape(n, n, n).astype(np.float64)
    K = k0.sum() + k1.sum()
    p1 = f[1] * ka[1] / (f[0] * ka[0] + f[1] * ka[1])
    assert abs(k1.sum() / K - p1) < 4 * math.sqrt(p1 * (1 - p1) / K)
    k = k0 + k1
    d = (np.arange(n) + 0.5) - n / 2
    X, Y, Z = np.meshgrid(d, d, d, indexing="ij")
    rr2 = Z ** 2 + Y ** 2 + X ** 2
    tot = (k * rr2).sum() / K
    sig = math.sqrt(((k * rr2 ** 2).sum() / K - tot ** 2) / K)
    r2_true = 2 * ell ** 2 / ((1 - a) * (1 - a * gbar))
    assert abs(tot - (r2_true + 0.25)) < 4 * sig, (tot, r2_true + 0.25, sig)
    r2_swapped = 2 * ell ** 2 / ((1 - a) * (1 - a * (f[0] * ks[0] * gg[1] + f[1] * ks[1] * gg[0]) / (f[0] * ks[0] + f[1] * ks[1])))
    assert abs(r2_swapped - r2_true) > 20 * sig           # the pin can tell the two assignments apart


def test_p22_mixture_component_order_is_a_relabelling(orc):
    """Readings Q35/Q36, the second component's share of the path (its frozen temperature index and the row it
    re-emits from): listing a mixture's components in the other order changes nothing physical.  A moderately thick
    sphere (tau ~ 4 at the source's peak) of a grey material and a kappa ~ nu^2 material, 30 % / 70 %: the escaping
    spectrum and both materials' radial temperature profiles of the run with the order (grey, nu^2) agree with those
    of the run with the order (nu^2, grey) within the counting noise.  Together with the pins of the one-material
    path (which component 0 is, bit for bit: P22 (i)) this pins component 1: a wrong mass in its Eq. 4 or a row of
    the other material moves its re-emission by 25 % in frequency."""
    n, N, Tstar = 16, 300_000, 2500.0
    lam = W.wavelength_grid_um(60, 0.1, 3000.0)
    nu = W.nu_from_lambda_um(lam)
    kabs = np.stack([np.full(len(nu), 40.0), 400.0 * (nu / nu[-1]) ** 2])
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    nu_peak = 2.82 * K_BOLTZ * Tstar / H_PLANCK
    k_peak = 0.3 * 40.0 + 0.7 * 400.0 * (nu_peak / nu[-1]) ** 2
    rho0 = 4.0 / (k_peak * n / 2 * h)
    rho = np.where(r < n / 2, rho0, 0.0).astype(np.float32)
    c = n / 2 * h
    zeros = np.zeros((2, len(nu)))
    runs = []
    for order, seed in (((0, 1), 2210), ((1, 0), 2211)):
        fr = [(0.3, 0.7)[m] for m in order]
        o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 2, nu, kabs, zeros, zeros,
                       W.temperature_grid(1000, 2.0, 3000.0), W.LSUN_ERG_S, Tstar, None, [c, c, c], [0.0, 1.0],
                       mixtures=([2], [list(order)], [fr]))
        res = o.run(N, seed=seed, n_threads=NTH)
        assert res["absorptions"] > 2 * N
        sed = o.read_raw()["sed"][0].astype(np.float64)
        T = [o.read(T_from_lucy=True)["T"].reshape(n, n, n).astype(np.float64),
             o.read_comp1(T_from_lucy=True)["T"].reshape(n, n, n).astype(np.float64)]
        Tm = {order[0]: T[0], order[1]: T[1]}               # by MATERIAL
        # ... and a frozen-temperature sweep (S12) at the Lucy temperatures of that run: its escaping spectrum
        o.run(N, seed=seed + 10, mode=orc.MODE_FROZEN_SWEEP, n_sweeps=1, sweep_T_from_lucy=1, reset=False, n_threads=NTH)
        sed_sweep = o.read_raw()["sed"][0].astype(np.float64)
        runs.append((sed, Tm, sed_sweep))
    (sA, TA, wA), (sB, TB, wB) = runs
    for a_, b_ in ((sA, sB), (wA, wB)):
        sel = (a_ + b_) >= 50
        chi2 = ((a_[sel] - b_[sel]) ** 2 / (a_[sel] + b_[sel])).sum()
        ndf = int(sel.sum())
        assert ndf >= 25 and chi2 < ndf + 5 * math.sqrt(2 * ndf), (chi2, ndf)
    for m in (0, 1):
        for r_lo in (2.0, 4.0, 6.0):
            s = (r >= r_lo) & (r < r_lo + 1.0)
            assert abs(TA[m][s].mean() / TB[m][s].mean() - 1) < 0.01, (m, r_lo, TA[m][s].mean(), TB[m][s].mean())
    s = (r >= 4.0) & (r < 5.0)
    assert TA[1][s].mean() / TA[0][s].mean() > 1.1        # the two materials' temperatures differ: the pin has teeth


# ------------------------------------------------------------------------------------------ P23 Eq. 9 hybrid (NEXT-4)
def test_p23_eq9_series_and_threshold(orc):
    """Sect. 3.1, readings Q37 / Q38.  (i) Eq. 9's 1 - e^-tau as the oracle evaluates it (series to
    tau^5) against -expm1(-tau) below the threshold; (ii) which cells are tallied: a slab of cells just below and one
    just above tau_max = sqrt(3) h rho max_nu(kabs + ksca) = 10^-2, and one far above: only the first is tallied, with
    every traversal's (1 - e^-tau_abs), which lies between the linear tally and the linear tally (1 - tau_max/2)."""
    for tau in (1e-9, 1e-6, 1e-4, 3e-3, 9.99e-3):
        assert abs(orc.eq9_value(tau) / -math.expm1(-tau) - 1) < 1e-12
    n = 12
    w = W.uniform_cube(n, tau_edge_V=1.0, albedo=0.4, g_const=0.3, n_nu=12, slope=1.0)
    kmax = float((w.kappa_abs + w.kappa_sca).max())
    rho_at = lambda tau: tau / (math.sqrt(3.0) * w.cell_size_cm * kmax)
    rho = np.zeros((n, n, n), np.float32)
    rho[:, :, 0:4] = rho_at(0.99e-2)
    rho[:, :, 4:8] = rho_at(1.01e-2)
    rho[:, :, 8:12] = rho_at(3.0)
    w.rho = rho
    N = 60_000
    lin = orc.Oracle.from_workload(w)
    lin.run(N, seed=230, absorb_and_stop=True, n_threads=NTH)
    hyb = orc.Oracle.from_workload(w)
    r = hyb.run(N, seed=230, absorb_and_stop=True, lucy_hybrid=True, n_threads=NTH)
    Ll = lin.read_raw()["lucy_fx"].reshape(n, n, n).astype(np.float64)
    Lh = hyb.read_raw()["lucy_fx"].reshape(n, n, n).astype(np.float64)
    assert np.array_equal(lin.read_raw()["k"], hyb.read_raw()["k"])          # the estimator does not touch the transport
    assert not Lh[:, :, 4:].any() and (Lh[:, :, 0:4] > 0).all()
    ratio = Lh[:, :, 0:4] / Ll[:, :, 0:4]
    assert (ratio < 1.0).all() and (ratio > 1.0 - 0.5e-2).all()
    assert r["lucy_adds"] > 0


def test_p23_hybrid_temperatures(orc):
    """Reading Q39 against radiative balance (the closed form of P8): in an optically thin sphere every cell is below
    the threshold, so in hybrid mode the Eq. 9 energy gives the output temperature AND the frozen per-epoch index
    B&W re-emits from: both follow T = T* (R*/2r)^(2/(4+beta)), although hardly any packet is ever absorbed there
    (the count-based index of those cells would sit at the bottom of the T grid).  A sphere 10^5 times denser next to
    it in the same run is above the threshold: no tally, temperature from its counts."""
    beta, Tstar, n, N = 1.0, 1500.0, 24, 600_000
    lam = W.wavelength_grid_um(160, 0.2, 1e5)
    nu = W.nu_from_lambda_um(lam)
    kabs = 100.0 * (nu / nu[-1]) ** beta
    h = W.AU_CM
    x = (np.arange(n) + 0.5) - n / 2
    r = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2)
    rho0 = 1e-3 / (kabs.max() * n / 2 * h)
    rho = np.where(r < n / 2, rho0, 0.0).astype(np.float32)
    L = W.LSUN_ERG_S
    c = n / 2 * h
    Tg = W.temperature_grid(1000, 2.0, 2000.0)
    o = orc.Oracle(n, n, n, h, rho, np.zeros(n ** 3, np.uint8), 1, nu, kabs[None], np.zeros((1, len(nu))),
                   np.zeros((1, len(nu))), Tg, L, Tstar, None, [c, c, c], [0.0, 1.0])
    res = o.run(N, seed=8, lucy_hybrid=True, n_threads=NTH)
    assert res["absorptions"] < 0.01 * N
    T = lib_T = o.read(T_from_lucy=2)["T"].reshape(n, n, n).astype(np.float64)
    tidx = o.read_raw()["tidx"].reshape(n, n, n)
    Rstar = math.sqrt(L / (4 * math.pi * SIGMA_SB * Tstar ** 4))
    for r_lo in (4.0, 7.0, 10.0):
        sel = (r >= r_lo) & (r < r_lo + 1.0)
        T_exp = Tstar * (Rstar / (2 * r[sel] * h)) ** (2 / (4 + beta))
        assert abs((T[sel] / T_exp).mean() - 1) < 0.01, r_lo
        # the index the LAST epoch re-emitted from (midpoint prediction of the tally at ~98 % of the run): first grid T above
        assert abs((Tg[tidx[sel]] / T_exp).mean() - 1) < 0.02, r_lo
    assert (o.read_raw()["k"].reshape(n, n, n)[(r >= 7.0) & (r < 8.0)] == 0).mean() > 0.9
    # a thick cell in the same kind of run: no tally, T from counts
    rho2 = rho.copy()
    rho2[n // 2 - 2:n // 2 + 2, n // 2 - 2:n // 2 + 2, n // 2 - 2:n // 2 + 2] = rho0 * 1e5
    o2 = orc.Oracle(n, n, n, h, rho2, np.zeros(n ** 3, np.uint8), 1, nu, kabs[None], np.zeros((1, len(nu))),
                    np.zeros((1, len(nu))), Tg, L, Tstar, None, [c, c, c], [0.0, 1.0])
    o2.run(60_000, seed=9, lucy_hybrid=True, n_threads=NTH)
    core = (slice(n // 2 - 2, n // 2 + 2),) * 3
    assert not o2.read_raw()["lucy_fx"].reshape(n, n, n)[core].any()
    Th, Tc = o2.read(T_from_lucy=2)["T"].reshape(n, n, n)[core], o2.read(T_from_lucy=False)["T"].reshape(n, n, n)[core]
    assert np.array_equal(Th, Tc) and (Tc > 0).all()
    # ... and a frozen-T sweep in hybrid mode takes the core's index from its counts, the thin cells' from their tally
    Tl = o2.read(T_from_lucy=2)["T"].reshape(n, n, n).astype(np.float64)
    o2.run(20_000, seed=11, mode=orc.MODE_FROZEN_SWEEP, n_sweeps=1, lucy_hybrid=True, reset=False, n_threads=NTH)
    t2 = o2.read_raw()["tidx"].reshape(n, n, n)
    assert (t2[core] > 0).all() and np.abs(Tg[t2[core]] / Tc - 1).max() < 0.02
    shell = (r >= 7.0) & (r < 8.0)
    assert abs((Tg[t2[shell]] / Tl[shell]).mean() - 1) < 0.02


# ------------------------------------------------------------------------------------------ P24 sub-cubes (NEXT-3)
def _fine_medium(nf_cells, seed, n_species=2):
    """A random clumpy medium on a fine grid: densities over two decades, a quarter of the cells empty."""
    rng = np.random.default_rng(seed)
    rho = (10.0 ** rng.uniform(-1.5, 0.5, (nf_cells,) * 3)).astype(np.float32)
    rho[rng.random((nf_cells,) * 3) < 0.25] = 0.0
    sp = rng.integers(0, n_species, (nf_cells,) * 3).astype(np.uint8)
    return rho, sp


def _two_species_cube(n, tau_edge):
    w = W.uniform_cube(n, tau_edge_V=tau_edge, albedo=0.5, g_const=0.4, n_nu=16, slope=1.0, source_offset_cells=(0.3, -0.2, 0.1))
    w.kappa_abs = np.vstack([w.kappa_abs, 0.5 * w.kappa_abs[:1]])
    w.kappa_sca = np.vstack([w.kappa_sca, 2.0 * w.kappa_sca[:1]])
    w.g = np.vstack([w.g, 0.0 * w.g[:1] - 0.2])
    w.n_species = 2
    return w


def _to_blocks(fine, n, R):
    """[nR]^3 array -> [n^3 cubes][R^3] in cube order (z, y, x) and sub-cube order (z, y, x)."""
    return fine.reshape(n, R, n, R, n, R).transpose(0, 2, 4, 1, 3, 5).reshape(n ** 3, R ** 3)


@pytest.mark.parametrize("R", [2, 4])
def test_p24_fully_refined_grid_is_the_fine_uniform_grid(orc, R):
    """Reading Q40 against the uniform-grid path (itself pinned by P2-P18): with EVERY cube divided into R^3 sub-cubes
    the run is the run on the (n R)^3 uniform grid of cell size h/R -- face coordinates c + k/R, chord lengths and
    volumes differ from the fine grid's by exact powers of two -- so every packet makes the same crossings, scatterings
    and absorptions and escapes into the same bin, and every sub-cube has the fine cell's count, tally and temperature
    index, bit for bit, through B&W epochs and a sweep."""
    n, N = 6, 20_000
    nfc = n * R
    fine = _two_species_cube(nfc, tau_edge=1.5)
    rho_f, sp_f = _fine_medium(nfc, 240 + R)
    rho_f *= np.float32(fine.rho.flat[0])
    fine.rho, fine.species = rho_f, sp_f
    coarse = _two_species_cube(n, tau_edge=1.5)
    coarse.cell_size_cm = fine.cell_size_cm * R
    coarse.source_pos_cm = fine.source_pos_cm
    coarse.rho = np.ones((n, n, n), np.float32)
    coarse.species = np.zeros((n, n, n), np.uint8)
    coarse.subgrid = (R, np.arange(n ** 3), _to_blocks(rho_f, n, R), _to_blocks(sp_f, n, R))
    of, oc = orc.Oracle.from_workload(fine), orc.Oracle.from_workload(coarse)
    for step in range(2):
        kw = dict(n_threads=NTH, digests=True) if step == 0 else dict(n_threads=NTH, digests=True, mode=orc.MODE_FROZEN_SWEEP, n_sweeps=1, reset=False)
        rf, rc = of.run(N, 2400 + step, **kw), oc.run(N, 2400 + step, **kw)
        for key in ("crossings", "dusty_crossings", "scatterings", "absorptions", "escapes", "direct_escapes", "lucy_adds"):
            assert rf[key] == rc[key], key
        for key in ("crossings", "scatterings", "absorptions", "escape_bin"):
            assert np.array_equal(rf["digests"][key], rc["digests"][key]), key
        F, Cc = of.read_raw(), oc.read_raw()
        assert np.array_equal(F["sed"], Cc["sed"])
        for key in ("k", "lucy_fx", "tidx"):
            assert not Cc[key][:n ** 3].any()                               # refined cubes hold nothing themselves
            assert np.array_equal(_to_blocks(F[key].reshape(nfc, nfc, nfc), n, R).reshape(-1), Cc[key][n ** 3:]), (step, key)
        assert F["k"].sum() > N / 4
    assert np.array_equal(_to_blocks(of.read()["T"].reshape(nfc, nfc, nfc), n, R).reshape(-1), oc.read()["T"][n ** 3:])


def test_p24_partly_refined_grid(orc):
    """Cubes of a coarse grid divided here and there (a third of them, R = 4), the others not: the medium is the same
    as the fine uniform grid's in which an undivided cube is R^3 equal cells, so the statistics agree -- absorptions
    per coarse cube, their split over the sub-cubes of the divided cubes (this is what a wrong sub-cube at the entry
    from an undivided cube, or a wrong row kept from a divided one, changes), and the escaping spectrum -- and the
    temperature of a sub-cube comes from its own volume (h/R)^3."""
    n, R, N = 6, 4, 200_000
    nfc = n * R
    rng = np.random.default_rng(77)
    refined = rng.random(n ** 3) < 0.35
    refined[(n ** 3) // 2 + n // 2] = True
    rho_f, sp_f = _fine_medium(nfc, 99)
    base = _two_species_cube(nfc, tau_edge=1.5)
    rho_f *= np.float32(base.rho.flat[0])
    rb, sb = _to_blocks(rho_f, n, R), _to_blocks(sp_f, n, R)
    rb[~refined] = rb[~refined][:, :1]                  # an undivided cube: one density, one species
    sb[~refined] = sb[~refined][:, :1]
    back = lambda blocks: blocks.reshape(n, n, n, R, R, R).transpose(0, 3, 1, 4, 2, 5).reshape(nfc, nfc, nfc)
    base.rho, base.species = np.ascontiguousarray(back(rb)), np.ascontiguousarray(back(sb))
    coarse = _two_species_cube(n, tau_edge=1.5)
    coarse.cell_size_cm = base.cell_size_cm * R
    coarse.source_pos_cm = base.source_pos_cm
    coarse.rho = np.where(refined, 1.0, rb[:, 0]).astype(np.float32).reshape(n, n, n)
    coarse.species = sb[:, 0].reshape(n, n, n).copy()
    idx = np.flatnonzero(refined)
    coarse.subgrid = (R, idx, rb[idx], sb[idx])
    of, oc = orc.Oracle.from_workload(base), orc.Oracle.from_workload(coarse)
    rf = of.run(N, 2411, n_threads=NTH, absorb_and_stop=True)
    rc = oc.run(N, 2412, n_threads=NTH, absorb_and_stop=True)
    assert rc["crossings"] < rf["crossings"]            # undivided cubes are crossed in one step
    kf = _to_blocks(of.read_raw()["k"].reshape(nfc, nfc, nfc), n, R).astype(np.float64)
    kc_raw = oc.read_raw()["k"].astype(np.float64)
    kc = np.zeros_like(kf)
    kc[~refined, 0] = kc_raw[:n ** 3][~refined]
    kc[idx] = kc_raw[n ** 3:].reshape(len(idx), R ** 3)
    a, b = kf.sum(axis=1), kc.sum(axis=1)               # per coarse cube
    sel = (a + b) >= 40
    chi2 = ((a[sel] - b[sel]) ** 2 / (a[sel] + b[sel])).sum()
    assert sel.sum() > 100 and chi2 < sel.sum() + 5 * math.sqrt(2 * sel.sum()), (chi2, sel.sum())
    a, b = kf[idx].reshape(-1), kc[idx].reshape(-1)     # per sub-cube of the divided cubes
    sel = (a + b) >= 30
    chi2 = ((a[sel] - b[sel]) ** 2 / (a[sel] + b[sel])).sum()
    assert sel.sum() > 300 and chi2 < sel.sum() + 5 * math.sqrt(2 * sel.sum()), (chi2, sel.sum())
    assert abs(rf["absorptions"] - rc["absorptions"]) < 5 * math.sqrt(2 * rf["absorptions"])
    # temperatures (full B&W runs): a divided cube's sub-cubes against the fine grid's cells (a wrong volume in Eq. 4,
    # h^3 for (h/R)^3, would shift every one of them by a factor 64^(1/5) or so)
    of.run(60_000, 2413, n_threads=NTH); oc.run(60_000, 2414, n_threads=NTH)
    Tf = _to_blocks(of.read(T_from_lucy=True)["T"].reshape(nfc, nfc, nfc).astype(np.float64), n, R)[idx].reshape(-1)
    Tc = oc.read(T_from_lucy=True)["T"][n ** 3:].astype(np.float64)
    ok = (Tf > 0) & (Tc > 0)
    assert ok.sum() > 1000 and abs(np.log(Tc[ok] / Tf[ok]).mean()) < 0.01 and abs(np.median(np.log(Tc[ok] / Tf[ok]))) < 0.01
