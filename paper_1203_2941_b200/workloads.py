"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic lives here).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It builds the
*inputs* of the transport problem -- density cube, species cube, frequency grid, opacity
tables, asymmetry factors, T grid, source description, escape-bin edges -- for the five
configurations named in BASELINE.json / SURVEY.md section 8(d).  It imports neither the
binding nor the oracle, draws its geometry random numbers from numpy's seeded generator,
and performs no transport, no Planck integrals, no sampling.

The inputs stand in for the paper's own workloads, whose opacity data are not available:
  * constant-density / r^-2 shell of PAPER.md:166 (Sect. 3.6, Table 1 workload),
  * the Pascucci disk of PAPER.md:236-263 (Sect. 5.2, Table 2, Eq. 18-19),
  * the clumpy AGN torus of PAPER.md:302-311 (Sect. 6, Eq. 21).
Recipe details are restated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# physical constants used only to express the inputs in cgs
AU_CM = 1.495978707e13
PC_CM = 3.0856775814913673e18
LSUN_ERG_S = 3.828e33
RSUN_CM = 6.957e10
SIGMA_SB = 5.670374419e-5
C_CM_S = 2.99792458e10
KAPPA_V_EXT = 3.5e4  # cm^2 g^-1 at 0.55 um, PAPER.md:295 (Sect. 6)
LAMBDA_V_UM = 0.55


@dataclasses.dataclass
class Workload:
    """Plain container of problem inputs (all numpy, host side)."""

    name: str
    nx: int
    ny: int
    nz: int
    cell_size_cm: float
    rho: np.ndarray  # float32 [nz][ny][nx], g cm^-3
    species: np.ndarray  # uint8   [nz][ny][nx]
    n_species: int
    nu_hz: np.ndarray  # float64 [n_nu], ascending
    kappa_abs: np.ndarray  # float64 [n_species][n_nu], cm^2 g^-1
    kappa_sca: np.ndarray  # float64 [n_species][n_nu]
    g: np.ndarray  # float64 [n_species][n_nu]
    T_grid: np.ndarray  # float64 [n_T], ascending, K
    L_erg_s: float
    T_star_K: float  # > 0: blackbody source; <= 0: use L_nu_weights
    L_nu_weights: np.ndarray | None  # float64 [n_nu] spectral shape L_nu(nu_j), or None
    source_pos_cm: tuple[float, float, float]
    abs_mu_edges: np.ndarray  # float64 [n_dir+1], ascending in |cos i|, 0..1
    n_packets: int  # the configuration's full packet count
    seed: int
    meta: dict = dataclasses.field(default_factory=dict)
    # NEXT-3: (n_components[n_species], material[n_species][2], mass fraction[n_species][2]): cell species x is a mixture
    # of one or two of the n_species materials (None: species x is material x)
    mixtures: tuple | None = None
    # NEXT-3: (R, cube[n_sub], rho_sub[n_sub][R^3], species_sub[n_sub][R^3]): the cubes with these cell indices are divided
    # into R^3 sub-cubes (z, y, x order) with their own densities and species; rho of such a cube must be > 0 (a placeholder)
    subgrid: tuple | None = None

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_nu(self) -> int:
        return int(self.nu_hz.shape[0])

    @property
    def n_dir(self) -> int:
        return int(self.abs_mu_edges.shape[0]) - 1


# ----------------------------------------------------------------------------- grids


def wavelength_grid_um(n: int, lam_min: float, lam_max: float) -> np.ndarray:
    """n log-spaced wavelengths, inclusive of both ends, ascending in lambda."""
    return np.exp(np.linspace(math.log(lam_min), math.log(lam_max), n))


def nu_from_lambda_um(lam_um: np.ndarray) -> np.ndarray:
    """Frequencies in Hz, returned ASCENDING (i.e. wavelength descending)."""
    nu = C_CM_S / (lam_um * 1e-4)
    return np.ascontiguousarray(nu[::-1])


def lambda_um_from_nu(nu_hz: np.ndarray) -> np.ndarray:
    return C_CM_S / nu_hz * 1e4


def temperature_grid(n_T: int = 1000, T_min: float = 2.0, T_max: float = 2000.0) -> np.ndarray:
    return np.exp(np.linspace(math.log(T_min), math.log(T_max), n_T))


# ----------------------------------------------------------------------------- dust tables


def _gauss_lnlam(lam_um: np.ndarray, centre_um: float, sigma_ln: float) -> np.ndarray:
    x = (np.log(lam_um) - math.log(centre_um)) / sigma_ln
    return np.exp(-0.5 * x * x)


def dust_powerlaw(lam_um: np.ndarray, slope: float, albedo_V: float, g_const: float | None):
    """kappa_abs, kappa_sca both proportional to lambda^slope with a constant albedo; constant g."""
    kext = KAPPA_V_EXT * (lam_um / LAMBDA_V_UM) ** slope
    ksca = albedo_V * kext
    kabs = kext - ksca
    g = np.full_like(lam_um, 0.5 if g_const is None else g_const)
    return kabs, ksca, g


def dust_silicate_like(lam_um: np.ndarray, slope: float = -1.6, bump10: float = 0.05, bump18: float = 0.02,
                       albedo_V: float = 0.5):
    """Synthetic silicate-like table: power law + Gaussian 9.7 / 18 um bumps."""
    shape_abs = (lam_um / LAMBDA_V_UM) ** slope + bump10 * _gauss_lnlam(lam_um, 9.7, 0.15) \
        + bump18 * _gauss_lnlam(lam_um, 18.0, 0.2)
    shape_sca = np.minimum(1.0, (lam_um / LAMBDA_V_UM) ** -4.0)
    kabs = (1.0 - albedo_V) * KAPPA_V_EXT * shape_abs
    ksca = albedo_V * KAPPA_V_EXT * shape_sca
    g = 0.7 * np.maximum(0.0, 1.0 - np.log10(lam_um / 0.1) / 2.0)
    g = np.minimum(g, 0.7)
    return kabs, ksca, g


def dust_carbon_like(lam_um: np.ndarray, slope: float = -1.2, albedo_V: float = 0.4):
    shape_abs = (lam_um / LAMBDA_V_UM) ** slope
    shape_sca = np.minimum(1.0, (lam_um / LAMBDA_V_UM) ** -4.0)
    kabs = (1.0 - albedo_V) * KAPPA_V_EXT * shape_abs
    ksca = albedo_V * KAPPA_V_EXT * shape_sca
    g = 0.6 * np.maximum(0.0, 1.0 - np.log10(lam_um / 0.1) / 2.0)
    g = np.minimum(g, 0.6)
    return kabs, ksca, g


def _tables_nu_ascending(per_species, lam_um):
    """Stack per-species (kabs, ksca, g) given on ascending lambda into [ns][n_nu] on ascending nu."""
    kabs = np.stack([t[0][::-1] for t in per_species]).astype(np.float64)
    ksca = np.stack([t[1][::-1] for t in per_species]).astype(np.float64)
    g = np.stack([t[2][::-1] for t in per_species]).astype(np.float64)
    return np.ascontiguousarray(kabs), np.ascontiguousarray(ksca), np.ascontiguousarray(g)


# ----------------------------------------------------------------------------- density helpers


def _cell_centres(n: int) -> np.ndarray:
    """Cell-centre coordinates in cell units relative to the grid centre."""
    return (np.arange(n, dtype=np.float64) + 0.5) - 0.5 * n


def _scale_to_tau_V(rho: np.ndarray, h_cm: float, tau_V: float, row=None) -> np.ndarray:
    """Scale rho so that KAPPA_V_EXT * sum(rho*h) along +x from the grid centre equals tau_V.

    'Voxelised optical depth along +x from the source': the row of cells
    ix >= nx/2 at iy = ny/2, iz = nz/2.
    """
    nz, ny, nx = rho.shape
    if row is None:
        row = rho[nz // 2, ny // 2, nx // 2:]
    col = float(np.sum(row.astype(np.float64))) * h_cm
    if col <= 0.0:
        raise ValueError("empty +x column; cannot normalise tau_V")
    return (rho.astype(np.float64) * (tau_V / (KAPPA_V_EXT * col))).astype(np.float32)


# ----------------------------------------------------------------------------- configs


def sphere32(tau_V: float = 1.0, n_packets: int = 100_000, n: int = 32, seed: int = 1) -> Workload:
    """Config 1: homogeneous sphere, 1 species, albedo 0.5, g 0.5, 5800 K source."""
    h = 100.0 * AU_CM / 16.0 * (32.0 / n)
    x = _cell_centres(n)
    r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
    rho = np.where(r2 < (0.5 * n) ** 2, 1.0, 0.0).astype(np.float32)
    rho = _scale_to_tau_V(rho, h, tau_V)
    lam = wavelength_grid_um(64, 0.1, 1000.0)
    kabs, ksca, g = _tables_nu_ascending([dust_powerlaw(lam, -1.5, 0.5, 0.5)], lam)
    c = 0.5 * n * h
    return Workload(
        name="sphere32" if n == 32 else f"sphere{n}", nx=n, ny=n, nz=n, cell_size_cm=h, rho=rho,
        species=np.zeros((n, n, n), np.uint8), n_species=1, nu_hz=nu_from_lambda_um(lam),
        kappa_abs=kabs, kappa_sca=ksca, g=g, T_grid=temperature_grid(), L_erg_s=LSUN_ERG_S,
        T_star_K=5800.0, L_nu_weights=None, source_pos_cm=(c, c, c),
        abs_mu_edges=np.array([0.0, 1.0]), n_packets=n_packets, seed=seed,
        meta={"tau_V": tau_V})


def shell128(tau_V: float = 10.0, n_packets: int = 10_000_000, n: int = 128, seed: int = 2) -> Workload:
    """Config 2: r^-2 shell, r_out = 100 r_in, silicate-like dust, 2500 K source."""
    r_out_cells = 0.5 * n
    h = 70.0 * AU_CM / r_out_cells
    r_in_cells = r_out_cells / 100.0
    x = _cell_centres(n).astype(np.float32)
    r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
    inside = (r2 > r_in_cells ** 2) & (r2 < r_out_cells ** 2)
    rho = np.where(inside, 1.0 / np.maximum(r2, 1e-30), 0.0).astype(np.float32)
    rho = _scale_to_tau_V(rho, h, tau_V)
    lam = wavelength_grid_um(100, 0.1, 1000.0)
    kabs, ksca, g = _tables_nu_ascending([dust_silicate_like(lam)], lam)
    c = 0.5 * n * h
    return Workload(
        name=f"shell{n}", nx=n, ny=n, nz=n, cell_size_cm=h, rho=rho,
        species=np.zeros((n, n, n), np.uint8), n_species=1, nu_hz=nu_from_lambda_um(lam),
        kappa_abs=kabs, kappa_sca=ksca, g=g, T_grid=temperature_grid(), L_erg_s=LSUN_ERG_S,
        T_star_K=2500.0, L_nu_weights=None, source_pos_cm=(c, c, c),
        abs_mu_edges=np.array([0.0, 1.0]), n_packets=n_packets, seed=seed,
        meta={"tau_V": tau_V})


def disk256(tau_V: float = 10.0, n_packets: int = 100_000_000, n: int = 256, seed: int = 3) -> Workload:
    """Config 3: flared disk (Eq. 18-19 with the config's exp(-z^2/2h^2)), 2 species."""
    half = 0.5 * n
    h = 1000.0 * AU_CM / half
    au_per_cell = 1000.0 / half
    x = _cell_centres(n).astype(np.float32) * np.float32(au_per_cell)  # AU
    rcyl = np.sqrt(x[None, :] ** 2 + x[:, None] ** 2)  # [ny][nx]
    rr = np.maximum(rcyl, np.float32(1e-6))
    hr = (125.0 * (rr / 500.0) ** 1.125).astype(np.float32)  # scale height, AU
    ok = (rcyl >= 1.0) & (rcyl <= 1000.0)
    rho = np.empty((n, n, n), np.float32)
    species = np.empty((n, n, n), np.uint8)
    for iz in range(n):
        z = x[iz]
        rho[iz] = np.where(ok, (500.0 / rr) * np.exp(-(z * z) / (2.0 * hr * hr)), 0.0)
        species[iz] = np.where(np.abs(z) <= hr, 0, 1)
    rho = _scale_to_tau_V(rho, h, tau_V)
    species[rho == 0.0] = 0
    lam = wavelength_grid_um(100, 0.1, 1000.0)
    kabs, ksca, g = _tables_nu_ascending([dust_silicate_like(lam), dust_carbon_like(lam)], lam)
    c = half * h
    L = 4.0 * math.pi * RSUN_CM ** 2 * SIGMA_SB * 5800.0 ** 4
    return Workload(
        name=f"disk{n}", nx=n, ny=n, nz=n, cell_size_cm=h, rho=rho, species=species, n_species=2,
        nu_hz=nu_from_lambda_um(lam), kappa_abs=kabs, kappa_sca=ksca, g=g, T_grid=temperature_grid(),
        L_erg_s=L, T_star_K=5800.0, L_nu_weights=None, source_pos_cm=(c, c, c),
        abs_mu_edges=np.linspace(0.0, 1.0, 11), n_packets=n_packets, seed=seed,
        meta={"tau_V": tau_V})


def _torus(n: int, n_clumps: int, clump_edge: int, n_nu: int, lognormal_tau: bool, n_packets: int,
           seed: int, geometry_seed: int, name: str) -> Workload:
    half = 0.5 * n
    h = 6.0 * PC_CM / half
    r_in = 0.4 / 6.0 * half  # cells
    r_out = half
    theta1 = math.radians(45.0)
    rng = np.random.Generator(np.random.Philox(key=geometry_seed))
    # clump centres, PAPER.md:304-309 (Eq. 21) with r = r_in + zeta1 (r_out - r_in)  (reading Q26)
    z1, z2, z3 = rng.random(n_clumps), rng.random(n_clumps), rng.random(n_clumps)
    kind = rng.integers(0, 2, n_clumps).astype(np.uint8)  # which silicate-like variant
    if lognormal_tau:
        tau_clump = 30.0 * np.exp(rng.standard_normal(n_clumps))  # median 30, sigma_ln 1
    else:
        tau_clump = np.full(n_clumps, 10.0)
    r = r_in + z1 * (r_out - r_in)
    phi = 2.0 * math.pi * z2
    theta = 0.5 * math.pi + (2.0 * z3 - 1.0) * theta1
    cx = half + r * np.sin(theta) * np.cos(phi)
    cy = half + r * np.sin(theta) * np.sin(phi)
    cz = half + r * np.cos(theta)
    # density of a clump: tau_V across its edge at the analytic V-band opacity
    rho_c = tau_clump / (KAPPA_V_EXT * clump_edge * h)
    rho_c_ref = 10.0 / (KAPPA_V_EXT * clump_edge * h) if not lognormal_tau else 30.0 / (KAPPA_V_EXT * clump_edge * h)
    # interclump medium: 1e-3 of the (reference) clump density inside the torus volume, carbon-like (species 2)
    x = _cell_centres(n).astype(np.float32)
    rho = np.empty((n, n, n), np.float32)
    species = np.empty((n, n, n), np.uint8)
    rxy2 = x[None, :] ** 2 + x[:, None] ** 2
    cos_t1 = math.cos(0.5 * math.pi - theta1)  # |cos theta| < sin(theta1) ... inside the torus wedge
    for iz in range(n):
        z = x[iz]
        r2 = rxy2 + z * z
        rr = np.sqrt(r2)
        inside = (rr > r_in) & (rr < r_out) & (np.abs(z) < cos_t1 * rr)
        rho[iz] = np.where(inside, np.float32(1e-3 * rho_c_ref), np.float32(0.0))
        species[iz] = np.where(inside, 2, 0)
    e = clump_edge
    for i in range(n_clumps):
        x0 = int(math.floor(cx[i] - 0.5 * e + 0.5))
        y0 = int(math.floor(cy[i] - 0.5 * e + 0.5))
        z0 = int(math.floor(cz[i] - 0.5 * e + 0.5))
        xs, ys, zs = max(x0, 0), max(y0, 0), max(z0, 0)
        xe, ye, ze = min(x0 + e, n), min(y0 + e, n), min(z0 + e, n)
        if xs >= xe or ys >= ye or zs >= ze:
            continue
        # overlaps are not additive: later clumps overwrite
        rho[zs:ze, ys:ye, xs:xe] = np.float32(rho_c[i])
        species[zs:ze, ys:ye, xs:xe] = kind[i]
    lam = wavelength_grid_um(n_nu, 0.01, 1000.0)
    tabs = [dust_silicate_like(lam, -1.6, 0.05, 0.02), dust_silicate_like(lam, -1.3, 0.02, 0.01),
            dust_carbon_like(lam)]
    kabs, ksca, g = _tables_nu_ascending(tabs, lam)
    nu = nu_from_lambda_um(lam)
    lam_nu = lambda_um_from_nu(nu)
    # central engine: F_nu ~ nu^-0.5 on 0.01-10 um, zero elsewhere (config 4)
    w = np.where((lam_nu >= 0.01 * (1 - 1e-12)) & (lam_nu <= 10.0 * (1 + 1e-12)), (nu / nu[-1]) ** -0.5, 0.0)
    c = half * h
    edges = np.cos(np.radians(10.0 * np.arange(9, -1, -1)))
    edges[0], edges[-1] = 0.0, 1.0
    return Workload(
        name=name, nx=n, ny=n, nz=n, cell_size_cm=h, rho=rho, species=species, n_species=3,
        nu_hz=nu, kappa_abs=kabs, kappa_sca=ksca, g=g, T_grid=temperature_grid(), L_erg_s=1e45,
        T_star_K=0.0, L_nu_weights=np.ascontiguousarray(w), source_pos_cm=(c, c, c),
        abs_mu_edges=edges, n_packets=n_packets, seed=seed,
        meta={"n_clumps": n_clumps, "clump_edge": clump_edge, "geometry_seed": geometry_seed})


def torus256(n_clumps: int = 5000, n_packets: int = 100_000_000, n: int = 256, seed: int = 4,
             geometry_seed: int = 1004) -> Workload:
    """Config 4: clumpy AGN torus, 3-cell cubic clumps, tau_V = 10 each."""
    edge = max(1, round(3 * n / 256))
    return _torus(n, n_clumps, edge, 120, False, n_packets, seed, geometry_seed, f"torus{n}")


def torus512(n_clumps: int = 20000, n_packets: int = 1_000_000_000, n: int = 512, seed: int = 5,
             geometry_seed: int = 1005) -> Workload:
    """Config 5: scale test, 512^3, lognormal clump tau_V, 200 wavelengths."""
    edge = max(1, round(6 * n / 512))
    return _torus(n, n_clumps, edge, 200, True, n_packets, seed, geometry_seed, f"torus{n}")


def uniform_cube(n: int, tau_edge_V: float, albedo: float, g_const: float, n_nu: int = 16,
                 T_star: float = 5800.0, slope: float = 0.0, n_packets: int = 100_000, seed: int = 7,
                 n_dir: int = 1, source_offset_cells=(0.0, 0.0, 0.0), nxyz=None) -> Workload:
    """Small uniform test cube: optical depth tau_edge_V from the centre to a face along an axis."""
    nx, ny, nz = (n, n, n) if nxyz is None else nxyz
    h = AU_CM
    rho0 = tau_edge_V / (KAPPA_V_EXT * 0.5 * nx * h) if tau_edge_V > 0 else 0.0
    rho = np.full((nz, ny, nx), rho0, np.float32)
    lam = wavelength_grid_um(n_nu, 0.1, 1000.0)
    kabs, ksca, g = _tables_nu_ascending([dust_powerlaw(lam, slope, albedo, g_const)], lam)
    c = (0.5 * nx * h + source_offset_cells[0] * h, 0.5 * ny * h + source_offset_cells[1] * h,
         0.5 * nz * h + source_offset_cells[2] * h)
    return Workload(
        name=f"cube{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, cell_size_cm=h, rho=rho,
        species=np.zeros((nz, ny, nx), np.uint8), n_species=1, nu_hz=nu_from_lambda_um(lam),
        kappa_abs=kabs, kappa_sca=ksca, g=g, T_grid=temperature_grid(), L_erg_s=LSUN_ERG_S,
        T_star_K=T_star, L_nu_weights=None, source_pos_cm=c,
        abs_mu_edges=np.linspace(0.0, 1.0, n_dir + 1), n_packets=n_packets, seed=seed,
        meta={"tau_edge_V": tau_edge_V, "albedo": albedo, "g": g_const, "slope": slope})


CONFIGS = {
    "sphere32": sphere32,
    "shell128": shell128,
    "disk256": disk256,
    "torus256": torus256,
    "torus512": torus512,
}


def make(name: str, **kw) -> Workload:
    return CONFIGS[name](**kw)
