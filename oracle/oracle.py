"""ctypes wrapper around the CPU oracle (oracle/mcrt_oracle.c).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from the CUDA package; inputs arrive as plain numpy arrays (a Workload-shaped object
with the attribute names of paper_1203_2941_b200/workloads.py is accepted by ``Oracle.from_workload``).
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

MODE_BW_EPOCH = 0
MODE_FROZEN_SWEEP = 1


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "packets", "crossings", "dusty_crossings", "flights", "scatterings", "absorptions", "escapes",
        "direct_escapes", "epochs", "lucy_adds")] + [("fx_bits", C.c_int32), ("overflow", C.c_int32)]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class Opts(C.Structure):
    _fields_ = [("mode", C.c_int32), ("B0", C.c_uint64), ("Bmax", C.c_uint64), ("n_sweeps", C.c_int32),
                ("sweep_T_from_lucy", C.c_int32), ("n_threads", C.c_int32), ("absorb_and_stop", C.c_int32),
                ("per_cell_redraw", C.c_int32), ("keep_fp64_lucy", C.c_int32), ("reset", C.c_int32),
                ("pass0", C.c_uint32), ("pid0", C.c_uint64), ("n_total", C.c_uint64), ("growth", C.c_double), ("carry_K", C.c_uint32), ("source_strata", C.c_uint32), ("lucy_hybrid", C.c_int32)]


SCA_EVENT_DTYPE = np.dtype([("cell", np.uint32), ("slot", np.uint16), ("q", np.int16, (3,))])

DIGEST_DTYPE = np.dtype([("hash", np.uint64), ("crossings", np.uint32), ("scatterings", np.uint32),
                         ("absorptions", np.uint32), ("escape_bin", np.uint32)])

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                 C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_double,
                                 C.c_double, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_state_create.restype = C.c_void_p
        L.orc_state_create.argtypes = [C.c_void_p]
        L.orc_state_destroy.argtypes = [C.c_void_p]
        L.orc_run.restype = C.c_int
        L.orc_run.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.POINTER(Opts), C.POINTER(Stats), C.c_void_p]
        L.orc_read_raw.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.orc_read.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_get_tables.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.orc_eq9_value.restype = C.c_double
        L.orc_eq9_value.argtypes = [C.c_double]
        L.orc_set_subgrid.restype = C.c_int
        L.orc_set_subgrid.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_mixtures.restype = C.c_int
        L.orc_set_mixtures.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_read_raw_comp1.restype = C.c_int
        L.orc_read_raw_comp1.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.orc_read_comp1.restype = C.c_int
        L.orc_read_comp1.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_planck.restype = C.c_double
        L.orc_planck.argtypes = [C.c_double, C.c_double]
        L.orc_dplanck_dT.restype = C.c_double
        L.orc_dplanck_dT.argtypes = [C.c_double, C.c_double]
        L.orc_bin_widths.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.orc_lower_bound.restype = C.c_int
        L.orc_lower_bound.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_isotropic.argtypes = [C.c_double, C.c_double, C.c_void_p]
        L.orc_hg_scatter.argtypes = [C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_dda_trace.restype = C.c_int
        L.orc_dda_trace.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                    C.c_void_p]
        L.orc_T_of_x.restype = C.c_double
        L.orc_T_of_x.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_fx_bits.restype = C.c_int
        L.orc_fx_bits.argtypes = [C.c_uint64]
        L.orc_default_schedule.argtypes = [C.c_uint64, C.c_void_p, C.c_void_p]
        L.orc_det_log.restype = C.c_double
        L.orc_det_log.argtypes = [C.c_double]
        L.orc_det_sincos.argtypes = [C.c_double, C.c_void_p, C.c_void_p]
        L.orc_max_threads.restype = C.c_int
        L.orc_scatter_store.restype = C.c_int
        L.orc_scatter_store.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint64]
        L.orc_scatter_events.restype = C.c_uint64
        L.orc_scatter_events.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.orc_phase_hg.restype = C.c_double
        L.orc_phase_hg.argtypes = [C.c_double, C.c_double]
        L.orc_ray_trace.restype = C.c_int
        L.orc_ray_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                    C.c_int, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def philox(ctr, key):
    c = np.ascontiguousarray(ctr, np.uint32)
    k = np.ascontiguousarray(key, np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def uniforms(seed, pid, draw, pas=0):
    out = np.zeros(2, np.float64)
    lib().orc_uniforms(seed, pid, draw, pas, _p(out))
    return out


def planck(nu, T):
    return lib().orc_planck(float(nu), float(T))


def dplanck_dT(nu, T):
    return lib().orc_dplanck_dT(float(nu), float(T))


def bin_widths(nu):
    nu = np.ascontiguousarray(nu, np.float64)
    out = np.zeros_like(nu)
    lib().orc_bin_widths(len(nu), _p(nu), _p(out))
    return out


def lower_bound(cdf, z):
    cdf = np.ascontiguousarray(cdf, np.float64)
    return lib().orc_lower_bound(_p(cdf), len(cdf), float(z))


def isotropic(z0, z1):
    out = np.zeros(3)
    lib().orc_isotropic(float(z0), float(z1), _p(out))
    return out


def hg_scatter(g, z0, z1, u):
    u = np.ascontiguousarray(u, np.float64)
    out = np.zeros(3)
    lib().orc_hg_scatter(float(g), float(z0), float(z1), _p(u), _p(out))
    return out


def det_log(z):
    return float(lib().orc_det_log(float(z)))


def det_sincos(z):
    out = np.zeros(2)
    lib().orc_det_sincos(float(z), _p(out[0:1]), _p(out[1:2]))
    return float(out[0]), float(out[1])


def dda_trace(nx, ny, nz, p, u, max_n=4096):
    p = np.ascontiguousarray(p, np.float64)
    u = np.ascontiguousarray(u, np.float64)
    cells = np.zeros(max_n, np.int64)
    ds = np.zeros(max_n, np.float64)
    n = lib().orc_dda_trace(nx, ny, nz, _p(p), _p(u), max_n, _p(cells), _p(ds))
    return cells[:n], ds[:n]


def fx_bits(n):
    return lib().orc_fx_bits(int(n))


def default_schedule(n):
    b = np.zeros(2, np.uint64)
    lib().orc_default_schedule(int(n), _p(b[0:1]), _p(b[1:2]))
    return int(b[0]), int(b[1])


def phase_hg(g, cos_beta):
    return lib().orc_phase_hg(float(g), float(cos_beta))


def eq9_value(tau):
    return lib().orc_eq9_value(float(tau))


def max_threads():
    return lib().orc_max_threads()


class Oracle:
    """One problem (grid + dust + source + escape bins) and its tally state."""

    def __init__(self, nx, ny, nz, h, rho, species, n_species, nu, kabs, ksca, g, Tgrid, L, Tstar, Lnu_w,
                 pos_cm, mu_edges, mixtures=None, subgrid=None):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.nc = self.nx * self.ny * self.nz
        self.ns, self.nf, self.nT = int(n_species), len(nu), len(Tgrid)
        self.ndir = len(mu_edges) - 1
        self._keep = [np.ascontiguousarray(rho, np.float32).reshape(-1),
                      np.ascontiguousarray(species, np.uint8).reshape(-1),
                      np.ascontiguousarray(nu, np.float64), np.ascontiguousarray(kabs, np.float64),
                      np.ascontiguousarray(ksca, np.float64), np.ascontiguousarray(g, np.float64),
                      np.ascontiguousarray(Tgrid, np.float64),
                      None if Lnu_w is None else np.ascontiguousarray(Lnu_w, np.float64),
                      np.ascontiguousarray(pos_cm, np.float64), np.ascontiguousarray(mu_edges, np.float64)]
        k = self._keep
        self._ctx = lib().orc_create(self.nx, self.ny, self.nz, float(h), _p(k[0]), _p(k[1]), self.ns, self.nf,
                                     _p(k[2]), _p(k[3]), _p(k[4]), _p(k[5]), self.nT, _p(k[6]), float(L),
                                     float(Tstar), _p(k[7]), _p(k[8]), self.ndir, _p(k[9]))
        self.mixtures = mixtures
        if mixtures is not None:
            # NEXT-3: the species byte of a cell names a mixture: (ncomp[n_mix], material[n_mix][2], fraction[n_mix][2])
            nc_, mat_, fr_ = (np.ascontiguousarray(mixtures[0], np.int32), np.ascontiguousarray(mixtures[1], np.int32),
                              np.ascontiguousarray(mixtures[2], np.float64))
            assert mat_.shape == (len(nc_), 2) and fr_.shape == (len(nc_), 2)
            rc = lib().orc_set_mixtures(self._ctx, len(nc_), _p(nc_), _p(mat_), _p(fr_))
            assert rc == 0, "bad mixture table"
        self.subgrid = subgrid
        if subgrid is not None:
            # NEXT-3: (R, cube[n_sub] cell indices of the refined cubes, rho_sub[n_sub][R^3], species_sub[n_sub][R^3]);
            # the sub-cubes are cells nc .. nc + n_sub R^3 - 1 of every per-cell output
            Rr, cube, rs, ss = subgrid
            cube = np.ascontiguousarray(cube, np.int64)
            rs = np.ascontiguousarray(rs, np.float32).reshape(len(cube), -1)
            ss = np.ascontiguousarray(ss, np.uint8).reshape(len(cube), -1)
            assert rs.shape == (len(cube), Rr ** 3) and ss.shape == rs.shape
            rc = lib().orc_set_subgrid(self._ctx, int(Rr), len(cube), _p(cube), _p(rs), _p(ss))
            assert rc == 0, "bad sub-grid"
            self.nc0, self.nc = self.nc, self.nc + len(cube) * Rr ** 3
        self._state = lib().orc_state_create(self._ctx)
        self.last_n = 0

    @classmethod
    def from_workload(cls, w):
        return cls(w.nx, w.ny, w.nz, w.cell_size_cm, w.rho, w.species, w.n_species, w.nu_hz, w.kappa_abs,
                   w.kappa_sca, w.g, w.T_grid, w.L_erg_s, w.T_star_K, w.L_nu_weights, w.source_pos_cm,
                   w.abs_mu_edges, mixtures=getattr(w, "mixtures", None), subgrid=getattr(w, "subgrid", None))

    def close(self):
        if self._state:
            lib().orc_state_destroy(self._state)
            self._state = None
        if self._ctx:
            lib().orc_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def tables(self):
        dnu = np.zeros(self.nf)
        J = np.zeros((self.ns, self.nT))
        cB = np.zeros((self.ns, self.nT, self.nf))
        cdB = np.zeros((self.ns, self.nT, self.nf))
        alb = np.zeros((self.ns, self.nf))
        src = np.zeros(self.nf)
        lib().orc_get_tables(self._ctx, _p(dnu), _p(J), _p(cB), _p(cdB), _p(alb), _p(src))
        return {"dnu": dnu, "J": J, "cdfB": cB, "cdfdB": cdB, "albedo": alb, "srccdf": src}

    def T_of_x(self, s, x):
        return lib().orc_T_of_x(self._ctx, int(s), float(x))

    def run(self, n_packets, seed, mode=MODE_BW_EPOCH, B0=0, Bmax=0, n_sweeps=0, sweep_T_from_lucy=1,
            n_threads=1, absorb_and_stop=False, per_cell_redraw=False, keep_fp64_lucy=False, reset=True,
            pass0=0, digests=False, pid0=0, n_total=0, growth=0.0, carry_K=0, source_strata=0, lucy_hybrid=False):
        o = Opts(mode, B0, Bmax, n_sweeps, int(sweep_T_from_lucy), n_threads, int(absorb_and_stop),
                 int(per_cell_redraw), int(keep_fp64_lucy), int(reset), pass0, int(pid0), int(n_total), float(growth), int(carry_K), int(source_strata), int(lucy_hybrid))
        st = Stats()
        dig = np.zeros(n_packets, DIGEST_DTYPE) if digests else None
        rc = lib().orc_run(self._state, int(n_packets), int(seed), C.byref(o), C.byref(st), _p(dig))
        self.last_n = int(n_packets)
        out = st.as_dict()
        out["rc"] = rc
        if digests:
            out["digests"] = dig
        return out

    def read_raw(self, fp64_lucy=False):
        k = np.zeros(self.nc, np.uint64)
        L = np.zeros(self.nc, np.int64)
        sed = np.zeros((self.ndir, self.nf), np.uint64)
        sedd = np.zeros((self.ndir, self.nf), np.uint64)
        tidx = np.zeros(self.nc, np.uint16)
        Ls = np.zeros(self.nc, np.float64) if fp64_lucy else None
        lib().orc_read_raw(self._state, _p(k), _p(L), _p(sed), _p(sedd), _p(tidx), _p(Ls))
        out = {"k": k, "lucy_fx": L, "sed": sed, "sed_direct": sedd, "tidx": tidx}
        if fp64_lucy:
            out["lucy_fp64"] = Ls
        return out

    def read_raw_comp1(self):
        """Raw tallies of the second component of the mixtures (NEXT-3)."""
        k = np.zeros(self.nc, np.uint64)
        L = np.zeros(self.nc, np.int64)
        tidx = np.zeros(self.nc, np.uint16)
        assert lib().orc_read_raw_comp1(self._state, _p(k), _p(L), _p(tidx)) == 0
        return {"k": k, "lucy_fx": L, "tidx": tidx}

    def read_comp1(self, T_from_lucy=False):
        Ec = np.zeros(self.nc)
        El = np.zeros(self.nc)
        T = np.zeros(self.nc, np.float32)
        assert lib().orc_read_comp1(self._state, _p(Ec), _p(El), _p(T), int(T_from_lucy)) == 0
        return {"E_count": Ec, "E_lucy": El, "T": T}

    def scatter_store(self, nu_bins, capacity):
        b = np.ascontiguousarray(nu_bins, np.int32)
        rc = lib().orc_scatter_store(self._state, len(b), _p(b), int(capacity))
        assert rc == 0
        self._sca_cap = int(capacity)

    def scatter_events(self):
        ev = np.zeros(self._sca_cap, SCA_EVENT_DTYPE)
        n = lib().orc_scatter_events(self._state, _p(ev), self._sca_cap)
        return ev[:min(n, self._sca_cap)], int(n)

    def ray_trace(self, e_z, e_x, nx, ny, pixel_cm, distance_cm, nu_bin, T_from_lucy=False):
        ez = np.ascontiguousarray(e_z, np.float64)
        ex = np.ascontiguousarray(e_x, np.float64)
        Fe, Fs = np.zeros((ny, nx)), np.zeros((ny, nx))
        rc = lib().orc_ray_trace(self._state, _p(ez), _p(ex), int(nx), int(ny), float(pixel_cm), float(distance_cm),
                                 int(nu_bin), int(T_from_lucy), _p(Fe), _p(Fs))
        assert rc == 0
        return Fe, Fs

    def read(self, T_from_lucy=False):
        Ec = np.zeros(self.nc)
        El = np.zeros(self.nc)
        T = np.zeros(self.nc, np.float32)
        sed = np.zeros((self.ndir, self.nf))
        lib().orc_read(self._state, _p(Ec), _p(El), _p(T), int(T_from_lucy), _p(sed))
        return {"E_count": Ec, "E_lucy": El, "T": T, "SED": sed}
