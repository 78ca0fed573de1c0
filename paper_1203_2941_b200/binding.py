"""Thin ctypes binding over libmcrt_b200.so -- argument marshalling only.

The functions carry the names of include/mcrt.h and do nothing but convert arguments; every step of the
transport runs in the CUDA kernels of csrc/mcrt.cu.  PyTorch is used here for device memory (the
workspace tensor), the current stream and pinned host buffers -- plumbing, not compute.

There is no CPU fallback: if the shared library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MCRT_B200_LIB") or os.path.join(_HERE, "lib", "libmcrt_b200.so")

MCRT_HOST, MCRT_DEVICE = 0, 1
MCRT_OK, MCRT_EINVAL, MCRT_ESTATE, MCRT_ENOMEM, MCRT_ECUDA, MCRT_EOVERFLOW = 0, -1, -2, -3, -4, -5
MCRT_MODE_BW_EPOCH, MCRT_MODE_FROZEN_T_SWEEP, MCRT_MODE_LIVE_BW = 0, 1, 2

EXPORTS = [
    "mcrt_workspace_bytes", "mcrt_grid_create", "mcrt_dust_tables", "mcrt_dust_mixtures", "mcrt_subgrid", "mcrt_read_subcells", "mcrt_source", "mcrt_escape_bins",
    "mcrt_default_opts", "mcrt_run", "mcrt_run_begin", "mcrt_run_step", "mcrt_run_end", "mcrt_exchange_begin",
    "mcrt_exchange_end", "mcrt_exchange_peer_sum", "mcrt_exchange_local", "mcrt_epoch_schedule", "mcrt_part_slice",
    "mcrt_measure_read_bandwidth", "mcrt_scatter_store", "mcrt_scatter_events", "mcrt_ray_trace", "mcrt_get_stats", "mcrt_read", "mcrt_read_component", "mcrt_read_raw", "mcrt_read_tables",
    "mcrt_philox_device", "mcrt_traj_math_device", "mcrt_traj_math_device_static", "mcrt_set_stream", "mcrt_launch_config", "mcrt_last_error", "mcrt_version",
    "mcrt_destroy",
]


class McrtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mcrt error {code}: {msg}")
        self.code = code


class RunOpts(C.Structure):
    _fields_ = [("mode", C.c_int32), ("epoch_B0", C.c_uint64), ("epoch_Bmax", C.c_uint64),
                ("n_sweeps", C.c_int32), ("sweep_T_from_lucy", C.c_int32), ("record_digests", C.c_int32),
                ("reset_tallies", C.c_int32), ("rng_pass", C.c_uint32), ("grid_blocks", C.c_int32),
                ("block_threads", C.c_int32), ("time_kernels", C.c_int32), ("first_packet_id", C.c_uint64),
                ("n_total", C.c_uint64), ("epoch_growth", C.c_double), ("part_index", C.c_int32),
                ("part_count", C.c_int32), ("source_strata", C.c_uint32), ("carry_interactions", C.c_uint32), ("no_hot_cells", C.c_int32), ("lucy_hybrid", C.c_int32), ("tau_redraw_per_cell", C.c_int32)]


class ImageOpts(C.Structure):
    _fields_ = [("e_z", C.c_double * 3), ("e_x", C.c_double * 3), ("nx", C.c_int32), ("ny", C.c_int32),
                ("pixel_cm", C.c_double), ("distance_cm", C.c_double), ("nu_bin", C.c_int32), ("T_from_lucy", C.c_int32)]


SCA_EVENT_DTYPE = np.dtype([("cell", np.uint32), ("slot", np.uint16), ("q", np.int16, (3,))])


class Exchange(C.Structure):
    _fields_ = [("n", C.c_int32), ("ptr", C.c_void_p * 8), ("words", C.c_uint64 * 8)]


class RunStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "packets", "crossings", "dusty_crossings", "flights", "scatterings", "absorptions", "escapes",
        "direct_escapes", "epochs", "lucy_adds", "gpu_launches")] + [("fx_bits", C.c_int32), ("overflow", C.c_int32),
                                                                     ("transport_ms", C.c_double),
                                                                     ("update_ms", C.c_double)]

    def as_dict(self):
        return {n: (float if t is C.c_double else int)(getattr(self, n)) for n, t in self._fields_}


DIGEST_DTYPE = np.dtype([("hash", np.uint64), ("crossings", np.uint32), ("scatterings", np.uint32),
                         ("absorptions", np.uint32), ("escape_bin", np.uint32)])

_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen the CUDA library; fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} not found: build it with `python -m paper_1203_2941_b200.build` "
            "(the product has no CPU fallback)")
    L = C.CDLL(path)
    vp, i, d, u64 = C.c_void_p, C.c_int, C.c_double, C.c_uint64
    L.mcrt_workspace_bytes.argtypes = [i, i, i, i, i, i, i, u64, C.POINTER(C.c_size_t)]
    L.mcrt_grid_create.argtypes = [C.POINTER(vp), i, i, i, d, vp, vp, i, i, vp, C.c_size_t]
    L.mcrt_dust_tables.argtypes = [vp, i, vp, vp, vp, vp, i, vp]
    L.mcrt_source.argtypes = [vp, d, d, vp, vp]
    L.mcrt_escape_bins.argtypes = [vp, i, vp]
    L.mcrt_default_opts.argtypes = [C.POINTER(RunOpts)]
    L.mcrt_default_opts.restype = None
    L.mcrt_run.argtypes = [vp, u64, u64, C.POINTER(RunOpts), C.POINTER(RunStats)]
    L.mcrt_run_begin.argtypes = [vp, u64, u64, C.POINTER(RunOpts)]
    L.mcrt_run_step.argtypes = [vp, C.POINTER(i)]
    L.mcrt_run_end.argtypes = [vp, C.POINTER(RunStats)]
    L.mcrt_exchange_begin.argtypes = [vp, C.POINTER(Exchange)]
    L.mcrt_exchange_end.argtypes = [vp]
    L.mcrt_exchange_peer_sum.argtypes = [vp, i, i, C.POINTER(Exchange), i]
    L.mcrt_exchange_local.argtypes = [C.POINTER(vp), i]
    L.mcrt_epoch_schedule.argtypes = [u64, u64, u64, d, vp, u64, C.POINTER(u64)]
    L.mcrt_part_slice.argtypes = [u64, i, i, C.POINTER(u64), C.POINTER(u64)]
    L.mcrt_measure_read_bandwidth.argtypes = [C.c_size_t, i, C.POINTER(d)]
    L.mcrt_scatter_store.argtypes = [vp, i, vp, u64]
    L.mcrt_scatter_events.argtypes = [vp, C.POINTER(u64), vp, u64, i]
    L.mcrt_ray_trace.argtypes = [vp, C.POINTER(ImageOpts), vp, vp, i]
    L.mcrt_get_stats.argtypes = [vp, C.POINTER(RunStats)]
    L.mcrt_read.argtypes = [vp, vp, vp, vp, vp, vp, i]
    L.mcrt_read_raw.argtypes = [vp, vp, vp, vp, vp, vp, vp, i]
    L.mcrt_read_component.argtypes = [vp, i, vp, vp, vp, vp, vp, vp, vp, i]
    L.mcrt_dust_mixtures.argtypes = [vp, vp, vp, vp]
    L.mcrt_subgrid.argtypes = [vp, i, u64, vp, vp, vp]
    L.mcrt_read_subcells.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i]
    L.mcrt_read_tables.argtypes = [vp] + [vp] * 6
    L.mcrt_philox_device.argtypes = [vp, vp, vp, u64]
    L.mcrt_traj_math_device.argtypes = [vp, vp, vp, vp, u64]
    L.mcrt_traj_math_device_static.argtypes = [vp, vp, vp, vp, u64]
    L.mcrt_set_stream.argtypes = [vp, vp]
    L.mcrt_launch_config.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(C.c_size_t)]
    L.mcrt_last_error.argtypes = [vp]
    L.mcrt_last_error.restype = C.c_char_p
    L.mcrt_version.restype = C.c_char_p
    L.mcrt_destroy.argtypes = [vp]
    L.mcrt_destroy.restype = None
    for name in EXPORTS:
        if name not in ("mcrt_default_opts", "mcrt_last_error", "mcrt_version", "mcrt_destroy"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _check(rc, ctx=None):
    if rc != MCRT_OK:
        msg = load_library().mcrt_last_error(ctx)
        raise McrtError(rc, msg.decode() if msg else "")


def _ptr(a):
    """Host numpy array / torch tensor / int / None -> void*."""
    if a is None:
        return None
    if isinstance(a, int):
        return C.c_void_p(a)
    if isinstance(a, np.ndarray):
        return a.ctypes.data_as(C.c_void_p)
    return C.c_void_p(a.data_ptr())  # torch tensor (host pinned or device)


# ---------------------------------------------------------------- functions, same names as the C ABI
def mcrt_version() -> str:
    return load_library().mcrt_version().decode()


def mcrt_workspace_bytes(nx, ny, nz, n_species, n_nu, n_T, n_dir, n_digests=0) -> int:
    out = C.c_size_t(0)
    _check(load_library().mcrt_workspace_bytes(nx, ny, nz, n_species, n_nu, n_T, n_dir, n_digests, C.byref(out)))
    return out.value


def mcrt_grid_create(nx, ny, nz, cell_size_cm, rho, species, n_species, where=MCRT_HOST, workspace=None,
                     workspace_bytes=0):
    ctx = C.c_void_p(None)
    _check(load_library().mcrt_grid_create(C.byref(ctx), nx, ny, nz, float(cell_size_cm), _ptr(rho), _ptr(species),
                                           n_species, where, _ptr(workspace), workspace_bytes))
    return ctx


def mcrt_dust_tables(ctx, nu_hz, kappa_abs, kappa_sca, g, T_grid):
    nu = np.ascontiguousarray(nu_hz, np.float64)
    ka = np.ascontiguousarray(kappa_abs, np.float64)
    ks = np.ascontiguousarray(kappa_sca, np.float64)
    gg = np.ascontiguousarray(g, np.float64)
    Tg = np.ascontiguousarray(T_grid, np.float64)
    _check(load_library().mcrt_dust_tables(ctx, len(nu), _ptr(nu), _ptr(ka), _ptr(ks), _ptr(gg), len(Tg), _ptr(Tg)), ctx)


def mcrt_source(ctx, L_erg_s, T_star_K, L_nu_weights, pos_cm):
    w = None if L_nu_weights is None else np.ascontiguousarray(L_nu_weights, np.float64)
    p = np.ascontiguousarray(pos_cm, np.float64)
    _check(load_library().mcrt_source(ctx, float(L_erg_s), float(T_star_K), _ptr(w), _ptr(p)), ctx)


def mcrt_escape_bins(ctx, abs_mu_edges):
    e = np.ascontiguousarray(abs_mu_edges, np.float64)
    _check(load_library().mcrt_escape_bins(ctx, len(e) - 1, _ptr(e)), ctx)


def mcrt_default_opts() -> RunOpts:
    o = RunOpts()
    load_library().mcrt_default_opts(C.byref(o))
    return o


def mcrt_run(ctx, n_packets, seed, opts: RunOpts | None = None, want_stats=True):
    st = RunStats()
    _check(load_library().mcrt_run(ctx, int(n_packets), int(seed), C.byref(opts) if opts is not None else None,
                                   C.byref(st) if want_stats else None), ctx)
    return st.as_dict() if want_stats else None


def mcrt_run_begin(ctx, n_packets, seed, opts: RunOpts | None = None):
    _check(load_library().mcrt_run_begin(ctx, int(n_packets), int(seed), C.byref(opts) if opts is not None else None), ctx)


def mcrt_run_step(ctx) -> bool:
    """One epoch / sweep; returns True when it was the last one."""
    done = C.c_int(0)
    _check(load_library().mcrt_run_step(ctx, C.byref(done)), ctx)
    return bool(done.value)


def mcrt_run_end(ctx, want_stats=True):
    st = RunStats()
    _check(load_library().mcrt_run_end(ctx, C.byref(st) if want_stats else None), ctx)
    return st.as_dict() if want_stats else None


def mcrt_exchange_begin(ctx) -> Exchange:
    ex = Exchange()
    _check(load_library().mcrt_exchange_begin(ctx, C.byref(ex)), ctx)
    return ex


def mcrt_exchange_end(ctx):
    _check(load_library().mcrt_exchange_end(ctx), ctx)


def mcrt_exchange_peer_sum(ctx, part_index, views, phase):
    arr = (Exchange * len(views))(*views)
    _check(load_library().mcrt_exchange_peer_sum(ctx, int(part_index), len(views), arr, int(phase)), ctx)


def mcrt_exchange_local(ctxs):
    arr = (C.c_void_p * len(ctxs))(*[c.value if isinstance(c, C.c_void_p) else c for c in ctxs])
    _check(load_library().mcrt_exchange_local(arr, len(ctxs)), ctxs[0])


def mcrt_epoch_schedule(n_packets, epoch_B0=0, epoch_Bmax=0, epoch_growth=0.0):
    n = C.c_uint64(0)
    _check(load_library().mcrt_epoch_schedule(int(n_packets), int(epoch_B0), int(epoch_Bmax), float(epoch_growth), None, 0,
                                              C.byref(n)))
    sizes = np.zeros(n.value, np.uint64)
    _check(load_library().mcrt_epoch_schedule(int(n_packets), int(epoch_B0), int(epoch_Bmax), float(epoch_growth), _ptr(sizes),
                                              n.value, C.byref(n)))
    return sizes


def mcrt_part_slice(count, part_index, part_count):
    lo, hi = C.c_uint64(0), C.c_uint64(0)
    _check(load_library().mcrt_part_slice(int(count), int(part_index), int(part_count), C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def mcrt_measure_read_bandwidth(nbytes, repeats=10) -> float:
    g = C.c_double(0.0)
    _check(load_library().mcrt_measure_read_bandwidth(int(nbytes), int(repeats), C.byref(g)))
    return g.value


_sca_capacity = {}   # context address -> capacity of its event list (to size the host buffer)


def mcrt_scatter_store(ctx, nu_bins, capacity):
    b = np.ascontiguousarray(nu_bins, np.int32)
    _check(load_library().mcrt_scatter_store(ctx, len(b), _ptr(b), int(capacity)), ctx)
    _sca_capacity[ctx.value] = int(capacity)


def mcrt_scatter_events(ctx, max_events):
    """(events kept, events counted)"""
    n = C.c_uint64(0)
    max_events = min(int(max_events), _sca_capacity.get(ctx.value, int(max_events)))
    ev = np.zeros(max_events, SCA_EVENT_DTYPE)
    _check(load_library().mcrt_scatter_events(ctx, C.byref(n), _ptr(ev), max_events, MCRT_HOST), ctx)
    return ev[:min(int(n.value), max_events)], int(n.value)


def mcrt_ray_trace(ctx, e_z, e_x, nx, ny, pixel_cm, distance_cm, nu_bin, T_from_lucy=False, scatter=True):
    o = ImageOpts()
    o.e_z[:] = [float(v) for v in e_z]
    o.e_x[:] = [float(v) for v in e_x]
    o.nx, o.ny, o.pixel_cm, o.distance_cm, o.nu_bin, o.T_from_lucy = int(nx), int(ny), float(pixel_cm), float(distance_cm), int(nu_bin), int(T_from_lucy)
    Fe = np.zeros((ny, nx))
    Fs = np.zeros((ny, nx)) if scatter else None
    _check(load_library().mcrt_ray_trace(ctx, C.byref(o), _ptr(Fe), _ptr(Fs), MCRT_HOST), ctx)
    return Fe, Fs


def mcrt_get_stats(ctx):
    st = RunStats()
    _check(load_library().mcrt_get_stats(ctx, C.byref(st)), ctx)
    return st.as_dict()


def mcrt_read(ctx, E_abs_count=None, E_abs_lucy=None, T_count=None, T_lucy=None, SED=None, where=MCRT_HOST):
    _check(load_library().mcrt_read(ctx, _ptr(E_abs_count), _ptr(E_abs_lucy), _ptr(T_count), _ptr(T_lucy), _ptr(SED),
                                    where), ctx)


def mcrt_dust_mixtures(ctx, n_components, material, fraction):
    nc_ = np.ascontiguousarray(n_components, np.int32)
    mat = np.ascontiguousarray(material, np.int32)
    fr = np.ascontiguousarray(fraction, np.float64)
    assert mat.shape == (len(nc_), 2) and fr.shape == (len(nc_), 2)
    _check(load_library().mcrt_dust_mixtures(ctx, _ptr(nc_), _ptr(mat), _ptr(fr)), ctx)


def mcrt_subgrid(ctx, R, cube, rho_sub, species_sub):
    cube = np.ascontiguousarray(cube, np.int64).reshape(-1)
    rs = np.ascontiguousarray(rho_sub, np.float32).reshape(len(cube), -1)
    ss = np.ascontiguousarray(species_sub, np.uint8).reshape(len(cube), -1)
    assert rs.shape == (len(cube), int(R) ** 3) and ss.shape == rs.shape
    _check(load_library().mcrt_subgrid(ctx, int(R), len(cube), _ptr(cube), _ptr(rs), _ptr(ss)), ctx)


def mcrt_read_subcells(ctx, E_abs_count=None, E_abs_lucy=None, T_count=None, T_lucy=None, k_abs=None, lucy_fx=None,
                       tidx=None, where=MCRT_HOST):
    _check(load_library().mcrt_read_subcells(ctx, _ptr(E_abs_count), _ptr(E_abs_lucy), _ptr(T_count), _ptr(T_lucy),
                                             _ptr(k_abs), _ptr(lucy_fx), _ptr(tidx), where), ctx)


def mcrt_read_component(ctx, component, E_abs_count=None, E_abs_lucy=None, T_count=None, T_lucy=None, k_abs=None,
                        lucy_fx=None, tidx=None, where=MCRT_HOST):
    _check(load_library().mcrt_read_component(ctx, int(component), _ptr(E_abs_count), _ptr(E_abs_lucy), _ptr(T_count),
                                              _ptr(T_lucy), _ptr(k_abs), _ptr(lucy_fx), _ptr(tidx), where), ctx)


def mcrt_read_raw(ctx, k_abs=None, lucy_fx=None, sed_counts=None, sed_direct=None, tidx=None, digests=None,
                  where=MCRT_HOST):
    _check(load_library().mcrt_read_raw(ctx, _ptr(k_abs), _ptr(lucy_fx), _ptr(sed_counts), _ptr(sed_direct), _ptr(tidx),
                                        _ptr(digests), where), ctx)


def mcrt_read_tables(ctx, dnu=None, J=None, cdf_B=None, cdf_dB=None, albedo=None, src_cdf=None):
    _check(load_library().mcrt_read_tables(ctx, _ptr(dnu), _ptr(J), _ptr(cdf_B), _ptr(cdf_dB), _ptr(albedo),
                                           _ptr(src_cdf)), ctx)


def mcrt_philox_device(ctr, key):
    c = np.ascontiguousarray(ctr, np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, np.uint32).reshape(-1, 2)
    out = np.zeros_like(c)
    _check(load_library().mcrt_philox_device(_ptr(c), _ptr(k), _ptr(out), len(c)))
    return out


def mcrt_traj_math_device(z):
    z = np.ascontiguousarray(z, np.float64).reshape(-1)
    ln, s, c = np.zeros_like(z), np.zeros_like(z), np.zeros_like(z)
    _check(load_library().mcrt_traj_math_device(_ptr(z), _ptr(ln), _ptr(s), _ptr(c), len(z)))
    return ln, s, c


MCRT_STATIC_MAX_N = 65536


def mcrt_traj_math_device_static(z):
    """mcrt_traj_math_device through the entry point that allocates nothing on the device (n <= MCRT_STATIC_MAX_N)."""
    z = np.ascontiguousarray(z, np.float64).reshape(-1)
    ln, s, c = np.zeros_like(z), np.zeros_like(z), np.zeros_like(z)
    _check(load_library().mcrt_traj_math_device_static(_ptr(z), _ptr(ln), _ptr(s), _ptr(c), len(z)))
    return ln, s, c


def mcrt_set_stream(ctx, cuda_stream: int):
    _check(load_library().mcrt_set_stream(ctx, C.c_void_p(cuda_stream)), ctx)


def mcrt_launch_config(ctx):
    b, t, s = C.c_int(0), C.c_int(0), C.c_size_t(0)
    _check(load_library().mcrt_launch_config(ctx, C.byref(b), C.byref(t), C.byref(s)), ctx)
    return b.value, t.value, s.value


def mcrt_last_error(ctx=None) -> str:
    msg = load_library().mcrt_last_error(ctx)
    return msg.decode() if msg else ""


def mcrt_destroy(ctx):
    load_library().mcrt_destroy(ctx)


# ---------------------------------------------------------------- convenience wrapper (marshalling only)
class Context:
    """Owns a torch workspace tensor and a library context for one Workload-shaped problem."""

    def __init__(self, w, n_digests=0, device="cuda:0", inputs_on_device=False, use_torch_stream=True):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_1203_2941_b200 has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.nx, self.ny, self.nz, self.ns = w.nx, w.ny, w.nz, w.n_species
        self.nc = w.nx * w.ny * w.nz
        self.nf, self.nT, self.ndir = len(w.nu_hz), len(w.T_grid), len(w.abs_mu_edges) - 1
        nbytes = mcrt_workspace_bytes(w.nx, w.ny, w.nz, w.n_species, self.nf, self.nT, self.ndir, n_digests)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        if inputs_on_device:
            rho = w.rho if hasattr(w.rho, "data_ptr") else torch.from_numpy(np.ascontiguousarray(w.rho)).to(self.device)
            sp = w.species if hasattr(w.species, "data_ptr") else torch.from_numpy(np.ascontiguousarray(w.species)).to(self.device)
            torch.cuda.synchronize()
            where = MCRT_DEVICE
        else:
            rho = w.rho if hasattr(w.rho, "data_ptr") else np.ascontiguousarray(w.rho, np.float32)
            sp = w.species if hasattr(w.species, "data_ptr") else np.ascontiguousarray(w.species, np.uint8)
            where = MCRT_HOST
        self.ctx = mcrt_grid_create(w.nx, w.ny, w.nz, w.cell_size_cm, rho, sp, w.n_species, where,
                                    self.workspace, nbytes)
        self.stream = None
        if use_torch_stream:
            self.stream = torch.cuda.current_stream(self.device)
            mcrt_set_stream(self.ctx, self.stream.cuda_stream)
        mcrt_dust_tables(self.ctx, w.nu_hz, w.kappa_abs, w.kappa_sca, w.g, w.T_grid)
        if getattr(w, "mixtures", None) is not None:
            mcrt_dust_mixtures(self.ctx, *w.mixtures)
        self.n_subcells = 0
        if getattr(w, "subgrid", None) is not None:
            mcrt_subgrid(self.ctx, *w.subgrid)
            self.n_subcells = len(w.subgrid[1]) * int(w.subgrid[0]) ** 3
        mcrt_source(self.ctx, w.L_erg_s, w.T_star_K, w.L_nu_weights, w.source_pos_cm)
        mcrt_escape_bins(self.ctx, w.abs_mu_edges)
        self.last_n = 0

    def run(self, n_packets, seed, want_stats=True, **kw):
        o = mcrt_default_opts()
        for k, v in kw.items():
            if not hasattr(o, k):
                raise TypeError(f"unknown run option {k}")
            setattr(o, k, v)
        self.last_n = int(n_packets)
        self._recorded = bool(o.record_digests)
        return mcrt_run(self.ctx, n_packets, seed, o, want_stats)

    def _opts(self, n_packets, kw):
        o = mcrt_default_opts()
        for k, v in kw.items():
            if not hasattr(o, k):
                raise TypeError(f"unknown run option {k}")
            setattr(o, k, v)
        self.last_n = int(n_packets)
        return o

    def run_begin(self, n_packets, seed, **kw):
        mcrt_run_begin(self.ctx, n_packets, seed, self._opts(n_packets, kw))

    def run_step(self):
        return mcrt_run_step(self.ctx)

    def run_end(self, want_stats=True):
        return mcrt_run_end(self.ctx, want_stats)

    def stats(self):
        return mcrt_get_stats(self.ctx)

    def read_raw(self, digests=False):
        k = np.zeros(self.nc, np.uint64)
        L = np.zeros(self.nc, np.int64)
        sed = np.zeros((self.ndir, self.nf), np.uint64)
        sedd = np.zeros((self.ndir, self.nf), np.uint64)
        tidx = np.zeros(self.nc, np.uint16)
        dig = np.zeros(self.last_n, DIGEST_DTYPE) if digests else None
        mcrt_read_raw(self.ctx, k, L, sed, sedd, tidx, dig)
        out = {"k": k, "lucy_fx": L, "sed": sed, "sed_direct": sedd, "tidx": tidx}
        if digests:
            out["digests"] = dig
        return out

    def read_subcells(self):
        """Outputs and raw tallies of the sub-cubes (mcrt_subgrid), in its order."""
        n = self.n_subcells
        Ec, El = np.zeros(n), np.zeros(n)
        Tc, Tl = np.zeros(n, np.float32), np.zeros(n, np.float32)
        k, L, tidx = np.zeros(n, np.uint64), np.zeros(n, np.int64), np.zeros(n, np.uint16)
        mcrt_read_subcells(self.ctx, Ec, El, Tc, Tl, k, L, tidx)
        return {"E_count": Ec, "E_lucy": El, "T_count": Tc, "T_lucy": Tl, "k": k, "lucy_fx": L, "tidx": tidx}

    def read_component(self, component):
        """Outputs and raw tallies of one component of the mixtures (mcrt_dust_mixtures)."""
        Ec, El = np.zeros(self.nc), np.zeros(self.nc)
        Tc, Tl = np.zeros(self.nc, np.float32), np.zeros(self.nc, np.float32)
        k, L, tidx = np.zeros(self.nc, np.uint64), np.zeros(self.nc, np.int64), np.zeros(self.nc, np.uint16)
        mcrt_read_component(self.ctx, component, Ec, El, Tc, Tl, k, L, tidx)
        return {"E_count": Ec, "E_lucy": El, "T_count": Tc, "T_lucy": Tl, "k": k, "lucy_fx": L, "tidx": tidx}

    def read(self):
        Ec, El = np.zeros(self.nc), np.zeros(self.nc)
        Tc, Tl = np.zeros(self.nc, np.float32), np.zeros(self.nc, np.float32)
        sed = np.zeros((self.ndir, self.nf))
        mcrt_read(self.ctx, Ec, El, Tc, Tl, sed)
        return {"E_count": Ec, "E_lucy": El, "T_count": Tc, "T_lucy": Tl, "SED": sed}

    def tables(self):
        t = {"dnu": np.zeros(self.nf), "J": np.zeros((self.ns, self.nT)), "cdfB": np.zeros((self.ns, self.nT, self.nf)),
             "cdfdB": np.zeros((self.ns, self.nT, self.nf)), "albedo": np.zeros((self.ns, self.nf)),
             "srccdf": np.zeros(self.nf)}
        mcrt_read_tables(self.ctx, t["dnu"], t["J"], t["cdfB"], t["cdfdB"], t["albedo"], t["srccdf"])
        return t

    def launch_config(self):
        return mcrt_launch_config(self.ctx)

    def close(self):
        if getattr(self, "ctx", None):
            mcrt_destroy(self.ctx)
            self.ctx = None
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run_parts_local(parts, n_packets, seed, **kw):
    """A partitioned run whose parts are Contexts of ONE process on ONE device: every part
    transports its slice of every epoch, then the tallies are summed with mcrt_exchange_local.  Returns the
    (global) statistics.  Argument marshalling only."""
    n = len(parts)
    for r, c in enumerate(parts):
        c.run_begin(n_packets, seed, part_index=r, part_count=n, **kw)
    done = False
    while not done:
        flags = [c.run_step() for c in parts]
        done = flags[0]
        assert all(f == done for f in flags)
        mcrt_exchange_local([c.ctx for c in parts])
    return [c.run_end() for c in parts][0]
