"""CPU-side checks of the boundary: the shared library loads and exports every symbol include/mcrt.h
declares; pure host entry points behave; nothing computes without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1203_2941_b200 import build

    return build.build()


def test_library_exports_every_declared_symbol(lib_path):
    hdr = open(os.path.join(ROOT, "include", "mcrt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(mcrt_[a-z_0-9]+)\s*\(", hdr)))
    assert len(declared) >= 15
    lib = ctypes.CDLL(lib_path)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in mcrt.h but not exported"
    from paper_1203_2941_b200 import binding

    assert sorted(binding.EXPORTS) == declared
    for name in declared:
        assert hasattr(binding, name), f"binding lacks {name}"


def test_pure_host_entry_points(lib_path):
    from paper_1203_2941_b200 import binding as B

    assert "sm_100a" in B.mcrt_version()
    o = B.mcrt_default_opts()
    assert o.mode == B.MCRT_MODE_BW_EPOCH and o.reset_tallies == 1 and o.sweep_T_from_lucy == 1
    n = B.mcrt_workspace_bytes(256, 256, 256, 3, 120, 1000, 9, 0)
    nc = 256 ** 3
    assert 5 * 8 * nc < n < 5 * 8 * nc + 64 * 2 ** 20
    assert B.mcrt_workspace_bytes(256, 256, 256, 3, 120, 1000, 9, 10 ** 6) - n >= 24 * 10 ** 6
    with pytest.raises(B.McrtError):
        B.mcrt_workspace_bytes(0, 1, 1, 1, 2, 2, 1, 0)
    # ragged sizes are padded to whole 4x4x4 bricks
    assert B.mcrt_workspace_bytes(5, 5, 5, 1, 2, 2, 1) > B.mcrt_workspace_bytes(4, 4, 4, 1, 2, 2, 1)


def test_no_cpu_fallback(lib_path):
    """Without a CUDA device the product must fail loudly, never compute on the CPU."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1203_2941_b200 import binding as B, workloads as W

    w = W.sphere32(n=8)
    with pytest.raises(B.McrtError) as e:
        B.mcrt_grid_create(8, 8, 8, w.cell_size_cm, w.rho, w.species, 1)
    assert e.value.code == B.MCRT_ECUDA
    with pytest.raises(RuntimeError):
        B.Context(w)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1203_2941_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("CPU oracle", "").replace("the oracle", "").replace("with the oracle", ""), f
    # and the oracle does not import the product
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1203_2941_b200" not in src and "from paper_1203_2941_b200" not in src
            assert "mcrt.h" not in src and "libmcrt" not in src


def test_workloads_are_seeded_and_shaped():
    from paper_1203_2941_b200 import workloads as W

    a, b = W.torus256(n_clumps=100, n=32), W.torus256(n_clumps=100, n=32)
    assert np.array_equal(a.rho, b.rho) and np.array_equal(a.species, b.species)
    c = W.torus256(n_clumps=100, n=32, geometry_seed=77)
    assert not np.array_equal(a.rho, c.rho)
    assert a.n_species == 3 and a.n_nu == 120 and a.n_dir == 9 and a.T_star_K <= 0 and a.L_nu_weights is not None
    assert np.all(np.diff(a.nu_hz) > 0) and np.all(np.diff(a.abs_mu_edges) > 0)
    assert (a.L_nu_weights > 0).sum() > 10 and (a.L_nu_weights == 0).sum() > 10
    s = W.sphere32()
    assert s.rho.shape == (32, 32, 32) and s.n_packets == 100_000 and s.n_nu == 64
    # tau_V normalisation: kappa_ext(V) * sum(rho h) along +x from the centre = 1
    col = s.rho[16, 16, 16:].astype(np.float64).sum() * s.cell_size_cm * W.KAPPA_V_EXT
    assert abs(col - 1.0) < 1e-6
    d = W.disk256(n=32)
    assert d.n_species == 2 and d.n_dir == 10 and set(np.unique(d.species)) <= {0, 1}
    sh = W.shell128(n=32)
    assert sh.rho[16, 16, 16] > sh.rho[16, 16, 30] > 0
    t5 = W.torus512(n_clumps=50, n=32)
    assert t5.n_nu == 200 and t5.n_species == 3
