"""Host logic of the CUDA path: csrc/dda.h (face parameters, O(1) jump over boxes of vacuum cells) compiled
for the host and checked against the oracle's plain cell-by-cell walk (oracle.dda_trace) on random and
degenerate rays: identical dusty-cell list, identical segment lengths BIT FOR BIT, identical face count."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1203_2941_b200", "csrc")


@pytest.fixture(scope="module")
def dda(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("dda") / "libdda_host.so")
    subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-Wall",
                    "-o", out, os.path.join(CSRC, "dda_host.cpp")], check=True)
    L = C.CDLL(out)
    L.mcrt_dda_host_trace.restype = C.c_int
    L.mcrt_dda_host_trace.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]

    def trace(n, dusty, msh, p, u, c0, use_jumps=1, max_n=8192):
        cells = np.zeros(max_n, np.int64)
        ds = np.zeros(max_n, np.float64)
        faces = C.c_uint64(0)
        te = C.c_double(0)
        nj = C.c_int(0)
        p = np.ascontiguousarray(p, np.float64); u = np.ascontiguousarray(u, np.float64)
        c0 = np.ascontiguousarray(c0, np.int32)
        k = L.mcrt_dda_host_trace(n[0], n[1], n[2], dusty.ctypes.data, msh, p.ctypes.data, u.ctypes.data, c0.ctypes.data,
                                  use_jumps, max_n, cells.ctypes.data, ds.ctypes.data, C.byref(faces), C.byref(te),
                                  C.byref(nj))
        assert k <= max_n
        return cells[:k], ds[:k], faces.value, te.value, nj.value

    return trace


def _start_cell(p, u):
    c = np.floor(p).astype(np.int64)
    on = p == np.floor(p)
    c[on & (u < 0)] -= 1
    return c


def test_jump_walk_equals_cell_walk_random(orc, dda):
    rng = np.random.default_rng(7)
    total_jumps = 0
    for case in range(300):
        n = rng.integers(1, 41, 3)
        msh = int(rng.integers(2, 4))
        fill = rng.choice([0.0, 0.002, 0.02, 0.3])
        dusty = (rng.random((n[2], n[1], n[0])) < fill).astype(np.uint8)
        if rng.random() < 0.5:  # a few solid blobs like clumps
            for _ in range(3):
                c = [rng.integers(0, n[a]) for a in range(3)]
                dusty[max(0, c[2] - 1):c[2] + 2, max(0, c[1] - 1):c[1] + 2, max(0, c[0] - 1):c[0] + 2] = 1
        for _ in range(40):
            p = rng.random(3) * n
            if rng.random() < 0.3:   # points on faces / edges / corners
                k = rng.integers(0, 3)
                p[k] = np.round(p[k])
                if rng.random() < 0.5:
                    p[(k + 1) % 3] = np.round(p[(k + 1) % 3])
            u = rng.normal(size=3)
            r = rng.random()
            if r < 0.15:
                u[rng.integers(0, 3)] = 0.0            # axis-parallel planes
            elif r < 0.25:
                u[rng.integers(0, 3)] *= 1e-12          # grazing
            elif r < 0.3:
                u = np.sign(u) * np.array([1.0, 1.0, 1.0])  # exact diagonals: ties on every face
            elif r < 0.35:
                a = rng.integers(0, 3); u = np.zeros(3); u[a] = rng.choice([-1.0, 1.0])
            elif r < 0.4:
                u[rng.integers(0, 3)] = rng.choice([-1.0, 1.0]) * 1e-300   # 1/u ~ 1e300: face parameters overflow
            if not np.any(u):
                u[0] = 1.0
            u = u / np.sqrt(np.sum(u * u))
            c0 = _start_cell(p, u)
            if np.any(c0 < 0) or np.any(c0 >= n):
                continue
            cells_o, ds_o = orc.dda_trace(int(n[0]), int(n[1]), int(n[2]), p, u, max_n=8192)
            keep = dusty.reshape(-1)[cells_o] != 0
            cells_j, ds_j, faces, te, nj = dda(n, dusty, msh, p, u, c0)
            cells_s, ds_s, faces_s, te_s, nj_s = dda(n, dusty, msh, p, u, c0, use_jumps=0)
            cells_c, ds_c, faces_c, te_c, nj_c = dda(n, dusty, msh, p, u, c0, use_jumps=2)   # distance-map cubes
            assert faces_c == faces and np.array_equal(cells_c, cells_j), (case, p, u)
            assert np.array_equal(ds_c.view(np.uint64), ds_j.view(np.uint64)), (case, p, u)
            assert np.float64(te_c).view(np.uint64) == np.float64(te_s).view(np.uint64), (case, p, u)
            assert nj_s == 0 and faces_s == len(cells_o) == faces, (case, p, u)
            assert np.array_equal(cells_j, cells_o[keep]), (case, p, u)
            assert np.array_equal(ds_j.view(np.uint64), ds_o[keep].view(np.uint64)), (case, p, u)
            assert np.array_equal(ds_s.view(np.uint64), ds_o[keep].view(np.uint64)), (case, p, u)
            assert np.float64(te).view(np.uint64) == np.float64(te_s).view(np.uint64), (case, p, u)
            total_jumps += nj
    assert total_jumps > 2000


def test_jump_walk_large_empty_grid(orc, dda):
    """256^3 with one dusty block: level-2 (64-cell) jumps; face counts in the hundreds."""
    rng = np.random.default_rng(11)
    n = np.array([256, 200, 130])
    dusty = np.zeros((n[2], n[1], n[0]), np.uint8)
    dusty[60:70, 90:110, 120:140] = 1
    for _ in range(300):
        p = np.array([128.0, 100.0, 65.0]) if rng.random() < 0.5 else rng.random(3) * n
        u = rng.normal(size=3)
        u /= np.sqrt(np.sum(u * u))
        c0 = _start_cell(p, u)
        cells_o, ds_o = orc.dda_trace(int(n[0]), int(n[1]), int(n[2]), p, u, max_n=8192)
        keep = dusty.reshape(-1)[cells_o] != 0
        cells_j, ds_j, faces, te, nj = dda(n, dusty, 2, p, u, c0)
        assert faces == len(cells_o)
        assert np.array_equal(cells_j, cells_o[keep])
        assert np.array_equal(ds_j.view(np.uint64), ds_o[keep].view(np.uint64))
        assert nj < faces / 4 + 8
