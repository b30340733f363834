"""The CUDA path's node-local functions (csrc/islbm_lattice.cuh), compiled for the
host by g++ as a TEST harness, against the oracle.  Lets the hand-factored MRT
collisions be checked on a box without a GPU; the product library never runs
this host build."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2509_01099_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "host_harness", "harness.cpp")
LIB = os.path.join(HERE, "host_harness", "libharness.so")
HDR = os.path.join(HERE, "..", "paper_2509_01099_b200", "csrc", "islbm_lattice.cuh")


@pytest.fixture(scope="module")
def harness():
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(HDR)):
        subprocess.run(["g++", "-O2", "-std=c++17", "-x", "c++", "-fPIC", "-shared", "-ffp-contract=off",
                        "-o", LIB, SRC], check=True)
    return C.CDLL(LIB)


def dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def node_params(o):
    p, m = o.params(), o.matrices()
    s_nu = m["S"][1]
    s_q = m["S"][4]
    return np.array([p["gbeta"], s_nu, s_q, m["Q"][1], m["Q"][-1], p["a_T"]])


@pytest.mark.parametrize("dim", [2, 3])
def test_factored_collision_matches_oracle(harness, dim):
    w = inputs.custom_workload("t", dim, 8, stretch=1.4, Ra=3e4)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    prm = node_params(o)
    rng = np.random.default_rng(dim)
    for _ in range(50):
        f = (1 + 0.1 * rng.uniform(-1, 1, o.qf)) / o.qf
        g = 0.3 * rng.uniform(-1, 1, o.qg)
        fo, go = o.collide_node(f, g)
        fh, gh = f.copy(), g.copy()
        harness.harness_collide(dim, dptr(fh), dptr(gh), dptr(prm))
        assert np.abs(fh - fo).max() < 2e-16 * 8
        assert np.abs(gh - go).max() < 2e-16 * 8
        # deviation form (fp32-storage kernels collide f - w without re-adding the rest weights)
        fd, gd = f.copy(), g.copy()
        harness.harness_collide_dev(dim, dptr(fd), dptr(gd), dptr(prm))
        assert np.abs(fd - fo).max() < 2e-16 * 8
        assert np.abs(gd - go).max() < 2e-16 * 8
        # fp32-storage form: fp32 deviations in and out.  2-D: flow arithmetic in fp64, so on fp32-representable inputs
        # the result is the oracle's, rounded once to fp32.  3-D (ISLBM_F_FP32_3D): every temporary in fp32, a few dozen
        # fp32 operations on values of the input's size: the bound is in units of the INPUT deviations' magnitude,
        # 16 x 2^-24 (measured over 9000 nodes with deviations of 0.5 %, 5 % and 15 % of the weights: 7.0)
        wts = np.empty(o.qf); e_ = np.empty(3 * o.qf, dtype=np.int32); opp_ = np.empty(o.qf, dtype=np.int32)
        harness.harness_tables(dim, e_.ctypes.data_as(C.POINTER(C.c_int)), opp_.ctypes.data_as(C.POINTER(C.c_int)), dptr(wts))
        dev32 = (f - wts).astype(np.float32)
        g32 = g.astype(np.float32)
        fo32, go32 = o.collide_node(wts + dev32.astype(np.float64), g32.astype(np.float64))
        d_io, g_io = dev32.copy(), g32.copy()
        harness.harness_collide_dev_f32(dim, d_io.ctypes.data_as(C.POINTER(C.c_float)), g_io.ctypes.data_as(C.POINTER(C.c_float)), dptr(prm))
        if dim == 2:
            assert np.abs(d_io.astype(np.float64) - (fo32 - wts)).max() <= 2.0 ** -24 * np.abs(fo32 - wts).max() * 1.01
        else:
            assert np.abs(d_io.astype(np.float64) - (fo32 - wts)).max() <= 16 * 2.0 ** -24 * np.abs(dev32).max()
        # temperature populations: the fp32-storage kernels collide them in fp32 (ISLBM_G_FP32: a dozen fp32 operations
        # on values of the input's size), so the bound is in units of the INPUT's magnitude: 16 x 2^-24 (measured over
        # 5000 far-from-equilibrium nodes: 7.7 in 2-D, 12.0 in 3-D)
        assert np.abs(g_io.astype(np.float64) - go32).max() <= 16 * 2.0 ** -24 * np.abs(g32).max()
        # the all-fp32 deviation-form collisions themselves (3-D: the default of the fp32-storage kernels, same call as
        # above; 2-D: the ISLBM_F_FP32_2D A/B switch): same bound (measured 7.0 in 3-D, 5.5 in 2-D)
        d_io, g_io = dev32.copy(), g32.copy()
        harness.harness_collide_dev_allf32(dim, d_io.ctypes.data_as(C.POINTER(C.c_float)), g_io.ctypes.data_as(C.POINTER(C.c_float)), dptr(prm))
        assert np.abs(d_io.astype(np.float64) - (fo32 - wts)).max() <= 16 * 2.0 ** -24 * np.abs(dev32).max()
        assert np.abs(g_io.astype(np.float64) - go32).max() <= 16 * 2.0 ** -24 * np.abs(g32).max()
        # fields from post-collision populations == fields of the pre-collision state
        out = np.empty(5)
        harness.harness_fields_post(dim, dptr(fh), dptr(gh), dptr(prm), dptr(out))
        o2 = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
        F = np.zeros((o.qf,) + o.shape) + f[:, None, None, None]
        G = np.zeros((o.qg,) + o.shape) + g[:, None, None, None]
        o2.set_populations(F, G)
        fl = o2.fields()
        ref = np.array([fl[k][0, 0, 0] for k in ("rho", "u", "v", "w", "T")])
        assert np.abs(out - ref).max() < 1e-15


@pytest.mark.parametrize("dim", [2, 3])
def test_direction_tables_match_oracle(harness, dim):
    w = inputs.custom_workload("t", dim, 4)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    ef, _ = o.velocities()
    e = np.empty((o.qf, 3), dtype=np.int32)
    opp = np.empty(o.qf, dtype=np.int32)
    wt = np.empty(o.qf)
    harness.harness_tables(dim, e.ctypes.data_as(C.POINTER(C.c_int)), opp.ctypes.data_as(C.POINTER(C.c_int)), dptr(wt))
    assert np.array_equal(e, ef)
    for q in range(o.qf):
        assert np.array_equal(ef[opp[q]], -ef[q])
    o.init(0, 0.0)
    f, _ = o.get_populations()
    assert np.allclose(wt, f[:, 0, 0, 0], atol=1e-16)


@pytest.mark.parametrize("dim", [2, 3])
def test_storage_planes_are_a_permutation_grouped_by_halo_shape(harness, dim):
    """plane_f / plane_g (csrc/islbm_lattice.cuh) must be a bijection onto 0..Q-1 whose consecutive runs are
    the groups one TMA box loads: same halo shape (which of e_x, e_y is non-zero) and same marching role
    (e_march == 0: read at the emitted slice; != 0: read at the stencil slices)."""
    w = inputs.custom_workload("t", dim, 4)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    ef, eg = o.velocities()
    qf, qg = o.qf, o.qg
    ip = C.POINTER(C.c_int)
    pf, pg, inv = np.empty(qf, np.int32), np.empty(qg, np.int32), np.empty(qf + qg, np.int32)
    harness.harness_planes(dim, pf.ctypes.data_as(ip), pg.ctypes.data_as(ip), inv.ctypes.data_as(ip))
    assert sorted(list(pf) + list(pg)) == list(range(qf + qg))
    for q in range(qf):
        assert inv[pf[q]] == q
    for q in range(qg):
        assert inv[pg[q]] == qf + q
    march = dim - 1                      # y in 2-D, z in 3-D
    inplane = [a for a in range(dim) if a != march]
    vel = {int(pf[q]): ef[q] for q in range(qf)}
    vel.update({int(pg[q]): eg[q] for q in range(qg)})
    key = lambda p: (bool(vel[p][march] != 0), tuple(bool(vel[p][a] != 0) for a in inplane))
    runs = []
    for p in range(qf + qg):
        if not runs or key(runs[-1][0]) != key(p):
            runs.append([p])
        else:
            runs[-1].append(p)
    assert [len(r) for r in runs] == ([2, 4, 4, 4] if dim == 2 else [2, 4, 4, 4, 4, 4, 4])
    assert len({key(r[0]) for r in runs}) == len(runs)
