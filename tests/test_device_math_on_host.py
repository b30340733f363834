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
