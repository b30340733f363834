"""ctypes loader for the CPU oracle (oracle/islbm_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs import this module.  It
imports nothing from paper_2509_01099_b200 (the CUDA path) and holds no
arithmetic of the method: it compiles the C file with gcc and marshals numpy
arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "islbm_oracle.c")
_HDR = os.path.join(_HERE, "islbm_oracle.h")
_LIB = os.path.join(_HERE, "libislbm_oracle.so")
_lock = threading.Lock()
_lib = None

# -ffp-contract=off: no FMA contraction, the oracle evaluates the formulas as written.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile oracle/islbm_oracle.c -> oracle/libislbm_oracle.so (gcc)."""
    with _lock:
        stale = (
            force
            or not os.path.exists(_LIB)
            or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
        )
        if stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True, cwd=_HERE)
            os.replace(tmp, _LIB)
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _ptr(a, typ=_dp):
    return None if a is None else a.ctypes.data_as(typ)


def load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    vp = C.c_void_p
    sig = {
        "oracle_create": (vp, [C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, C.c_double, C.c_double, C.c_double, C.c_double]),
        "oracle_destroy": (None, [vp]),
        "oracle_set_threads": (None, [vp, C.c_int]),
        "oracle_get_threads": (C.c_int, [vp]),
        "oracle_set_buoyancy_scale": (None, [vp, C.c_double]),
        "oracle_set_reference_temperature": (None, [vp, C.c_double]),
        "oracle_set_stencil": (None, [vp, C.c_int]),
        "oracle_init": (None, [vp, C.c_ulonglong, C.c_double]),
        "oracle_set_populations": (None, [vp, _dp, _dp]),
        "oracle_get_populations": (None, [vp, _dp, _dp]),
        "oracle_get_post_collision": (None, [vp, _dp, _dp]),
        "oracle_set_post_collision": (None, [vp, _dp, _dp]),
        "oracle_collide": (None, [vp]),
        "oracle_stream": (None, [vp]),
        "oracle_step": (None, [vp, C.c_int]),
        "oracle_step_node": (None, [vp, C.c_int, C.c_int, C.c_int, _dp, _dp]),
        "oracle_fields": (None, [vp, _dp, _dp, _dp, _dp, _dp]),
        "oracle_nusselt": (None, [vp, _dp]),
        "oracle_nusselt_middle": (C.c_double, [vp]),
        "oracle_mass": (None, [vp, _dp]),
        "oracle_qf": (C.c_int, [vp]),
        "oracle_qg": (C.c_int, [vp]),
        "oracle_get_velocities": (None, [vp, _ip, _ip]),
        "oracle_get_matrices": (None, [vp, _dp, _dp, _dp, _dp, _dp, _dp]),
        "oracle_get_params": (None, [vp, _dp]),
        "oracle_get_weights": (None, [vp, C.c_int, C.c_int, _ip, _dp]),
        "oracle_meq": (None, [vp, C.c_double, _dp, _dp]),
        "oracle_neq": (None, [vp, C.c_double, _dp, _dp]),
        "oracle_mforce": (None, [vp, _dp, _dp, _dp]),
        "oracle_collide_node": (None, [vp, _dp, _dp, _dp, _dp]),
        "oracle_wall_derivative": (C.c_double, [C.c_double, C.c_double, C.c_double, C.c_double]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


PARAM_NAMES = ("U", "H_lu", "nu", "alpha", "gbeta", "tau_f", "a_T", "omega_bc", "dt_star", "L_eff_x", "L_eff_y", "L_eff_z")
NUSSELT_NAMES = ("Nu_hot", "Nu_cold", "Re", "u2", "Nu_vol")


def wall_derivative(q, phi_wall, phi1, phi2):
    return load().oracle_wall_derivative(q, phi_wall, phi1, phi2)


class Oracle:
    """One cavity on the CPU.  coords: list of 2 or 3 fp64 arrays (x, y[, z])."""

    def __init__(self, coords, delta, Ra, Pr, Ma, threads=1):
        self.lib = load()
        self.dim = len(coords)
        self.coords = [np.ascontiguousarray(c, dtype=np.float64) for c in coords]
        n = [len(c) for c in self.coords] + [1] * (3 - self.dim)
        self.n = tuple(n)
        xs = self.coords + [None] * (3 - self.dim)
        self.h = self.lib.oracle_create(self.dim, n[0], n[1], n[2], _ptr(xs[0]), _ptr(xs[1]), _ptr(xs[2]),
                                        float(delta), float(Ra), float(Pr), float(Ma))
        if not self.h:
            raise ValueError("oracle_create rejected the input")
        self.qf = self.lib.oracle_qf(self.h)
        self.qg = self.lib.oracle_qg(self.h)
        self.shape = (n[2], n[1], n[0])  # [z][y][x]
        self.set_threads(threads)

    def close(self):
        if getattr(self, "h", None):
            self.lib.oracle_destroy(self.h)
            self.h = None

    __del__ = close

    # -- state ---------------------------------------------------------------
    def set_threads(self, n):
        self.lib.oracle_set_threads(self.h, int(n))

    @property
    def threads(self):
        return self.lib.oracle_get_threads(self.h)

    def set_buoyancy_scale(self, s):
        self.lib.oracle_set_buoyancy_scale(self.h, float(s))

    def set_stencil(self, kind):
        self.lib.oracle_set_stencil(self.h, int(kind))

    def set_reference_temperature(self, T0):
        self.lib.oracle_set_reference_temperature(self.h, float(T0))

    def init(self, seed=0, amp=1e-3):
        self.lib.oracle_init(self.h, int(seed), float(amp))

    def _alloc(self):
        return (np.empty((self.qf,) + self.shape), np.empty((self.qg,) + self.shape))

    def set_populations(self, f, g):
        f = np.ascontiguousarray(f, dtype=np.float64)
        g = np.ascontiguousarray(g, dtype=np.float64)
        assert f.shape == (self.qf,) + self.shape and g.shape == (self.qg,) + self.shape
        self.lib.oracle_set_populations(self.h, _ptr(f), _ptr(g))

    def get_populations(self):
        f, g = self._alloc()
        self.lib.oracle_get_populations(self.h, _ptr(f), _ptr(g))
        return f, g

    def get_post_collision(self):
        f, g = self._alloc()
        self.lib.oracle_get_post_collision(self.h, _ptr(f), _ptr(g))
        return f, g

    def set_post_collision(self, fp, gp):
        fp = np.ascontiguousarray(fp, dtype=np.float64)
        gp = np.ascontiguousarray(gp, dtype=np.float64)
        assert fp.shape == (self.qf,) + self.shape and gp.shape == (self.qg,) + self.shape
        self.lib.oracle_set_post_collision(self.h, _ptr(fp), _ptr(gp))

    # -- the step ------------------------------------------------------------
    def collide(self):
        self.lib.oracle_collide(self.h)

    def stream(self):
        self.lib.oracle_stream(self.h)

    def step(self, n=1):
        self.lib.oracle_step(self.h, int(n))

    def step_node(self, ix, iy, iz=0):
        of, og = np.empty(self.qf), np.empty(self.qg)
        self.lib.oracle_step_node(self.h, int(ix), int(iy), int(iz), _ptr(of), _ptr(og))
        return of, og

    def collide_node(self, f, g):
        f = np.ascontiguousarray(f, dtype=np.float64)
        g = np.ascontiguousarray(g, dtype=np.float64)
        fp, gp = np.empty(self.qf), np.empty(self.qg)
        self.lib.oracle_collide_node(self.h, _ptr(f), _ptr(g), _ptr(fp), _ptr(gp))
        return fp, gp

    # -- diagnostics ---------------------------------------------------------
    def fields(self):
        out = [np.empty(self.shape) for _ in range(5)]
        self.lib.oracle_fields(self.h, *[_ptr(a) for a in out])
        return dict(zip(("rho", "u", "v", "w", "T"), out))

    def nusselt(self):
        out = np.empty(5)
        self.lib.oracle_nusselt(self.h, _ptr(out))
        return dict(zip(NUSSELT_NAMES, out.tolist()))

    def nusselt_middle(self):
        return float(self.lib.oracle_nusselt_middle(self.h))

    def mass(self):
        out = np.empty(2)
        self.lib.oracle_mass(self.h, _ptr(out))
        return {"weighted": out[0], "plain": out[1]}

    # -- introspection for the pins -----------------------------------------
    def params(self):
        out = np.empty(12)
        self.lib.oracle_get_params(self.h, _ptr(out))
        return dict(zip(PARAM_NAMES, out.tolist()))

    def velocities(self):
        ef = np.empty((self.qf, 3), dtype=np.int32)
        eg = np.empty((self.qg, 3), dtype=np.int32)
        self.lib.oracle_get_velocities(self.h, _ptr(ef, _ip), _ptr(eg, _ip))
        return ef, eg

    def matrices(self):
        M, Mi, S = np.empty((self.qf, self.qf)), np.empty((self.qf, self.qf)), np.empty(self.qf)
        N, Ni, Q = np.empty((self.qg, self.qg)), np.empty((self.qg, self.qg)), np.empty(self.qg)
        self.lib.oracle_get_matrices(self.h, _ptr(M), _ptr(Mi), _ptr(S), _ptr(N), _ptr(Ni), _ptr(Q))
        return dict(M=M, Minv=Mi, S=S, N=N, Ninv=Ni, Q=Q)

    def weights(self, axis, c):
        """base[n], w[n,3] for velocity component c in {-1,+1} along axis."""
        n = self.n[axis]
        base = np.empty(n, dtype=np.int32)
        w = np.empty((n, 3))
        self.lib.oracle_get_weights(self.h, int(axis), 1 if c > 0 else 0, _ptr(base, _ip), _ptr(w))
        return base, w

    def meq(self, rho, u):
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.empty(self.qf)
        self.lib.oracle_meq(self.h, float(rho), _ptr(u), _ptr(out))
        return out

    def neq(self, T, u):
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.empty(self.qg)
        self.lib.oracle_neq(self.h, float(T), _ptr(u), _ptr(out))
        return out

    def mforce(self, u, F):
        u = np.ascontiguousarray(u, dtype=np.float64)
        F = np.ascontiguousarray(F, dtype=np.float64)
        out = np.empty(self.qf)
        self.lib.oracle_mforce(self.h, _ptr(u), _ptr(F), _ptr(out))
        return out
