"""Thin Python binding of the C-ABI in include/islbm.h (argument marshalling only).

PyTorch supplies device memory and the CUDA stream; every step of the path runs
in the kernels of libislbm.so.  There is no fallback: if the library has not been
built, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libislbm.so")

D2Q9_D2Q5, D3Q19_D3Q7 = 0, 1
F64, F32_STORAGE = 0, 1
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED, KERNEL_UNIFORM_SHIFT = 0, 1, 2, 3

EXPORTS = (
    "islbm_workspace_bytes", "islbm_create", "islbm_create_slab", "islbm_halo", "islbm_halo_layout", "islbm_slab_set_peer", "islbm_diag_sums", "islbm_diag_from_sums",
    "islbm_residual_sums", "islbm_destroy", "islbm_get_params", "islbm_init",
    "islbm_set_populations", "islbm_set_populations_host", "islbm_get_populations", "islbm_step", "islbm_fields", "islbm_nusselt", "islbm_nusselt_static", "islbm_nusselt_middle",
    "islbm_steady_residual", "islbm_set_buoyancy_scale", "islbm_set_reference_temperature", "islbm_set_stencil", "islbm_set_kernel", "islbm_set_tuning", "islbm_launch_count",
    "islbm_kernel_name", "islbm_last_error", "islbm_version",
)


class _Mesh(C.Structure):
    _fields_ = [("dim", C.c_int), ("n", C.c_int * 3), ("x", C.POINTER(C.c_double) * 3), ("delta", C.c_double)]


class _Slab(C.Structure):
    _fields_ = [("lo_is_wall", C.c_int), ("hi_is_wall", C.c_int), ("L_eff_global", C.c_double), ("node_offset", C.c_longlong)]


class _Halo(C.Structure):
    _fields_ = [("is_wall", C.c_int), ("first_plane", C.c_int), ("n_planes", C.c_int), ("plane_pitch_bytes", C.c_size_t),
                ("layer_bytes", C.c_size_t), ("send_offset", C.c_size_t), ("recv_offset", C.c_size_t)]


class _HaloLayout(C.Structure):
    _fields_ = [("is_wall", C.c_int), ("cur", C.c_int), ("ghost_offset", C.c_size_t * 2), ("plane_pitch_bytes", C.c_size_t),
                ("layer_bytes", C.c_size_t), ("flag_offset", C.c_size_t), ("steps", C.c_longlong)]


class _Params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("U", "H_lu", "nu", "alpha", "gbeta", "tau_f", "a_T", "omega_bc", "dt_star")] + [
        ("L_eff", C.c_double * 3)]


class IslbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"islbm error {code}: {msg}")
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.islbm_workspace_bytes.argtypes = [C.POINTER(_Mesh), C.c_int, C.c_int, C.POINTER(C.c_size_t)]
    lib.islbm_create.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.c_int, C.c_double, C.c_double, C.c_double,
                                 C.c_int, vp, C.c_size_t, vp]
    lib.islbm_create_slab.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.c_int, C.c_double, C.c_double, C.c_double,
                                      C.c_int, vp, C.c_size_t, vp, C.POINTER(_Slab)]
    lib.islbm_halo.argtypes = [vp, C.c_int, C.POINTER(_Halo)]
    lib.islbm_halo_layout.argtypes = [vp, C.c_int, C.POINTER(_HaloLayout)]
    lib.islbm_slab_set_peer.argtypes = [vp, C.c_int, vp, C.POINTER(_HaloLayout)]
    lib.islbm_diag_sums.argtypes = [vp, dp]
    lib.islbm_diag_from_sums.argtypes = [vp, dp, dp]
    lib.islbm_residual_sums.argtypes = [vp, dp, C.POINTER(C.c_int)]
    lib.islbm_destroy.argtypes = [vp]
    lib.islbm_destroy.restype = None
    lib.islbm_get_params.argtypes = [vp, C.POINTER(_Params)]
    lib.islbm_init.argtypes = [vp, C.c_ulonglong, C.c_double]
    lib.islbm_set_populations.argtypes = [vp, vp, vp]
    lib.islbm_set_populations_host.argtypes = [vp, vp, vp]
    lib.islbm_get_populations.argtypes = [vp, vp, vp]
    lib.islbm_step.argtypes = [vp, C.c_int]
    lib.islbm_fields.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.islbm_nusselt.argtypes = [vp, dp]
    lib.islbm_nusselt_static.argtypes = [vp, dp]
    lib.islbm_nusselt_middle.argtypes = [vp, dp]
    lib.islbm_steady_residual.argtypes = [vp, dp]
    lib.islbm_set_buoyancy_scale.argtypes = [vp, C.c_double]
    lib.islbm_set_reference_temperature.argtypes = [vp, C.c_double]
    lib.islbm_set_stencil.argtypes = [vp, C.c_int]
    lib.islbm_set_kernel.argtypes = [vp, C.c_int]
    lib.islbm_set_tuning.argtypes = [vp, C.c_char_p, C.c_int]
    lib.islbm_launch_count.argtypes = [vp]
    lib.islbm_launch_count.restype = C.c_longlong
    lib.islbm_kernel_name.argtypes = [vp]
    lib.islbm_kernel_name.restype = C.c_char_p
    lib.islbm_last_error.restype = C.c_char_p
    lib.islbm_version.restype = C.c_char_p
    return lib


lib = _load()


def _check(rc):
    if rc != 0:
        raise IslbmError(rc, lib.islbm_last_error().decode())


def _mesh_struct(coords, delta):
    dim = len(coords)
    arrs = [np.ascontiguousarray(c, dtype=np.float64) for c in coords]
    m = _Mesh()
    m.dim = dim
    for a in range(3):
        m.n[a] = len(arrs[a]) if a < dim else 1
        m.x[a] = arrs[a].ctypes.data_as(C.POINTER(C.c_double)) if a < dim else None
    m.delta = float(delta)
    return m, arrs   # keep arrs alive while m is used


def workspace_bytes(coords, delta, precision=F64):
    m, _keep = _mesh_struct(coords, delta)
    out = C.c_size_t(0)
    _check(lib.islbm_workspace_bytes(C.byref(m), D2Q9_D2Q5 if m.dim == 2 else D3Q19_D3Q7, precision, C.byref(out)))
    return out.value


def _dev_ptr(t, n_expected=None):
    if t is None:
        return None
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    if n_expected is not None:
        assert t.numel() == n_expected, (t.shape, n_expected)
    return C.c_void_p(t.data_ptr())


class Islbm:
    """islbm_create / islbm_step / islbm_fields / islbm_nusselt on one CUDA device."""

    def __init__(self, coords, delta, Ra, Pr, Ma, precision=F64, device="cuda", stream=None, guard_bytes=0, slab=None):
        """slab = None, or dict(lo_is_wall, hi_is_wall, L_eff_global, node_offset): a slab of a larger cavity whose
        slowest-axis coordinates include one ghost layer at each non-wall end (islbm_create_slab)."""
        self.dim = len(coords)
        self.precision = precision
        self.device = torch.device(device)
        m, keep = _mesh_struct(coords, delta)
        self.n = tuple(m.n)
        self.shape = (self.n[2], self.n[1], self.n[0])
        self.nodes = self.n[0] * self.n[1] * self.n[2]
        self.qf, self.qg = (9, 5) if self.dim == 2 else (19, 7)
        lattice = D2Q9_D2Q5 if self.dim == 2 else D3Q19_D3Q7
        nbytes = C.c_size_t(0)
        _check(lib.islbm_workspace_bytes(C.byref(m), lattice, precision, C.byref(nbytes)))
        # owned here; guard_bytes (a multiple of 256) adds canary bands around the workspace for the out-of-bounds test
        assert guard_bytes % 256 == 0
        self.guard_bytes = guard_bytes
        self._alloc = torch.full((nbytes.value + 2 * guard_bytes,), 0xA5, dtype=torch.uint8, device=self.device) \
            if guard_bytes else torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
        self.workspace = self._alloc[guard_bytes:guard_bytes + nbytes.value]
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.h = C.c_void_p()
        if slab is None:
            _check(lib.islbm_create(C.byref(self.h), C.byref(m), lattice, float(Ra), float(Pr), float(Ma), precision,
                                    C.c_void_p(self.workspace.data_ptr()), nbytes.value, C.c_void_p(self.stream.cuda_stream)))
        else:
            sl = _Slab(int(slab["lo_is_wall"]), int(slab["hi_is_wall"]), float(slab["L_eff_global"]), int(slab["node_offset"]))
            _check(lib.islbm_create_slab(C.byref(self.h), C.byref(m), lattice, float(Ra), float(Pr), float(Ma), precision,
                                         C.c_void_p(self.workspace.data_ptr()), nbytes.value,
                                         C.c_void_p(self.stream.cuda_stream), C.byref(sl)))
        del keep

    def _out(self, shape):
        """Output tensor for a library call: allocated by torch's caching allocator on the CURRENT stream but written
        by kernels on the handle's stream, so the allocator is told about that use (no re-use while they run)."""
        t = torch.empty(shape, dtype=torch.float64, device=self.device)
        if self.stream != torch.cuda.current_stream(self.device):
            t.record_stream(self.stream)
        return t

    def guards_intact(self):
        """True if no kernel wrote into the canary bands around the workspace."""
        g = self.guard_bytes
        return bool((self._alloc[:g] == 0xA5).all().item() and (self._alloc[self._alloc.numel() - g:] == 0xA5).all().item())

    def close(self):
        if getattr(self, "h", None):
            lib.islbm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def params(self):
        p = _Params()
        _check(lib.islbm_get_params(self.h, C.byref(p)))
        d = {k: getattr(p, k) for k, _ in _Params._fields_ if k != "L_eff"}
        d.update(L_eff_x=p.L_eff[0], L_eff_y=p.L_eff[1], L_eff_z=p.L_eff[2])
        return d

    def set_buoyancy_scale(self, s):
        _check(lib.islbm_set_buoyancy_scale(self.h, float(s)))

    def set_reference_temperature(self, T0):
        _check(lib.islbm_set_reference_temperature(self.h, float(T0)))

    def set_stencil(self, kind):
        _check(lib.islbm_set_stencil(self.h, int(kind)))

    def set_kernel(self, which):
        _check(lib.islbm_set_kernel(self.h, int(which)))

    def set_tuning(self, **kv):
        for k, v in kv.items():
            _check(lib.islbm_set_tuning(self.h, k.encode(), int(v)))

    @property
    def kernel_name(self):
        return lib.islbm_kernel_name(self.h).decode()

    @property
    def launch_count(self):
        return int(lib.islbm_launch_count(self.h))

    def init(self, seed=0, noise_amp=1e-3):
        _check(lib.islbm_init(self.h, int(seed), float(noise_amp)))

    def set_populations(self, f, g):
        _check(lib.islbm_set_populations(self.h, _dev_ptr(f, self.qf * self.nodes), _dev_ptr(g, self.qg * self.nodes)))

    def set_populations_host(self, f, g):
        """f, g: HOST torch tensors (pinned for asynchronous copies) or numpy arrays, fp64, dense [q][z][y][x]."""
        def hp(a, n):
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float64 and a.flags.c_contiguous and a.size == n
                return C.c_void_p(a.ctypes.data)
            assert (not a.is_cuda) and a.dtype == torch.float64 and a.is_contiguous() and a.numel() == n
            return C.c_void_p(a.data_ptr())
        _check(lib.islbm_set_populations_host(self.h, hp(f, self.qf * self.nodes), hp(g, self.qg * self.nodes)))

    def get_populations(self):
        f = self._out((self.qf,) + self.shape)
        g = self._out((self.qg,) + self.shape)
        _check(lib.islbm_get_populations(self.h, _dev_ptr(f), _dev_ptr(g)))
        return f, g

    def step(self, n=1):
        _check(lib.islbm_step(self.h, int(n)))

    def fields(self, names=("rho", "u", "v", "w", "T")):
        out = {k: self._out(self.shape) for k in names if not (k == "w" and self.dim == 2)}
        _check(lib.islbm_fields(self.h, *[_dev_ptr(out.get(k)) for k in ("rho", "u", "v", "w", "T")]))
        return out

    def nusselt(self):
        out = (C.c_double * 5)()
        _check(lib.islbm_nusselt(self.h, out))
        return dict(zip(("Nu_hot", "Nu_cold", "Re", "u2", "Nu_vol"), list(out)))

    def nusselt_static(self):
        """islbm_nusselt with its scratch in a static device array of the library: allocates nothing (at most 33 554 432 nodes)."""
        out = (C.c_double * 5)()
        _check(lib.islbm_nusselt_static(self.h, out))
        return dict(zip(("Nu_hot", "Nu_cold", "Re", "u2", "Nu_vol"), list(out)))

    def halo(self, side):
        """(is_wall, [send views], [recv views]) of the current state: uint8 views of the workspace, one per plane."""
        hi = _Halo()
        _check(lib.islbm_halo(self.h, int(side), C.byref(hi)))
        send = [self.workspace[hi.send_offset + p * hi.plane_pitch_bytes: hi.send_offset + p * hi.plane_pitch_bytes + hi.layer_bytes]
                for p in range(hi.n_planes)]
        recv = [self.workspace[hi.recv_offset + p * hi.plane_pitch_bytes: hi.recv_offset + p * hi.plane_pitch_bytes + hi.layer_bytes]
                for p in range(hi.n_planes)]
        return bool(hi.is_wall), send, recv

    def halo_layout(self, side):
        """Plain dict (picklable) describing this handle's ghost layer of `side` inside its workspace."""
        hl = _HaloLayout()
        _check(lib.islbm_halo_layout(self.h, int(side), C.byref(hl)))
        return dict(is_wall=bool(hl.is_wall), cur=hl.cur, ghost_offset=[hl.ghost_offset[0], hl.ghost_offset[1]],
                    plane_pitch_bytes=hl.plane_pitch_bytes, layer_bytes=hl.layer_bytes, flag_offset=hl.flag_offset,
                    steps=hl.steps)

    def set_peer(self, side, peer_workspace_ptr, layout):
        """peer_workspace_ptr: device address of the neighbour's workspace as mapped in this process (0 detaches);
        layout: the neighbour's halo_layout() of its facing side."""
        if not peer_workspace_ptr:
            _check(lib.islbm_slab_set_peer(self.h, int(side), None, None))
            return
        hl = _HaloLayout(int(layout["is_wall"]), int(layout["cur"]), (C.c_size_t * 2)(*layout["ghost_offset"]),
                         layout["plane_pitch_bytes"], layout["layer_bytes"], layout["flag_offset"], int(layout["steps"]))
        _check(lib.islbm_slab_set_peer(self.h, int(side), C.c_void_p(int(peer_workspace_ptr)), C.byref(hl)))

    def diag_sums(self):
        s = (C.c_double * 8)()
        _check(lib.islbm_diag_sums(self.h, s))
        return list(s)

    def diag_from_sums(self, sums):
        s = (C.c_double * 8)(*[float(v) for v in sums])
        out = (C.c_double * 6)()
        _check(lib.islbm_diag_from_sums(self.h, s, out))
        return dict(zip(("Nu_hot", "Nu_cold", "Re", "u2", "Nu_vol", "Nu_middle"), list(out)))

    def residual_sums(self):
        s = (C.c_double * 4)()
        first = C.c_int(0)
        _check(lib.islbm_residual_sums(self.h, s, C.byref(first)))
        return list(s), bool(first.value)

    def nusselt_middle(self):
        out = C.c_double(0.0)
        _check(lib.islbm_nusselt_middle(self.h, C.byref(out)))
        return out.value

    def steady_residual(self):
        out = (C.c_double * 2)()
        _check(lib.islbm_steady_residual(self.h, out))
        return out[0], out[1]
