"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol
include/islbm.h declares, and its host logic (argument validation, workspace
sizing) behaves as the header says.  No compute call is made (no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import __graft_entry__ as graft
from paper_2509_01099_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    graft.build()
    from paper_2509_01099_b200 import islbm
    return islbm


def declared_functions():
    src = open(os.path.join(ROOT, "include", "islbm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(islbm_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(binding):
    names = declared_functions()
    assert len(names) >= 15
    for name in names:
        assert hasattr(binding.lib, name), name
    assert set(names) == set(binding.EXPORTS)


def test_header_is_plain_c99():
    """include/islbm.h is a C header: it must parse as C99 on its own (no C++ or torch types in the boundary)."""
    import subprocess
    hdr = os.path.join(ROOT, "include", "islbm.h")
    r = subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-fsyntax-only", "-x", "c", hdr],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_version_and_cubin_arch(binding):
    assert b"sm_100a" in binding.lib.islbm_version()
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_library_holds_tma_and_mbarrier_instructions(binding):
    """The step kernels are TMA-staged: the sm_100a SASS must contain bulk-tensor loads and mbarrier waits."""
    import subprocess
    sass = subprocess.run(["cuobjdump", "-sass", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "UTMALDG" in sass and "SYNCS" in sass
    assert "USETMAXREG" in sass      # the fp64 3-D kernel's producer warpgroup donates its registers (setmaxnreg)
    assert "FFMA2" in sass           # packed fp32 interpolation of the fp32-storage kernels (fma.rn.f32x2)
    assert "STAS.64" in sass and "UCGABAR_ARV" in sass   # the cluster kernel: st.async into a neighbour CTA's shared memory, barrier.cluster
    for kern in ("k_step_zmarch", "k_step_ymarch", "k_step_shift", "k_step_generic", "k_nusselt_partial", "k_multistep_cluster2"):
        assert kern in sass, kern


def test_workspace_bytes_scales_with_mesh(binding):
    w = inputs.workload("c1_64sq")
    b64 = binding.workspace_bytes(w.coords, w.delta, binding.F64)
    b32 = binding.workspace_bytes(w.coords, w.delta, binding.F32_STORAGE)
    pops = 2 * 14 * 64 * 64
    assert b64 >= pops * 8 and b32 >= pops * 4 and b32 < b64
    w3 = inputs.custom_workload("t", 3, 16)
    assert binding.workspace_bytes(w3.coords, w3.delta) >= 2 * 26 * 16**3 * 8


def _mesh(binding, coords, delta):
    return binding._mesh_struct(coords, delta)


def test_create_validates_arguments_before_touching_the_device(binding):
    lib = binding.lib
    x, d = inputs.tanh_mesh(16, 1.2)
    h = C.c_void_p()
    fake_ws = C.c_void_p(256)      # never dereferenced: validation fails first
    big = C.c_size_t(1 << 40)

    def create(coords, delta, lattice=0, Ra=1e5, Pr=0.71, Ma=0.17, prec=0, ws=fake_ws, nbytes=big):
        m, keep = _mesh(binding, coords, delta)
        return lib.islbm_create(C.byref(h), C.byref(m), lattice, Ra, Pr, Ma, prec, ws, nbytes, None)

    assert create([x, x], d, lattice=1) == -1                        # lattice/dim mismatch
    assert create([x, x, x], d, lattice=0) == -1
    assert create([x[:2], x], d) == -1                               # n < 3
    assert create([x, x], d, prec=7) == -1
    assert create([x, x[::-1].copy()], d) == -2                      # not increasing
    assert create([x, x], 2 * d) == -2                               # spacing < delta
    assert b"delta" in lib.islbm_last_error()
    assert create([x, x], d, Ra=-1.0) == -3
    assert create([x, x], d, Ra=1e-3) == -3                          # a_T out of range (huge diffusivity)
    assert create([x, x], d, ws=None) == -4
    assert create([x, x], d, ws=C.c_void_p(8)) == -4                 # misaligned
    assert create([x, x], d, nbytes=C.c_size_t(1024)) == -4          # too small
    assert b"workspace too small" in lib.islbm_last_error()
    assert not h.value


def test_null_handles_are_rejected(binding):
    lib = binding.lib
    assert lib.islbm_step(None, 1) == -1
    assert lib.islbm_init(None, 0, 0.0) == -1
    out = (C.c_double * 5)()
    assert lib.islbm_nusselt(None, out) == -1
    assert lib.islbm_launch_count(None) == 0


def test_binding_fails_loudly_without_the_library(tmp_path):
    import subprocess
    import sys
    code = ("import importlib.util, sys; sys.path.insert(0, %r);"
            "import paper_2509_01099_b200.islbm as m; m.LIB_PATH = '/nonexistent/libislbm.so';"
            "m._load()" % ROOT)
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True)
    assert r.returncode != 0 and "no CPU fallback" in r.stderr


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2509_01099_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                for needle in ("import oracle", "from oracle", "libislbm_oracle", "islbm_oracle.h", "oracle_step",
                               "oracle.oracle", "Oracle("):
                    assert needle not in txt, (fn, needle)
    # and the oracle never imports the CUDA path
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            code = "\n".join(l for l in txt.splitlines() if l.lstrip().startswith(("import ", "from ", "#include")))
            assert "paper_2509" not in code and "libislbm.so" not in txt and "csrc" not in code


def test_workload_recipes():
    for name in inputs.workload_names():
        w = inputs.workload(name)
        x = w.coords[0]
        assert x[0] == pytest.approx(0.0, abs=1e-15) and x[-1] == pytest.approx(1.0) and np.all(np.diff(x) >= w.delta * (1 - 1e-12))
        u = inputs.workload(name + "_uniform")
        assert np.allclose(np.diff(u.coords[0]), u.delta)
    f, g = inputs.random_state((1, 8, 8), 9, 5, seed=1)
    f2, _ = inputs.random_state((1, 8, 8), 9, 5, seed=1)
    assert np.array_equal(f, f2) and f.min() > 0
