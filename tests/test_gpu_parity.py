"""Parity of the CUDA path (through the C-ABI binding) with the CPU oracle.

Tolerances (BASELINE.json north_star): fp64 populations after 1 step: max abs
difference per population plane / max abs oracle value of that plane <= 1e-12;
u, v, w (normalised by max |u|) and T (normalised by Delta_T = 1) after 1000
steps <= 1e-9; fp32-storage path: u and T after 1000 steps <= 1e-5.
"""
import math
import os
import zlib

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.oracle import Oracle  # noqa: E402
from paper_2509_01099_b200 import inputs  # noqa: E402

NTHREADS = max(1, min(32, len(os.sched_getaffinity(0))))
SQ3 = math.sqrt(3.0)


@pytest.fixture(scope="module")
def islbm():
    import __graft_entry__ as graft
    graft.build()
    from paper_2509_01099_b200 import islbm as mod
    assert torch.cuda.is_available()
    return mod


def pair(islbm, coords, delta, Ra, Pr=0.71, Ma=0.1 * SQ3, precision=0, kernel=0, threads=NTHREADS):
    sim = islbm.Islbm(coords, delta, Ra, Pr, Ma, precision=precision)
    if kernel:
        sim.set_kernel(kernel)
    orc = Oracle(coords, delta, Ra, Pr, Ma, threads=threads)
    return sim, orc


def plane_err(a, b):
    """max over planes of max|a-b| / max|b| (reading A17)."""
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    return float((np.abs(a - b).max(1) / np.abs(b).max(1)).max())


def elem_err(a, b, floor=0.1):
    """max ELEMENT-WISE relative error |a-b| / max(|b|, floor * max|b| over the plane) — for the flow populations.
    Near equilibrium f_q ~ w_q > 0 everywhere and this is the plain element-wise relative error north_star asks for;
    on the far-from-equilibrium random states (all f_q = 1/Q: over-relaxation with s = 1.7 sends the diagonal
    populations through zero, where a few-ulp absolute error has no relative meaning) elements below 10 % of the plane
    maximum are measured against that floor.  The
    plane-normalised metric above is kept for g, which crosses zero everywhere (reading A17)."""
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    den = np.maximum(np.abs(b), floor * np.abs(b).max(1, keepdims=True))
    return float((np.abs(a - b) / den).max())


def ragged_coords(dim, ns, stretches):
    out = []
    for n, s in zip(ns[:dim], stretches[:dim]):
        out.append(inputs.tanh_mesh(n, s)[0])
    delta = min(float(np.diff(c).min()) for c in out)
    return out, delta


def kernels_for(islbm, sim):
    """(kernel, tuning) variants valid for this mesh: the generic kernel, the TMA-staged kernel in the
    launch configurations bench.py can select (strip width, chunk length incl. ragged chunks, L2 policies,
    serpentine order, order of the first ring fill), and the pure-shift kernel on uniform meshes."""
    ks = [(islbm.KERNEL_GENERIC, {})]
    try:
        sim.set_kernel(islbm.KERNEL_TILED)
        ks.append((islbm.KERNEL_TILED, {}))
        ks.append((islbm.KERNEL_TILED, dict(chunk=5, load_policy=1, store_policy=2, l2promo=3, pdl=0, fill=2)))
        ks.append((islbm.KERNEL_TILED, dict(chunk=2, fill=1)))
        ks.append((islbm.KERNEL_TILED, dict(chunk=1)))                            # one emitted layer per CTA
        if sim.dim == 3:
            ks.append((islbm.KERNEL_TILED, dict(shape3d=3, chunk=3)))
            ks.append((islbm.KERNEL_TILED, dict(shape3d=4, fill=2)))
            ks.append((islbm.KERNEL_TILED, dict(shape3d=5)))
            ks.append((islbm.KERNEL_TILED, dict(walls=1, chunk=6)))      # separate boundary kernel over the shell (A/B variant)
            for tune in (dict(shape3d=1), dict(shape3d=2, chunk=7)):      # wide tiles: fp32 storage only (shared memory)
                try:
                    sim.set_tuning(**tune)
                    sim.set_kernel(islbm.KERNEL_TILED)
                    ks.append((islbm.KERNEL_TILED, tune))
                except islbm.IslbmError:
                    pass
            sim.set_tuning(**DEFAULT_TUNING)
        if sim.dim == 2:
            ks.append((islbm.KERNEL_TILED, dict(tx2d=128, chunk=7, serpentine=1)))
            ks.append((islbm.KERNEL_TILED, dict(tx2d=224, chunk=3)))
            ks.append((islbm.KERNEL_TILED, dict(tx2d=224, chunk=0, serpentine=1, load_policy=1)))
            ks.append((islbm.KERNEL_TILED, dict(ring2d=3, rows2d=3, rows2d1=5)))
            ks.append((islbm.KERNEL_TILED, dict(ring2d=4, chunk=9, serpentine=1, fill=2)))
            ks.append((islbm.KERNEL_TILED, dict(ring2d=3, chunk=2, pdl=0)))
            ks.append((islbm.KERNEL_TILED, dict(cluster=2)))      # tiny meshes: per-step launches instead of the cluster kernel
    except islbm.IslbmError:
        pass
    try:
        sim.set_kernel(islbm.KERNEL_UNIFORM_SHIFT)
        ks.append((islbm.KERNEL_UNIFORM_SHIFT, {}))
    except islbm.IslbmError:
        pass
    sim.set_kernel(islbm.KERNEL_AUTO)
    return ks


DEFAULT_TUNING = dict(chunk=0, l2promo=0, load_policy=0, store_policy=0, tx2d=0, serpentine=0, shape3d=0, pdl=1, fill=0,
                      ring2d=0, rows2d=0, rows2d1=0, walls=0, graph=0, cluster=0)


def select(sim, k, tune):
    sim.set_tuning(**{**DEFAULT_TUNING, **tune})
    sim.set_kernel(k)


# ---------------------------------------------------------------------------
# one step from a far-from-equilibrium random state: every population
# ---------------------------------------------------------------------------
CASES_1STEP = [
    ("2d_64sq_c1", 2, (64, 64, 1), (1.2, 1.2, 0)),
    ("2d_ragged_70x45", 2, (70, 45, 1), (1.6, 1.1, 0)),
    ("2d_ragged_131x67", 2, (131, 67, 1), (1.3, 1.9, 0)),
    ("2d_strips_300x40", 2, (300, 40, 1), (1.5, 1.3, 0)),
    ("2d_strips_516x37", 2, (516, 37, 1), (1.8, 1.2, 0)),
    ("2d_strips_258x9", 2, (258, 9, 1), (1.4, 0.8, 0)),
    ("2d_strips_130x3", 2, (130, 3, 1), (1.4, 0.5, 0)),
    ("2d_tiled_4x4", 2, (4, 4, 1), (0.5, 0.5, 0)),
    ("2d_min_3x3", 2, (3, 3, 1), (0.5, 0.5, 0)),
    ("2d_thin_3x40", 2, (3, 40, 1), (0.5, 1.5, 0)),
    ("3d_ragged_37x21x19", 3, (37, 21, 19), (1.5, 1.2, 1.7)),
    ("3d_ragged_66x10x35", 3, (66, 10, 35), (1.1, 1.4, 1.3)),
    ("3d_tiled_64x24x40", 3, (64, 24, 40), (1.3, 1.2, 1.5)),
    ("3d_tiled_34x18x7", 3, (34, 18, 7), (1.2, 1.1, 0.9)),
    ("3d_tiled_96x50x33", 3, (96, 50, 33), (1.6, 1.4, 1.2)),
    ("3d_tiled_4x4x3", 3, (4, 4, 3), (0.5, 0.5, 0.5)),
    ("3d_clamp_33x17x9", 3, (33, 17, 9), (1.2, 1.3, 1.1)),
    ("3d_clamp_65x9x5", 3, (65, 9, 5), (1.4, 0.9, 0.7)),
    ("3d_min_3x3x3", 3, (3, 3, 3), (0.5, 0.5, 0.5)),
    ("3d_thin_5x3x33", 3, (5, 3, 33), (0.7, 0.5, 1.5)),
]


@pytest.mark.parametrize("name,dim,ns,st", CASES_1STEP, ids=[c[0] for c in CASES_1STEP])
def test_one_step_all_populations(islbm, name, dim, ns, st):
    coords, delta = ragged_coords(dim, ns, st)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    Ra = 0.71 * (0.1 * H_lu / 0.03) ** 2            # nu = 0.03 l.u. whatever the mesh
    sim, orc = pair(islbm, coords, delta, Ra=Ra)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=zlib.crc32(name.encode()) % 1000, amp=0.05)
    orc.set_populations(f0, g0)
    orc.step(1)
    fo, go = orc.get_populations()
    orc.step(2)
    fo3, go3 = orc.get_populations()
    variants = kernels_for(islbm, sim)
    assert any(k == islbm.KERNEL_TILED for k, _ in variants), "the TMA kernel must take every mesh with n >= 3"
    for k, tune in variants:
        select(sim, k, tune)
        sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
        f_back, g_back = sim.get_populations()            # before any step: the input itself
        assert np.array_equal(f_back.cpu().numpy(), f0) and np.array_equal(g_back.cpu().numpy(), g0)
        sim.step(1)
        f1, g1 = sim.get_populations()
        ef, eg = elem_err(f1.cpu().numpy(), fo), plane_err(g1.cpu().numpy(), go)      # f: every element (north_star)
        assert ef <= 1e-12 and eg <= 1e-12, (name, sim.kernel_name, tune, ef, eg)
        # second and third step (ping-pong both ways)
        sim.step(2)
        f3, g3 = sim.get_populations()
        ef, eg = elem_err(f3.cpu().numpy(), fo3), plane_err(g3.cpu().numpy(), go3)
        assert ef <= 3e-12 and eg <= 3e-12, (name, sim.kernel_name, tune, ef, eg)


@pytest.mark.parametrize("dim,ns,st", [(2, (132, 45, 1), (1.5, 1.2, 0)), (2, (520, 21, 1), (1.7, 1.1, 0)),
                                       (2, (131, 67, 1), (1.3, 1.9, 0)), (3, (36, 18, 9), (1.3, 1.2, 1.1)),
                                       (3, (68, 27, 20), (1.5, 1.1, 1.4)), (3, (37, 21, 19), (1.5, 1.2, 1.7)),
                                       (3, (33, 17, 9), (1.2, 1.3, 1.1))])
def test_fp32_storage_every_kernel_three_steps(islbm, dim, ns, st):
    """fp32 storage of f_q - w_q and g_q (flow collision in fp64 in 2-D, in fp32 in 3-D; the TMA kernels interpolate
    in fp32): every kernel variant against the fp64 oracle.
    Tolerance: 3 steps x one fp32 rounding (2^-24 relative to |f_q - w_q| <= 0.4) per stored value, amplified
    by the 9-point interpolation weights (|w| sums <= ~2): 2e-6 of the plane maximum (measured in 3-D: 6.3e-7 to
    6.7e-7 for the TMA kernels, 7e-8 for the generic kernel, which interpolates in fp64)."""
    coords, delta = ragged_coords(dim, ns, st)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    Ra = 0.71 * (0.1 * H_lu / 0.03) ** 2
    sim, orc = pair(islbm, coords, delta, Ra=Ra, precision=1)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=11 + dim, amp=0.05)
    orc.set_populations(f0, g0)
    orc.step(3)
    fo, go = orc.get_populations()
    variants = kernels_for(islbm, sim)
    assert any(k == islbm.KERNEL_TILED for k, _ in variants)
    for k, tune in variants:
        select(sim, k, tune)
        sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
        sim.step(3)
        f3, g3 = sim.get_populations()
        ef, eg = plane_err(f3.cpu().numpy(), fo), plane_err(g3.cpu().numpy(), go)
        assert ef <= 2e-6 and eg <= 2e-6, (sim.kernel_name, tune, ef, eg)


@pytest.mark.parametrize("dim,ns,prec", [(2, (70, 45, 1), 0), (3, (37, 21, 19), 0), (3, (33, 17, 9), 1), (2, (3, 3, 1), 0)])
def test_set_populations_host_equals_device_path(islbm, dim, ns, prec):
    """islbm_set_populations_host (slab-staged H2D inside the library; numpy = pageable, torch pinned) gives the
    same state, bit for bit, as islbm_set_populations with device arrays; ragged slabs included."""
    coords, delta = ragged_coords(dim, ns, (1.3, 1.2, 1.1))
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    mk = lambda: islbm.Islbm(coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2, 0.71, 0.1 * SQ3, precision=prec)
    a, b = mk(), mk()
    f0, g0 = inputs.random_state(a.shape, a.qf, a.qg, seed=5, amp=0.05)
    a.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
    fp = torch.from_numpy(f0).pin_memory()
    for fh, gh in ((f0, g0), (fp, torch.from_numpy(g0).pin_memory())):
        b.steady_residual() if b.launch_count else None       # dirty the staging (snapshot) area between uploads
        b.set_populations_host(fh, gh)
        fa, ga = a.get_populations()
        fb, gb = b.get_populations()
        assert torch.equal(fa, fb) and torch.equal(ga, gb)
        b.step(3)
    a.step(3)
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert torch.equal(fa, fb) and torch.equal(ga, gb)
    assert b.steady_residual() == (1.0, 1.0)                 # the upload invalidated the Eq. 30 snapshot


@pytest.mark.parametrize("name,dim,ns,st", CASES_1STEP, ids=[c[0] for c in CASES_1STEP])
def test_upwind_stencil_parity(islbm, name, dim, ns, st):
    """A2 alternative ({j-2,j-1,j} for c = +1, {j,j+1,j+2} for c = -1): the TMA kernels of that
    stencil (2-row halo, split z-stencil groups) and the generic kernel against the oracle's table-driven stream, on
    the same 20 meshes and tuning variants as the central stencil, 1e-12 after one step and 3e-12 after three."""
    coords, delta = ragged_coords(dim, ns, st)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    sim, orc = pair(islbm, coords, delta, Ra=0.71 * (0.1 * H_lu / 0.03) ** 2)
    sim.set_stencil(1)
    orc.set_stencil(1)
    assert sim.kernel_name in ("tiled_ymarch_tma_upwind", "tiled_zmarch_tma_upwind")
    with pytest.raises(islbm.IslbmError):
        sim.set_kernel(islbm.KERNEL_UNIFORM_SHIFT)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=zlib.crc32(name.encode()) % 1000 + 1, amp=0.05)
    orc.set_populations(f0, g0)
    orc.step(1)
    fo, go = orc.get_populations()
    orc.step(2)
    fo3, go3 = orc.get_populations()
    variants = kernels_for(islbm, sim)
    assert sum(k == islbm.KERNEL_TILED for k, _ in variants) >= 3
    for k, tune in variants:
        select(sim, k, tune)
        assert sim.kernel_name.endswith("upwind") == (k != islbm.KERNEL_GENERIC)
        sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
        sim.step(1)
        f1, g1 = sim.get_populations()
        ef, eg = elem_err(f1.cpu().numpy(), fo), plane_err(g1.cpu().numpy(), go)
        assert ef <= 1e-12 and eg <= 1e-12, (name, sim.kernel_name, tune, ef, eg)
        sim.step(2)
        f3, g3 = sim.get_populations()
        ef, eg = elem_err(f3.cpu().numpy(), fo3), plane_err(g3.cpu().numpy(), go3)
        assert ef <= 3e-12 and eg <= 3e-12, (name, sim.kernel_name, tune, ef, eg)
    with pytest.raises(islbm.IslbmError):
        sim.set_stencil(0)                      # the state exists: too late


@pytest.mark.parametrize("dim,ns,st", [(2, (132, 45, 1), (1.5, 1.2, 0)), (2, (131, 67, 1), (1.3, 1.9, 0)),
                                       (3, (36, 18, 9), (1.3, 1.2, 1.1)), (3, (68, 27, 20), (1.5, 1.1, 1.4)),
                                       (3, (37, 21, 19), (1.5, 1.2, 1.7))])
def test_upwind_stencil_fp32_storage(islbm, dim, ns, st):
    """Upwind stencil with fp32 storage (packed f32x2 interpolation, stencil sets in shared memory): 2e-6 after 3 steps."""
    coords, delta = ragged_coords(dim, ns, st)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    sim, orc = pair(islbm, coords, delta, Ra=0.71 * (0.1 * H_lu / 0.03) ** 2, precision=1)
    sim.set_stencil(1)
    orc.set_stencil(1)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=13 + dim, amp=0.05)
    orc.set_populations(f0, g0)
    orc.step(3)
    fo, go = orc.get_populations()
    for k, tune in kernels_for(islbm, sim):
        select(sim, k, tune)
        sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
        sim.step(3)
        f3, g3 = sim.get_populations()
        ef, eg = plane_err(f3.cpu().numpy(), fo), plane_err(g3.cpu().numpy(), go)
        assert ef <= 2e-6 and eg <= 2e-6, (sim.kernel_name, tune, ef, eg)


def test_upwind_stencil_1000_steps_and_slab_refusal(islbm):
    """Upwind stencil on config 1 from the seeded start: fields and diagnostics 1e-9 after 1000 steps; a slab handle
    (one ghost layer) refuses the stencil."""
    w = inputs.workload("c1_64sq")
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.set_stencil(1)
    orc.set_stencil(1)
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    sim.step(1000)
    orc.step(1000)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    _diag_close(sim, orc)
    from paper_2509_01099_b200 import slab
    cav = slab.SlabCavity(w.coords, w.delta, w.Ra, w.Pr, w.Ma, 0, 2, exchange=lambda: None)
    with pytest.raises(islbm.IslbmError):
        cav.sim.set_stencil(1)


def test_uniform_mesh_one_step(islbm):
    for dim, n in ((2, 32), (3, 16)):
        w = inputs.custom_workload("u", dim, n, mesh="uniform", Ra=1e4)
        sim, orc = pair(islbm, w.coords, w.delta, w.Ra)
        f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=dim, amp=0.05)
        orc.set_populations(f0, g0)
        orc.step(1)
        fo, go = orc.get_populations()
        variants = kernels_for(islbm, sim)
        assert (islbm.KERNEL_UNIFORM_SHIFT, {}) in variants
        for k, tune in variants:
            select(sim, k, tune)
            sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
            sim.step(1)
            f1, g1 = sim.get_populations()
            assert elem_err(f1.cpu().numpy(), fo) <= 1e-12 and plane_err(g1.cpu().numpy(), go) <= 1e-12, (dim, k, tune)
        # mass is conserved to round-off on the uniform mesh (pin P4 on the GPU path)
        sim.step(200)
        rho = sim.fields(("rho",))["rho"]
        assert abs(rho.sum().item() - f0.sum()) / f0.sum() < 1e-13


# ---------------------------------------------------------------------------
# BASELINE.json config 1: 1000 steps, populations and fields
# ---------------------------------------------------------------------------
def field_err(sim, orc, floor=1e-4):
    """u, v, w normalised by max|u| (reading A17), T by Delta_T = 1.  `floor` (lattice units) bounds the velocity
    normaliser from below: the runs that start from rest + 1e-3 noise have |u| ~ 1e-7..1e-4 l.u. for the first
    hundreds of steps, and the few-ulp ABSOLUTE error of sum(e f)/rho (~1e-16) would read as 1e-9 relative to
    that; 1e-4 l.u. = 1e-3 U.  Tests of a developed flow (|u| ~ 0.1 U) pass floor=0."""
    fs, fo = sim.fields(), orc.fields()
    umax = max(max(np.abs(fo[k]).max() for k in ("u", "v", "w")), floor)
    assert umax > 0.0
    out = {k: float(np.abs(fs[k].cpu().numpy() - fo[k]).max() / umax) for k in fs if k in ("u", "v", "w")}
    out["T"] = float(np.abs(fs["T"].cpu().numpy() - fo["T"]).max())      # Delta_T = 1
    out["rho"] = float(np.abs(fs["rho"].cpu().numpy() - fo["rho"]).max())
    return out


def test_config1_init_and_1000_steps(islbm):
    w = inputs.workload("c1_64sq")
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    ps, po = sim.params(), orc.params()
    for k in po:
        assert ps[k] == pytest.approx(po[k], rel=1e-14), k
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    f, g = sim.get_populations()
    fo, go = orc.get_populations()
    assert np.abs(f.cpu().numpy() - fo).max() < 1e-16 and np.abs(g.cpu().numpy() - go).max() < 1e-18
    sim.step(1)
    orc.step(1)
    f, g = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f.cpu().numpy(), fo) <= 1e-12 and plane_err(g.cpu().numpy(), go) <= 1e-12
    sim.step(999)
    orc.step(999)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    f, g = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f.cpu().numpy(), fo) <= 1e-9 and plane_err(g.cpu().numpy(), go) <= 1e-9
    ns, no = sim.nusselt(), orc.nusselt()
    for k in no:
        assert ns[k] == pytest.approx(no[k], rel=1e-9, abs=1e-12), k
    assert sim.nusselt_middle() == pytest.approx(orc.nusselt_middle(), rel=1e-9, abs=1e-12)   # Eq. 33, even n


def test_config1_fp32_storage_1000_steps(islbm):
    w = inputs.workload("c1_64sq")
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=1)
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    sim.step(1000)
    orc.step(1000)
    err = field_err(sim, orc)
    assert err["u"] <= 1e-5 and err["v"] <= 1e-5 and err["T"] <= 1e-5, err


def test_3d_small_200_steps_fields_and_nusselt(islbm):
    w = inputs.custom_workload("c4_small", 3, 32, stretch=1.5, Ra=1e5)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.init(0, 1e-3)
    orc.init(0, 1e-3)
    sim.step(200)
    orc.step(200)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    ns, no = sim.nusselt(), orc.nusselt()
    for k in no:
        assert ns[k] == pytest.approx(no[k], rel=1e-9, abs=1e-12), k
    assert sim.nusselt_middle() == pytest.approx(orc.nusselt_middle(), rel=1e-9, abs=1e-12)
    # fp32 storage, 3-D
    sim32 = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=1)
    sim32.init(0, 1e-3)
    sim32.step(200)
    e32 = field_err(sim32, orc)
    assert e32["u"] <= 1e-5 and e32["v"] <= 1e-5 and e32["w"] <= 1e-5 and e32["T"] <= 1e-5, e32


# ---------------------------------------------------------------------------
# BASELINE.json configs 2-5 at full size, in the launch configuration bench.py times
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("name,steps", [("c2_512sq", 20), ("c3_1024sq", 5), ("c4_128cu", 3),
                                        ("c2_512sq_uniform", 5)])
def test_full_size_configs_few_steps(islbm, name, steps):
    w = inputs.workload(name)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    sim.step(1)
    orc.step(1)
    f, g = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f.cpu().numpy(), fo) <= 1e-12 and plane_err(g.cpu().numpy(), go) <= 1e-12
    del f, g
    sim.step(steps - 1)
    orc.step(steps - 1)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-10, err
    ns, no = sim.nusselt(), orc.nusselt()
    assert ns["Nu_hot"] == pytest.approx(no["Nu_hot"], rel=1e-10)


@pytest.mark.parametrize("name,steps", [("c2_512sq", 1000)])
def test_full_size_configs_long_runs(islbm, name, steps):
    """north_star: 1e-9 on u, v and T after 1000 steps, at BASELINE.json's full size with the OpenMP oracle."""
    w = inputs.workload(name)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma, threads=len(os.sched_getaffinity(0)))
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    sim.step(steps)
    orc.step(steps)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    ns, no = sim.nusselt(), orc.nusselt()
    for k in no:
        assert ns[k] == pytest.approx(no[k], rel=1e-9, abs=1e-12), k
    # islbm_step(0) is a no-op
    f0, g0 = sim.get_populations()
    sim.step(0)
    f1, g1 = sim.get_populations()
    assert torch.equal(f0, f1) and torch.equal(g0, g1)


def _long_3d(islbm, name, steps):
    w = inputs.workload(name)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma, threads=len(os.sched_getaffinity(0)))
    sim32 = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=1)
    assert sim.kernel_name == "tiled_zmarch_tma" and sim32.kernel_name == "tiled_zmarch_tma"
    for s_ in (sim, sim32, orc):
        s_.init(w.seed, w.noise_amp)
        s_.step(steps)
    err = field_err(sim, orc)
    e32 = field_err(sim32, orc)
    ns, no = sim.nusselt(), orc.nusselt()
    print("LONG", name, steps, "steps: fp64", err, "fp32", e32, "Nu/Re", ns, no)
    assert max(err.values()) <= 1e-9, err
    assert max(e32[k] for k in ("u", "v", "w", "T")) <= 1e-5, e32
    for k in no:
        assert ns[k] == pytest.approx(no[k], rel=1e-9, abs=1e-12), k
    assert sim.nusselt_middle() == pytest.approx(orc.nusselt_middle(), rel=1e-9, abs=1e-12)


def test_config4_128cu_1000_steps_fp64_and_fp32(islbm):
    """BASELINE.json config 4 at full size and the full 1000 steps of north_star: fp64 within 1e-9 and fp32 storage
    within 1e-5 on u, v, w, T; every diagnostic within 1e-9 (about 3 min of OpenMP oracle on the GPU box)."""
    _long_3d(islbm, "c4_128cu", 1000)


def test_config5_256cu_100_steps_fp64_and_fp32(islbm):
    """BASELINE.json config 5 at full size, launch configuration of bench.py, the 100 steps SURVEY.md 8(d) prescribes
    for it (about 2 min of OpenMP oracle); the full 1000 steps are the opt-in test below (21 min of oracle: beyond
    the driver's pytest limit; its last result line is committed in profiles/r2_long_parity.md)."""
    _long_3d(islbm, "c5_256cu", 100)


@pytest.mark.skipif(os.environ.get("ISLBM_LONG") != "1", reason="~21 min of host oracle time; set ISLBM_LONG=1")
def test_config5_256cu_1000_steps_fp64_and_fp32_long(islbm):
    """north_star bar on config 5 at full size and the full 1000 steps.  Opt-in (the OpenMP oracle needs ~20 min for
    256^3 x 1000 on 16 host threads); result of the last run: profiles/r2_long_parity.md."""
    _long_3d(islbm, "c5_256cu", 1000)


def test_config3_1024sq_1000_steps_fp64_and_fp32(islbm):
    """BASELINE.json config 3 at full size, 1000 steps: fp64 within 1e-9 and fp32 storage within 1e-5 on u, v, T."""
    w = inputs.workload("c3_1024sq")
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma, threads=len(os.sched_getaffinity(0)))
    sim32 = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=1)
    assert sim.kernel_name.startswith("tiled_ymarch_tma") and sim32.kernel_name.startswith("tiled_ymarch_tma")
    for s_ in (sim, sim32, orc):
        s_.init(w.seed, w.noise_amp)
        s_.step(1000)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    e32 = field_err(sim32, orc)
    assert e32["u"] <= 1e-5 and e32["v"] <= 1e-5 and e32["T"] <= 1e-5, e32


def test_config5_256cu_sampled_nodes(islbm):
    """256^3: the oracle computes sampled nodes one by one (oracle_step_node) from the
    seeded initial state; walls, edges, corners and tile seams are all in the sample."""
    w = inputs.workload("c5_256cu")
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    orc = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.init(w.seed, w.noise_amp)
    orc.init(w.seed, w.noise_amp)
    sim.step(1)
    f, g = sim.get_populations()
    n = 256
    special = [0, 1, 2, 7, 8, 15, 16, 31, 32, 33, 63, 64, 127, 128, 191, 192, 253, 254, 255]
    rng = np.random.default_rng(5)
    pts = [(a, b, c) for a in (0, 1, 128, 254, 255) for b in (0, 31, 32, 255) for c in (0, 8, 255)]
    pts += [tuple(rng.choice(special, 3)) for _ in range(300)]
    pts += [tuple(rng.integers(0, n, 3)) for _ in range(700)]
    idx = torch.tensor(pts, device="cuda")
    fs = f[:, idx[:, 2], idx[:, 1], idx[:, 0]].cpu().numpy()
    gs = g[:, idx[:, 2], idx[:, 1], idx[:, 0]].cpu().numpy()
    fo = np.empty_like(fs)
    go = np.empty_like(gs)
    for k, (ix, iy, iz) in enumerate(pts):
        fo[:, k], go[:, k] = orc.step_node(int(ix), int(iy), int(iz))
    assert elem_err(fs, fo) <= 1e-12 and plane_err(gs, go) <= 1e-12
    # properties that hold at any size: rho ~ 1, T within the noise amplitude, everything finite
    fl = sim.fields(("rho", "T"))
    assert torch.isfinite(fl["rho"]).all() and (fl["rho"] - 1).abs().max().item() < 1e-6
    assert fl["T"].abs().max().item() < 0.2     # one anti-bounce-back kick of omega*T_w at the x-walls


# ---------------------------------------------------------------------------
# Eq. 28 with q != 1 (paper-mode erf mesh, hand-made mesh) and developed flows against the oracle
# ---------------------------------------------------------------------------
def _diag_close(sim, orc, rel=1e-9):
    ns, no = sim.nusselt(), orc.nusselt()
    for k in no:                                           # Nu_hot, Nu_cold, Re, u2, Nu_vol
        assert ns[k] == pytest.approx(no[k], rel=rel, abs=1e-12), (k, ns[k], no[k])
    nm_s, nm_o = sim.nusselt_middle(), orc.nusselt_middle()
    assert nm_s == pytest.approx(nm_o, rel=rel, abs=1e-12), ("Nu_middle", nm_s, nm_o)
    return ns


@pytest.mark.parametrize("kind,dim,n", [("erf", 2, 129), ("wallgap", 2, 40), ("erf", 3, 49), ("wallgap", 3, 22)])
def test_q_not_one_meshes_populations_fields_and_all_six_diagnostics(islbm, kind, dim, n):
    """Meshes on which q of Eq. 28 is NOT 1: the paper's erf mesh with delta = y_1 (paper mode,
    Ma = 0.1, T0 = T_cold) and the hand-made mesh with q = 2.5 at the hot and 1.75 at the cold wall.  Populations
    1e-12 after one step from a far-from-equilibrium state; fields and all six diagnostics (Nu_hot, Nu_cold, <Re>,
    <u*^2>, <Nu>, Nu_middle) 1e-9 after 300 steps from the seeded start.  The oracle side of Eq. 28 at q != 1 is pinned by
    test_P6b / test_P6c (tests/test_oracle_pins.py); a swapped or inverted q on the CUDA side fails here."""
    if kind == "erf":
        x, delta = inputs.erf_mesh(n, 1.5)
        Ma, T0 = 0.1, -0.5
    else:
        x, delta = inputs.wallgap_mesh(n)
        Ma, T0 = 0.1 * SQ3, 0.0
    coords = [x.copy() for _ in range(dim)]
    q_lo, q_hi = (x[1] - x[0]) / delta, (x[-1] - x[-2]) / delta
    assert q_lo > 1.005 and q_hi > 1.005
    H_lu = (x[-1] - x[0] + delta) / delta
    # erf: the paper's Ra for these grids; hand-made mesh (H_lu = 52 / 29 l.u.): Ra such that nu = 0.03 l.u.
    Ra = (1e6 if dim == 2 else 1e5) if kind == "erf" else 0.71 * (0.1 * H_lu / 0.03) ** 2
    sim, orc = pair(islbm, coords, delta, Ra, 0.71, Ma)
    sim.set_reference_temperature(T0)
    orc.set_reference_temperature(T0)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=17 + dim, amp=0.05)
    orc.set_populations(f0, g0)
    sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
    sim.step(1)
    orc.step(1)
    f1, g1 = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f1.cpu().numpy(), fo) <= 1e-12 and plane_err(g1.cpu().numpy(), go) <= 1e-12
    _diag_close(sim, orc)                                   # far from equilibrium: every term of every sum is O(1)
    sim.init(0, 1e-3)
    orc.init(0, 1e-3)
    sim.step(300)
    orc.step(300)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    ns = _diag_close(sim, orc)
    assert ns["Nu_hot"] > 1.5                               # the wall layer is developing: a curved profile at the wall


@pytest.mark.parametrize("dim,n,Ra", [(2, 64, 1e5), (3, 32, 1e5)])
def test_developed_flow_parity_1000_steps(islbm, dim, n, Ra):
    """The nonlinear regime: config 1 (64^2, Ra = 1e5) and a 32^3 cavity are run on the GPU to the steady-state
    criterion of Eq. 30, that state (f_t, g_t) is injected into the oracle, and both sides then
    take 1000 steps: populations, fields (velocity normaliser NOT floored: |u| ~ 0.2 U) and all six diagnostics within
    1e-9.  (The seeded-start tests above stay in the conduction transient, |u| <= 1e-4 l.u.)"""
    w = inputs.workload("c1_64sq") if dim == 2 else inputs.custom_workload("dev3", 3, n, stretch=1.5, Ra=Ra)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.init(w.seed, w.noise_amp)
    sim.steady_residual()
    for _ in range(400):
        sim.step(2000)
        ru, rT = sim.steady_residual()
        if ru < 1e-9 and rT < 1e-9:
            break
    assert ru < 1e-6 and rT < 1e-6, (ru, rT)               # developed (steady to 1e-9 in practice)
    f, g = sim.get_populations()
    orc.set_populations(f.cpu().numpy(), g.cpu().numpy())
    sim32 = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=1)      # fp32 storage from the same developed state
    sim32.set_populations(f, g)
    nu0 = sim.nusselt()
    assert nu0["Nu_hot"] > 2.0 and nu0["Re"] > 5.0          # a convecting cavity, not the conduction transient
    sim.step(1)
    orc.step(1)
    f1, g1 = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f1.cpu().numpy(), fo) <= 1e-12 and plane_err(g1.cpu().numpy(), go) <= 1e-12
    sim.step(999)
    orc.step(999)
    err = field_err(sim, orc, floor=0.0)
    assert max(err.values()) <= 1e-9, err
    f1, g1 = sim.get_populations()
    fo, go = orc.get_populations()
    assert elem_err(f1.cpu().numpy(), fo) <= 1e-9 and plane_err(g1.cpu().numpy(), go) <= 1e-9
    _diag_close(sim, orc)
    # fp32 storage in the nonlinear regime: north_star's 1e-5 on u, v, w and T after the same 1000 steps, and the
    # diagnostics of a convecting cavity to 1e-5 relative
    sim32.step(1000)
    e32 = field_err(sim32, orc, floor=0.0)
    assert max(e32[k] for k in e32 if k != "rho") <= 1e-5, e32
    n32, no = sim32.nusselt(), orc.nusselt()
    for k in no:
        assert n32[k] == pytest.approx(no[k], rel=1e-5), (k, n32[k], no[k])


def test_paper_mode_convergence_order(islbm, golden):
    """three paper-mode grids with refinement ratio 2 (129, 257, 513 points of
    Eq. 26, a = 1.5, Ma = 0.1, Ra = 1e6, T0 = T_cold; the paper's triple is 257, 513, 1025), each run to Eq. 30
    (about 50 s on the B200).  65 points are not yet in the asymptotic range at Ra = 1e6: the triple 65 / 129 / 257
    gives p = 1.6-1.8 (measured, profiles/attempts.md).  Observed order p of Eq. 35 for the
    domain-integrated <Nu> and for Nu_hot in [2.2, 3.2] (the paper: "nearly third-order ... in domain-integrated
    quantities", p = 2.6 for <Nu>), and the Richardson value of Nu_hot (Eq. 36) within 0.1 % of the 8.8206 Table 2
    prints as its own grid-independent value."""
    vals = {}
    for npts in (129, 257, 513):
        w = inputs.custom_workload("conv", 2, npts, mesh="erf", stretch=1.5, Ra=1e6, Ma=0.1)
        sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
        sim.set_reference_temperature(-0.5)
        sim.init(0, 0.0)
        sim.steady_residual()
        for _ in range(1500):
            sim.step(2000)
            ru, rT = sim.steady_residual()
            if ru < 1e-9 and rT < 1e-9:
                break
        assert ru < 1e-9 and rT < 1e-9, (npts, ru, rT)
        nu = sim.nusselt()
        vals[npts] = (nu["Nu_vol"], nu["Nu_hot"], sim.nusselt_middle())
        sim.close()
    print("CONVERGENCE", vals)
    order = lambda k: math.log(abs((vals[129][k] - vals[257][k]) / (vals[257][k] - vals[513][k]))) / math.log(2.0)
    p_vol, p_hot, p_mid = order(0), order(1), order(2)
    assert 2.2 <= p_vol <= 3.2 and 2.2 <= p_hot <= 3.2 and 2.2 <= p_mid <= 3.2, (p_vol, p_hot, p_mid)
    rp = 2.0 ** p_hot
    nu_hot_inf = (rp * vals[513][1] - vals[257][1]) / (rp - 1.0)                 # Eq. 36
    assert nu_hot_inf == pytest.approx(golden["table2"]["Ra1e6"]["inf"][1], rel=1e-3)


# ---------------------------------------------------------------------------
# method-level properties on the GPU path
# ---------------------------------------------------------------------------
def test_conduction_fixed_point_on_gpu(islbm):
    """Pin P5 on the CUDA path: buoyancy off, linear-T state, stretched mesh."""
    w = inputs.custom_workload("p5", 2, 48, stretch=1.6, Ra=1e5)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra)
    sim.set_buoyancy_scale(0.0)
    p = orc.params()
    qk = 3.0 - SQ3
    x = w.coords[0]
    G = -1.0 / p["H_lu"]
    T = 0.5 + G * (x - (x[0] - w.delta / 2)) / w.delta
    wr = np.full(5, p["omega_bc"] / 2)
    wr[0] = 1 - wr[1:].sum()
    ex = np.array([0, 1, 0, -1, 0])
    f0 = np.empty((9,) + orc.shape)
    f0[:] = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None, None]
    g0 = np.empty((5,) + orc.shape)
    for i in range(5):
        g0[i] = (wr[i] * T - wr[i] / qk * ex[i] * G)[None, None, :]
    sim.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
    sim.step(1000)
    f1, g1 = sim.get_populations()
    assert np.abs(f1.cpu().numpy() - f0).max() < 1e-13 and np.abs(g1.cpu().numpy() - g0).max() < 1e-13
    nu = sim.nusselt()
    assert nu["Nu_hot"] == pytest.approx(1.0, abs=1e-10) and nu["Nu_cold"] == pytest.approx(1.0, abs=1e-10)


def test_more_than_2_pow_31_elements_per_buffer(islbm):
    """Maximum sizes: 640 x 640 x 224 nodes = 2.39e9 stored values per buffer (> 2^31, 19 GB), so every index must be
    64-bit.  The oracle would need 76 GB of host memory at this size; the check is the TMA kernel (tensor-map
    coordinates) against the generic kernel (explicit 64-bit indices), which share no indexing code and are each
    checked against the oracle at small sizes, plus size-independent properties of the state."""
    free, _ = torch.cuda.mem_get_info()
    if free < 110e9:
        pytest.skip("needs 110 GB of free device memory")
    ns = (640, 640, 224)
    coords = [inputs.tanh_mesh(n, 1.6)[0] for n in ns]
    delta = min(float(np.diff(c).min()) for c in coords)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    sim = islbm.Islbm(coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2, 0.71, 0.1 * SQ3)
    assert sim.nodes * 26 > 2 ** 31 and sim.kernel_name == "tiled_zmarch_tma"
    sim.init(7, 1e-3)
    sim.step(2)
    f_t, g_t = sim.get_populations()
    sim.init(7, 1e-3)
    sim.set_kernel(islbm.KERNEL_GENERIC)
    sim.step(2)
    f_g, g_g = sim.get_populations()
    for a, b in ((f_t, f_g), (g_t, g_g)):
        for q in range(a.shape[0]):
            assert (a[q] - b[q]).abs().max().item() <= 1e-13 * max(b[q].abs().max().item(), 1e-30), q
    del f_g, g_g
    assert torch.isfinite(f_t).all() and torch.isfinite(g_t).all()
    assert abs(f_t.sum(0).mean().item() - 1.0) < 1e-9                     # rho ~ 1 everywhere
    assert (f_t[:, -1, -1, -1] > 0).all() and g_t[:, -1, -1, -1].abs().max().item() < 1.0   # the very last node was written


@pytest.mark.parametrize("dim,ns,prec", [(2, (70, 45), 0), (2, (131, 67), 1), (2, (3, 3), 0), (3, (37, 21, 19), 0),
                                         (3, (33, 17, 9), 1), (3, (64, 24, 40), 0), (3, (3, 3, 3), 1)])
def test_no_kernel_writes_outside_the_workspace(islbm, dim, ns, prec):
    """Canary bands of 1 MiB on both sides of the workspace stay intact through every kernel variant, the
    reductions, the residual and get/set (compute-sanitizer is not available on the GPU pool)."""
    coords, delta = ragged_coords(dim, ns + (1,), (1.3, 1.2, 1.1))
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    sim = islbm.Islbm(coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2, 0.71, 0.1 * SQ3, precision=prec, guard_bytes=1 << 20)
    sim.init(0, 1e-3)
    for k, tune in kernels_for(islbm, sim):
        select(sim, k, tune)
        sim.step(3)
        f, g = sim.get_populations()
        sim.set_populations(f, g)
        sim.step(2)
    sim.nusselt(), sim.nusselt_middle(), sim.steady_residual(), sim.steady_residual(), sim.fields()
    torch.cuda.synchronize()
    assert sim.guards_intact()
    # the upwind-stencil kernels (2-row halo boxes, half-group boxes, per-lane window offsets) on the same mesh
    up = islbm.Islbm(coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2, 0.71, 0.1 * SQ3, precision=prec, guard_bytes=1 << 20)
    up.set_stencil(1)
    up.init(0, 1e-3)
    for k, tune in kernels_for(islbm, up):
        select(up, k, tune)
        up.step(3)
        f, g = up.get_populations()
        up.set_populations(f, g)
        up.step(2)
    up.nusselt(), up.nusselt_static(), up.fields()
    torch.cuda.synchronize()
    assert up.guards_intact()


@pytest.mark.parametrize("dim,ns,prec", [(2, (64, 64), 0), (2, (70, 45), 1), (3, (37, 21, 19), 0)])
def test_graph_replay_equals_plain_launches_bitwise(islbm, dim, ns, prec):
    """islbm_step(n >= 32) on a small mesh replays a captured CUDA graph of 32 PDL-chained step kernels: identical
    bits to launching the kernels one by one (graph = 2), whatever mix of call sizes, and after re-planning."""
    coords, delta = ragged_coords(dim, ns + (1,), (1.3, 1.2, 1.1))
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    mk = lambda: islbm.Islbm(coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2, 0.71, 0.1 * SQ3, precision=prec)
    a, b = mk(), mk()
    a.set_tuning(cluster=2)                                    # (the 64^2 fp64 case would otherwise take the cluster kernel)
    b.set_tuning(graph=2, cluster=2)
    for s_ in (a, b):
        s_.init(1, 1e-3)
    for n in (100, 1, 33, 64, 7):
        l0 = a.launch_count
        a.step(n)
        b.step(n)
        assert a.launch_count - l0 == n                        # the count is of kernels, not of host launches
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert torch.equal(fa, fb) and torch.equal(ga, gb)
    a.set_tuning(chunk=3)                                      # re-plan: the captured graph is dropped
    a.step(70)
    b.step(70)
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert torch.equal(fa, fb) and torch.equal(ga, gb)


@pytest.mark.parametrize("nx,ny", [(64, 64), (32, 32), (48, 48), (16, 64), (128, 32), (20, 6), (7, 4), (84, 6)])
def test_cluster_multistep_kernel_equals_per_step_launches_bitwise(islbm, nx, ny):
    """Tiny 2-D fp64 meshes: islbm_step(n >= 2) runs all n steps in ONE launch of a thread-block cluster (bands of whole
    rows, state in distributed shared memory, halo rows by remote shared-memory stores, one cluster barrier per step).
    Same bits as the per-step TMA kernel (cluster = 2) from a far-from-equilibrium state, whatever mix of call sizes,
    and 1e-12 against the oracle after 3 steps; every cluster size from 2 to 16 CTAs and bands of 2 to 8 rows."""
    coords = [inputs.tanh_mesh(nx, 1.3)[0], inputs.tanh_mesh(ny, 1.6)[0]]
    delta = min(float(np.diff(c).min()) for c in coords)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    Ra = 0.71 * (0.1 * H_lu / 0.03) ** 2
    a, orc = pair(islbm, coords, delta, Ra=Ra)
    b = islbm.Islbm(coords, delta, Ra, 0.71, 0.1 * SQ3)
    b.set_tuning(cluster=2)
    f0, g0 = inputs.random_state(orc.shape, orc.qf, orc.qg, seed=3, amp=0.05)
    orc.set_populations(f0, g0)
    for s_ in (a, b):
        s_.set_populations(torch.from_numpy(f0).cuda(), torch.from_numpy(g0).cuda())
    l0 = a.launch_count
    a.step(3)
    assert a.launch_count - l0 == 1
    b.step(3)
    orc.step(3)
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert torch.equal(fa, fb) and torch.equal(ga, gb)
    fo, go = orc.get_populations()
    assert elem_err(fa.cpu().numpy(), fo) <= 3e-12 and plane_err(ga.cpu().numpy(), go) <= 3e-12
    for n in (2, 1, 37, 100, 5):
        a.step(n)
        b.step(n)
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert torch.equal(fa, fb) and torch.equal(ga, gb)
    for s_ in (a, b):                      # a long run from the rest + noise start (the random state does not stay finite)
        s_.init(1, 1e-3)
        s_.step(1000)
    fa, ga = a.get_populations()
    fb, gb = b.get_populations()
    assert bool(torch.isfinite(fa).all()) and torch.equal(fa, fb) and torch.equal(ga, gb)
    na, nb = a.nusselt(), b.nusselt()
    assert na == nb


def test_state_errors_and_launch_accounting(islbm):
    w = inputs.custom_workload("s", 2, 16)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    with pytest.raises(islbm.IslbmError) as e:
        sim.step(1)
    assert e.value.code == -6
    sim.init(0, 1e-3)
    n0 = sim.launch_count
    sim.step(10)
    assert sim.launch_count - n0 == 1          # 16^2 fp64: the multi-step cluster kernel, one launch for the ten steps
    sim.set_tuning(cluster=2)
    n0 = sim.launch_count
    sim.step(10)
    assert sim.launch_count - n0 >= 10
    with pytest.raises(islbm.IslbmError):
        sim.set_buoyancy_scale(0.5)
    r0 = sim.steady_residual()
    sim.step(10)
    r1 = sim.steady_residual()
    assert r0 == (1.0, 1.0) and 0 < r1[1] < 10 and r1[0] >= 0


def test_tuning_and_kernel_selection_errors(islbm):
    w = inputs.custom_workload("e", 2, 24, stretch=1.4, Ra=1e5)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    for bad in (dict(nonsense=1), dict(tx2d=100), dict(chunk=-1)):
        with pytest.raises(islbm.IslbmError) as e:
            sim.set_tuning(**bad)
        assert e.value.code == -1
    with pytest.raises(islbm.IslbmError):
        sim.set_kernel(7)
    with pytest.raises(islbm.IslbmError) as e:
        sim.set_kernel(islbm.KERNEL_UNIFORM_SHIFT)           # stretched mesh: the pure shift is not valid
    assert "delta" in str(e.value)
    with pytest.raises(islbm.IslbmError):
        sim.nusselt_middle()                                  # no state yet
    sim.init(0, 1e-3)
    sim.set_tuning(chunk=1000)                                # clamped to the longest supported chunk
    sim.step(3)
    assert np.isfinite(sim.nusselt_middle())


def test_steady_residual_matches_definition(islbm):
    """Eq. 30 on the device vs the same sums formed from islbm_fields outputs."""
    w = inputs.custom_workload("r", 2, 40, stretch=1.4, Ra=1e5)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.init(0, 1e-3)
    sim.step(300)
    a = sim.fields()
    sim.steady_residual()
    sim.step(50)
    b = sim.fields()
    ru, rT = sim.steady_residual()
    du = torch.sqrt((b["u"] - a["u"]) ** 2 + (b["v"] - a["v"]) ** 2).sum() / torch.sqrt(a["u"] ** 2 + a["v"] ** 2).sum()
    dT = (b["T"] - a["T"]).abs().sum() / a["T"].abs().sum()
    assert ru == pytest.approx(du.item(), rel=1e-10) and rT == pytest.approx(dT.item(), rel=1e-10)


# ---------------------------------------------------------------------------
# end-to-end pin against values the paper prints (A2, A7, A22)
# ---------------------------------------------------------------------------
def test_paper_mode_table2_ra1e6_257(islbm, golden):
    """Paper mode: erf mesh Eq. 26 with a = 1.5 (257 points, fluid nodes 1..255, delta = y_1), Ma = 0.1, Ra = 1e6,
    reference temperature T0 = T_cold (the paper's T* in [0,1], reading A9), run on the CUDA path to the steady-state
    criterion of Eq. 30, against Table 2 and Table 3.
    <Nu>, Nu_hot, Nu_middle within 0.3 % (the paper's own 257^2 -> infinity spread is 0.1-0.35 %); the printed <Re>
    matches sqrt(Ra/Pr) * sqrt(<u*^2>_V) (reading A22), not the mean speed of Eq. 34 as printed."""
    ref = golden["table2"]["Ra1e6"]["257"]
    w = inputs.custom_workload("paper", 2, 257, mesh="erf", stretch=1.5, Ra=1e6, Ma=0.1)
    assert len(w.coords[0]) == 255
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.set_reference_temperature(-0.5)
    sim.init(0, 0.0)
    sim.steady_residual()
    for _ in range(1500):                       # at most 3e6 steps; converges after ~1.45e6
        sim.step(2000)
        ru, rT = sim.steady_residual()
        if ru < 1e-9 and rT < 1e-9:
            break
    assert ru < 1e-9 and rT < 1e-9
    nu = sim.nusselt()
    nm = sim.nusselt_middle()
    assert nu["Nu_vol"] == pytest.approx(ref[0], rel=3e-3)
    assert nu["Nu_hot"] == pytest.approx(ref[1], rel=3e-3)
    assert nm == pytest.approx(ref[2], rel=3e-3)
    assert nu["Nu_cold"] == pytest.approx(nu["Nu_hot"], rel=2e-6)          # steady state: what enters leaves
    assert nm == pytest.approx(nu["Nu_vol"], rel=5e-4)                     # every vertical plane carries the same flux
    # with T0 = T_cold the estimator <Nu> = sqrt(RaPr)<u*T*> + 1 sits a resolution-independent 0.025 below the wall
    # value (weak compressibility: <u*>_V != 0 multiplies the 0.5 offset of T*); Nu_hot itself does not depend on T0
    assert 0.015 < nu["Nu_hot"] - nu["Nu_vol"] < 0.035
    re_rms = math.sqrt(1e6 / 0.71 * nu["u2"])
    assert re_rms == pytest.approx(ref[3], rel=3e-3)
    assert nu["Re"] < 0.8 * ref[3]                                        # Eq. 34 as printed is a different number
    # cell-centre values, Table 3: T_c on the paper's [0,1] scale = ours + 0.5, u_c in free-fall units;
    # node 127 of the 255 fluid nodes sits at x* = y* = 0.5 exactly.  With T0 = mean the solution is centro-symmetric
    # (T_c = 0.5, u_c = 0 to round-off); the paper's non-zero values are the signature of T0 = T_cold.  The paper's
    # own u_c moves by 9 % from 257^2 to infinity (-1.2163e-4 -> -1.3320e-4): 15 % tolerance; v_c (1e-5) is not asserted.
    c3 = golden["table3"]["Ra1e6"]["257"]
    fl = sim.fields(("u", "v", "T"))
    U = sim.params()["U"]
    T_c = fl["T"][0, 127, 127].item() + 0.5
    assert T_c < 0.4999 and T_c == pytest.approx(c3["T_c"], abs=3e-4)
    assert fl["u"][0, 127, 127].item() / U == pytest.approx(c3["u_c"], rel=0.15)
    assert fl["v"][0, 127, 127].item() > 0.0


def test_paper_mode_table2_ra1e7_513(islbm, golden):
    """A second Rayleigh number end to end: paper mode (erf a = 1.5, Ma = 0.1, T0 = T_cold), Ra = 1e7 on the 513-point
    mesh, run to the Eq. 30 criterion (5.4e6 steps, about a minute), against Table 2 and Table 3
    (PAPER.md:371): Nu_hot 0.2 %, <Nu> and Nu_middle 0.3 % (the estimator offset of reading A9), rms <Re> (A22) 0.2 %."""
    ref = golden["table2"]["Ra1e7"]["513"]
    w = inputs.custom_workload("paper7", 2, 513, mesh="erf", stretch=1.5, Ra=1e7, Ma=0.1)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.set_reference_temperature(-0.5)
    sim.init(0, 0.0)
    sim.steady_residual()
    for _ in range(4000):
        sim.step(2000)
        ru, rT = sim.steady_residual()
        if ru < 1e-9 and rT < 1e-9:
            break
    assert ru < 1e-9 and rT < 1e-9
    nu = sim.nusselt()
    nm = sim.nusselt_middle()
    print("TABLE2 Ra1e7 513", nu, nm, math.sqrt(1e7 / 0.71 * nu["u2"]), ref)
    assert nu["Nu_hot"] == pytest.approx(ref[1], rel=2e-3)
    assert nu["Nu_vol"] == pytest.approx(ref[0], rel=3e-3)
    assert nm == pytest.approx(ref[2], rel=3e-3)
    assert nu["Nu_cold"] == pytest.approx(nu["Nu_hot"], rel=5e-6)
    assert math.sqrt(1e7 / 0.71 * nu["u2"]) == pytest.approx(ref[3], rel=2e-3)


def test_reference_temperature_parity_and_symmetry(islbm):
    """T0 = T_cold (paper) against the oracle; T0 = mean keeps the centro-symmetry T(1-x,1-y) = -T(x,y)."""
    w = inputs.custom_workload("t0", 2, 41, stretch=1.4, Ra=1e5)
    sim, orc = pair(islbm, w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sim.set_reference_temperature(-0.5)
    orc.set_reference_temperature(-0.5)
    sim.init(0, 1e-3)
    orc.init(0, 1e-3)
    sim.step(300)
    orc.step(300)
    err = field_err(sim, orc)
    assert max(err.values()) <= 1e-9, err
    ns, no = sim.nusselt(), orc.nusselt()
    for k in no:
        assert ns[k] == pytest.approx(no[k], rel=1e-9, abs=1e-12), k
    assert sim.nusselt_middle() == pytest.approx(orc.nusselt_middle(), rel=1e-9, abs=1e-12)
    with pytest.raises(islbm.IslbmError):
        sim.set_reference_temperature(0.25)         # state already holds the force
    sym = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    sym.init(0, 0.0)
    sym.step(2000)
    T = sym.fields(("T",))["T"][0]
    assert (T + torch.flip(T, (0, 1))).abs().max().item() < 1e-12 and T.abs().max().item() > 0.3


def test_paper_mode_table4_ra1e5_129_fp32_storage(islbm, golden):
    """The same 3-D paper-mode case on the fp32-storage path, whose 3-D kernels do ALL node arithmetic in fp32
    (interpolation and both collisions): 4e5 steps from rest (the fp64 run meets Eq. 30 at 1e-9 after
    3.8e5), then the Table 4 values within the tolerances of the fp64 test.  The Eq. 30 residuals of an
    fp32 state floor at its rounding noise, so they are only required to be small, not 1e-9."""
    ref = golden["table4"]["Ra1e5"]["129"]
    w = inputs.custom_workload("paper3", 3, 129, mesh="erf", stretch=1.5, Ra=1e5, Ma=0.1)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=islbm.F32_STORAGE)
    assert sim.kernel_name == "tiled_zmarch_tma"
    sim.set_reference_temperature(-0.5)
    sim.init(0, 0.0)
    sim.step(398000)
    sim.steady_residual()
    sim.step(2000)
    ru, rT = sim.steady_residual()
    nu = sim.nusselt()
    re_rms = math.sqrt(1e5 / 0.71 * nu["u2"])
    print("T4 fp32", nu, re_rms, "residuals", ru, rT, "Table 4", ref)
    assert ru < 1e-5 and rT < 1e-5
    assert nu["Nu_vol"] == pytest.approx(ref[0], rel=3e-3)
    assert nu["Nu_hot"] == pytest.approx(ref[1], rel=6e-3)
    assert nu["Nu_cold"] == pytest.approx(nu["Nu_hot"], rel=1e-4)
    assert re_rms == pytest.approx(ref[3], rel=3e-3)


def test_paper_mode_table4_ra1e5_129(islbm, golden):
    """3-D paper mode (erf a = 1.5, 129 points -> 127^3 fluid nodes, Ma = 0.1, Ra = 1e5) to the Eq. 30 criterion
    against Table 4: <Nu> within 0.3 %, Nu_hot within 0.6 % (the paper's Nu_hot falls by 0.24 %
    from 129^3 to 181^3), <Re> in its rms form (A22) within 0.3 %.  ~3e5 steps of the z-marching TMA kernel."""
    ref = golden["table4"]["Ra1e5"]["129"]
    w = inputs.custom_workload("paper3", 3, 129, mesh="erf", stretch=1.5, Ra=1e5, Ma=0.1)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    assert sim.kernel_name == "tiled_zmarch_tma"
    sim.set_reference_temperature(-0.5)         # the paper's T* in [0,1] (reading A9)
    sim.init(0, 0.0)
    sim.steady_residual()
    for _ in range(400):
        sim.step(2000)
        ru, rT = sim.steady_residual()
        if ru < 1e-9 and rT < 1e-9:
            break
    assert ru < 1e-9 and rT < 1e-9
    nu = sim.nusselt()
    assert nu["Nu_vol"] == pytest.approx(ref[0], rel=3e-3)
    assert nu["Nu_hot"] == pytest.approx(ref[1], rel=6e-3)
    assert nu["Nu_cold"] == pytest.approx(nu["Nu_hot"], rel=1e-6)
    assert math.sqrt(1e5 / 0.71 * nu["u2"]) == pytest.approx(ref[3], rel=3e-3)
    # reading A10: Eq. 42 prints sqrt(u*^2 + v*^2) in 3-D; the library takes the full speed.  Both forms from the fields
    # with the Eq. 29 weights (ghost coordinates one delta outside, normalised by the effective lengths): the full
    # speed reproduces the library's <u*^2> and Table 4's <Re>; the two-component form as printed does not.
    flA = sim.fields(("u", "v", "w"))
    xx = np.asarray(w.coords[0])
    xe = np.concatenate(([xx[0] - w.delta], xx, [xx[-1] + w.delta]))
    w1 = torch.from_numpy(0.5 * (xe[2:] - xe[:-2])).cuda()
    W = w1[:, None, None] * w1[None, :, None] * w1[None, None, :]
    vol = (xx[-1] - xx[0] + w.delta) ** 3
    Ulu = sim.params()["U"]
    u2_full = ((flA["u"] ** 2 + flA["v"] ** 2 + flA["w"] ** 2) * W).sum().item() / vol / Ulu ** 2
    u2_uv = ((flA["u"] ** 2 + flA["v"] ** 2) * W).sum().item() / vol / Ulu ** 2
    assert u2_full == pytest.approx(nu["u2"], rel=1e-10)
    re_uv = math.sqrt(1e5 / 0.71 * u2_uv)
    print("A10", math.sqrt(1e5 / 0.71 * u2_full), re_uv, ref[3])
    assert abs(re_uv / ref[3] - 1.0) > 2 * abs(math.sqrt(1e5 / 0.71 * u2_full) / ref[3] - 1.0)
    # cell-centre values, Table 5: node 63 of the 127 sits at 0.5 exactly.  The vorticity there
    # (3-point Lagrange derivative on the stretched mesh, free-fall units) is physics: within 0.5 %.  T_c - 0.5, u_c
    # and v_c are the O(Ma^2) signature of T0 = T_cold in a weakly compressible model; ours come out at 0.78-0.86 of
    # the paper's (mesh-converged: 181^3 moves them by 0.3 %, and no relaxation rate of reading A7 moves them by more
    # than 0.1 %), so signs and magnitude only.
    c5 = golden["table5"]["Ra1e5"]["129"]
    fl = sim.fields(("u", "v", "w", "T"))
    U = sim.params()["U"]
    x = np.asarray(w.coords[0])
    c = 63
    assert x[c] == pytest.approx(0.5, abs=1e-15)
    hm, hp = x[c] - x[c - 1], x[c + 1] - x[c]
    cm, c0, cp = -hp / (hm * (hm + hp)), (hp - hm) / (hm * hp), hm / (hp * (hm + hp))

    def ddx(f, axis):                                     # fields are [z][y][x]
        i = [c, c, c]
        lo, hi = list(i), list(i)
        lo[axis] -= 1
        hi[axis] += 1
        return (cm * f[tuple(lo)] + c0 * f[tuple(i)] + cp * f[tuple(hi)]).item() / U

    om = (ddx(fl["w"], 1) - ddx(fl["v"], 0), ddx(fl["u"], 0) - ddx(fl["w"], 2), ddx(fl["v"], 2) - ddx(fl["u"], 1))
    assert math.sqrt(sum(o * o for o in om)) == pytest.approx(c5["omega_c"], rel=5e-3)
    assert abs(om[0]) < 1e-9 and abs(om[1]) < 1e-9 and abs(fl["w"][c, c, c].item()) < 1e-12     # mid-plane symmetry in z
    T_c = fl["T"][c, c, c].item() + 0.5
    assert T_c < 0.4998 and T_c == pytest.approx(c5["T_c"], abs=2e-4)
    assert fl["u"][c, c, c].item() / U == pytest.approx(c5["u_c"], rel=0.2)
    assert fl["v"][c, c, c].item() / U == pytest.approx(c5["v_c"], rel=0.25)


def test_command_line_driver(islbm, capsys):
    """python -m paper_2509_01099_b200.run: a short paper-mode run prints parameters and a diagnostics line per report."""
    import json as _json
    from paper_2509_01099_b200 import run
    run.main(["--paper", "--dim", "2", "--points", "65", "--Ra", "1e5", "--steps", "400", "--every", "200"])
    lines = [_json.loads(l) for l in capsys.readouterr().out.strip().splitlines()]
    assert lines[0]["T0"] == -0.5 and lines[0]["kernel"].startswith("tiled_ymarch_tma") and lines[0]["nodes"] == 63 * 63
    assert [l["step"] for l in lines[1:]] == [200, 400]
    assert all(np.isfinite(l["Nu_hot"]) and l["Re_rms"] >= l["Re"] for l in lines[1:])
    # --time: one JSON line with the timing of a tuning variant (the A/B rows of profiles/attempts.md)
    run.main(["--workload", "c1_64sq", "--time", "64", "--tune", "chunk=2", "--tune", "graph=2", "--stencil", "1"])
    t = _json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert t["kernel"] == "tiled_ymarch_tma_upwind" and t["tune"] == ["chunk=2", "graph=2"] and 0.5 < t["us_per_step"] < 100
    assert t["MLUPS"] == pytest.approx(64 * 64 / t["us_per_step"])
