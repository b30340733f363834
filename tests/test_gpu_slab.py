"""Slab decomposition on ONE GPU: K slab handles in one process, halo exchanged by direct copies, against the
single-domain handle (bit for bit on the owned layers) and against the oracle.  No rank waits on another: the
slabs are stepped one after the other on the same stream."""
import math
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.oracle import Oracle  # noqa: E402
from paper_2509_01099_b200 import inputs, slab  # noqa: E402

SQ3 = math.sqrt(3.0)


@pytest.fixture(scope="module")
def islbm():
    import __graft_entry__ as graft
    graft.build()
    from paper_2509_01099_b200 import islbm as mod
    return mod


def mesh(dim, ns, st):
    coords = [inputs.tanh_mesh(n, s)[0] for n, s in zip(ns[:dim], st[:dim])]
    delta = min(float(np.diff(c).min()) for c in coords)
    H_lu = (coords[1][-1] - coords[1][0] + delta) / delta
    return coords, delta, 0.71 * (0.1 * H_lu / 0.03) ** 2


@pytest.mark.parametrize("fused", [False, True], ids=["exchange", "fused"])
@pytest.mark.parametrize("dim,ns,world,prec,kernel", [
    (2, (70, 45), 2, 0, 0), (2, (70, 45), 4, 0, 0), (2, (131, 20), 5, 1, 0), (2, (40, 33), 3, 0, 1),
    (3, (40, 24, 37), 3, 0, 0), (3, (33, 17, 9), 2, 1, 0), (3, (36, 18, 16), 8, 0, 0), (3, (20, 12, 11), 2, 0, 1)])
def test_slabs_equal_the_single_domain_bitwise(islbm, dim, ns, world, prec, kernel, fused):
    coords, delta, Ra = mesh(dim, ns, (1.4, 1.2, 1.3))
    Ma = 0.1 * SQ3
    whole = islbm.Islbm(coords, delta, Ra, 0.71, Ma, precision=prec)
    slabs = [slab.SlabCavity(coords, delta, Ra, 0.71, Ma, r, world, precision=prec, exchange=lambda: None) for r in range(world)]
    if kernel:
        whole.set_kernel(kernel)
        for s in slabs:
            s.sim.set_kernel(kernel)
    whole.init(3, 1e-3)
    for s in slabs:
        s.init(3, 1e-3)
        assert whole.params()["H_lu"] == s.sim.params()["H_lu"]
    if fused:
        slab.connect_local(slabs)        # the step kernels store the halo into the neighbours' ghost layers themselves
    halo = (lambda: None) if fused else (lambda: slab.exchange_local(slabs))
    for _ in range(7):
        whole.step(1)
        for s in slabs:
            s.sim.step(1)
        halo()
    fw = whole.fields()
    fw_pop, gw_pop = whole.get_populations()
    for s in slabs:
        lo, hi = s.own
        fl = s.sim.fields()
        for k in fl:
            ref = fw[k][..., lo:hi, :] if dim == 2 else fw[k][lo:hi]
            assert torch.equal(s.owned(fl[k]), ref), (k, s.rank)
        fp, gp = s.sim.get_populations()
        reff = fw_pop[..., lo:hi, :] if dim == 2 else fw_pop[:, lo:hi]
        assert torch.equal(s.owned(fp), reff)
    # diagnostics: partial sums added over the slabs == the single-domain reduction (different summation order)
    total = np.sum([s.sim.diag_sums() for s in slabs], axis=0)
    d = slabs[0].sim.diag_from_sums(total)
    nu = whole.nusselt()
    for k in nu:
        assert d[k] == pytest.approx(nu[k], rel=1e-11, abs=1e-13), k
    assert d["Nu_middle"] == pytest.approx(whole.nusselt_middle(), rel=1e-11, abs=1e-13)
    # Eq. 30 residual from sums
    r0 = [s.sim.residual_sums() for s in slabs]
    whole.steady_residual()
    assert all(first for _, first in r0)
    whole.step(1)
    for s in slabs:
        s.sim.step(1)
    halo()
    sums = np.sum([s.sim.residual_sums()[0] for s in slabs], axis=0)
    ru, rT = whole.steady_residual()
    assert sums[0] / sums[1] == pytest.approx(ru, rel=1e-10) and sums[2] / sums[3] == pytest.approx(rT, rel=1e-10)
    with pytest.raises(islbm.IslbmError):
        slabs[0].sim.nusselt()


def test_fused_exchange_is_one_launch_per_step_and_flags_count_steps(islbm):
    """Fused exchange with the neighbour-only device-side synchronisation: one kernel per slab and step and no other
    launch (no collective, no exchange pass); each slab's step flags hold the number of steps its neighbours have
    finished; a neighbour at a different step count is refused; a buffer-parity difference between neighbours (one
    of them re-initialised after an odd number of steps) is handled (it used to corrupt silently)."""
    coords, delta, Ra = mesh(3, (40, 24, 21), (1.4, 1.2, 1.3))
    Ma = 0.1 * SQ3
    whole = islbm.Islbm(coords, delta, Ra, 0.71, Ma)
    slabs = [slab.SlabCavity(coords, delta, Ra, 0.71, Ma, r, 3, exchange=lambda: None) for r in range(3)]
    whole.init(5, 1e-3)
    for s in slabs:
        s.init(5, 1e-3)
    slabs[1].sim.step(1)                   # slab 1: one step on its own, then a fresh state: cur = 1, steps = 0
    with pytest.raises(islbm.IslbmError) as e:
        slab.connect_local(slabs)          # step counts 0 / 1 / 0
    assert e.value.code == -6 and "steps" in str(e.value)
    slabs[1].init(5, 1e-3)
    assert [s.sim.halo_layout(0)["cur"] for s in slabs] == [0, 1, 0]
    slab.connect_local(slabs)
    l0 = [s.sim.launch_count for s in slabs]
    for _ in range(6):
        whole.step(1)
        for s in slabs:                    # in turn on one stream: every flag is set before the kernel that reads it
            s.sim.step(1)
    assert [s.sim.launch_count - a for s, a in zip(slabs, l0)] == [6, 6, 6]
    torch.cuda.synchronize()
    for r, s in enumerate(slabs):
        lay = [s.sim.halo_layout(side) for side in (0, 1)]
        flags = [int(s.sim.workspace[l["flag_offset"]:l["flag_offset"] + 8].view(torch.int64).item()) for l in lay]
        assert (r == 0 or flags[0] == 6) and (r == 2 or flags[1] == 6), (r, flags)      # wall sides have no flag
        assert lay[0]["steps"] == 6
    fw = whole.fields()
    for s in slabs:
        lo, hi = s.own
        fl = s.sim.fields()
        for k in fl:
            assert torch.equal(s.owned(fl[k]), fw[k][lo:hi]), (k, s.rank)


def test_fused_exchange_wait_is_bounded(islbm):
    """A neighbour that never steps must not hang the GPU: the boundary CTAs of the waiting slab give up after
    `slab_wait_ms` (200 ms here; default 10 s), count the time-out, and the next synchronising slab call reports it."""
    import time
    coords, delta, Ra = mesh(3, (40, 24, 21), (1.4, 1.2, 1.3))
    slabs = [slab.SlabCavity(coords, delta, Ra, 0.71, 0.1 * SQ3, r, 2, exchange=lambda: None) for r in range(2)]
    for s in slabs:
        s.init(5, 1e-3)
    slabs[0].sim.set_tuning(slab_wait_ms=200)
    slab.connect_local(slabs)
    slabs[0].sim.step(1)                       # step 1 needs the neighbour's step 0: there from the start
    slabs[0].sim.diag_sums()                   # fine so far
    t0 = time.time()
    slabs[0].sim.step(1)                       # step 2 needs the neighbour's step 1, which never comes
    with pytest.raises(islbm.IslbmError) as e:
        slabs[0].sim.diag_sums()
    dt = time.time() - t0
    assert e.value.code == -6 and "gave up waiting" in str(e.value)
    assert 0.15 < dt < 5.0, dt
    for s in slabs:
        s.close()


def test_slabs_against_the_oracle(islbm):
    coords, delta, Ra = mesh(3, (24, 16, 21), (1.3, 1.2, 1.4))
    orc = Oracle(coords, delta, Ra, 0.71, 0.1 * SQ3, threads=max(1, min(16, len(os.sched_getaffinity(0)))))
    slabs = [slab.SlabCavity(coords, delta, Ra, 0.71, 0.1 * SQ3, r, 3, exchange=lambda: None) for r in range(3)]
    orc.init(0, 1e-3)
    for s in slabs:
        s.init(0, 1e-3)
    orc.step(20)
    for _ in range(20):
        for s in slabs:
            s.sim.step(1)
        slab.exchange_local(slabs)
    fo = orc.fields()
    umax = max(np.abs(fo[k]).max() for k in ("u", "v", "w"))
    for s in slabs:
        lo, hi = s.own
        fl = s.sim.fields()
        for k in ("u", "v", "w"):
            assert np.abs(s.owned(fl[k]).cpu().numpy() - fo[k][lo:hi]).max() <= 1e-10 * max(umax, 1e-4)
        assert np.abs(s.owned(fl["T"]).cpu().numpy() - fo["T"][lo:hi]).max() <= 1e-12


_IPC_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2509_01099_b200 import inputs, slab, islbm
rank, world = int(os.environ["RANK"]), 2
dist.init_process_group(backend="gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
coords = [inputs.tanh_mesh(n, s)[0] for n, s in zip((40, 24, 22), (1.4, 1.2, 1.3))]
delta = min(float(np.diff(c).min()) for c in coords)
H = (coords[1][-1] - coords[1][0] + delta) / delta
Ra = 0.71 * (0.1 * H / 0.03) ** 2
cav = slab.SlabCavity(coords, delta, Ra, 0.71, 0.1 * 3 ** 0.5, rank, world)
cav.init(3, 1e-3)
cav.connect_ipc()                       # CUDA IPC mapping of the neighbour's workspace + fused exchange
cav.step(6)
d = cav.diagnostics()
lo, hi = cav.own
T = cav.owned(cav.sim.fields(("T",))["T"]).cpu().numpy()
np.save({out!r} + f"_{{rank}}.npy", T)
print(json.dumps(dict(rank=rank, own=[lo, hi], **d)))
dist.barrier()
cav.close()
dist.destroy_process_group()
"""


def test_two_processes_one_gpu_fused_exchange_over_cuda_ipc(islbm, tmp_path):
    """Two ranks as two PROCESSES sharing the one GPU: control plane gloo, data plane CUDA IPC (each rank's step
    kernel stores its boundary layer into the other process's workspace and publishes its step flag there).  The
    ranks share ONE GPU here, so connect_ipc orders the steps by a host barrier after a device synchronise (its
    default for a non-NCCL backend): every flag is already set when the kernel that reads it starts, and no kernel
    ever waits on another process's kernel (B200_PROFILING.md: such waits on one GPU can time out the context
    switch).  Result against the single-domain run."""
    import subprocess, sys, json
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    port = 29900 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_IPC_WORKER.format(root=root, port=port, out=str(tmp_path / "T")))
    procs = [subprocess.Popen([sys.executable, str(script)], env={**os.environ, "RANK": str(r)}, stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for p in procs:
        so, se = p.communicate(timeout=600)
        assert p.returncode == 0, se[-2000:]
        outs.append(json.loads(so.strip().splitlines()[-1]))
    coords, delta, Ra = mesh(3, (40, 24, 22), (1.4, 1.2, 1.3))
    whole = islbm.Islbm(coords, delta, Ra, 0.71, 0.1 * SQ3)
    whole.init(3, 1e-3)
    whole.step(6)
    Tw = whole.fields(("T",))["T"].cpu().numpy()
    nu = whole.nusselt()
    for o in outs:
        lo, hi = o["own"]
        assert np.array_equal(np.load(str(tmp_path / "T") + f"_{o['rank']}.npy"), Tw[lo:hi])
        for k in nu:
            assert o[k] == pytest.approx(nu[k], rel=1e-11, abs=1e-13), k
