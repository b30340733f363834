"""Host logic of the slab decomposition on CPU: index arithmetic and the halo-exchange schedule over a
world-size-2 and world-size-3 gloo group (plain CPU tensors stand in for the workspace views)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2509_01099_b200 import inputs, slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_split_covers_every_layer_once():
    for n, w in ((10, 1), (10, 3), (7, 7), (256, 8), (37, 4)):
        r = slab.split(n, w)
        assert r[0][0] == 0 and r[-1][1] == n and all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [hi - lo for lo, hi in r]
        assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        slab.split(3, 4)


@pytest.mark.parametrize("dim,n,world", [(2, 45, 2), (3, 19, 3), (3, 16, 8)])
def test_slab_inputs_ghosts_offsets_and_extent(dim, n, world):
    x, delta = inputs.tanh_mesh(n, 1.4)
    coords = [inputs.tanh_mesh(12, 1.2)[0] for _ in range(dim - 1)] + [x]
    covered = []
    for r in range(world):
        local, sl, own, (glo, ghi) = slab.slab_inputs(coords, delta, r, world)
        lo, hi = own
        assert (glo, ghi) == (int(r > 0), int(r < world - 1))
        assert sl["lo_is_wall"] == (r == 0) and sl["hi_is_wall"] == (r == world - 1)
        assert np.array_equal(local[-1], x[lo - glo: hi + ghi])
        for a in range(dim - 1):
            assert np.array_equal(local[a], coords[a])
        assert sl["L_eff_global"] == pytest.approx(x[-1] - x[0] + delta, rel=1e-15)
        assert sl["node_offset"] == (lo - glo) * 12 ** (dim - 1)
        covered += list(range(lo, hi))
    assert covered == list(range(n))


def test_slab_inputs_refuse_slabs_thinner_than_the_stencil():
    x, delta = inputs.tanh_mesh(8, 1.2)
    with pytest.raises(ValueError):
        slab.slab_inputs([x, x, x], delta, 0, 8)      # 1 owned + 1 ghost layer < 3


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2509_01099_b200 import slab
rank, world = int(os.environ["RANK"]), {world}
dist.init_process_group(backend="gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
P = 3
mk = lambda v: [torch.full((5,), float(v + p)) for p in range(P)]
send_lo, send_hi = mk(100 * rank + 10), mk(100 * rank + 20)
recv_lo, recv_hi = mk(-1), mk(-1)
slab.exchange_p2p(send_lo, recv_lo, send_hi, recv_hi, rank, world)
print(json.dumps({{"rank": rank, "recv_lo": [t[0].item() for t in recv_lo], "recv_hi": [t[0].item() for t in recv_hi]}}))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_schedule_over_gloo(tmp_path, world):
    port = 29700 + (os.getpid() + world) % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT, port=port, world=world))
    procs = [subprocess.Popen([sys.executable, str(script)], env={**os.environ, "RANK": str(r)}, stdout=subprocess.PIPE, text=True)
             for r in range(world)]
    outs = {}
    for p in procs:
        o = json.loads(p.communicate(timeout=300)[0].strip().splitlines()[-1])
        outs[o["rank"]] = o
    for r in range(world):
        # my low ghost holds the high send layers of rank r-1; my high ghost the low send layers of rank r+1
        want_lo = [100 * (r - 1) + 20 + p for p in range(3)] if r > 0 else [-1 + p for p in range(3)]
        want_hi = [100 * (r + 1) + 10 + p for p in range(3)] if r < world - 1 else [-1 + p for p in range(3)]
        assert outs[r]["recv_lo"] == want_lo and outs[r]["recv_hi"] == want_hi
