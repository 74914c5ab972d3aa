"""CPU, gloo, world_size 2 and 3: the host-side logic of the time-direction domain decomposition
(paper_2503_16994_b200/slab.py): who owns which slices, which face lands where on the
periodic ring (including world_size 2, where both neighbours are the same peer), the one-off gauge halo, the
all-reduce of CG scalars.  The kernels themselves are covered on the GPU by tests/test_gpu_slab.py."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import json, os, sys
sys.path.insert(0, %r)
import torch
import torch.distributed as dist
from paper_2503_16994_b200 import slab
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
xch = slab.FaceExchange()
L = (2, 2, 2, 4 * world)
ns = 8
# faces: value = 100 * sender + (1: its send_lo, 2: its send_hi)
send_lo = torch.full((6 * ns,), 100.0 * rank + 1, dtype=torch.float64)
send_hi = torch.full((6 * ns,), 100.0 * rank + 2, dtype=torch.float64)
recv_lo, recv_hi = torch.zeros_like(send_lo), torch.zeros_like(send_lo)
xch(send_lo, send_hi, recv_lo, recv_hi)
# gauge halo: slab links filled with their global time coordinate
T = slab.slab_extent(L[3], world)
t0 = slab.slab_origin(L[3], world, rank)
U = torch.empty((T * ns, 4, 3, 3), dtype=torch.complex128)
for t in range(T):
    U[t * ns:(t + 1) * ns] = float(t0 + t)
halo_lo, halo_hi = slab.gauge_halo_exchange(U, L, xch)
s = xch.allreduce_sum(torch.tensor([float(rank + 1)], dtype=torch.float64))
# a lattice with open time boundaries: the chain is not closed
xo = slab.FaceExchange(periodic=False)
olo, ohi = torch.full_like(send_lo, -1.0), torch.full_like(send_lo, -1.0)
xo(send_lo, send_hi, olo, ohi)
oh_lo, oh_hi = slab.gauge_halo_exchange(U, L, xo)
open(os.path.join(%r, "rank%%d.json" %% rank), "w").write(json.dumps({"rank": rank, "world": world, "t0": t0, "T": T, "below": xch.below, "above": xch.above,
                  "recv_lo": sorted(set(recv_lo.tolist())), "recv_hi": sorted(set(recv_hi.tolist())),
                  "halo_lo": sorted(set(halo_lo.real.flatten().tolist())),
                  "halo_hi": sorted(set(halo_hi.real.flatten().tolist())), "sum": s.item(),
                  "open_nbr": [xo.below, xo.above], "open_lo": sorted(set(olo.tolist())), "open_hi": sorted(set(ohi.tolist())),
                  "open_halo": [None if h is None else sorted(set(h.real.flatten().tolist())) for h in (oh_lo, oh_hi)],
                  "edges": slab.slab_edges(world, rank, 1)}))
dist.barrier()
dist.destroy_process_group()
'''


@pytest.mark.parametrize("world,port", [(2, 29551), (3, 29552)])
def test_face_exchange_on_the_time_ring(tmp_path, world, port):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % (ROOT, str(tmp_path)))   # every rank writes its own file: stdout lines can interleave
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    rows = {}
    for r in range(world):
        d = json.loads((tmp_path / ("rank%d.json" % r)).read_text())
        rows[d["rank"]] = d
    assert sorted(rows) == list(range(world))
    L4 = 4 * world
    for r, d in rows.items():
        below, above = (r - 1) % world, (r + 1) % world
        assert (d["below"], d["above"]) == (below, above)
        assert (d["t0"], d["T"]) == (4 * r, 4)
        assert d["recv_lo"] == [100.0 * below + 2]     # the rank below's send_hi (its last slice)
        assert d["recv_hi"] == [100.0 * above + 1]     # the rank above's send_lo (its first slice)
        assert d["halo_lo"] == [float((4 * r - 1) % L4)]
        assert d["halo_hi"] == [float((4 * r + 4) % L4)]
        assert d["sum"] == world * (world + 1) / 2
        # open lattice: first rank has nobody below, last nobody above; those receive buffers stay untouched
        first, last = r == 0, r == world - 1
        assert d["open_nbr"] == [None if first else below, None if last else above]
        assert d["open_lo"] == ([-1.0] if first else [100.0 * below + 2])
        assert d["open_hi"] == ([-1.0] if last else [100.0 * above + 1])
        assert d["open_halo"] == [None if first else [float(4 * r - 1)], None if last else [float(4 * r + 4)]]
        assert d["edges"] == (1 if first else 0) | (2 if last else 0)


def test_slab_bookkeeping():
    from paper_2503_16994_b200 import slab

    assert slab.slab_extent(96, 8) == 12 and slab.slab_origin(96, 8, 3) == 36
    assert slab.ring_neighbours(4, 0) == (3, 1) and slab.ring_neighbours(1, 0) == (0, 0)
    th = slab.slab_theta((0.5, 0.5, 0.5, 3.0), 96, 8)
    assert th[:3] == [0.5, 0.5, 0.5] and abs(th[3] / 12 - 3.0 / 96) < 1e-15   # same phase per link
    for L4, w in ((96, 5), (8, 4), (12, 2 * 3)):
        with pytest.raises(ValueError):
            slab.slab_extent(L4, w)


def test_single_rank_exchange_is_the_periodic_wrap():
    import torch
    from paper_2503_16994_b200 import slab

    xch = slab.FaceExchange()
    assert (xch.world, xch.below, xch.above) == (1, 0, 0)
    a, b = torch.arange(6.0), torch.arange(6.0) + 10
    ra, rb = torch.zeros(6), torch.zeros(6)
    xch(a, b, ra, rb)
    assert torch.equal(rb, a) and torch.equal(ra, b)   # recv_hi = send_lo, recv_lo = send_hi
