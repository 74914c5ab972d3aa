"""-m gpu, one process per GPU (as many as the box has, up to 4): the time-direction domain decomposition with one process per
GPU over NCCL -- slab.FaceExchange's batch_isend_irecv ring, the side-stream overlap of slab.SlabDirac and the
callbacks of lqcd_cg_solve_slab -- against the oracle on the whole lattice.  On the one-GPU boxes of this build the
same kernels and the same exchange pattern are covered by tests/test_gpu_slab.py (slabs one after the other,
threads as ranks) and tests/test_slab_dist.py (gloo); there this file runs a single rank, and it is the check of the
NCCL ring to run when several GPUs are there."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import json, os, sys
sys.path.insert(0, %(root)r)
import numpy as np
import torch
import torch.distributed as dist
from paper_2503_16994_b200 import binding as B, slab, synth

rank, world, local = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"]), int(os.environ["LOCAL_RANK"])
torch.cuda.set_device(local)
dist.init_process_group("nccl", device_id=torch.device("cuda", local))
L, kappa, csw, theta = (8, 4, 4, 4 * world), 0.125, 1.0, (0.3, -0.2, 0.1, np.pi)
U = synth.smooth_gauge(L, 151)                      # every rank draws the same seeded whole-lattice inputs ...
b = synth.gaussian_spinor(L, 152)
ns, T = L[0] * L[1] * L[2], slab.slab_extent(L[3], world)
lo, hi = rank * T * ns, (rank + 1) * T * ns         # ... and keeps its own time slab
g = slab.slab_geom_create(L, world, theta, device=local, rank=rank)
Uc = torch.from_numpy(U[lo:hi]).cuda()
dU = B.alloc_field(g, B.FIELD_GAUGE)
B.gauge_import(g, Uc, dU)
xch = slab.FaceExchange()
halo_lo, halo_hi = slab.gauge_halo_exchange(Uc, L, xch)
dA = B.alloc_field(g, B.FIELD_CLOVER)
B.clover_build_slab(g, kappa, csw, dU, halo_lo, halo_hi, dA)
src, dst = B.alloc_field(g, B.FIELD_SPINOR), B.alloc_field(g, B.FIELD_SPINOR)
B.spinor_import(g, torch.from_numpy(b[lo:hi]).cuda(), src)
D = slab.SlabDirac(g, kappa, dU, dA, exchange=xch)
out = {}
canon = torch.empty((hi - lo, 4, 3), dtype=torch.complex128, device="cuda")
for name, dagger in (("dw", False), ("dwdag", True)):
    D.apply(src, dst, dagger)
    B.spinor_export(g, dst, canon)
    torch.cuda.synchronize()
    out[name] = canon.cpu().numpy().copy()
comm = slab.SlabCommunicator(g, xch)
ws = B.alloc_field(g, B.FIELD_WORKSPACE)
info = slab.cg_solve_slab(g, kappa, dU, dA, src, dst, ws, comm, tol=1e-10, maxiter=4000)
B.spinor_export(g, dst, canon)
torch.cuda.synchronize()
out["x"] = canon.cpu().numpy().copy()
np.savez(os.path.join(%(tmp)r, "rank%%d.npz" %% rank), lo=lo, hi=hi, iters=info["iters"], **out)
dist.barrier()
dist.destroy_process_group()
'''


@pytest.mark.timeout(900)
def test_slab_dw_and_cg_over_nccl(tmp_path):
    # one GPU: a single rank still runs the whole worker under an NCCL process group (communicator, callbacks, solver,
    # the slab as its own neighbour); the send/recv ring itself needs >= 2 GPUs
    world = max(1, min(torch.cuda.device_count(), 4))
    import oracle
    from paper_2503_16994_b200 import synth

    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT, "tmp": str(tmp_path)})
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    run = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                          "--master-addr", "127.0.0.1", "--master-port", "29561", str(script)],
                         capture_output=True, text=True, timeout=800, env=env)
    assert run.returncode == 0, run.stderr[-3000:]
    L, kappa, csw, theta = (8, 4, 4, 4 * world), 0.125, 1.0, (0.3, -0.2, 0.1, np.pi)
    U = synth.smooth_gauge(L, 151)
    b = synth.gaussian_spinor(L, 152)
    A = oracle.clover_blocks(L, U, kappa, csw)
    got = {k: np.empty_like(b) for k in ("dw", "dwdag", "x")}
    iters = set()
    for r in range(world):
        z = np.load(tmp_path / ("rank%d.npz" % r))
        for k in got:
            got[k][int(z["lo"]):int(z["hi"])] = z[k]
        iters.add(int(z["iters"]))
    V = b.shape[0]
    for k, dagger in (("dw", False), ("dwdag", True)):
        ref = oracle.dw(L, U, b, kappa, A, theta=theta, dagger=dagger)
        err = np.linalg.norm((got[k] - ref).reshape(V, -1), axis=1) / np.linalg.norm(ref.reshape(V, -1), axis=1)
        assert err.max() <= 1e-12
    xo, it_o, _, _ = oracle.cg(L, U, b, kappa, A, theta=theta, tol=1e-10)
    assert np.linalg.norm(got["x"] - xo) / np.linalg.norm(xo) <= 1e-8
    assert len(iters) == 1 and abs(iters.pop() - it_o) <= 2
