"""Multi-GPU host path with the REAL library as the compute step.

dist.sharded_apply / sharded_expect split the alpha rows over the ranks, each rank computes its slab with
bs_apply_rows on cuda:0 and the slabs are exchanged.  Only one GPU exists here, so the ranks are processes that share
cuda:0: their kernels are independent (nothing waits on another rank inside a kernel) and the collectives run over
gloo on host tensors, with the device work inside the apply_rows callback.  World sizes 1, 2 and 3 (ragged slabs),
checked against the oracle; the same callback drives `bench.py --sharded` over NCCL.
"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, os.path.join(sys.argv[1], 'tests'))
import numpy as np, torch, torch.distributed as dist
import synth_inputs as si
from oracle import oracle as orc
from paper_2606_28952_b200 import bs
from paper_2606_28952_b200.dist import sharded_apply, sharded_expect
dist.init_process_group("gloo")
rank = dist.get_rank()
torch.cuda.set_device(0)
cases = [("mol", 9, 3, 5), ("mol", 12, 6, 6), ("hub", 10, 5, 4)]
for kind, n, na, nb in cases:
    if kind == "mol":
        h, g = si.integrals(n, 1002 if n == 12 else 79)
        ref, op = orc.molecular_h(h, g), bs.bs_jw_molecular(h, g)
    else:
        ref, op = orc.hubbard_h(n, 1.0, 4.0), bs.bs_jw_hubbard(n, 1.0, 4.0)
    osec, sec = orc.Sector(n, na, nb), bs.bs_sector_build(n, na, nb)
    psi = si.random_state(osec.dim, 2001)
    Db = osec.dim_beta
    def apply_rows(pin, pout, lo, hi):        # host tensors in and out, the slab itself by the library on cuda:0
        d_in = pin.cuda(); d_out = torch.full_like(d_in, float('nan'))
        bs.bs_apply_rows(op, sec, d_in, d_out, lo, hi)
        got = d_out.cpu()
        assert torch.isnan(got[:lo * Db].real).all() and torch.isnan(got[hi * Db:].real).all()   # nothing else written
        pout[lo * Db:hi * Db] = got[lo * Db:hi * Db]
    t_in = torch.from_numpy(psi.copy())
    t_out = torch.full_like(t_in, float('nan'))
    sharded_apply(apply_rows, t_in, t_out, osec.dim_alpha, Db)
    want = osec.apply_grouped(ref, psi)
    err = np.linalg.norm(t_out.numpy() - want) / np.linalg.norm(want)
    assert err <= 1e-12, (rank, kind, n, err)
    e = sharded_expect(apply_rows, t_in, torch.zeros_like(t_in), osec.dim_alpha, Db)
    assert abs(e - orc.vdot(psi, want)) <= 1e-10, (rank, e)
dist.barrier()
dist.destroy_process_group()
print("RANK_OK", rank)
"""


@pytest.mark.parametrize("world", [1, 2, 3])
def test_sharded_apply_with_library(world, tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 29700 + world + (os.getpid() % 200)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), ROOT]
    env = dict(os.environ, OMP_NUM_THREADS="4")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, env=env)
    assert r.returncode == 0 and r.stdout.count("RANK_OK") == world, r.stdout[-2000:] + r.stderr[-3000:]
