"""Two-GPU parity of the x-slab sharded path over NCCL: torchrun with two
ranks, each evaluating its slab in the CUDA kernels, all-gather of F and all-reduce of dL/dv, against the single-GPU
whole-grid result.  Skips cleanly on a box with fewer than two GPUs (the build and its driver run on one)."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import paper_2303_10440_b200 as dm
from paper_2303_10440_b200.sharding import sharded_mesh_ft_backward, sharded_mesh_ft_forward
from workloads import build_workload
from workloads.configs import spectrum_cotangent
local = int(os.environ["LOCAL_RANK"])
torch.cuda.set_device(local)
dist.init_process_group("nccl", device_id=torch.device("cuda", local))
for cfg, grid in ((2, (30, 16, 16)), (4, (32, 24, 16))):      # 30 rows over 2 ranks; a surface-mode aggregate
    w = build_workload(cfg, subdiv_override=2, grid_override=grid)
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    vd = torch.as_tensor(w.vertices, device="cuda")
    Gd = torch.as_tensor(spectrum_cotangent(w), device="cuda")
    F_ref = plan.mesh_ft_forward(vd).clone()
    dv_ref = plan.mesh_ft_backward(vd, Gd).clone()
    F = sharded_mesh_ft_forward(plan, vd)
    dv = sharded_mesh_ft_backward(plan, vd, Gd)
    assert float((F - F_ref).abs().max()) <= 1e-6 * float(F_ref[0, 0, 0].abs()), "the slabs of F must tile the whole-grid spectrum"
    rel = float(torch.linalg.norm(dv - dv_ref) / torch.linalg.norm(dv_ref))
    assert rel <= 1e-5, rel
    plan.close()
dist.barrier()
dist.destroy_process_group()
print("NCCL_SLAB_OK")
'''


def test_two_rank_slab_sharding_over_nccl(tmp_path):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs on one node")
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29541", str(script)],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.count("NCCL_SLAB_OK") == 2, r.stdout[-2000:] + r.stderr[-2000:]
