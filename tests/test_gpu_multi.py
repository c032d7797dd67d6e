"""-m gpu tests of the multi-GPU mode (replicas / batch shards, one process per GPU, no data-path
collective).  They need two CUDA devices and are skipped on a one-GPU box; the rank / shard arithmetic itself is covered
on the CPU by tests/test_multiproc.py (gloo, world size 2)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import rel_l2, oracle_problem

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _two_devices():
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    import paper_2605_28800_b200 as fe
    fe.load()
    return fe


def test_two_grids_on_two_devices_in_one_process():
    """The one-time kernel set-up (dynamic shared-memory limits, persistent grid sizes) is per device: a second Grid on
    cuda:1 must run the same kernels as the first one on cuda:0, each shard against the oracle."""
    fe = _two_devices()
    from paper_2605_28800_b200 import parallel as par
    w = fi.open_batio3("two_dev", (64, 32, 32), 2, "f64", 77)
    for rank in (0, 1):
        mine = par.shard_members(w.batch, rank, 2)
        ws = fi.Workload(name=w.name, n=w.n, d=w.d, periodic=w.periodic, pbc_images=w.pbc_images, batch=len(mine),
                         dtype=w.dtype, materials=[w.materials[b] for b in mine], globals_=[w.globals_[b] for b in mine],
                         matmap=w.matmap, P0=w.P0[mine.start:mine.stop], dt=w.dt, integrator=w.integrator)
        g = fe.Grid.from_workload(ws, device="cuda:%d" % rank)
        g.precompute_tensor()
        P = g.state(ws.P0)
        assert P.device.index == rank
        for i, b in enumerate(mine):
            o = orc.Oracle(oracle_problem(w, b), elec="fft")
            assert rel_l2(g.rhs(P).cpu().numpy()[i], o.rhs(w.P0[b])) < 1e-10
        g.step(P, ws.dt, 8, fe.FE_EULER, fe.FE_TERM_ALL)          # long enough for the graph replay path
        assert np.isfinite(P.cpu().numpy()).all()
        g.close()


def test_bench_launcher_starts_one_rank_per_gpu():
    """`python bench.py --gpus 2` outside torchrun starts two ranks itself and reports n_gpus = 2 (weak scaling)."""
    _two_devices()
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "4", "--warmup", "3",
                        "--workload", "cfg3", "--no-cpu", "--no-cufft"], capture_output=True, text=True, env=env,
                       timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["value"] > 0
