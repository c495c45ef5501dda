"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the path shards replicas by rank with no data-path
collective, so the only cross-rank logic is the max-over-ranks timing, the whole-job value,
and the rule that rank 0 alone prints the line of the reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
mine = [10.0 + 5.0 * rank, 3.0 - rank, 7.0]            # rank 1 is slower on the first, faster on the second
red = bench.max_over_ranks(mine, world, torch.device("cpu"))
dist.barrier()
if rank == 0:
    print(json.dumps({{"red": red, "value": bench.whole_job_value(512 * 100, world, red[0])}}))
dist.destroy_process_group()
"""


def _torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29731"] + args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_whole_job_value_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    p = _torchrun([str(script)])
    assert p.returncode == 0, p.stderr[-2000:]
    line = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(line) == 1, "exactly one rank prints"
    d = json.loads(line[0])
    assert d["red"] == [15.0, 3.0, 7.0]
    assert d["value"] == pytest.approx(2 * 512 * 100 / 15e-3)


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    p = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "0", "--steps", "2", "--warmup", "3",
                   "--ref-budget", "2"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0


_MW_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2301_04835_b200.multiwalker import deposit_hill_all_ranks
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")

class FakeCtx:                       # stands in for psg.Context on CPU tensors: records what the helper asks the library for
    def __init__(self): self.centres, self.heights = [], []
    def hill_heights(self, xi, mask, out):
        out.copy_(100.0 * (rank + 1) + xi[:, 0])          # any rank-dependent numbers
        if mask is not None: out[mask == 0] = 0.0
    def append_hills(self, c, h):
        self.centres.append(c.clone()); self.heights.append(h.clone())

ctx = FakeCtx()
R, n_cv = 3, 2
xi = torch.arange(R * n_cv, dtype=torch.float32).reshape(R, n_cv) + 10.0 * rank
mask = torch.tensor([1, 0, 1], dtype=torch.uint8) if rank == 1 else None
n = deposit_hill_all_ranks(ctx, xi, mask)
out = dict(rank=rank, n=n, centres=ctx.centres[0].tolist(), heights=ctx.heights[0].tolist())
gathered = [None] * world
dist.all_gather_object(gathered, out)
if rank == 0:
    print(json.dumps(gathered))
dist.destroy_process_group()
"""


def test_multiwalker_deposit_gathers_in_rank_order_gloo(tmp_path):
    """deposit_hill_all_ranks: every rank appends the (centre, height) pairs of ALL walkers, rank 0's first,
    with the zero heights of masked-out walkers kept in place for the library to skip; both ranks append the same list"""
    script = tmp_path / "mw_worker.py"
    script.write_text(_MW_WORKER.format(root=ROOT))
    p = _torchrun([str(script)])
    assert p.returncode == 0, p.stderr[-2000:]
    line = [l for l in p.stdout.splitlines() if l.startswith("[")]
    assert len(line) == 1
    r0, r1 = json.loads(line[0])
    assert r0["n"] == r1["n"] == 6
    assert r0["centres"] == r1["centres"] and r0["heights"] == r1["heights"]
    assert r0["centres"] == [[0.0, 1.0], [2.0, 3.0], [4.0, 5.0], [10.0, 11.0], [12.0, 13.0], [14.0, 15.0]]
    assert r0["heights"] == [100.0, 102.0, 104.0, 210.0, 0.0, 214.0]


def test_multiwalker_deposit_single_process():
    """without an initialised process group the helper is the two library calls back to back"""
    import torch
    from paper_2301_04835_b200.multiwalker import deposit_hill_all_ranks

    class Ctx:
        def hill_heights(self, xi, mask, out):
            out.fill_(1.5)

        def append_hills(self, c, h):
            self.got = (c.clone(), h.clone())

    c = Ctx()
    xi = torch.ones((4, 2))
    assert deposit_hill_all_ranks(c, xi) == 4
    assert torch.equal(c.got[0], xi) and torch.equal(c.got[1], torch.full((4,), 1.5))


_ABF_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2301_04835_b200.multiwalker import abf_step_all_ranks
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")

class FakeCtx:                       # stands in for psg.Context on CPU tensors: a 6-bin grid, one CV
    n_cv = 1
    def __init__(self): self.hist = torch.zeros(6, dtype=torch.int32); self.fsum = torch.zeros(6); self.calls = []
    def abf_n_bins(self): return 6
    def abf_accumulate_delta(self, pos, fs, dh, df):
        dh.zero_(); df.zero_()
        for b, f in zip(pos.tolist(), fs.tolist()):      # "positions" are the bins here
            dh[int(b)] += 1; df[int(b)] += f
        self.calls.append("acc")
    def abf_apply_grid_delta(self, dh, df, pos, force):
        self.hist += dh; self.fsum += df
        force += self.fsum[pos.long()] / self.hist[pos.long()].clamp(min=1)
        self.calls.append("apply")

ctx = FakeCtx()
pos = torch.tensor([0.0, 2.0, 2.0]) if rank == 0 else torch.tensor([2.0, 5.0, 0.0])
fs = torch.tensor([1.0, 2.0, 3.0]) * (rank + 1)
force = torch.zeros(3)
for _ in range(2):
    abf_step_all_ranks(ctx, pos, force, fs)
out = dict(rank=rank, hist=ctx.hist.tolist(), fsum=ctx.fsum.tolist(), force=force.tolist(), calls=ctx.calls)
gathered = [None] * world
dist.all_gather_object(gathered, out)
if rank == 0:
    print(json.dumps(gathered))
dist.destroy_process_group()
"""


def test_multiwalker_abf_all_reduces_the_grid_deltas_gloo(tmp_path):
    """abf_step_all_ranks: both ranks end with the grid ONE context holding all six replicas would build --
    the all-reduce sums the per-step histogram / force-sum contributions before anyone reads a mean force"""
    script = tmp_path / "abf_worker.py"
    script.write_text(_ABF_WORKER.format(root=ROOT))
    p = _torchrun([str(script)])
    assert p.returncode == 0, p.stderr[-2000:]
    line = [l for l in p.stdout.splitlines() if l.startswith("[")]
    assert len(line) == 1
    r0, r1 = json.loads(line[0])
    assert r0["hist"] == r1["hist"] == [4, 0, 6, 0, 0, 2]                  # two steps of {0: 2, 2: 3, 5: 1}
    assert r0["fsum"] == r1["fsum"] == [2 * (1.0 + 6.0), 0.0, 2 * (2.0 + 3.0 + 2.0), 0.0, 0.0, 2 * 4.0]
    assert r0["calls"] == ["acc", "apply", "acc", "apply"]
    # step 1 means: bin 0 -> 7/2, bin 2 -> 7/3, bin 5 -> 4; step 2: 14/4, 14/6, 8/2: the same numbers
    assert r0["force"] == pytest.approx([7.0, 14 / 3, 14 / 3]) and r1["force"] == pytest.approx([14 / 3, 8.0, 7.0])
