"""Host logic of the N > 1 bench path on CPU (gloo, world_size 2): the by-view split of SURVEY.md 8(e) -- every rank
renders its own view of its own replica and the step ends with one all-reduce (sum) of the flat gradient buffer; the
whole-job value is all ranks' pixels over the max-over-ranks time. Also: the reference arm runs on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2311_18482_b200 import inputs
    scene = inputs.unbounded_scene(n=64, width=64, height=64, focal=46.0)   # the bench workload's camera family
    cam = bench.view_for_rank(scene, rank)
    t_local = 0.010 * (rank + 1)          # rank 1 is the slow one
    pixels = cam.width * cam.height * 5   # 5 steps

    def reduce_max(t):
        tt = torch.tensor([t], dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        return float(tt.item())

    agg = bench.aggregate(pixels, t_local, world, reduce_max)
    # the one exchange step of the by-view split: the eight gradient arrays live in ONE flat buffer (binding.Grads),
    # summed over the views with a single all-reduce
    from types import SimpleNamespace
    from paper_2311_18482_b200 import binding
    gr = binding.Grads(SimpleNamespace(n=scene.n, sh_stored=16, F=8), device="cpu")
    rng = np.random.default_rng(rank)
    for k in binding.Grads.FIELDS:
        getattr(gr, k).copy_(torch.from_numpy(rng.standard_normal(tuple(getattr(gr, k).shape)).astype(np.float32)))
    dist.all_reduce(gr.flat, op=dist.ReduceOp.SUM)
    ok = True
    rngs = [np.random.default_rng(r_) for r_ in range(world)]
    for k in binding.Grads.FIELDS:
        shape = tuple(getattr(gr, k).shape)
        want = sum(g_.standard_normal(shape).astype(np.float32) for g_ in rngs)
        ok = ok and np.allclose(getattr(gr, k).numpy(), want, atol=1e-6)
        ok = ok and getattr(gr, k).data_ptr() % 16 == 0
    json.dump(dict(rank=rank, w2c=[float(v) for v in cam.world_to_cam], seconds=agg["seconds"], mpix_s=agg["mpix_s"], grads_ok=bool(ok)),
              open(os.path.join(out_dir, f"r{rank}.json"), "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_weak_scaling_aggregate(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(world)]
    # both ranks agree on the max-over-ranks time and on the whole-job throughput
    assert r[0]["seconds"] == pytest.approx(0.020) and r[1]["seconds"] == pytest.approx(0.020)
    expect = 64 * 64 * 5 * world / 0.020 / 1e6
    assert r[0]["mpix_s"] == pytest.approx(expect) and r[1]["mpix_s"] == pytest.approx(expect)
    assert r[0]["grads_ok"] and r[1]["grads_ok"]   # every gradient array = sum over the ranks, on both ranks
    # each rank renders a different view: rank 0 the configured camera, rank 1 the same camera rotated about y
    from paper_2311_18482_b200 import inputs
    cam0 = inputs.unbounded_scene(n=64, width=64, height=64, focal=46.0).cameras[0]
    assert np.allclose(r[0]["w2c"], cam0.world_to_cam)
    assert not np.allclose(r[1]["w2c"], r[0]["w2c"])
    R1 = np.array(r[1]["w2c"]).reshape(3, 4)[:, :3]
    assert np.allclose(R1 @ R1.T, np.eye(3), atol=1e-6)   # still a rigid camera


def test_single_rank_aggregate_needs_no_collective():
    import bench
    agg = bench.aggregate(1_000_000, 0.5, 1)
    assert agg["seconds"] == 0.5 and agg["mpix_s"] == pytest.approx(2.0)


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_gpus_flag_spawns_the_ranks_itself_and_prints_one_line():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment starts the two ranks itself
    (torch.distributed.run on 127.0.0.1) and rank 0 prints ONE JSON line with n_gpus = 2. --dry-host keeps it on the CPU
    (gloo): the spawn, the per-rank views, the asynchronous gradient all-reduce waited for after the stand-in decode stage
    and the max-over-ranks aggregate all run; no kernel does."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-host", "--steps", "3", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["dry_host"] is True and out["steps"] == 3
    assert out["grads_allreduce_ok"] is True        # every element = 1 + 2: both ranks' gradients were summed
    assert out["distinct_views"] == 2 and out["seconds_max_over_ranks"] > 0
