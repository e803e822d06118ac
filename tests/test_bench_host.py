"""CPU: host-side logic of bench.py — replica aggregation over torch.distributed (gloo, world_size 2), byte/flop
accounting of the per-step roofline (pinned to the paper's P:85 numbers through oracle.accounting)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # replicas only: every rank serves the same number of requests; tokens add up, time is the max over ranks
    assert bench.shard_requests(3, world) == [3, 3]
    tok, sec = bench.aggregate(128.0 * (rank + 1), 1.0 + 0.5 * rank, dist)
    out.put((rank, tok, sec))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, tok, sec in res:
        assert tok == 128.0 + 256.0 and sec == 1.5        # whole-job tokens ÷ max-over-ranks time


def test_aggregate_single_process():
    import bench
    assert bench.aggregate(10.0, 2.0, None) == (10.0, 2.0)


def test_step_work_matches_paper_byte_count():
    """DS-1 decode touches 27 x 6 experts x 3*2048*1408*2 B = 2673 MiB of expert weights per token."""
    import bench
    import synth
    from oracle.accounting import decode_expert_bytes_per_token, step_roofline_seconds
    s = synth.get_config("c3").shape
    n_moe = s.n_layers - s.n_dense_layers
    b0, f0 = bench.step_work(s, 1, 100, 0, 0)
    b1, f1 = bench.step_work(s, 1, 100, n_moe * s.top_k, 0)
    assert b1 - b0 == decode_expert_bytes_per_token(27, 6, 2048, 1408, 2)
    assert round((b1 - b0) / 2 ** 20) == 2673
    # needed-but-not-resident experts are also WRITTEN into the slot region
    b2, _ = bench.step_work(s, 1, 100, n_moe * s.top_k, 10)
    assert b2 - b1 == 10 * 3 * 2048 * 1408 * 2
    t, bound, terms = bench.roofline_time(1e9, 6.4e9, 1e12, 50.0, 6400.0, 1000.0)
    t2, bound2, _ = step_roofline_seconds(1e9, 6.4e9, 1e12, 50e9, 6400e9, 1000e12)
    assert bound == bound2 == "h2d" and abs(t - t2) < 1e-12 and abs(t - 0.02) < 1e-12


def test_shared_expert_buffer_matches_private_copy(tmp_path):
    """bench.py --gpus N: local rank 0 draws the routed experts into a shared mapping, the other ranks map it."""
    import synth
    cfg = synth.get_config("c1b")
    ref = synth.make_weights(cfg, pin=False)
    s = cfg.shape
    n = (s.n_layers - s.n_dense_layers) * s.n_experts * 3 * s.hidden * s.expert_inter
    path = str(tmp_path / "experts.bin")
    a = torch.from_file(path, shared=True, size=n, dtype=torch.bfloat16).view_as(ref.experts)
    wa = synth.make_weights(cfg, pin=False, experts_buf=a, fill_experts=True)
    b = torch.from_file(path, shared=True, size=n, dtype=torch.bfloat16).view_as(ref.experts)
    wb = synth.make_weights(cfg, pin=False, experts_buf=b, fill_experts=False)
    assert torch.equal(wa.experts, ref.experts) and torch.equal(wb.experts, ref.experts)
    assert all(torch.equal(wb.dense[k], ref.dense[k]) for k in ref.dense)


def _replica_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import synth
    cfg = synth.get_config("c1b")
    w = bench.replica_weights(cfg, "skip", rank, world, dist, tag=f"test{port}")
    # what a replica hands to the engine: the expert images (shared mapping) and its own dense tensors
    out.put((rank, float(w.experts.double().sum()), float(w.experts[1, 3, 17:4000].double().abs().sum()),
             float(w.dense["l0.router"].double().sum()), w.experts.data_ptr() % 4096))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_share_one_expert_copy_two_ranks_gloo():
    """bench.py --gpus N: two CPU-side ranks go through the /dev/shm path of replica_weights — local rank 0 draws the
    routed experts into the mapping, rank 1 maps what rank 0 drew; both see the bytes of a private copy."""
    import synth
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_replica_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = synth.make_weights(synth.get_config("c1b"), pin=False)
    want = (float(ref.experts.double().sum()), float(ref.experts[1, 3, 17:4000].double().abs().sum()),
            float(ref.dense["l0.router"].double().sum()))
    for r in res:
        assert r[1:4] == want
        assert r[4] == 0                                   # page-aligned mapping (cudaHostRegister needs that)
    assert not [f for f in os.listdir("/dev/shm") if f.startswith(f"promoe_experts_test{port}")]   # unlinked after mapping


def test_gpus_flag_spawns_one_rank_per_gpu():
    """`python bench.py --gpus N` without a launcher starts N ranks itself."""
    import bench
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "2"])
    assert cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
