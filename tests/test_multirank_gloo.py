"""N > 1 host logic on CPU (gloo, world_size 2): the path shards by tokens with no data-path collective
(DESIGN.md 9); bench.py only needs a barrier and a max-over-ranks of the device time."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle
    from bm_inputs import CONFIGS, bf16_bits, make_layer
    assert bench.dist_env() == (rank, rank, world)
    # max over ranks of a per-rank time, as the timed loop uses it
    t = bench.max_over_ranks(0.010 * (rank + 1), world, torch.device("cpu"))
    assert abs(t - 0.010 * world) < 1e-12
    bench.barrier(world)
    # every rank: same layer (seed 0), its own tokens (x seed = rank), as DeviceLayer builds them
    cfg = CONFIGS["tiny"]
    L = make_layer(cfg, 0)
    if rank != 0:
        L.x = make_layer(cfg, rank, weights=False).x
    r = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), None, cfg.K, L.group_map.numpy(), cfg.G)
    out = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2))
    np.save(os.path.join(out_dir, f"out{rank}.npy"), out)
    torch.save(L.x, os.path.join(out_dir, f"x{rank}.pt"))
    # whole-job throughput = units all ranks processed / max time
    total = torch.tensor([float(cfg.T)], dtype=torch.float64)
    dist.all_reduce(total)
    assert total.item() == cfg.T * world
    dist.destroy_process_group()


def test_two_ranks_gloo_sharding_needs_no_collective(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    # the union of the ranks' batches, run as ONE batch, gives the same rows: tokens are independent,
    # so sharding them across ranks needs no exchange step
    import oracle
    from bm_inputs import CONFIGS, bf16_bits, make_layer
    cfg = CONFIGS["tiny"]
    L = make_layer(cfg, 0)
    xs = [torch.load(tmp_path / f"x{r}.pt") for r in range(world)]
    outs = [np.load(tmp_path / f"out{r}.npy") for r in range(world)]
    assert not torch.equal(xs[0], xs[1])
    x_all = torch.cat(xs)
    r = oracle.route(bf16_bits(x_all), bf16_bits(L.W_router), None, cfg.K, L.group_map.numpy(), cfg.G)
    out_all = oracle.moe_forward(bf16_bits(x_all), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2))
    assert (out_all == np.concatenate(outs)).all()


def test_reference_arm_nonzero_ranks_exit_without_work(monkeypatch, capsys):
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setenv("LOCAL_RANK", "1")

    class A:
        config, steps, warmup = "tiny", 1, 0
    bench.run_reference(A())
    assert capsys.readouterr().out == ""


# ---------------------------------------------------------------------------------------------------
# tensor parallelism over F (NEXT-4): the decomposition and the host plumbing, on CPU
# ---------------------------------------------------------------------------------------------------
def _tp_worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from bm_inputs import bf16_bits, make_layer, LayerConfig
    from paper_2607_04164_b200.tp import shard_f
    cfg = LayerConfig("tp", T=24, D=64, F=88, E=8, K=3, G=4, S=1, zipf_s=1.0)      # F = 11 units of 8: uneven shards
    L = make_layer(cfg, 0)
    W1r, W3r, W2r = shard_f(L.W1, L.W3, L.W2, rank, world)
    r = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), L.router_bias.numpy(), cfg.K, L.group_map.numpy(), cfg.G)
    part = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(W1r), bf16_bits(W3r), bf16_bits(W2r), cfg.S)
    t = torch.from_numpy(part)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)            # the one exchange step of the TP layer
    np.save(os.path.join(out_dir, f"tp{rank}.npy"), t.numpy())
    np.save(os.path.join(out_dir, f"f{rank}.npy"), np.array([W1r.shape[1]]))
    dist.destroy_process_group()


def test_tensor_parallel_over_f_two_ranks_gloo(tmp_path):
    """SwiGLU is elementwise over F, so the layer is the sum over ranks of the layer on each rank's F shard
    (include/bm.h: bm_moe_forward_f32): oracle partials, summed with a gloo all-reduce, equal the unsharded oracle."""
    world, port = 2, _free_port()
    mp.spawn(_tp_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    import oracle
    from bm_inputs import bf16_bits, make_layer, LayerConfig
    cfg = LayerConfig("tp", T=24, D=64, F=88, E=8, K=3, G=4, S=1, zipf_s=1.0)
    L = make_layer(cfg, 0)
    r = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), L.router_bias.numpy(), cfg.K, L.group_map.numpy(), cfg.G)
    full = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), cfg.S)
    outs = [np.load(tmp_path / f"tp{k}.npy") for k in range(world)]
    fs = [int(np.load(tmp_path / f"f{k}.npy")[0]) for k in range(world)]
    assert sum(fs) == cfg.F and all(f % 8 == 0 and f > 0 for f in fs)
    assert (outs[0] == outs[1]).all()
    assert np.abs(outs[0] - full).max() <= 1e-12 * (1 + np.abs(full).max())


def test_shard_bounds_cover_f_exactly():
    from paper_2607_04164_b200.tp import shard_bounds
    for F, world in [(88, 2), (1408, 8), (14336, 8), (64, 8), (1408, 3)]:
        cuts = [shard_bounds(F, r, world) for r in range(world)]
        assert cuts[0][0] == 0 and cuts[-1][1] == F
        assert all(cuts[i][1] == cuts[i + 1][0] for i in range(world - 1))
        sizes = [hi - lo for lo, hi in cuts]
        assert all(s % 8 == 0 and s > 0 for s in sizes) and max(sizes) - min(sizes) <= 8
