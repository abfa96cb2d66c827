"""World-size-2 gloo test of the data-parallel host logic (no GPU): a minibatch sharded over two
processes, each computing its shard's gradient (here with the oracle standing in for the CUDA
kernels), then the sum all-reduce, must equal the single-process full-minibatch gradient."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_2505_07814_b200.parallel import shard_range  # noqa: E402


def test_shard_range_partitions():
    for B in (0, 1, 5, 64, 1023):
        for world in (1, 2, 3, 8):
            parts = [shard_range(B, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out_dir):
    import oracle
    from paper_2505_07814_b200 import parallel, synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = synth.get_config(1)
    geom = oracle.Geometry(cfg.dz, cfg.lam, cfg.dx)
    tr, ev = synth.truth(cfg), synth.eval_point(cfg, "A")
    B = 7
    idx = synth.minibatch(cfg, 0, cfg.B)[:B]
    meas = synth.poisson_amplitudes(cfg, oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][idx], None, geom), idx)
    pos = ev["positions"][idx]
    g_obj = torch.zeros(ev["object"].shape, dtype=torch.complex128)
    g_probe = torch.zeros(ev["probe"].shape, dtype=torch.complex128)
    g_pos = torch.zeros(B, 2, dtype=torch.float64)
    loss = torch.zeros(1, dtype=torch.float64)

    def compute(lo, hi):
        g = oracle.grad_batch(ev["object"], ev["probe"], pos[lo:hi], None, meas[lo:hi], geom)
        g_obj.copy_(torch.from_numpy(g["g_object"]))
        g_probe.copy_(torch.from_numpy(g["g_probe"]))
        g_pos[lo:hi] = torch.from_numpy(g["g_positions"])
        loss[0] = g["loss"]

    lo, hi = parallel.sharded_gradient(compute, B, g_obj, g_probe, g_pos, None, loss)
    assert (lo, hi) == parallel.shard_range(B, rank, world)
    if rank == 0:
        full = oracle.grad_batch(ev["object"], ev["probe"], pos, None, meas, geom)
        np.testing.assert_allclose(g_obj.numpy(), full["g_object"], rtol=1e-11, atol=1e-11)
        np.testing.assert_allclose(g_probe.numpy(), full["g_probe"], rtol=1e-11, atol=1e-11)
        np.testing.assert_allclose(g_pos.numpy(), full["g_positions"], rtol=1e-11, atol=1e-11)
        assert np.isclose(loss.item(), full["loss"], rtol=1e-12)
        open(os.path.join(out_dir, "ok"), "w").write("ok")
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharded_gradient_equals_full_batch(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert (tmp_path / "ok").exists()
