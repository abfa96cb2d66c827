"""The data-parallel path with the real kernels: two processes, each with its own plan on
cuda:0, run pty_forward_loss + pty_backward on their shard of one minibatch through parallel.sharded_gradient and sum
the partial gradients with one all-reduce; rank 0 compares the result with the oracle's full-minibatch gradient.
The box has one GPU, so both ranks share it and the exchange goes through gloo; the ranks' kernels never wait on one
another (the only coupling is the host-side collective after each rank's stream has drained).  With one GPU per rank
the same code runs over NCCL (bench.py --gpus N)."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

pytestmark = pytest.mark.gpu

LOSS_RTOL, GRAD_RTOL = 1e-4, 1e-3


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out_dir):
    import sys
    here = os.path.dirname(os.path.abspath(__file__))
    sys.path[:0] = [os.path.dirname(here), here]
    import oracle
    from cases import geom_of, make_case, rel_l2
    from paper_2505_07814_b200 import binding as pty, parallel, synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    cfg = synth.get_config(3, Nz=3, M=2, tilt_mode=1, true_tilt=(3e-4, -2e-4), eval_tilt=(1e-4, 2e-4))
    B = 7                                              # shards of 4 and 3 positions
    idx = synth.minibatch(cfg, 0, cfg.B)[:B]
    tr, ev = synth.truth(cfg), synth.eval_point(cfg, "A")
    geom = geom_of(cfg)
    meas = synth.poisson_amplitudes(cfg, oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][idx], tr["tilt"], geom), idx)
    pos = np.ascontiguousarray(ev["positions"][idx])
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    obj, probe, dpos, dmeas, tilt = dev(ev["object"]), dev(ev["probe"]), dev(pos), dev(meas), dev(np.asarray(ev["tilt"], np.float32))
    lo, hi = parallel.shard_range(B, rank, world)
    plan = pty.plan_for(cfg, Bmax=hi - lo)
    g_obj, g_probe = torch.zeros_like(obj), torch.zeros_like(probe)
    g_pos, g_tilt = torch.zeros(B, 2, device="cuda"), torch.zeros(2, device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")

    def compute(a, b):
        plan.forward_loss(obj, probe, dpos[a:b], tilt, dmeas[a:b], loss)
        plan.backward(obj, probe, dpos[a:b], tilt, dmeas[a:b], g_obj, g_probe, g_pos[a:b], g_tilt, flags=pty.PTY_BWD_REUSE_FORWARD)
        assert plan.status()[0] == 0

    assert parallel.sharded_gradient(compute, B, g_obj, g_probe, g_pos, g_tilt, loss) == (lo, hi)
    torch.cuda.synchronize()
    if rank == 0:
        ref = oracle.grad_batch(ev["object"], ev["probe"], pos, ev["tilt"], meas, geom)
        assert abs(loss.item() - ref["loss"]) <= LOSS_RTOL * ref["loss"]
        errs = {"g_object": rel_l2(g_obj.cpu().numpy(), ref["g_object"]), "g_probe": rel_l2(g_probe.cpu().numpy(), ref["g_probe"]),
                "g_positions": rel_l2(g_pos.cpu().numpy(), ref["g_positions"]), "g_tilt": rel_l2(g_tilt.cpu().numpy(), ref["g_tilt"].sum(0))}
        assert all(v <= GRAD_RTOL for v in errs.values()), errs
        open(os.path.join(out_dir, "ok"), "w").write(repr(errs))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_two_ranks_on_one_gpu_through_sharded_gradient(tmp_path):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    build.build()
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok").exists()
    print((tmp_path / "ok").read_text())
