"""Worker of tests/test_gpu_cluster_order.py: runs the N = 256 cluster kernels many times on a case whose outputs
receive exactly one contribution each and prints, as one JSON line, the distinct SHA-256 digests seen per output.
The library under test is the one PTY_LIB names (paper_2505_07814_b200/binding.py).  Usage: worker.py <iterations>."""
import hashlib
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2505_07814_b200 import binding as pty, synth  # noqa: E402


def main(iterations):
    cfg = synth.get_config(5, M=1, Nz=4)          # 256^2 window, 4-CTA cluster, three propagations per pass
    g = 256 * np.arange(4, dtype=np.float32) + 16.0
    yy, xx = np.meshgrid(g, g, indexing="ij")     # 16 patches that do not overlap: one contribution per g_object pixel
    rng = np.random.default_rng(33)
    pos = (np.stack([yy.ravel(), xx.ravel()], 1) + rng.uniform(-0.4, 0.4, (16, 2))).astype(np.float32)
    ev = synth.eval_point(cfg, "A")
    B = len(pos)
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    obj, probe = dev(ev["object"][:cfg.Nz]), dev(ev["probe"][:1])
    dpos, meas = dev(pos), dev(np.sqrt(rng.poisson(3.0, (B, cfg.N, cfg.N))).astype(np.float32))
    tilt = dev(np.asarray(ev["tilt"], np.float32)) if cfg.tilt_mode else None
    plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, 1, cfg.N, B, cfg.dz, cfg.lam, cfg.dx, tilt_mode=cfg.tilt_mode)
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    lpp, inten = torch.zeros(B, device="cuda"), torch.zeros(B, cfg.N, cfg.N, device="cuda")
    g_obj, g_pos = torch.zeros_like(obj), torch.zeros(B, 2, device="cuda")
    side, junk = torch.cuda.Stream(), torch.randn(4096, 4096, device="cuda")
    seen = {"intensity": set(), "loss_per_pos": set(), "g_object": set()}
    for it in range(iterations):
        if it % 2:                                 # every other pass shares the SMs with a GEMM: different CTA timing
            with torch.cuda.stream(side):
                for _ in range(2):
                    junk = junk @ junk * 1e-3
        plan.forward_loss(obj, probe, dpos, tilt, meas, loss, lpp, inten)
        plan.backward(obj, probe, dpos, tilt, meas, g_obj, None, g_pos, flags=pty.PTY_BWD_REUSE_FORWARD)
        assert plan.status()[0] == 0
        for name, t in (("intensity", inten), ("loss_per_pos", lpp), ("g_object", g_obj)):
            seen[name].add(hashlib.sha256(t.cpu().numpy().tobytes()).hexdigest())
    torch.cuda.synchronize()
    print(json.dumps({"lib": os.path.basename(pty.LIB_PATH), "iterations": iterations,
                      "digests": {k: sorted(v) for k, v in seen.items()}}))


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 40)
