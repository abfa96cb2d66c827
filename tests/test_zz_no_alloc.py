"""pty_ortho_probe_noalloc: the probe-mode orthogonalisation for callers that cannot allocate.

Every other call of include/pty.h needs a plan, and a plan needs a device workspace that the caller allocates.  A host
application whose memory pool took the whole GPU at start-up, or a hook that is handed the probe and a stream and
nothing else, cannot provide one; for them the library keeps a fixed 33 KB scratch array of its own (M <= 32 modes) and
this entry point allocates nothing.  The array is shared by all calls and keeps the last call's contents, so the test
makes two calls in a row with different mode counts and window sizes, and checks both against the plan-based path
(pty_constrain with ortho_probe) -- same kernels, so the bound is rounding-tight -- and against the oracle's unique
quantities at the tolerances of tests/test_gpu_features.py::test_probe_orthogonalisation.

This file is named to be collected last: with `pytest -x` a failure here hides no other test.  It needs nothing from
the tests before it and passes in a fresh process as well.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import constraints as oc  # noqa: E402
from cases import rel_l2  # noqa: E402
from paper_2505_07814_b200 import synth  # noqa: E402


@pytest.fixture(scope="module")
def pty():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    build.build()
    from paper_2505_07814_b200 import binding
    return binding


def mixed_probe(c, M, seed):
    """M strongly non-orthogonal modes with the window of config c."""
    cfg = synth.get_config(c, M=M)
    rng = np.random.default_rng(seed)
    mix = rng.standard_normal((M, M)) + 1j * rng.standard_normal((M, M))
    return cfg, np.tensordot(mix, synth.make_probe(cfg), axes=1).astype(np.complex64)


def test_two_calls_in_a_row_match_the_plan_path(pty):
    # second call: fewer modes and a smaller window than the first, so that stale scratch contents would show
    for call, (c, M, seed) in enumerate(((4, 12, 5), (1, 5, 6))):
        cfg, P = mixed_probe(c, M, seed)
        via_plan = torch.from_numpy(P).cuda()
        plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, 1, cfg.dz, cfg.lam, cfg.dx)
        plan.constrain(probe=via_plan, ortho_probe=True)
        no_alloc = torch.from_numpy(P).cuda()
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        pty.ortho_probe_noalloc(no_alloc)
        torch.cuda.synchronize()
        if call > 0:      # the first call may load kernels onto the device; after that the free memory must not move
            assert torch.cuda.mem_get_info()[0] >= free_before, "pty_ortho_probe_noalloc took device memory"
        Q, Q_plan = no_alloc.cpu().numpy(), via_plan.cpu().numpy()
        assert rel_l2(Q, Q_plan) <= 1e-6, (call, rel_l2(Q, Q_plan))
        # and the unique parts against the oracle: powers, mutual orthogonality
        Q_ref, lam_ref = oc.orthogonalize_modes(P)
        qf = Q.reshape(M, -1).astype(np.complex128)
        G = np.conj(qf) @ qf.T
        lam = np.real(np.diag(G))
        np.testing.assert_allclose(lam, lam_ref, rtol=1e-4, atol=1e-6 * lam_ref[0])
        assert np.max(np.abs(G - np.diag(lam))) <= 1e-5 * lam_ref[0]
        plan.close()


def test_sizes_beyond_the_fixed_scratch_are_refused(pty):
    too_many = torch.zeros(pty.ORTHO_NOALLOC_MAX_MODES + 1, 8, 8, dtype=torch.complex64, device="cuda")
    with pytest.raises(pty.PtyError) as e:
        pty.ortho_probe_noalloc(too_many)
    assert e.value.code == pty.PTY_ERR_UNSUPPORTED and "limit: 32 modes" in str(e.value)
    assert torch.count_nonzero(too_many).item() == 0
    at_limit = torch.randn(pty.ORTHO_NOALLOC_MAX_MODES, 8, 8, dtype=torch.complex64, device="cuda")
    pty.ortho_probe_noalloc(at_limit)                       # the stated maximum itself works
    qf = at_limit.cpu().numpy().reshape(pty.ORTHO_NOALLOC_MAX_MODES, -1).astype(np.complex128)
    G = np.conj(qf) @ qf.T
    assert np.max(np.abs(G - np.diag(np.diag(G)))) <= 1e-5 * np.max(np.real(np.diag(G)))
