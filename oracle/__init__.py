"""Float64 CPU oracle for the multislice-ptychography hot path (PtyRAD, arxiv 2505.07814).

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (the package
``paper_2505_07814_b200`` and its CUDA library) imports, links or calls this
package.  It may be used by ``tests/``, by ``__graft_entry__.smoke()`` and by
the ``cpu_baseline`` / ``--impl reference`` legs of ``bench.py``.

It shares no code with the CUDA path: no kernels, headers, tables, constants
or helpers.  Only the seeded input generators (``paper_2505_07814_b200.synth``,
which holds none of the method's arithmetic) feed both sides.

Every function cites the passage of ``/root/reference/PAPER.md`` it follows.
Parity status: every function here (``multislice``, ``losses``, ``constraints``) is pinned by ``tests/test_oracle_*.py``
(brute-force DFT, closed forms, invariants, adjoint dot-products, central
finite differences, torch.autograd third opinion); nothing is "parity unpinned".
"""
from .multislice import *  # noqa: F401,F403
from . import constraints, losses  # noqa: F401  (NEXT-2 / NEXT-3: Eq. 5-9, amplitude-phase, constraints)
