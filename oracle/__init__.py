"""CPU oracle for the tomoCAM hot path (arXiv 2304.12934) -- TEST INFRASTRUCTURE ONLY.

Plain, slow, float64 numpy restatement of what the CUDA path computes, written
from /root/reference/PAPER.md ("P:L<n>" = line number there) and the readings
listed in DESIGN.md.  It shares no code with ``paper_2304_12934_b200/`` and is
never imported by it.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.

Modules
  direct.py   (D1)/(D2): direct non-uniform DFT of the Fourier-slice Radon pair,
              and the Dirichlet-kernel closed form of the same matrix
              (eqs. (3), (5), (6)).           pinned
  analytic.py closed-form projections (Gaussian, ellipse) and a ray-driven
              line-integral projector (eq. (2)).                 pinned
  nufft.py    the NUFFT approximation, step by step (eqs. (6)-(8) and
              "reverse order").              pinned (vs direct.py)
  prior.py    qGGMRF prior value and gradient (eqs. (12)-(13)). pinned
  mbir.py     monotone accelerated gradient with restart (eq. (9)-(10),
              P:L99-103).  The paper only CITES the optimiser, so the
              iterate sequence is PARITY UNPINNED against the paper; the loop is
              pinned by invariants only (monotone F, first iterate, lstsq limit).
"""
