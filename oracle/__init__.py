"""FP64 CPU oracle for the PTEFIT per-slice Picard iteration (arxiv 2601.12378).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It shares no code with ``paper_2601_12378_b200`` (the CUDA path) and imports nothing
from it; the only module both sides use is ``synth`` (seeded input generators).

Every function cites the passage of ``PAPER.md`` (arxiv 2601.12378) it follows, or the
DESIGN.md reading where the paper is silent.  Plain numpy/scipy in float64, no
blocking, fusion or reordering beyond what the cited definition states.

Pin status:
  greens   : pinned (quadrature of Eq. 3-5, golden values, reciprocity, B = curl psi)
  gs_solve : pinned (Solov'ev closed form, dense solve, discrete residual)
  search   : fit/classification pinned (exact quadratics, brute force); bilinear pinned (exact on
             a linear field), cold_start pinned (hand values), limiter-vertex validity pinned by
             constructed fluxes (behind an X-point: rejected; in front: wins);
             the plasma-region rule itself = DESIGN.md reading, **parity unpinned by the paper**
  basis    : pinned (Eq. 10 closed forms at hand-computable points); tension-spline cardinals
             pinned (tau->0 = scipy natural CubicSpline, tau->inf = hat functions, partition of
             unity, the defining ODE by finite differences, C2 at the knots) -- the spline terms
             are BASELINE.json's, not the paper's: **parity unpinned by the paper**
  lsq      : pinned (normal-equation identity, exact-data recovery, chi^2 follows the chi-square
             law with M - nb degrees of freedom on forward-chain data + noise)
  picard   : pinned (fixed-point property, exact-data recovery in one iteration, warm = continued
             cold start); no printed example in the paper
"""
