"""fp64 CPU oracle for the micromagnetic hot path of arXiv 1406.7635 ("MuMax3").

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline`
/ `--impl reference` legs of `bench.py` may import this package; the product
(`paper_1406_7635_b200/`) never does, and this package never imports the product.  It is a
plain, slow, numpy/fp64 restatement of what the paper defines; citations `Lnnn` are lines
of /root/reference/PAPER.md.

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`):
  demag tensor  - cube factors 1/3 (Table I), trace rule, point-dipole far field
                  (Fig. 4), thin-film / rod limits and Tables II-III (L151-L171),
                  analytic-vs-quadrature cross-check, direct sum vs FFT convolution
  exchange      - zero for uniform m; spiral energy (L204, L723); Eq. 9 -> Eq. 6 limit
  anisotropy    - Eq. 19<->20 and 22<->23 energy identities, finite-difference gradient
  torque / RK45 - Larmor precession m_x = cos(gamma B t) (Fig. 3 L97), 5th-order
                  convergence (Fig. 10), |m| = 1, energy non-increasing with damping
  parity unpinned (shared rule only): the step-size controller's
                  exponent/clamps and the Euclidean error norm; the 5 ns relax duration of C2.
"""
from .sim import RefSim, MM_DEMAG, MM_EXCH, MM_ANIS, MM_ZEEMAN, MM_ALL

__all__ = ["RefSim", "MM_DEMAG", "MM_EXCH", "MM_ANIS", "MM_ZEEMAN", "MM_ALL"]
