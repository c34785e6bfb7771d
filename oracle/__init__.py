"""CPU oracle for the coupled T-matrix multiple-scattering solve of arXiv 2107.09879.

TEST INFRASTRUCTURE ONLY.  Plain, slow, double-precision restatement of the paper's
equations (Appendix I-II, IV) used to check the CUDA path.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import anything from this package; the product (``paper_2107_09879_b200``)
never does, and this package never imports the product.

Every function cites the PAPER.md passage it follows.  Readings of garbled or silent
passages are listed in DESIGN.md ("Readings") and referenced here as R1..R19.

Parity pins (tests/test_oracle_*.py, ``-m "not gpu"``):
  special functions -> mpmath; Wigner 3j -> orthogonality + sympy; VSWF -> numerical
  curl identities; translation block -> pointwise addition theorem against direct VSWF
  evaluation; Mie T -> textbook extinction + Rayleigh limit + unitarity; incident
  coefficients -> field reconstruction; assembled solve -> N=1 Mie, extinction=scattering,
  adjoint bilinear identity, hand-rolled LU; matrix-free C matvec -> dense assembly; null-field T
  (nullfield.py) -> Lorenz-Mie limit, displaced sphere through the regular translation operator,
  losslessness / reciprocity / mirror structure; shape derivative -> Mie radius derivative.
"""
