"""CPU FP64 oracle for the PAW-FE R-ChFSI filter path (arxiv/paper_2604_26037).

THIS PACKAGE IS TEST INFRASTRUCTURE.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  The product
(``paper_2604_26037_b200``) never imports, links or executes anything here, and this package never
imports the product.  The two share no code; only ``pawfe_inputs`` (seeded data, no method
arithmetic) serves both.

It is a plain, slow, obviously-correct restatement of what the path computes, in FP64 NumPy/SciPy:
explicit sparse operators assembled from their definitions, the filter written line by line from
Algorithm 2 of the paper, and a dense brute-force eigensolve for tiny meshes.  Each function cites
the PAPER.md passage (or DESIGN.md reading) it follows.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``) -- see DESIGN.md "Oracle pins":
  gll/gauss rules ............ textbook tables, exactness degree
  K, M, M_D .................. K 1 = 0, 1^T M 1 = 1^T M_D 1 = volume, symmetry
  H_loc (V=0) ................ free-electron k^2/2 (periodic) / particle-in-a-box (Dirichlet) spectra
  cell-wise vs assembled ..... sum_e scatter(H^e gather(X)) == CSR product
  H, S ....................... Hermitian, S positive definite
  S^-1 approx (Eq. 28-29) .... exact Woodbury inverse of M_D + C dS C^T for one atom
  projector integrals ........ partition of unity: sum_J C_J,alpha = integral of p_alpha (closed form)
  filter (Alg. 2) ............ == plain Chebyshev filter Eq. 19-20 with exact S^-1; eigenpair fixed point
  outer loop (Alg. 1) ........ lowest Ritz values == dense eigh(H, S) on config 0
  complex path ............... H(k) Hermitian, k=0 reproduces real matrices, 1/2|k+G|^2 spectrum
Round 2 (tests/test_oracle_pins_r2.py; each verified to turn red under the mutation named):
  potential cell matrix ...... 0th / 1st / 2nd moments of V^e == closed Gaussian moments (x<->z mirror of the points)
  lumped mass ................ composite GLL rule: exact to degree 2p-1, Lobatto remainder at 2p (uniform weights)
  k-term of H^e .............. k with three different components, per-axis +-G plane waves (G_x <-> G_z swap)
  operators.apply_H_rows ..... == rows of the assembled product on config 0, complex and Dirichlet twins (dropped cell)
  operators.apply_HSinv_rows . == rows of apply_H(apply_Sinv(X)) on the same cases (atom reached through a neighbour cell)
  paw.projector_overlap_matrix == brute-force 3-D Gram matrix of the projector functions (the <p|p> variant of L228)
With these, no function on the path is "parity unpinned".
"""
