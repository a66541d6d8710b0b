"""CPU oracle for the SplitSolve hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may
import anything from here.  The product (`paper_1812_01396_b200/`, `libsplitsolve.so`) never does,
and this package never imports the product or its CUDA binding.  Inputs are plain numpy arrays
handed in by the caller.

What the oracle computes is the *plain definition* of the result the paper's method reaches
("solving such a system is equivalent to obtaining the first and last block columns
of T^-1 and multiplying them with the non-zero rows of Inj"):

    T = E*S - H - Sigma^RB                (Eq. 5; where Sigma_L / Sigma_R sit: L148)
    X = T^-1 Inj                          (Eq. 5)
    G_1N = (T^-1)_{1,nb}                  (Eq. 4)
    T(E) = Re Tr(Gamma_L G_1N Gamma_R G_1N^H),  Gamma = i (Sigma - Sigma^H)   (BASELINE.json north_star;
                                          the paper only plots T(E): Fig. 1(b) caption L23, L85)

It assembles the FULL matrix and runs LU with partial pivoting on it -- dense (`dense.py`, Tier A), or
the same matrix in LAPACK band storage (`banded.py`, Tier B) for sizes whose dense form does not fit.
No block recursion, no Schur sweeps, no Sherman-Morrison-Woodbury: nothing of Algorithm 1 (L159-165)
or Eq. 11-13 (L135-139) is used here, so an error in the method's algebra cannot hide in the oracle.
`stepwise.py` additionally restates Eq. 11-13 / Algorithm 1 step by step in the paper's notation,
only so that the tests can pin the paper's algebra (and our readings of its garbled spots) to the
plain definition.

Arithmetic: complex128 (fp64 re/im) throughout, as the paper (DP flops, L266) and BASELINE.json fix.

Pin status (tests/test_oracle_pins.py, all `-m "not gpu"`):
  dense.assemble_T / solve / transmission : pinned (brute-force inverse, hand-written Gaussian
      elimination, closed-form perfect chain X_j = e^{ikj}, T = bs; 1-D single-impurity textbook
      transmission; T_LR = T_RL at Im E = 0 and the eta-identity at Im E != 0; 0 <= T <= bs;
      Sigma = 0 / decoupled => T = 0)
  dense.inverse_columns                  : pinned (A * [Q|P] = [e_1|e_nb]; P_1 = Q_nb^H at real E)
  banded.*                               : pinned to dense.* on C0-sized and medium inputs + closed form C1
  residual.backward_error                : pinned to the dense residual on small inputs
  stepwise.*                             : pinned to dense.* (it is itself only a cross-check)
  observables.density                    : pinned (closed-form perfect chain rho_i = sum_e w_e; brute-force loop)
  observables.bond_current               : pinned (conservation at Im E = 0; perfect chain J = 2 bs sin k; brute-force loop)
No function here is "parity unpinned".
"""
