"""fp64 CPU oracle for the tomographic reconstruction hot path of arXiv:1806.07938.

THIS PACKAGE IS TEST INFRASTRUCTURE.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` leg may import it.  It shares no
code with `paper_1806_07938_b200/` (the CUDA path) and never imports it; the only
module both sides use is `tomo_inputs/` (seeded inputs, no method arithmetic).

What it computes (each module cites the passage it follows, PAPER.md L<line>):

  vonkarman.py   D_phi(r) of Eq.53 (L619), phase covariance C_phi
  geometry.py    subaperture / phase-point grids, pupil masks (Fig.2)
  covariance.py  linear-stencil slope models (Eq.47-48, Eq.54-55), dense C_ss (Eq.14,
                 L136-158) and C_os (Eq.15-17) built from POSITIONS
  fftmodel.py    FFT slope model Eq.41-46 (L534-572): the continuous integrals, evaluated in physical space (edge-averaged
                 structure function, Gauss-Legendre panels); shares no grid with the library's FFT-based builder
  projectors.py  W, Z, M = I - Z Z^+ (Eq.33-36)
  solver.py      direct solve of Eq.5/Eq.12, textbook CG and MINRES (S2.G L337, L426), Eq.13
  toeplitz.py    the paper's 2RBT product Eq.18-28 step by step, generators, op counts
  directsum.py   matrix-free direct-sum MVM for ELT sizes (directsum.c, OpenMP)
  system.py      assembles a TomoConfig into the operator A, rhs and projections
  layered.py     layered-phase (MCAO) variant of L199 / L516: Sigma_{phi_k s} of each layer on its meta-pupil grid from
                 positions, no I'_k, no sum over layers; ray tracing of the layers (reading G31)
  loworder.py    low-order NGS tip/tilt path (paper-silent, L321/L412; reading G30): MMSE estimator of the aperture-mean
                 slopes from positions, tilt add-back

Pins (tests/test_oracle_*.py, `-m "not gpu"`): closed forms of D_phi, the Kolmogorov
limit, the PSD integral, printed formulas Eq.50-52 / Eq.56-62 against the generic
stencil evaluation, symmetry/PSD of C_ss, dense == paper's index maps == 2-D FFT
product, projector identities, CG -> Cholesky, MINRES = the least-squares minimiser over the
Krylov space (brute force) = scipy's minres, LGS ground-layer identity, the
paper's printed closed-form counts (L150, L177, L197, L270, L280, L295), the telescoping
closed form of the aperture-mean Hudgin slope variance (loworder.py); the FFT slope model against Eq.43 / Eq.46 as
printed, summed over frequency grids refined to convergence, and against adaptive quadrature (test_oracle_fftmodel.py);
the layered variant against the joint Gaussian model written out sample by sample with the phase covariance, against the
LTAO covariances through ray tracing on grid-aligned directions, and against the 2RBT product (test_oracle_layered.py).

Parity unpinned: absolute WFE in nm (Table 3) and the curves of Fig.9-15 are not
reproduced; nothing in this package depends on them.
"""
