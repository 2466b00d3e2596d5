"""CPU oracle for the BLTC Yukawa convolution -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product package (paper_2003_01833_b200) never does, and this
package never imports the product's CUDA binding.  See oracle/direct_sum.c (the definition,
PAPER.md:371 Eq. (32) with Eq. (18),(20),(21)) and oracle/bltc_cpu.c (Algorithm 3,
PAPER.md:437-462, step by step).

NEXT-1: oracle/coulomb_sum.c is the Hartree-potential direct sum with the Gaussian
singularity subtraction (Eq. (19),(23),(24)) and oracle_bltc_eval_coulomb in
oracle/bltc_cpu.c evaluates it through the same treecode; pinned by tests/test_oracle_pins_coulomb.py.

Pinned by tests/test_oracle_pins.py (closed forms, invariants, limits); nothing here is
"parity unpinned" except the two items DESIGN.md lists (BLTC error magnitude at theta=0.7,
n=8 for the Yukawa kernel; numerical values on molecules -- the paper prints neither).
"""
from .cpu_oracle import (build, direct, coulomb_direct, OraclePlan, kernel_value, n_threads)  # noqa: F401
