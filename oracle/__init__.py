"""CPU oracle for the nao_* hot path -- TEST INFRASTRUCTURE ONLY (see nao_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
"""
from .oracle import (build_oracle_lib, geneig, geneig_lowdin, fermi, density, solve_problem,  # noqa: F401
                     cholesky, heev, energy_density, fold_density, geneig_lowdin_pruned)
