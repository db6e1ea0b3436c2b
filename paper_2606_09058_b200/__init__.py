"""B200-native (sm_100a) generalized eigensolver + Fermi level + density matrix for NAO-based DFT
(arxiv/paper_2606_09058 hot path).  See include/nao.h for the C-ABI and DESIGN.md for the design.

`paper_2606_09058_b200.synth` (input generator) is importable without CUDA; everything else needs libnao.so.
"""
from .binding import (NAO_REAL, NAO_COMPLEX, NAO_S_FACTORED, NAO_NC_BLOCK_S, NAO_TRD_ONE_STAGE,  # noqa: F401
                      NAO_TRD_TWO_STAGE, NAO_LOWDIN, NAO_PRUNED_LEVEL, NAO_STREAM_GROUPS_2, NAO_STREAM_GROUPS_4, NAO_STREAM_GROUPS_8, EXPORTS, NaoError, lib, geneig, geneig_workspace, fermi_mu, fermi_mu_static, FERMI_STATIC_MAX_STATES, density_matrix,
                      gemm, potrf_trtri, heev, stedc, occupied_count, scf_step, energy_weights, fold_density, set_lowdin_threshold, solve_host, dmma_peak, launch_count, version, profile_enable, profile_read, profile_kernel,
                      profile_kernel_launches)
