"""B200-native local-energy hot path of arxiv 2208.05637 (MADE neural quantum states for quantum chemistry).

Public API = thin binding over the C ABI in include/nqs.h:
    ham_compile / ham_compile_packed -> Hamiltonian
    made_create                      -> Made
    made_logpsi, pauli_contract, local_energy, local_energy_host, energy_grad, made_sample,
    weighted_stats_static (allocation-free statistics)
The CUDA library is loaded on first use and there is no CPU fallback.
"""
from .binding import (PATH_AUTO, PATH_SIMT, PATH_TC, NqsError, Hamiltonian, Made, ham_compile, ham_compile_text,
                      ham_compile_packed, made_create, made_logpsi, pauli_contract, local_energy,
                      local_energy_host, energy_grad, made_sample, kernel_launch_count, lib, LIB_PATH,
                      weighted_stats_static, STATS_STATIC_MAX_ROWS)

__all__ = ["PATH_AUTO", "PATH_SIMT", "PATH_TC", "NqsError", "Hamiltonian", "Made", "ham_compile", "ham_compile_text",
           "ham_compile_packed", "made_create", "made_logpsi", "pauli_contract", "local_energy",
           "local_energy_host", "energy_grad", "made_sample", "kernel_launch_count", "lib", "LIB_PATH",
           "weighted_stats_static", "STATS_STATIC_MAX_ROWS"]
