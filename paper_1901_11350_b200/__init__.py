"""B200-native LLG hot path of arXiv 1901.11350 (Spirit): C-ABI CUDA library + thin Python binding.

    from paper_1901_11350_b200 import SpinSystem
    s = SpinSystem(bravais, basis, n_cells, periodic); s.hamiltonian_set_pairs(...); s.llg_iterate(1000)

The package never imports `oracle` (the CPU checker) and has no CPU fallback.
"""
from .binding import EXPORTS, SpinError, SpinSystem, lib, spin_ipc_close, spin_ipc_export, spin_ipc_open, spin_jit_compiler_info, version

__all__ = ["SpinSystem", "SpinError", "lib", "version", "spin_jit_compiler_info", "EXPORTS", "spin_ipc_export", "spin_ipc_open", "spin_ipc_close"]
