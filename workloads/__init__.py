"""Seeded synthetic inputs shared by the oracle's tests and the CUDA path's tests (data only)."""
from .synthetic import (MAT_H, MAT_S, System, gamma_table, hash_uniform_np, hash_uniform_torch,
                        make_system, to_scipy)

__all__ = ["MAT_H", "MAT_S", "System", "gamma_table", "hash_uniform_np", "hash_uniform_torch",
           "make_system", "to_scipy"]
