"""ORACLE -- test infrastructure only (see iris_oracle.cpp header).

ctypes wrapper around the float64 scalar C++ oracle.  Imports nothing from the CUDA package.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
"""
from .wrapper import Oracle, build_oracle, oracle_lib_path

__all__ = ["Oracle", "build_oracle", "oracle_lib_path"]
