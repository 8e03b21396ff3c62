"""CPU oracle of the TPC sector track finder - TEST INFRASTRUCTURE, not the product.

Import only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs.
"""
from .oracle import Oracle, build_oracle, oracle_lib_path  # noqa: F401
