"""CPU oracle (test infrastructure only -- see oracle/qmmm_oracle.c).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this.
"""
from .qmmm_oracle import build, field, potential_terms, OracleResult  # noqa: F401
