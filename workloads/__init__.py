"""Seeded synthetic input generators (spaces, constraint programs, objective tables).

This package is the ONLY code shared between the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_28372_b200/``).  It holds none of the method's arithmetic: no enumeration, no
validity test, no repair, no operator, no RNG used by the method.  It only *describes* inputs:
parameter domains, constraint programs (as postfix int32 words, the input format declared in
``include/cao.h``), hand-written Python predicates of the same constraints (used by the tests'
brute-force reference), and a seeded objective table built from a valid-row table handed in by
the caller.
"""
from .rpn import P, C, Expr, MIN, MAX, AND, OR, NOT, OPCODES  # noqa: F401
from .spaces import Space, Workload, space_cfg0, space_cfg1, space_cfg2, space_cfg3, \
    random_tiny_space, WORKLOADS, CFG3_SEED0_TABLE, splitmix64_stream  # noqa: F401
from .objective import objective_table, test_objective_37  # noqa: F401
