"""fp64 CPU oracle for MSA -- test infrastructure only (see msa_oracle.c header)."""
from .msa_oracle import build, e4m3_to_double, forward, forward_problem, num_threads  # noqa: F401
