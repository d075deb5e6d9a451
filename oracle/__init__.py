"""CPU oracle for the GENE ExB nonlinearity -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_1310_1485_b200 (the CUDA path) and neither
imports the other.  See oracle/gene_nl_oracle.c for what is computed and the citations.
"""
from .gene_nl_oracle import (  # noqa: F401
    DFT_NAIVE,
    DFT_RECURSIVE,
    build,
    dft,
    nl_convolution_modes,
    nl_convolution_plane,
    nl_pseudospectral,
    nlx_convolution_plane,
    nlx_pseudospectral,
    num_threads,
)
