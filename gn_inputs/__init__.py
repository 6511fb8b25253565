"""Seeded synthetic inputs (geometry, graph, fp32 weights, classes, parameter tables).

Inputs only: nothing here computes a delay, quantises a weight, steps a vertex or draws the
method's drive/noise numbers.  The oracle (``oracle/``) and the CUDA library
(``paper_0908_3934_b200/``) both consume what this package returns and never import each other.
"""
from .generate import build_lib, geometric_network, Network  # noqa: F401
from .configs import make_config, hh_class, as_hodgkin_huxley, CONFIG_NAMES, MASTER_SEED  # noqa: F401
from . import paper_test_set  # noqa: F401  (the paper's 80-network test set, regenerated: PAPER.md:388-450)
