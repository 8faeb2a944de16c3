"""Seeded synthetic problem generators (inputs only).

This package produces the matrices, connectivities, diagonals and starting
blocks that BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2503_22652_b200/``) consume.  It holds none of the method's
arithmetic: no Chebyshev recurrence, no filter, no Rayleigh-Ritz.  Neither
``oracle/`` nor the CUDA package is imported from here.

Recipes follow BASELINE.json ``configs`` and SURVEY.md section 8(c)/(d)
(readings S14-S16); the paper's own controlled experiment family is
PAPER.md:269-285 (section 4.1.1).
"""
from .dense import (haar_orthogonal, config1_dense_standard, config2_dense_generalized,
                    e1_standard, e1_generalized)
from .laplacian import laplacian3d_csr, config3_sparse_laplacian, laplacian3d_exact_eigs
from .fe import (gll_nodes_weights, fe_reference_matrices, fe_problem, config4_fe, config5_fe)
from .noise import counter_gaussian


def start_block(m, block, seed):
    """Seeded Gaussian starting block X0 [m][block] (Algorithm 1 Step 0)."""
    import numpy as np
    return np.random.default_rng(seed).standard_normal((m, block))

__all__ = [
    "haar_orthogonal", "config1_dense_standard", "config2_dense_generalized",
    "e1_standard", "e1_generalized", "laplacian3d_csr", "config3_sparse_laplacian",
    "laplacian3d_exact_eigs", "gll_nodes_weights", "fe_reference_matrices", "fe_problem",
    "config4_fe", "config5_fe", "counter_gaussian", "start_block",
]
