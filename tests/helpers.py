"""Test helpers: build oracle operators from a workload dict (tests may import oracle/)."""
import numpy as np

from oracle import chfsi_oracle as orc


def oracle_ops(prob):
    """(A, B, Dinv) oracle operator objects for a workload dict."""
    return orc.operators_from_workload(prob)


def rel_fro(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def small_dense_generalized(m, seed):
    """Small SPD-B generalized dense problem with a diagonal approximate inverse."""
    rng = np.random.default_rng(seed)
    F = rng.standard_normal((m, m))
    A = (F + F.T) / np.sqrt(2.0 * m) + np.diag(np.linspace(0.0, 10.0, m))
    F = rng.standard_normal((m, m))
    B = np.eye(m) + 0.1 * (F + F.T) / np.sqrt(2.0 * m)
    return dict(kind="dense", m=m, A=A, B=B, dinv=1.0 / np.diag(B).copy())
