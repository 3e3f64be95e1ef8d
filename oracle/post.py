"""Oracle of the host post-processing step (test infrastructure only): compliance contribution tensor, Eq. 23 of
the paper: S* = S1 + phi H with S = C^-1, written out with numpy's inverse."""
import numpy as np


def contribution_tensor(C_eff, C_matrix, phi):
    return (np.linalg.inv(np.asarray(C_eff, dtype=np.float64)) - np.linalg.inv(np.asarray(C_matrix, dtype=np.float64))) / phi
