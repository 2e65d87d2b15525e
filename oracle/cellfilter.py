"""Cell filter of CFNEB -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Follows PAPER.md "Cell Filter", Eq. 10-17, in the paper's notation:
row-vector convention, h rows = lattice vectors, D = h0^-1 h,
R~ = s h0 = R D^-1 (Eq. 10), B = D D^T (Eq. 15).  Readings: SURVEY.md A7-A9, A13.
"""
import numpy as np

CELL_FIXED = 0
CELL_B = 1  # Eq. 17, rotation-free (default)
CELL_D = 2  # Eq. 14


def input_mapping(R, h, h0):
    """O0 (Eq. 10, 15): D = h0^-1 h; B = D D^T; R~ = R D^-1.  Returns (R~, B, D)."""
    D = np.linalg.solve(h0, h)  # h0^-1 h
    B = D @ D.T
    Rt = R @ np.linalg.inv(D)
    return Rt, B, D


def cell_map(B):
    """O1 (reading A8): D := sqrt(B), the unique symmetric positive-definite root.

    B = D D^T is invariant under h -> h Q; taking the symmetric root drops the rotation.
    """
    w, U = np.linalg.eigh(0.5 * (B + B.T))
    if not np.all(w > 0.0):
        raise ValueError("B is not positive definite")
    return (U * np.sqrt(w)) @ U.T


def generalized_force(F, V, D, lam=1.0, cell_mode=CELL_B):
    """O4: generalized force conjugate to (R~, lam*B) -- Eq. 17, as printed (A9: no 1/2).

    atoms: F D^T (Eq. 12);  cell: D^-T V D^-1 / lam (Eq. 16-17), or D^-T V / lam for
    CELL_D (Eq. 13-14), or 0 for CELL_FIXED.  Returns (N+3, 3).
    """
    G_atoms = F @ D.T
    Dinv = np.linalg.inv(D)
    if cell_mode == CELL_B:
        G_cell = Dinv.T @ V @ Dinv / lam
    elif cell_mode == CELL_D:
        G_cell = Dinv.T @ V / lam
    else:
        G_cell = np.zeros((3, 3))
    return np.vstack([G_atoms, G_cell])


def pack(Rt, C, lam=1.0):
    """Generalized coordinate X = [R~ ; lam*C], (N+3) x 3 (Eq. 11 / Eq. 17; A13). C = B or D."""
    return np.vstack([Rt, lam * C])


def unpack(X, lam=1.0):
    """Inverse of pack: (R~, C)."""
    return X[:-3], X[-3:] / lam
