"""Packed form of the oracle's Jacobian (TEST INFRASTRUCTURE ONLY; see oracle/__init__.py).

The packed Jacobian of include/tfa.h (second option) is a re-arrangement of the BSR values, not new
arithmetic: the diagonal blocks in an array of their own, and of every off-diagonal block only the entries the flux
Jacobian can fill -- fields 8x8, ions 5x5, electrons 5x5, each row-major, in that order (114 of 324).  This module
writes that arrangement out from the oracle's BSR output, calling nothing but numpy, and insists that what it drops
is exactly 0.0 (pinned separately: tests/test_oracle_assembly.py::test_flux_jacobian_block_structure).
"""
import numpy as np

NEQ = 18
FIELDS = list(range(8))
IONS = [8, 10, 11, 12, 16]          # rho_i, u_i (3), T_i
ELECTRONS = [9, 13, 14, 15, 17]     # rho_e, u_e (3), T_e
GROUPS = (FIELDS, IONS, ELECTRONS)
PACKED_BLOCK = sum(len(g) ** 2 for g in GROUPS)   # 114


def pack_bsr(vals, rowptr, col):
    """vals [nnzb][18][18] in the pattern (rowptr, col) -> (diag [n][18][18], offd [nnzb - n][114])."""
    vals = np.asarray(vals)
    n = len(rowptr) - 1
    rows = np.repeat(np.arange(n), np.diff(rowptr))
    is_diag = rows == np.asarray(col)
    assert is_diag.sum() == n, "every row has exactly one diagonal block"
    diag = vals[is_diag].copy()
    off = vals[~is_diag]                          # BSR order with the diagonal blocks taken out
    keep = np.zeros((NEQ, NEQ), dtype=bool)
    parts = []
    for g in GROUPS:
        keep[np.ix_(g, g)] = True
        parts.append(off[:, g][:, :, g].reshape(len(off), -1))
    assert not off[:, ~keep].any(), "an off-diagonal block has a non-zero outside the 8x8 + 5x5 + 5x5 pattern"
    return diag, np.concatenate(parts, axis=1)


def unpack_bsr(diag, offd, rowptr, col):
    """The inverse arrangement: (diag, offd) -> vals [nnzb][18][18]."""
    n = len(rowptr) - 1
    rows = np.repeat(np.arange(n), np.diff(rowptr))
    is_diag = rows == np.asarray(col)
    vals = np.zeros((len(col), NEQ, NEQ))
    vals[is_diag] = diag
    off = np.zeros((len(offd), NEQ, NEQ))
    p = 0
    for g in GROUPS:
        k = len(g)
        blk = offd[:, p:p + k * k].reshape(-1, k, k)
        for a, ra in enumerate(g):
            off[:, ra, g] = blk[:, a, :]
        p += k * k
    vals[~is_diag] = off
    return vals
