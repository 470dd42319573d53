"""CPU oracle of the linear-solve step (TEST INFRASTRUCTURE ONLY; see oracle/__init__.py).

Restarted GMRES with right preconditioning, written out step by step after the textbook algorithm (Saad,
"Iterative Methods for Sparse Linear Systems", Alg. 9.5 with the Givens-rotation least-squares update of
section 6.5.3), which is the method the paper names (restarted GMRES + Jacobi-type preconditioner, PAPER.md L28,
L392).  The sparse matrix-vector product and the small dense inverses are library primitives (scipy / numpy).

Pins (tests/test_solve.py, -m "not gpu"): on well-conditioned systems the result equals the direct sparse
solution (scipy `spsolve`) within the stopping tolerance; GMRES(n) without restart reaches the exact solution of
an n x n system in at most n iterations; the residual norms of the recurrence equal the true ones.
"""
import numpy as np
import scipy.sparse as sp

NEQ = 18


def bsr_matrix(vals, rowptr, col):
    n = len(rowptr) - 1
    return sp.bsr_matrix((np.asarray(vals), np.asarray(col), np.asarray(rowptr)), shape=(NEQ * n, NEQ * n))


def block_jacobi(vals, rowptr, col):
    """Inverses of the diagonal blocks, [n][18][18]."""
    n = len(rowptr) - 1
    out = np.empty((n, NEQ, NEQ))
    for i in range(n):
        b = rowptr[i] + int(np.nonzero(col[rowptr[i]:rowptr[i + 1]] == i)[0][0])
        out[i] = np.linalg.inv(vals[b])
    return out


def apply_block_diag(dinv, v):
    return np.einsum("irc,ic->ir", dinv, v.reshape(-1, NEQ)).ravel()


def gmres(A, b, x0=None, dinv=None, restart=30, max_iters=300, rtol=1e-8):
    """Solve A x = b: A M^-1 u = b, x = x0 + M^-1 u.  Returns (x, iterations, relative true residual,
    list of the recurrence's residual estimates)."""
    n = b.shape[0]
    x = np.zeros(n) if x0 is None else np.array(x0, dtype=np.float64)
    Minv = (lambda v: apply_block_diag(dinv, v)) if dinv is not None else (lambda v: v)
    bnorm = np.linalg.norm(b)
    if bnorm == 0.0:
        return np.zeros(n), 0, 0.0, []
    iters, est = 0, []
    while True:
        r = b - A @ x
        beta = np.linalg.norm(r)
        rel = beta / bnorm
        if rel <= rtol or iters >= max_iters:
            return x, iters, rel, est
        m = restart
        V = np.zeros((m + 1, n))
        H = np.zeros((m + 1, m))
        cs, sn, g = np.zeros(m), np.zeros(m), np.zeros(m + 1)
        V[0] = r / beta
        g[0] = beta
        k = 0
        while k < m and iters < max_iters:
            w = A @ Minv(V[k])
            for j in range(k + 1):               # modified Gram-Schmidt
                H[j, k] = V[j] @ w
                w = w - H[j, k] * V[j]
            H[k + 1, k] = np.linalg.norm(w)
            if H[k + 1, k] > 0.0:
                V[k + 1] = w / H[k + 1, k]
            for j in range(k):                   # previous rotations on the new column
                t = cs[j] * H[j, k] + sn[j] * H[j + 1, k]
                H[j + 1, k] = -sn[j] * H[j, k] + cs[j] * H[j + 1, k]
                H[j, k] = t
            den = np.hypot(H[k, k], H[k + 1, k])
            cs[k], sn[k] = (H[k, k] / den, H[k + 1, k] / den) if den > 0.0 else (1.0, 0.0)
            H[k, k], H[k + 1, k] = den, 0.0
            g[k + 1] = -sn[k] * g[k]
            g[k] = cs[k] * g[k]
            k += 1
            iters += 1
            est.append(abs(g[k]) / bnorm)
            if abs(g[k]) <= rtol * bnorm:
                break
        y = np.linalg.solve(np.triu(H[:k, :k]), g[:k]) if k > 0 else np.zeros(0)
        x = x + Minv(V[:k].T @ y)


def jvp(rhs_fn, P, v, eps):
    """Matrix-free Jacobian action ("Jacobian-free" variant): (R~(P + eps v) - R~(P)) / eps with
    rhs_fn(P) = -R~(P) the oracle's residual-only assembly (gradient and limiter recomputed, not frozen)."""
    return -(rhs_fn(P + eps * v) - rhs_fn(P)) / eps
