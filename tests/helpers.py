"""Test-side helpers: golden-file reader, brute-force connectivity, tolerance checkers."""
import os
import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden_sections(name):
    out, cur = {}, None
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if not line:
                continue
            if line.startswith("["):
                cur = line.strip("[]")
                out[cur] = []
            else:
                out[cur].append([float(x) if ("." in x or "e" in x) else int(x) for x in line.split()])
    return out


def brute_connectivity(cell_nodes):
    """O(n^2)-style set arithmetic, independent of the sort-based builders.

    Returns faces (sorted (lo,hi) -> [cells]), face-neighbour sets, vertex-neighbour sets.
    """
    nc = len(cell_nodes)
    edge_cells = {}
    for c in range(nc):
        a = [int(x) for x in cell_nodes[c]]
        for k in range(3):
            key = (min(a[k], a[(k + 1) % 3]), max(a[k], a[(k + 1) % 3]))
            edge_cells.setdefault(key, []).append(c)
    faces = sorted(edge_cells.items())
    node_cells = {}
    for c in range(nc):
        for v in cell_nodes[c]:
            node_cells.setdefault(int(v), set()).add(c)
    vert_nb = [sorted(set().union(*[node_cells[int(v)] for v in cell_nodes[c]]) - {c}) for c in range(nc)]
    face_nb = [set() for _ in range(nc)]
    for _, cs in faces:
        if len(cs) == 2:
            face_nb[cs[0]].add(cs[1])
            face_nb[cs[1]].add(cs[0])
    return faces, face_nb, vert_nb


def check_connectivity_against_brute(mesh_get, sizes, cell_nodes):
    """mesh_get(name)->array, sizes=(nc,nf,nnzb,nst).  Bit-exact comparison with brute force."""
    nc, nf, nnzb, nst = sizes
    faces, face_nb, vert_nb = brute_connectivity(cell_nodes)
    assert nf == len(faces)
    fc = mesh_get("face_cells")
    exp_fc = np.array([[min(cs), max(cs) if len(cs) == 2 else -1] for _, cs in faces], dtype=np.int32)
    np.testing.assert_array_equal(fc, exp_fc)
    cf = mesh_get("cell_faces")
    key_to_face = {k: i for i, (k, _) in enumerate(faces)}
    for c in range(nc):
        a = [int(x) for x in cell_nodes[c]]
        for k in range(3):
            key = (min(a[k], a[(k + 1) % 3]), max(a[k], a[(k + 1) % 3]))
            assert cf[c, k] == key_to_face[key]
    sp, si = mesh_get("stencil_ptr"), mesh_get("stencil_idx")
    assert sp[0] == 0 and sp[-1] == nst == sum(len(v) for v in vert_nb)
    for c in range(nc):
        assert list(si[sp[c]:sp[c + 1]]) == vert_nb[c]
    rp, col = mesh_get("bsr_rowptr"), mesh_get("bsr_col")
    assert rp[0] == 0 and rp[-1] == nnzb
    for c in range(nc):
        assert list(col[rp[c]:rp[c + 1]]) == sorted(face_nb[c] | {c})


def rcm_reference(rowptr, col):
    """Serial reverse Cuthill-McKee per DESIGN.md S11, written independently in Python."""
    n = len(rowptr) - 1
    nbrs = [[int(j) for j in col[rowptr[i]:rowptr[i + 1]] if j != i] for i in range(n)]
    deg = [len(x) for x in nbrs]
    seen = [False] * n
    order = []
    while len(order) < n:
        start = min((i for i in range(n) if not seen[i]), key=lambda i: (deg[i], i))
        seen[start] = True
        order.append(start)
        head = len(order) - 1
        while head < len(order):
            v = order[head]
            head += 1
            for w in sorted((w for w in nbrs[v] if not seen[w]), key=lambda w: (deg[w], w)):
                seen[w] = True
                order.append(w)
    return np.array(order[::-1], dtype=np.int32)


def bandwidth(rowptr, col):
    rows = np.repeat(np.arange(len(rowptr) - 1), np.diff(rowptr))
    return int(np.abs(rows - col).max())


# ---- tolerances of BASELINE.json north_star, as read in DESIGN.md (S18) ----
RES_TOL = 1e-12   # relative to the per-variable max of the oracle's sum-of-|terms| scale
JAC_TOL = 1e-8    # relative to the row-maximum magnitude of the oracle's Jacobian row


def residual_error(rhs, rhs_ref, scale_ref):
    """max over variables of  max_i |rhs - ref| / max_i scale  (S18)."""
    num = np.abs(rhs - rhs_ref).max(axis=0)
    den = scale_ref.max(axis=0)
    den = np.where(den > 0, den, 1.0)
    return float((num / den).max())


def jacobian_error_rows(vals_rows, ref_rows):
    """vals_rows, ref_rows: [n_rows][nblk][18][18].  Error relative to each scalar row's max |entry|."""
    diff = np.abs(vals_rows - ref_rows).max(axis=(1, 3))         # [n_rows][18]
    rowmax = np.abs(ref_rows).max(axis=(1, 3))
    rowmax = np.where(rowmax > 0, rowmax, 1.0)
    return float((diff / rowmax).max())


def bsr_to_rows(vals, rowptr, rows=None):
    """[nnzb][18][18] -> zero-padded [n_rows][4][18][18] (blocks in BSR order)."""
    n = len(rowptr) - 1
    rows = np.arange(n) if rows is None else np.asarray(rows)
    out = np.zeros((len(rows), 4, 18, 18))
    for q, i in enumerate(rows):
        b, e = rowptr[i], rowptr[i + 1]
        out[q, :e - b] = vals[b:e]
    return out


def bsr_to_dense(vals, rowptr, col):
    n = len(rowptr) - 1
    A = np.zeros((n * 18, n * 18))
    for i in range(n):
        for q in range(rowptr[i], rowptr[i + 1]):
            j = col[q]
            A[18 * i:18 * i + 18, 18 * j:18 * j + 18] = vals[q]
    return A
