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


def cells_as_lists(cell_nodes, cell_ptr=None):
    """Corner lists of every cell: [nc][3] array, or flat array + CSR pointer for mixed meshes."""
    if cell_ptr is None:
        return [[int(x) for x in row] for row in cell_nodes]
    return [[int(x) for x in cell_nodes[cell_ptr[c]:cell_ptr[c + 1]]] for c in range(len(cell_ptr) - 1)]


def brute_connectivity(cell_nodes, cell_ptr=None):
    """O(n^2)-style set arithmetic, independent of the sort-based builders.

    Returns faces (sorted (lo,hi) -> [cells]), face-neighbour sets, vertex-neighbour sets.
    """
    cells = cells_as_lists(cell_nodes, cell_ptr)
    nc = len(cells)
    edge_cells = {}
    for c, a in enumerate(cells):
        for k in range(len(a)):
            key = (min(a[k], a[(k + 1) % len(a)]), max(a[k], a[(k + 1) % len(a)]))
            edge_cells.setdefault(key, []).append(c)
    faces = sorted(edge_cells.items())
    node_cells = {}
    for c, a in enumerate(cells):
        for v in a:
            node_cells.setdefault(v, set()).add(c)
    vert_nb = [sorted(set().union(*[node_cells[v] for v in cells[c]]) - {c}) for c in range(nc)]
    face_nb = [set() for _ in range(nc)]
    for _, cs in faces:
        if len(cs) == 2:
            face_nb[cs[0]].add(cs[1])
            face_nb[cs[1]].add(cs[0])
    return faces, face_nb, vert_nb


def check_connectivity_against_brute(mesh_get, sizes, cell_nodes, cell_ptr=None):
    """mesh_get(name)->array, sizes=(nc,nf,nnzb,nst).  Bit-exact comparison with brute force."""
    nc, nf, nnzb, nst = sizes
    cells = cells_as_lists(cell_nodes, cell_ptr)
    faces, face_nb, vert_nb = brute_connectivity(cell_nodes, cell_ptr)
    assert nf == len(faces)
    fc = mesh_get("face_cells")
    exp_fc = np.array([[min(cs), max(cs) if len(cs) == 2 else -1] for _, cs in faces], dtype=np.int32)
    np.testing.assert_array_equal(fc, exp_fc)
    cf = mesh_get("cell_faces")
    assert cf.shape == (nc, max(len(a) for a in cells))
    key_to_face = {k: i for i, (k, _) in enumerate(faces)}
    for c, a in enumerate(cells):
        for k in range(len(a)):
            key = (min(a[k], a[(k + 1) % len(a)]), max(a[k], a[(k + 1) % len(a)]))
            assert cf[c, k] == key_to_face[key]
        assert (cf[c, len(a):] == -1).all()
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


def jacobian_error_blocks(vals, ref, rowptr):
    """vals, ref: [nnzb][18][18] in the same BSR pattern.  Same measure as jacobian_error_rows (error relative to
    the scalar row's largest |entry| over all blocks of the BSR row), vectorised for large meshes."""
    n = len(rowptr) - 1
    rows = np.repeat(np.arange(n), np.diff(rowptr))
    diff = np.zeros((n, 18))
    rowmax = np.zeros((n, 18))
    np.maximum.at(diff, rows, np.abs(vals - ref).max(axis=2))
    np.maximum.at(rowmax, rows, np.abs(ref).max(axis=2))
    return float((diff / np.where(rowmax > 0, rowmax, 1.0)).max())


def jacobian_error_padded(vals, ref_rows, rowptr):
    """vals: [nblk][18][18], the blocks of consecutive BSR rows (rowptr relative to the first of them);
    ref_rows: the oracle's zero-padded [n_rows][B][18][18] for the same rows."""
    n = len(rowptr) - 1
    cnt = np.diff(rowptr)
    rows = np.repeat(np.arange(n), cnt)
    slot = np.arange(len(rows)) - np.repeat(rowptr[:-1], cnt)
    ref = ref_rows[rows, slot]
    assert not ref_rows[np.arange(ref_rows.shape[1])[None, :] >= cnt[:, None]].any(), "padding blocks must be zero"
    return jacobian_error_blocks(vals, ref, rowptr)


def bsr_to_rows(vals, rowptr, rows=None, width=None):
    """[nnzb][18][18] -> zero-padded [n_rows][width][18][18] (blocks in BSR order; width = the longest row)."""
    n = len(rowptr) - 1
    rows = np.arange(n) if rows is None else np.asarray(rows)
    width = max(4, int(np.diff(rowptr).max())) if width is None else width
    out = np.zeros((len(rows), width, 18, 18))
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
