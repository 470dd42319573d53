"""ctypes binding of oracle/tfo.cpp (TEST INFRASTRUCTURE ONLY; see oracle/tfo.h)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# TFO_SANITIZE=1: an AddressSanitizer + UndefinedBehaviorSanitizer build of the oracle; run the
# CPU tests with  LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 TFO_SANITIZE=1
_SANITIZE = os.environ.get("TFO_SANITIZE", "0") == "1"
_SO = os.path.join(_HERE, "liboracle_tfo_san.so" if _SANITIZE else "liboracle_tfo.so")
NEQ = 18


class PhysicsC(C.Structure):
    _fields_ = [("gamma_gas", C.c_double), ("mass_ratio", C.c_double), ("c", C.c_double),
                ("gamma_psi", C.c_double), ("chi_phi", C.c_double), ("rusanov_alpha", C.c_double)]


class Numerics(C.Structure):
    _fields_ = [("fd_delta", C.c_double), ("fd_ref", C.c_double * NEQ), ("venkat_K", C.c_double),
                ("lsq_weight_power", C.c_double), ("ausm_Kp", C.c_double), ("ausm_Ku", C.c_double),
                ("ausm_sigma", C.c_double), ("ausm_beta", C.c_double), ("ausm_Minf", C.c_double * 2),
                ("term_mask", C.c_int32), ("pad_", C.c_int32)]


MESH_ITEMS = dict(face_cells=(0, np.int32), cell_faces=(1, np.int32), stencil_ptr=(2, np.int32),
                  stencil_idx=(3, np.int32), bsr_rowptr=(4, np.int32), bsr_col=(5, np.int32),
                  perm=(6, np.int32), volume=(7, np.float64), face_normal_len=(8, np.float64),
                  centroid=(9, np.float64), face_nodes=(10, np.int32), bfaces=(12, np.int32),
                  bc_tags=(13, np.int32))
BC_TRANSMISSIVE, BC_GHOST, BC_WALL = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain -O2, no fast-math, no FMA contraction)."""
    src = os.path.join(_HERE, "tfo.cpp")
    hdr = os.path.join(_HERE, "tfo.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC",
           "-shared", "-Wall", "-o", _SO, src]
    if _SANITIZE:
        cmd[3:3] = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_void_p
        L.tfo_last_error.restype = C.c_char_p
        L.tfo_mesh_create.argtypes = [C.POINTER(vp), C.c_int64, vp, C.c_int64, vp, vp]
        L.tfo_mesh_create_poly.argtypes = [C.POINTER(vp), C.c_int64, vp, C.c_int64, vp, vp, vp]
        L.tfo_mesh_info.argtypes = [vp, C.POINTER(C.c_int32), C.POINTER(C.c_int64)]
        L.tfo_mesh_set_bc.argtypes = [vp, vp, vp]
        L.tfo_wall_ghost.argtypes = [vp, C.c_double, C.c_double, vp]
        L.tfo_wall_ghost.restype = None
        L.tfo_mesh_reorder.argtypes = [vp, C.c_int, vp]
        L.tfo_mesh_sizes.argtypes = [vp] + [C.POINTER(C.c_int64)] * 4
        L.tfo_mesh_get.argtypes = [vp, C.c_int, vp, C.c_int64]
        L.tfo_mesh_destroy.argtypes = [vp]
        L.tfo_mesh_destroy.restype = None
        L.tfo_default_physics.argtypes = [C.POINTER(PhysicsC)]
        L.tfo_default_numerics.argtypes = [C.POINTER(Numerics), C.POINTER(PhysicsC)]
        L.tfo_gradients.argtypes = [vp, C.POINTER(Numerics), vp, vp, vp]
        L.tfo_assemble.argtypes = [vp, C.POINTER(PhysicsC), C.POINTER(Numerics), vp, vp, vp, C.c_double,
                                   vp, vp, vp, C.c_int64, vp]
        L.tfo_residual_frozen.argtypes = [vp, C.POINTER(PhysicsC), C.POINTER(Numerics), vp, vp, vp, vp, vp,
                                          C.c_double, vp]
        L.tfo_flux_maxwell.argtypes = [C.POINTER(PhysicsC), vp, vp, C.c_double, C.c_double, vp]
        L.tfo_flux_ausm.argtypes = [C.POINTER(PhysicsC), C.POINTER(Numerics), C.c_int, vp, vp, C.c_double,
                                    C.c_double, vp]
        L.tfo_flux_face.argtypes = [C.POINTER(PhysicsC), C.POINTER(Numerics), vp, vp, C.c_double, C.c_double, vp]
        L.tfo_phys_flux.argtypes = [C.POINTER(PhysicsC), vp, C.c_double, C.c_double, vp]
        L.tfo_source.argtypes = [C.POINTER(PhysicsC), vp, vp]
        L.tfo_cons.argtypes = [C.POINTER(PhysicsC), vp, vp]
        L.tfo_dcons_dprim.argtypes = [C.POINTER(PhysicsC), vp, vp]
        L.tfo_num_threads.restype = C.c_int
        L.tfo_ausm_split.argtypes = [C.c_double, C.c_double, C.c_double, vp]
        L.tfo_ausm_split.restype = None
        _ = dp, ip
        _lib = L
    return _lib


def _chk(rc: int):
    if rc != 0:
        raise RuntimeError(f"oracle error {rc}: {lib().tfo_last_error().decode()}")


def _p(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def physics_c(ph=None) -> PhysicsC:
    """PhysicsC from any object with the six attribute names (e.g. workloads.Physics) or defaults."""
    p = PhysicsC()
    lib().tfo_default_physics(C.byref(p))
    if ph is not None:
        for name, _ in PhysicsC._fields_:
            setattr(p, name, float(getattr(ph, name)))
    return p


def default_numerics(ph: PhysicsC | None = None, **over) -> Numerics:
    ph = ph or physics_c()
    n = Numerics()
    lib().tfo_default_numerics(C.byref(n), C.byref(ph))
    for k, v in over.items():
        if k in ("fd_ref", "ausm_Minf"):
            arr = getattr(n, k)
            for i, x in enumerate(v):
                arr[i] = float(x)
        else:
            setattr(n, k, v)
    return n


def num_threads() -> int:
    return int(lib().tfo_num_threads())


def set_num_threads(n: int):
    lib().tfo_set_num_threads(C.c_int(int(n)))


class OracleMesh:
    def __init__(self, node_xy, cell_nodes, cell_xy=None, cell_ptr=None):
        """Triangles: cell_nodes [nc][3].  Mixed triangles / quadrilaterals: cell_ptr [nc+1] and flat cell_nodes,
        cell_xy [cell_ptr[nc]][2]."""
        self._h = C.c_void_p()
        node_xy = _f64(node_xy)
        cell_nodes = np.ascontiguousarray(cell_nodes, dtype=np.int32)
        cxy = None if cell_xy is None else _f64(cell_xy)
        if cell_ptr is None:
            _chk(lib().tfo_mesh_create(C.byref(self._h), node_xy.shape[0], _p(node_xy), cell_nodes.shape[0],
                                       _p(cell_nodes), _p(cxy)))
        else:
            cp = np.ascontiguousarray(cell_ptr, dtype=np.int32)
            _chk(lib().tfo_mesh_create_poly(C.byref(self._h), node_xy.shape[0], _p(node_xy), cp.shape[0] - 1,
                                            _p(cp), _p(cell_nodes), _p(cxy)))
        self._sizes()

    @classmethod
    def from_input(cls, mi) -> "OracleMesh":
        return cls(mi.node_xy, mi.cell_nodes, mi.cell_xy, getattr(mi, "cell_ptr", None))

    def _sizes(self):
        v = [C.c_int64() for _ in range(4)]
        _chk(lib().tfo_mesh_sizes(self._h, *[C.byref(x) for x in v]))
        self.n_cells, self.n_faces, self.nnzb, self.n_stencil = [int(x.value) for x in v]
        mf, nb = C.c_int32(), C.c_int64()
        _chk(lib().tfo_mesh_info(self._h, C.byref(mf), C.byref(nb)))
        self.max_faces, self.n_bfaces = int(mf.value), int(nb.value)

    def set_bc(self, tags, ghost=None):
        """tags [n_bfaces] in the order of get("bfaces"); ghost [n_bfaces][18] for the BC_GHOST faces."""
        tags = np.ascontiguousarray(tags, dtype=np.int32)
        assert tags.shape == (self.n_bfaces,)
        gh = None if ghost is None else _f64(ghost)
        assert gh is None or gh.shape == (self.n_bfaces, NEQ)
        _chk(lib().tfo_mesh_set_bc(self._h, _p(tags), _p(gh)))

    def reorder(self, kind: str = "rcm", perm=None):
        k = {"none": 0, "rcm": 1, "user": 2}[kind]
        pp = None if perm is None else np.ascontiguousarray(perm, dtype=np.int32)
        _chk(lib().tfo_mesh_reorder(self._h, k, _p(pp)))
        self._sizes()

    def get(self, name: str) -> np.ndarray:
        which, dt = MESH_ITEMS[name]
        n = dict(face_cells=2 * self.n_faces, face_nodes=2 * self.n_faces, cell_faces=self.max_faces * self.n_cells,
                 stencil_ptr=self.n_cells + 1, stencil_idx=self.n_stencil, bsr_rowptr=self.n_cells + 1,
                 bsr_col=self.nnzb, perm=self.n_cells, volume=self.n_cells, face_normal_len=3 * self.n_faces,
                 centroid=2 * self.n_cells, bfaces=self.n_bfaces, bc_tags=self.n_bfaces)[name]
        out = np.empty(n, dtype=dt)
        _chk(lib().tfo_mesh_get(self._h, which, _p(out), out.nbytes))
        shape = dict(face_cells=(-1, 2), face_nodes=(-1, 2), cell_faces=(-1, self.max_faces),
                     face_normal_len=(-1, 3), centroid=(-1, 2)).get(name)
        return out.reshape(shape) if shape else out

    def close(self):
        if self._h:
            lib().tfo_mesh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def gradients(mesh: OracleMesh, nu: Numerics, state):
    state = _f64(state)
    grad = np.empty((mesh.n_cells, NEQ, 2))
    phi = np.empty((mesh.n_cells, NEQ))
    _chk(lib().tfo_gradients(mesh._h, C.byref(nu), _p(state), _p(grad), _p(phi)))
    return grad, phi


def assemble(mesh: OracleMesh, ph: PhysicsC, nu: Numerics, state, state_n=None, state_nm1=None, dt=1e-3,
             rows=None, jacobian=True):
    """Returns (rhs, scale, vals).  rows=None: vals[nnzb][18][18]; else compact, zero-padded
    vals[n_rows][max_faces + 1][18][18]."""
    state = _f64(state)
    state_n = state if state_n is None else _f64(state_n)
    state_nm1 = state if state_nm1 is None else _f64(state_nm1)
    if rows is None:
        n = mesh.n_cells
        vals = np.empty((mesh.nnzb, NEQ, NEQ)) if jacobian else None
        rr, nr = None, 0
    else:
        rr = np.ascontiguousarray(rows, dtype=np.int32)
        n = nr = rr.shape[0]
        vals = np.empty((n, mesh.max_faces + 1, NEQ, NEQ)) if jacobian else None
    rhs = np.empty((n, NEQ))
    scale = np.empty((n, NEQ))
    _chk(lib().tfo_assemble(mesh._h, C.byref(ph), C.byref(nu), _p(state), _p(state_n), _p(state_nm1),
                            float(dt), _p(rhs), _p(scale), _p(vals), nr, _p(rr)))
    return rhs, scale, vals


def residual_frozen(mesh, ph, nu, state, grad, phi, state_n=None, state_nm1=None, dt=1e-3):
    state = _f64(state)
    state_n = state if state_n is None else _f64(state_n)
    state_nm1 = state if state_nm1 is None else _f64(state_nm1)
    grad, phi = _f64(grad), _f64(phi)
    rhs = np.empty((mesh.n_cells, NEQ))
    _chk(lib().tfo_residual_frozen(mesh._h, C.byref(ph), C.byref(nu), _p(state), _p(grad), _p(phi),
                                   _p(state_n), _p(state_nm1), float(dt), _p(rhs)))
    return rhs


def flux_maxwell(ph, UL, UR, nx, ny):
    UL, UR = _f64(UL), _f64(UR)
    H = np.empty(8)
    lib().tfo_flux_maxwell(C.byref(ph), _p(UL), _p(UR), nx, ny, _p(H))
    return H


def flux_ausm(ph, nu, s, PL, PR, nx, ny):
    PL, PR = _f64(PL), _f64(PR)
    H = np.empty(5)
    lib().tfo_flux_ausm(C.byref(ph), C.byref(nu), int(s), _p(PL), _p(PR), nx, ny, _p(H))
    return H


def flux_face(ph, nu, PL, PR, nx, ny):
    PL, PR = _f64(PL), _f64(PR)
    H = np.empty(NEQ)
    lib().tfo_flux_face(C.byref(ph), C.byref(nu), _p(PL), _p(PR), nx, ny, _p(H))
    return H


def phys_flux(ph, P, nx, ny):
    P = _f64(P)
    F = np.empty(NEQ)
    lib().tfo_phys_flux(C.byref(ph), _p(P), nx, ny, _p(F))
    return F


def wall_ghost(P, nx, ny):
    P = _f64(P)
    G = np.empty(NEQ)
    lib().tfo_wall_ghost(_p(P), float(nx), float(ny), _p(G))
    return G


def source(ph, P):
    P = _f64(P)
    S = np.empty(NEQ)
    lib().tfo_source(C.byref(ph), _p(P), _p(S))
    return S


def cons(ph, P):
    P = _f64(P)
    U = np.empty(NEQ)
    lib().tfo_cons(C.byref(ph), _p(P), _p(U))
    return U


def dcons_dprim(ph, P):
    P = _f64(P)
    D = np.empty((NEQ, NEQ))
    lib().tfo_dcons_dprim(C.byref(ph), _p(P), _p(D))
    return D


def ausm_split(M, alpha=3.0 / 16.0, beta=0.125):
    out = np.empty(4)
    lib().tfo_ausm_split(float(M), float(alpha), float(beta), _p(out))
    return out
