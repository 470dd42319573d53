"""Thin Python binding of include/tfa.h — argument marshalling only.

Same names as the C entry points (``mesh_create``, ``mesh_reorder``, ``set_physics``,
``assemble``, ...).  PyTorch supplies device memory and the stream; every step of the path runs
in libtfa's CUDA kernels.
"""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import _lib
from ._lib import NEQ, BLOCK, Physics, Numerics, TfaError  # noqa: F401

MESH_ITEMS = dict(face_cells=(0, np.int32), cell_faces=(1, np.int32), stencil_ptr=(2, np.int32),
                  stencil_idx=(3, np.int32), bsr_rowptr=(4, np.int32), bsr_col=(5, np.int32),
                  perm=(6, np.int32), volume=(7, np.float64), face_normal_len=(8, np.float64),
                  centroid=(9, np.float64), face_nodes=(10, np.int32), cell_nbr=(11, np.int32),
                  bfaces=(12, np.int32), bc_tags=(13, np.int32))
_REORDER = {"none": 0, "rcm": 1, "user": 2, "morton": 3}
BC_TRANSMISSIVE, BC_GHOST, BC_WALL = 0, 1, 2
PACKED_BLOCK = 114
STATIC_MAX_STENCIL = 2097152   # tfa.h TFA_STATIC_MAX_STENCIL


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _hp(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t: torch.Tensor | None):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise ValueError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _fp(t: torch.Tensor | None):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise ValueError("expected a contiguous float32 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def default_physics(src=None) -> Physics:
    p = Physics()
    _lib.load().tfa_default_physics(C.byref(p))
    if src is not None:
        for name, _ in Physics._fields_:
            setattr(p, name, float(getattr(src, name)))
    return p


def default_numerics(ph: Physics | None = None, **over) -> Numerics:
    ph = ph or default_physics()
    n = Numerics()
    _lib.load().tfa_default_numerics(C.byref(n), C.byref(ph))
    for k, v in over.items():
        if k in ("fd_ref", "ausm_Minf"):
            arr = getattr(n, k)
            for i, x in enumerate(v):
                arr[i] = float(x)
        else:
            setattr(n, k, v)
    return n


class Mesh:
    """Owner of a ``tfa_mesh*`` (tfa_mesh_create / tfa_mesh_destroy)."""

    def __init__(self, node_xy, cell_nodes, cell_xy=None, cell_ptr=None):
        """Triangles: cell_nodes [nc][3] (tfa_mesh_create).  Mixed triangles / quadrilaterals: cell_ptr [nc+1] and
        flat cell_nodes, cell_xy [cell_ptr[nc]][2] (tfa_mesh_create_poly)."""
        lib = _lib.load()
        self._h = C.c_void_p()
        node_xy = np.ascontiguousarray(node_xy, dtype=np.float64)
        cell_nodes = np.ascontiguousarray(cell_nodes, dtype=np.int32)
        cxy = None if cell_xy is None else np.ascontiguousarray(cell_xy, dtype=np.float64)
        if cell_ptr is None:
            _lib.check(lib.tfa_mesh_create(C.byref(self._h), node_xy.shape[0], _hp(node_xy), cell_nodes.shape[0],
                                           _hp(cell_nodes), _hp(cxy), _stream()))
        else:
            cp = np.ascontiguousarray(cell_ptr, dtype=np.int32)
            _lib.check(lib.tfa_mesh_create_poly(C.byref(self._h), node_xy.shape[0], _hp(node_xy), cp.shape[0] - 1,
                                                _hp(cp), _hp(cell_nodes), _hp(cxy), _stream()))
        self._sizes()

    @classmethod
    def from_input(cls, mi) -> "Mesh":
        return cls(mi.node_xy, mi.cell_nodes, mi.cell_xy, getattr(mi, "cell_ptr", None))

    @classmethod
    def _borrowed(cls, handle, keep_alive) -> "Mesh":
        """View of a tfa_mesh* owned by another object (a Shard), which `keep_alive` keeps alive."""
        m = cls.__new__(cls)
        m._h = C.c_void_p(handle)
        m._owner = keep_alive
        m._sizes()
        return m

    def _sizes(self):
        v = [C.c_int64() for _ in range(4)]
        _lib.check(_lib.load().tfa_mesh_sizes(self._h, *[C.byref(x) for x in v]))
        self.n_cells, self.n_faces, self.nnzb, self.n_stencil = [int(x.value) for x in v]
        mf, nb = C.c_int32(), C.c_int64()
        _lib.check(_lib.load().tfa_mesh_info(self._h, C.byref(mf), C.byref(nb)))
        self.max_faces, self.n_bfaces = int(mf.value), int(nb.value)

    def set_bc(self, tags):
        """tfa_mesh_set_bc: tags [n_bfaces] (BC_*) in the order of get("bfaces")."""
        tags = np.ascontiguousarray(tags, dtype=np.int32)
        if tags.shape != (self.n_bfaces,):
            raise ValueError("one tag per boundary face")
        _lib.check(_lib.load().tfa_mesh_set_bc(self._h, _hp(tags), _stream()))

    def reorder(self, kind: str = "rcm", perm=None):
        pp = None if perm is None else np.ascontiguousarray(perm, dtype=np.int32)
        _lib.check(_lib.load().tfa_mesh_reorder(self._h, _REORDER[kind], _hp(pp), _stream()))
        self._sizes()

    def get(self, name: str) -> np.ndarray:
        which, dt = MESH_ITEMS[name]
        F = self.max_faces
        n = dict(face_cells=2 * self.n_faces, face_nodes=2 * self.n_faces, cell_faces=F * self.n_cells,
                 cell_nbr=F * self.n_cells, stencil_ptr=self.n_cells + 1, stencil_idx=self.n_stencil,
                 bsr_rowptr=self.n_cells + 1, bsr_col=self.nnzb, perm=self.n_cells, volume=self.n_cells,
                 face_normal_len=3 * self.n_faces, centroid=2 * self.n_cells, bfaces=self.n_bfaces,
                 bc_tags=self.n_bfaces)[name]
        out = np.empty(n, dtype=dt)
        _lib.check(_lib.load().tfa_mesh_get(self._h, which, _hp(out), out.nbytes))
        shape = dict(face_cells=(-1, 2), face_nodes=(-1, 2), cell_faces=(-1, F), cell_nbr=(-1, F),
                     face_normal_len=(-1, 3), centroid=(-1, 2)).get(name)
        return out.reshape(shape) if shape else out

    def device_ptr(self, name: str) -> int:
        return int(_lib.load().tfa_mesh_device_ptr(self._h, MESH_ITEMS[name][0]) or 0)

    def close(self):
        if getattr(self, "_h", None):
            if getattr(self, "_owner", None) is None:
                _lib.load().tfa_mesh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Context:
    """Owner of a ``tfa_ctx*``: physics + numerics constants and the per-mesh workspace."""

    def __init__(self, physics=None, numerics: Numerics | None = None):
        self._h = C.c_void_p()
        _lib.check(_lib.load().tfa_ctx_create(C.byref(self._h)))
        self.physics = physics if isinstance(physics, Physics) else default_physics(physics)
        self.set_physics(self.physics)
        self.set_numerics(numerics or default_numerics(self.physics))

    def set_physics(self, p: Physics):
        _lib.check(_lib.load().tfa_set_physics(self._h, C.byref(p)))
        self.physics = p

    def set_numerics(self, n: Numerics):
        _lib.check(_lib.load().tfa_set_numerics(self._h, C.byref(n)))
        self.numerics = n

    def set_ghost_states(self, ghost: torch.Tensor | None):
        """tfa_set_ghost_states: ghost [n_bfaces][18] device tensor, read (not copied) by later assemblies; the
        binding keeps a reference so that it stays alive."""
        self._ghost = ghost
        n = 0 if ghost is None else ghost.shape[0]
        _lib.check(_lib.load().tfa_set_ghost_states(self._h, _dp(ghost), n))

    def gradients(self, mesh: Mesh, state: torch.Tensor):
        grad = torch.empty((mesh.n_cells, NEQ, 2), dtype=torch.float64, device=state.device)
        phi = torch.empty((mesh.n_cells, NEQ), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_gradients(self._h, mesh._h, _dp(state), _dp(grad), _dp(phi), _stream()))
        return grad, phi

    def assemble(self, mesh: Mesh, state, state_n=None, state_nm1=None, dt=1e-3, rhs=None, vals=None,
                 jacobian=True):
        """tfa_assemble on device tensors.  Returns (rhs, vals); asynchronous on the current stream."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if rhs is None:
            rhs = torch.empty((mesh.n_cells, NEQ), dtype=torch.float64, device=state.device)
        if vals is None and jacobian:
            vals = torch.empty((mesh.nnzb, NEQ, NEQ), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_assemble(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt),
                                            _dp(rhs), _dp(vals) if jacobian else None, _stream()))
        return rhs, vals

    def assemble_packed(self, mesh: Mesh, state, state_n=None, state_nm1=None, dt=1e-3, rhs=None, diag=None, offd=None):
        """tfa_assemble_packed: returns (rhs, diag [n_cells][18][18], offd [nnzb - n_cells][114])."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if rhs is None:
            rhs = torch.empty((mesh.n_cells, NEQ), dtype=torch.float64, device=state.device)
        if diag is None:
            diag = torch.empty((mesh.n_cells, NEQ, NEQ), dtype=torch.float64, device=state.device)
        if offd is None:
            offd = torch.empty((mesh.nnzb - mesh.n_cells, PACKED_BLOCK), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_assemble_packed(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt),
                                                   _dp(rhs), _dp(diag), _dp(offd), _stream()))
        return rhs, diag, offd

    def block_jacobi_packed(self, mesh: Mesh, diag, dinv=None):
        if dinv is None:
            dinv = torch.empty_like(diag)
        _lib.check(_lib.load().tfa_block_jacobi_packed(self._h, mesh._h, _dp(diag), _dp(dinv), _stream()))
        return dinv

    def gmres_packed(self, mesh: Mesh, diag, offd, b, x=None, dinv=None, restart=30, max_iters=300, rtol=1e-8):
        if x is None:
            x = torch.zeros_like(b)
        info = (C.c_double * 2)()
        _lib.check(_lib.load().tfa_gmres_packed(self._h, mesh._h, _dp(diag), _dp(offd), _dp(dinv), _dp(b), _dp(x),
                                                int(restart), int(max_iters), float(rtol), info, _stream()))
        return x, int(info[0]), float(info[1])

    def gmres_packed_f32(self, mesh: Mesh, diag, offd, diag32, offd32, b, x=None, dinv32=None, restart=30,
                         max_iters=300, rtol=1e-8):
        """tfa_gmres_packed_f32: Krylov cycles on the FP32 copies (packed_to_f32, to_f32), restarts in FP64."""
        if x is None:
            x = torch.zeros_like(b)
        info = (C.c_double * 2)()
        _lib.check(_lib.load().tfa_gmres_packed_f32(self._h, mesh._h, _dp(diag), _dp(offd), _fp(diag32), _fp(offd32),
                                                    _fp(dinv32), _dp(b), _dp(x), int(restart), int(max_iters),
                                                    float(rtol), info, _stream()))
        return x, int(info[0]), float(info[1])

    def assemble_gradient(self, mesh: Mesh, state):
        """tfa_assemble_gradient: step a2 only; the face states stay in the context (face_states)."""
        _lib.check(_lib.load().tfa_assemble_gradient(self._h, mesh._h, _dp(state), _stream()))

    def face_states(self, mesh: Mesh) -> torch.Tensor:
        """tfa_face_states as a tensor view [n_cells][F][18] of the context's buffer (no copy)."""
        ptr = _lib.load().tfa_face_states(self._h)
        n = mesh.n_cells * mesh.max_faces * NEQ
        if not ptr or n == 0:
            return torch.empty((0, mesh.max_faces, NEQ), dtype=torch.float64, device="cuda")
        iface = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False), "version": 3, "strides": None}
        holder = type("_FaceStates", (), {"__cuda_array_interface__": iface})()
        return torch.as_tensor(holder, device="cuda").view(mesh.n_cells, mesh.max_faces, NEQ)

    def face_states_static(self, mesh: Mesh, state, out=None) -> torch.Tensor:
        """tfa_face_states_static: step a2 into the caller's [n_cells][F][18] buffer with the scratch in the library's
        static device array (no allocation in the call when `out` is given; STATIC_MAX_STENCIL entries at most)."""
        if out is None:
            out = torch.empty((mesh.n_cells, mesh.max_faces, NEQ), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_face_states_static(self._h, mesh._h, _dp(state), _dp(out), _stream()))
        return out

    def assemble_faces(self, mesh: Mesh, state, state_n=None, state_nm1=None, dt=1e-3, rhs=None, vals=None):
        """tfa_assemble_faces: steps a3..a7 on the context's face states.  vals must be given (its size is the
        caller's business: a shard's value array holds the owned rows only)."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if rhs is None:
            rhs = torch.empty((mesh.n_cells, NEQ), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_assemble_faces(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt),
                                                  _dp(rhs), _dp(vals), _stream()))
        return rhs, vals

    def assemble_faces_packed(self, mesh: Mesh, state, state_n, state_nm1, dt, rhs, diag, offd):
        """tfa_assemble_faces_packed: steps a3..a7 on the context's face states, packed output (diag, offd given)."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if rhs is None:
            rhs = torch.empty((mesh.n_cells, NEQ), dtype=torch.float64, device=state.device)
        _lib.check(_lib.load().tfa_assemble_faces_packed(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1),
                                                         float(dt), _dp(rhs), _dp(diag), _dp(offd), _stream()))
        return rhs, diag, offd

    def assemble_host(self, mesh: Mesh, state, state_n, state_nm1, dt, rhs, vals):
        """tfa_assemble_host on HOST buffers (numpy arrays or CPU tensors, ideally pinned)."""
        def hp(x):
            if x is None:
                return None
            if isinstance(x, torch.Tensor):
                assert not x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
                return C.c_void_p(x.data_ptr())
            assert x.dtype == np.float64 and x.flags.c_contiguous
            return _hp(x)
        _lib.check(_lib.load().tfa_assemble_host(self._h, mesh._h, hp(state), hp(state_n), hp(state_nm1), float(dt),
                                                 hp(rhs), hp(vals), _stream()))
        return rhs, vals

    def block_jacobi(self, mesh: Mesh, vals, dinv=None):
        """tfa_block_jacobi: inverses of the diagonal blocks, [n_cells][18][18]."""
        if dinv is None:
            dinv = torch.empty((mesh.n_cells, NEQ, NEQ), dtype=torch.float64, device=vals.device)
        _lib.check(_lib.load().tfa_block_jacobi(self._h, mesh._h, _dp(vals), _dp(dinv), _stream()))
        return dinv

    def gmres(self, mesh: Mesh, vals, b, x=None, dinv=None, restart=30, max_iters=300, rtol=1e-8):
        """tfa_gmres: returns (x, iterations, relative residual).  x (initial guess) is updated in place."""
        if x is None:
            x = torch.zeros_like(b)
        info = (C.c_double * 2)()
        _lib.check(_lib.load().tfa_gmres(self._h, mesh._h, _dp(vals), _dp(dinv), _dp(b), _dp(x), int(restart),
                                         int(max_iters), float(rtol), info, _stream()))
        return x, int(info[0]), float(info[1])

    def implicit_step(self, mesh: Mesh, state, state_n, state_nm1, dt, work=None, max_newton=3, newton_tol=0.0,
                      restart=30, max_iters=300, rtol=1e-8, matrix_free=False):
        """tfa_implicit_step: Newton sub-iterations of one BDF2 step; `state` (initial guess) is updated in place to
        P^{n+1}.  Returns (newton_iterations, last relative update, gmres_iterations, last linear residual) and the
        work dictionary (rhs, vals, dinv, dP), which may be passed in again.  matrix_free: False (assembled BSR
        matrix), True (tfa_gmres_jfnk) or "packed_f32" (mode 2: packed Jacobian + mixed-precision solve)."""
        if work is None:
            f = dict(dtype=torch.float64, device=state.device)
            work = dict(rhs=torch.empty((mesh.n_cells, NEQ), **f), vals=torch.empty((mesh.nnzb, NEQ, NEQ), **f),
                        dinv=torch.empty((mesh.n_cells, NEQ, NEQ), **f), dP=torch.empty((mesh.n_cells, NEQ), **f))
        info = (C.c_double * 4)()
        _lib.check(_lib.load().tfa_implicit_step(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt),
                                                 _dp(work["rhs"]), _dp(work["vals"]), _dp(work["dinv"]), _dp(work["dP"]),
                                                 int(max_newton), float(newton_tol), int(restart), int(max_iters),
                                                 float(rtol), 2 if matrix_free == "packed_f32" else int(bool(matrix_free)), info,
                                                 _stream()))
        return (int(info[0]), float(info[1]), int(info[2]), float(info[3])), work

    def jvp(self, mesh: Mesh, state, v, state_n=None, state_nm1=None, dt=1e-3, eps=0.0, out=None):
        """tfa_jvp: (dR~/dP) v by a forward difference of the residual (matrix-free)."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if out is None:
            out = torch.empty_like(v)
        _lib.check(_lib.load().tfa_jvp(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt), _dp(v),
                                       _dp(out), float(eps), _stream()))
        return out

    def gmres_jfnk(self, mesh: Mesh, state, b, state_n=None, state_nm1=None, dt=1e-3, x=None, dinv=None, restart=30,
                   max_iters=300, rtol=1e-8):
        """tfa_gmres_jfnk: returns (x, iterations, relative residual)."""
        state_n = state if state_n is None else state_n
        state_nm1 = state if state_nm1 is None else state_nm1
        if x is None:
            x = torch.zeros_like(b)
        info = (C.c_double * 2)()
        _lib.check(_lib.load().tfa_gmres_jfnk(self._h, mesh._h, _dp(state), _dp(state_n), _dp(state_nm1), float(dt),
                                              _dp(dinv), _dp(b), _dp(x), int(restart), int(max_iters), float(rtol),
                                              info, _stream()))
        return x, int(info[0]), float(info[1])

    def check(self):
        _lib.check(_lib.load().tfa_check(self._h, _stream()))

    def timing_enable(self, on: bool = True):
        _lib.check(_lib.load().tfa_timing_enable(self._h, int(on)))

    def timing_read(self):
        """(ms_gradient_kernel, ms_assembly_kernel, n_calls) accumulated since the last read."""
        ms = (C.c_double * 2)()
        n = C.c_int()
        _lib.check(_lib.load().tfa_timing_read(self._h, ms, C.byref(n)))
        return float(ms[0]), float(ms[1]), int(n.value)

    @property
    def launches_per_assemble(self) -> int:
        return int(_lib.load().tfa_launches_per_assemble(self._h))

    def close(self):
        if getattr(self, "_h", None):
            _lib.load().tfa_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------------
# sharding over several GPUs: one process per GPU, neighbour-only exchanges
# ------------------------------------------------------------------------------------------------
PART_LOCAL_TO_GLOBAL, PART_SEND_STATE, PART_RECV_STATE, PART_SEND_FACE, PART_RECV_FACE = range(5)
HALO_STATE, HALO_FACE = 0, 1


class Partition:
    """tfa_partition_*: the host-only half of the sharding (no CUDA call): which cells a rank owns, which ghosts it
    keeps, and the per-peer send / receive lists of the two halo exchanges."""

    def __init__(self, cell_nbr=None, stencil_ptr=None, stencil_idx=None, n_ranks=1, rank=0, _handle=None, _owner=None):
        lib = _lib.load()
        self._owner = _owner
        if _handle is not None:
            self._h = C.c_void_p(_handle)
        else:
            nbr = np.ascontiguousarray(cell_nbr, dtype=np.int32)
            sp = np.ascontiguousarray(stencil_ptr, dtype=np.int32)
            si = np.ascontiguousarray(stencil_idx, dtype=np.int32)
            self._h = C.c_void_p()
            _lib.check(lib.tfa_partition_create(C.byref(self._h), nbr.shape[0], nbr.shape[1] if nbr.ndim == 2 else 3,
                                                _hp(nbr), _hp(sp), _hp(si), int(n_ranks), int(rank)))
        v = [C.c_int64() for _ in range(4)]
        _lib.check(lib.tfa_partition_sizes(self._h, *[C.byref(x) for x in v]))
        self.n_local, self.n_owned, self.first_owned_local, self.first_owned_global = [int(x.value) for x in v]
        self.n_ranks, self.rank = int(n_ranks), int(rank)

    def list(self, which: int, peer: int = 0) -> np.ndarray:
        lib = _lib.load()
        n = int(lib.tfa_partition_count(self._h, which, peer))
        if n < 0:
            raise ValueError("unknown list or peer")
        out = np.empty(n, dtype=np.int32)
        _lib.check(lib.tfa_partition_get(self._h, which, peer, _hp(out), n))
        return out

    @property
    def local_to_global(self) -> np.ndarray:
        return self.list(PART_LOCAL_TO_GLOBAL)

    def count(self, which: int, peer: int) -> int:
        return int(_lib.load().tfa_partition_count(self._h, which, peer))

    def close(self):
        if getattr(self, "_h", None):
            if self._owner is None:
                _lib.load().tfa_partition_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def exchange_halo(part: Partition, kind: int, width: int, pack, unpack, new_buffer, group=None):
    """One neighbour-only halo exchange over torch.distributed (NCCL send/recv on GPUs; any backend works).

    pack(peer, buf) fills buf [count][width] with the rows `peer` needs; unpack(peer, buf) stores the rows received
    from it; new_buffer(rows, width) allocates a buffer on the right device.  Only peers that share cells are
    contacted; there is no reduction and no collective."""
    import torch.distributed as dist
    send_which = PART_SEND_STATE if kind == HALO_STATE else PART_SEND_FACE
    recv_which = PART_RECV_STATE if kind == HALO_STATE else PART_RECV_FACE
    ops, recvs = [], []
    for peer in range(part.n_ranks):
        if peer == part.rank:
            continue
        ns, nr = part.count(send_which, peer), part.count(recv_which, peer)
        if nr:
            rb = new_buffer(nr, width)
            recvs.append((peer, rb))
            ops.append(dist.P2POp(dist.irecv, rb, peer, group))
        if ns:
            sb = new_buffer(ns, width)
            pack(peer, sb)
            ops.append(dist.P2POp(dist.isend, sb, peer, group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for peer, rb in recvs:
        unpack(peer, rb)


class Shard:
    """tfa_shard_*: rank `rank`'s part of a global mesh: the local mesh (owned + ghost cells), the block range of
    the owned rows and the device-side pack / unpack of the halos."""

    def __init__(self, global_mesh: Mesh, n_ranks: int, rank: int):
        lib = _lib.load()
        self._h = C.c_void_p()
        _lib.check(lib.tfa_shard_create(C.byref(self._h), global_mesh._h, int(n_ranks), int(rank), _stream()))
        self.mesh = Mesh._borrowed(lib.tfa_shard_mesh(self._h), self)
        self.part = Partition(n_ranks=n_ranks, rank=rank, _handle=lib.tfa_shard_partition(self._h), _owner=self)
        a, b = C.c_int64(), C.c_int64()
        _lib.check(lib.tfa_shard_info(self._h, C.byref(a), C.byref(b)))
        self.nnzb_owned, self.block_offset = int(a.value), int(b.value)
        self.bface_global = np.empty(self.mesh.n_bfaces, dtype=np.int32)
        _lib.check(lib.tfa_shard_bface_global(self._h, _hp(self.bface_global), self.mesh.n_bfaces))

    def pack(self, kind: int, peer: int, src: torch.Tensor, buf: torch.Tensor):
        _lib.check(_lib.load().tfa_shard_pack(self._h, kind, peer, _dp(src), _dp(buf), _stream()))

    def unpack(self, kind: int, peer: int, buf: torch.Tensor, dst: torch.Tensor):
        _lib.check(_lib.load().tfa_shard_unpack(self._h, kind, peer, _dp(buf), _dp(dst), _stream()))

    def _width(self, kind: int) -> int:
        return NEQ if kind == HALO_STATE else self.mesh.max_faces * NEQ

    def exchange(self, kind: int, tensor: torch.Tensor, group=None):
        """Halo exchange of `tensor` ([n_local][18] states or [n_local][F][18] face states) with the other ranks."""
        exchange_halo(self.part, kind, self._width(kind),
                      lambda peer, buf: self.pack(kind, peer, tensor, buf),
                      lambda peer, buf: self.unpack(kind, peer, buf, tensor),
                      lambda n, w: torch.empty((n, w), dtype=torch.float64, device=tensor.device), group)

    def owned_bsr_pattern(self):
        """(rowptr [n_owned + 1], col [nnzb_owned]) of the owned rows; columns are local cell ids."""
        rp = self.mesh.get("bsr_rowptr")
        o0 = self.part.first_owned_local
        return (rp[o0:o0 + self.part.n_owned + 1] - self.block_offset,
                self.mesh.get("bsr_col")[self.block_offset:self.block_offset + self.nnzb_owned])

    def assemble(self, ctx: Context, state, state_n=None, state_nm1=None, dt=1e-3, rhs=None, vals=None, exchange=None):
        """One sharded assembly (include/tfa.h): state halo, gradient kernel, face-state halo, flux / Jacobian
        kernel.  `exchange(kind, tensor)` defaults to the torch.distributed exchange of this shard."""
        exchange = exchange or self.exchange
        if vals is None:
            vals = torch.empty((self.nnzb_owned, NEQ, NEQ), dtype=torch.float64, device=state.device)
        exchange(HALO_STATE, state)
        ctx.assemble_gradient(self.mesh, state)
        exchange(HALO_FACE, ctx.face_states(self.mesh))
        return ctx.assemble_faces(self.mesh, state, state_n, state_nm1, dt, rhs, vals)

    def assemble_packed(self, ctx: Context, state, state_n=None, state_nm1=None, dt=1e-3, rhs=None, diag=None, offd=None,
                        exchange=None):
        """The same sharded assembly with the packed Jacobian of the owned rows: diag [n_owned][18][18],
        offd [nnzb_owned - n_owned][114] (tfa_assemble_faces_packed)."""
        exchange = exchange or self.exchange
        f = dict(dtype=torch.float64, device=state.device)
        if diag is None:
            diag = torch.empty((self.part.n_owned, NEQ, NEQ), **f)
        if offd is None:
            offd = torch.empty((self.nnzb_owned - self.part.n_owned, PACKED_BLOCK), **f)
        exchange(HALO_STATE, state)
        ctx.assemble_gradient(self.mesh, state)
        exchange(HALO_FACE, ctx.face_states(self.mesh))
        return ctx.assemble_faces_packed(self.mesh, state, state_n, state_nm1, dt, rhs, diag, offd)

    def close(self):
        if getattr(self, "_h", None):
            self.mesh._h = C.c_void_p()
            self.part._h = C.c_void_p()
            _lib.load().tfa_shard_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def exchange_in_process(shards, kind: int, tensors):
    """The halo exchange among shards that live in ONE process on one GPU (tests and debugging; the kernels of
    the ranks do not wait on each other, so running them one after another is legitimate): the same pack and unpack
    kernels, with a device buffer standing in for the wire."""
    n = len(shards)
    which = PART_SEND_STATE if kind == HALO_STATE else PART_SEND_FACE
    for r in range(n):
        for p in range(n):
            cnt = shards[r].part.count(which, p) if p != r else 0
            if cnt:
                buf = torch.empty((cnt, shards[r]._width(kind)), dtype=torch.float64, device=tensors[r].device)
                shards[r].pack(kind, p, tensors[r], buf)
                shards[p].unpack(kind, r, buf, tensors[p])


def probe_dfma(grid: int, iters: int, sink: torch.Tensor):
    _lib.check(_lib.load().tfa_probe_dfma(int(grid), int(iters), _dp(sink), _stream()))
    return grid * 256 * iters * 8 * 2   # flops


def probe_copy(src: torch.Tensor, dst: torch.Tensor):
    n = src.numel()
    _lib.check(_lib.load().tfa_probe_copy(_dp(src), _dp(dst), n, _stream()))
    return 16 * n                       # bytes read + written


def probe_math(x: torch.Tensor):
    """(sqrt, reciprocal) of x as the AUSM flux kernel computes them."""
    s, r = torch.empty_like(x), torch.empty_like(x)
    _lib.check(_lib.load().tfa_probe_math(_dp(x), _dp(s), _dp(r), x.numel(), _stream()))
    return s, r


def packed_spmv(mesh: Mesh, diag, offd, x, y=None):
    """tfa_packed_spmv: y = A x on the packed Jacobian."""
    if y is None:
        y = torch.empty_like(x)
    _lib.check(_lib.load().tfa_packed_spmv(mesh._h, _dp(diag), _dp(offd), _dp(x), _dp(y), _stream()))
    return y


PACKED_BLOCK_F32 = 116


def to_f32(src, dst=None):
    """tfa_to_f32: an FP32 copy of an FP64 device array."""
    if dst is None:
        dst = torch.empty(src.shape, dtype=torch.float32, device=src.device)
    _lib.check(_lib.load().tfa_to_f32(_dp(src), _fp(dst), src.numel(), _stream()))
    return dst


def packed_to_f32(mesh: Mesh, diag, offd):
    """tfa_packed_to_f32: FP32 copies of the packed Jacobian for gmres_packed_f32 (off-diagonal blocks 116 apart)."""
    diag32 = torch.empty((mesh.n_cells, NEQ, NEQ), dtype=torch.float32, device=diag.device)
    offd32 = torch.empty((mesh.nnzb - mesh.n_cells, PACKED_BLOCK_F32), dtype=torch.float32, device=diag.device)
    _lib.check(_lib.load().tfa_packed_to_f32(mesh._h, _dp(diag), _dp(offd), _fp(diag32), _fp(offd32), _stream()))
    return diag32, offd32


def packed_to_bsr(mesh: Mesh, diag, offd, vals=None):
    """tfa_packed_to_bsr: the packed Jacobian expanded into the mesh's BSR value array."""
    if vals is None:
        vals = torch.empty((mesh.nnzb, NEQ, NEQ), dtype=torch.float64, device=diag.device)
    _lib.check(_lib.load().tfa_packed_to_bsr(mesh._h, _dp(diag), _dp(offd), _dp(vals), _stream()))
    return vals


def bsr_spmv(mesh: Mesh, vals: torch.Tensor, x: torch.Tensor, y: torch.Tensor | None = None):
    """tfa_bsr_spmv: y = A x in the mesh's BSR pattern."""
    if y is None:
        y = torch.empty_like(x)
    _lib.check(_lib.load().tfa_bsr_spmv(mesh._h, _dp(vals), _dp(x), _dp(y), _stream()))
    return y


# C-style aliases, same names as the ABI
def mesh_create(node_xy, cell_nodes, cell_xy=None) -> Mesh:
    return Mesh(node_xy, cell_nodes, cell_xy)


def mesh_create_poly(node_xy, cell_ptr, cell_nodes, cell_xy=None) -> Mesh:
    return Mesh(node_xy, cell_nodes, cell_xy, cell_ptr)


def mesh_set_bc(mesh: Mesh, tags):
    mesh.set_bc(tags)


def set_ghost_states(ctx: Context, ghost):
    ctx.set_ghost_states(ghost)


def mesh_reorder(mesh: Mesh, kind="rcm", perm=None):
    mesh.reorder(kind, perm)


def ctx_create(physics=None, numerics=None) -> Context:
    return Context(physics, numerics)


def set_physics(ctx: Context, p: Physics):
    ctx.set_physics(p)


def set_numerics(ctx: Context, n: Numerics):
    ctx.set_numerics(n)


def assemble(ctx: Context, mesh: Mesh, state, state_n=None, state_nm1=None, dt=1e-3, **kw):
    return ctx.assemble(mesh, state, state_n, state_nm1, dt, **kw)


def destroy(obj):
    obj.close()
