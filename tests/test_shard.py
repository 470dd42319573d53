"""Sharding of the assembly over several GPUs.

CPU tests (-m "not gpu"): the host-only partitioner (tfa_partition_*) on the oracle's connectivity -- ownership,
ghost layers and the symmetry of the halo lists against set arithmetic done here -- and the exchange plumbing
(api.exchange_halo over torch.distributed) with two gloo processes.  GPU tests: the sharded assembly of 2, 3 and 5
ranks emulated in one process on one GPU gives, row for row and bit for bit, the single-GPU assembly; and the
oracle's rows.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def connectivity(orc, mi, rcm=True):
    """(cell_nbr, stencil_ptr, stencil_idx, OracleMesh) of a mesh, from the oracle (bit-identical to the CUDA
    builder's by tests/test_gpu_parity.py)."""
    o = orc.OracleMesh.from_input(mi)
    if rcm:
        o.reorder("rcm")
    cf, fc = o.get("cell_faces"), o.get("face_cells")
    me = np.arange(o.n_cells)[:, None]
    pair = fc[np.maximum(cf, 0)]
    nbr = np.where(pair[:, :, 0] == me, pair[:, :, 1], pair[:, :, 0])
    nbr = np.where(cf >= 0, nbr, -1).astype(np.int32)
    return nbr, o.get("stencil_ptr"), o.get("stencil_idx"), o


def shard_mesh(W, kind):
    if kind == "delaunay":
        return W.delaunay_mesh(23, 17, *W.GEM_DOMAIN, jitter=0.3, seed=4, shuffle_cells=True)
    if kind == "periodic":
        return W.split_quad_mesh(12, 9)
    return W.quad_mesh(11, 8, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False, jitter=0.2, seed=6, tri_every=3)


@pytest.mark.parametrize("kind", ["delaunay", "periodic", "mixed"])
@pytest.mark.parametrize("n_ranks", [1, 2, 3, 7])
def test_partition_lists_against_set_arithmetic(orc, W, kind, n_ranks):
    from paper_1809_02532_b200 import api
    nbr, sp, si, o = connectivity(orc, shard_mesh(W, kind))
    nc = o.n_cells
    parts = [api.Partition(nbr, sp, si, n_ranks, r) for r in range(n_ranks)]
    owner = np.empty(nc, dtype=np.int64)
    covered = 0
    for r, p in enumerate(parts):
        c0, n = p.first_owned_global, p.n_owned
        assert c0 == covered and abs(n - nc / n_ranks) < 1.0        # contiguous, balanced chunks
        owner[c0:c0 + n] = r
        covered += n
    assert covered == nc
    for r, p in enumerate(parts):
        l2g = p.local_to_global
        assert (np.diff(l2g) > 0).all()                               # local order = global order
        own = np.arange(p.first_owned_global, p.first_owned_global + p.n_owned)
        np.testing.assert_array_equal(l2g[p.first_owned_local:p.first_owned_local + p.n_owned], own)
        # ghosts = vertex neighbours of owned cells that are not owned
        reach = set()
        for i in own:
            reach.update(int(j) for j in si[sp[i]:sp[i + 1]])
        ghosts = sorted(reach - set(own.tolist()))
        assert sorted(set(l2g.tolist()) - set(own.tolist())) == ghosts
        face_ghosts = sorted({int(j) for i in own for j in nbr[i] if j >= 0 and owner[j] != r})
        for q in range(n_ranks):
            rs, rf = l2g[p.list(api.PART_RECV_STATE, q)], l2g[p.list(api.PART_RECV_FACE, q)]
            assert list(rs) == [g for g in ghosts if owner[g] == q]
            assert list(rf) == [g for g in face_ghosts if owner[g] == q]
            # what q sends to r is what r receives from q, in the same order
            pq = parts[q]
            np.testing.assert_array_equal(pq.local_to_global[pq.list(api.PART_SEND_STATE, r)], rs)
            np.testing.assert_array_equal(pq.local_to_global[pq.list(api.PART_SEND_FACE, r)], rf)
        assert p.count(api.PART_SEND_STATE, r) == 0 and p.count(api.PART_RECV_STATE, r) == 0
    with pytest.raises(api.TfaError):
        api.Partition(nbr, sp, si, 2, 2)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import oracle
    from paper_1809_02532_b200 import api, workloads as W
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mi = shard_mesh(W, "mixed")
    nbr, sp, si, o = connectivity(oracle, mi)
    part = api.Partition(nbr, sp, si, world, rank)
    l2g = part.local_to_global
    F = nbr.shape[1]
    rng = np.random.default_rng(5)
    gstate = rng.normal(size=(o.n_cells, 18))                       # the "global" arrays every rank can rebuild
    gface = rng.normal(size=(o.n_cells, F * 18))
    o0, n = part.first_owned_local, part.n_owned
    ok = True
    for kind, glob, width in ((api.HALO_STATE, gstate, 18), (api.HALO_FACE, gface, F * 18)):
        loc = torch.full((part.n_local, width), float("nan"), dtype=torch.float64)
        loc[o0:o0 + n] = torch.from_numpy(glob[l2g[o0:o0 + n]])     # a rank knows its own cells only
        send = api.PART_SEND_STATE if kind == api.HALO_STATE else api.PART_SEND_FACE
        recv = api.PART_RECV_STATE if kind == api.HALO_STATE else api.PART_RECV_FACE
        api.exchange_halo(part, kind, width,
                          lambda peer, buf: buf.copy_(loc[torch.from_numpy(part.list(send, peer).astype(np.int64))]),
                          lambda peer, buf: loc.index_copy_(0, torch.from_numpy(part.list(recv, peer).astype(np.int64)), buf),
                          lambda rows, w: torch.empty((rows, w), dtype=torch.float64))
        got = loc.numpy()
        filled = ~np.isnan(got[:, 0])
        expect_filled = np.zeros(part.n_local, dtype=bool)
        expect_filled[o0:o0 + n] = True
        for q in range(world):
            expect_filled[part.list(recv, q)] = True
        ok &= bool((filled == expect_filled).all()) and bool((got[filled] == glob[l2g][filled]).all())
        if kind == api.HALO_STATE:
            ok &= bool(filled.all())                                 # every ghost state arrives
    out.put((rank, ok, part.n_local, part.n_owned))
    dist.barrier()
    dist.destroy_process_group()


def test_halo_exchange_two_gloo_processes():
    """world_size = 2 over gloo on CPU: after the state exchange every ghost row holds its owner's values; after the
    face exchange exactly the face-neighbour ghosts do."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(g[1] for g in got), got
    assert sum(g[3] for g in got) == shard_mesh(__import__("paper_1809_02532_b200.workloads", fromlist=["x"]), "mixed").n_cells
    assert all(g[2] > g[3] for g in got)                            # each rank keeps ghosts


# ------------------------------------------------------------------------------------------
# GPU: the sharded assembly, ranks emulated one after another in one process on one GPU
# ------------------------------------------------------------------------------------------
def sharded_assembly(api, gmesh, n_ranks, P, Pn, Pnm1, dt, ghost=None, numerics=None, packed=None):
    """Assemble with n_ranks shards of `gmesh` living in this process; the halos travel through the library's pack
    and unpack kernels (api.exchange_in_process).  Returns per rank (shard, rhs, vals) and the local states."""
    import torch
    shards = [api.Shard(gmesh, n_ranks, r) for r in range(n_ranks)]
    ctxs = [api.Context(numerics=numerics) for _ in range(n_ranks)]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    nan = float("nan")
    loc, locn, locm = [], [], []
    for s in shards:
        l2g, o0, n = s.part.local_to_global, s.part.first_owned_local, s.part.n_owned
        st = torch.full((s.part.n_local, 18), nan, dtype=torch.float64, device="cuda")
        st[o0:o0 + n] = dev(P[l2g[o0:o0 + n]])                        # a rank knows the state of its own cells
        loc.append(st)
        locn.append(dev(Pn[l2g]))
        locm.append(dev(Pnm1[l2g]))
    if ghost is not None:
        for s, c in zip(shards, ctxs):
            gl = np.zeros((s.mesh.n_bfaces, 18))
            real = s.bface_global >= 0
            gl[real] = ghost[s.bface_global[real]]
            c.set_ghost_states(dev(gl))
    api.exchange_in_process(shards, api.HALO_STATE, loc)
    for s, c, st in zip(shards, ctxs, loc):
        assert not bool(torch.isnan(st).any())                        # every ghost state arrived
        c.assemble_gradient(s.mesh, st)
    faces = [c.face_states(s.mesh) for s, c in zip(shards, ctxs)]
    api.exchange_in_process(shards, api.HALO_FACE, faces)
    out = []
    for s, c, st, sn, sm in zip(shards, ctxs, loc, locn, locm):
        vals = torch.full((s.nnzb_owned, 18, 18), nan, dtype=torch.float64, device="cuda")
        rhs, _ = c.assemble_faces(s.mesh, st, sn, sm, dt, vals=vals)
        c.check()
        if packed is not None:   # the packed Jacobian of the owned rows, from the same face states
            n = s.part.n_owned
            pd = torch.full((n, 18, 18), nan, dtype=torch.float64, device="cuda")
            po = torch.full((s.nnzb_owned - n, 114), nan, dtype=torch.float64, device="cuda")
            rhs_p, _, _ = c.assemble_faces_packed(s.mesh, st, sn, sm, dt, None, pd, po)
            c.check()
            packed.append((rhs_p, pd, po))
        out.append((s, rhs, vals))
    return out, loc


@pytest.mark.gpu
@pytest.mark.parametrize("kind", ["delaunay", "periodic", "mixed"])
@pytest.mark.parametrize("n_ranks", [2, 3, 5])
def test_sharded_assembly_equals_the_single_gpu_assembly_bit_for_bit(orc, W, kind, n_ranks):
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    mi = shard_mesh(W, kind)
    g = api.Mesh.from_input(mi)
    g.reorder("rcm")
    perm = g.get("perm")
    rng = np.random.default_rng(3)
    ghost = None
    if g.n_bfaces:
        g.set_bc((np.arange(g.n_bfaces) % 3).astype(np.int32))
        from conftest import random_state
        ghost = random_state(rng, g.n_bfaces)
    cen = mi.centroids()[perm]
    P = W.gem_state(cen) + rng.uniform(-1e-3, 1e-3, (g.n_cells, 18))
    Pn, Pnm1 = W.perturb(P, 1, 1e-4), W.perturb(P, 2, 1e-4)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ctx = api.Context()
    if ghost is not None:
        ctx.set_ghost_states(dev(ghost))
    rhs_g, vals_g = ctx.assemble(g, dev(P), dev(Pn), dev(Pnm1), 1e-3)
    ctx.check()
    rp_g, col_g = g.get("bsr_rowptr"), g.get("bsr_col")
    packed = []
    out, _ = sharded_assembly(api, g, n_ranks, P, Pn, Pnm1, 1e-3, ghost, packed=packed)
    # the packed output of a shard (tfa_assemble_faces_packed): the rank's pieces of the single-GPU packed arrays
    _, diag_g, offd_g = ctx.assemble_packed(g, dev(P), dev(Pn), dev(Pnm1), 1e-3)
    for (s, rhs, vals), (rhs_p, pd, po) in zip(out, packed):
        o0, n, c0 = s.part.first_owned_local, s.part.n_owned, s.part.first_owned_global
        assert not bool(torch.isnan(pd).any()) and not bool(torch.isnan(po).any())
        assert torch.equal(rhs_p[o0:o0 + n], rhs[o0:o0 + n])
        assert torch.equal(pd, diag_g[c0:c0 + n])
        assert torch.equal(po, offd_g[int(rp_g[c0]) - c0:int(rp_g[c0 + n]) - (c0 + n)])
    rows_seen = 0
    for s, rhs, vals in out:
        assert not bool(torch.isnan(vals).any()), "an owned block was not written"
        l2g, o0, n = s.part.local_to_global, s.part.first_owned_local, s.part.n_owned
        c0 = s.part.first_owned_global
        assert torch.equal(rhs[o0:o0 + n], rhs_g[c0:c0 + n])
        assert s.nnzb_owned == rp_g[c0 + n] - rp_g[c0]
        assert torch.equal(vals, vals_g[int(rp_g[c0]):int(rp_g[c0 + n])])
        rp, col = s.owned_bsr_pattern()
        np.testing.assert_array_equal(rp, rp_g[c0:c0 + n + 1] - rp_g[c0])
        np.testing.assert_array_equal(l2g[col], col_g[rp_g[c0]:rp_g[c0 + n]])      # local columns name the same cells
        rows_seen += n
    assert rows_seen == g.n_cells
    # and against the oracle (the single-GPU result is compared with it elsewhere; once more, through the shards)
    from helpers import residual_error, jacobian_error_blocks, RES_TOL, JAC_TOL
    o = orc.OracleMesh.from_input(mi)
    o.reorder("rcm")
    if ghost is not None:
        o.set_bc((np.arange(g.n_bfaces) % 3).astype(np.int32), ghost)
    ph_o = orc.physics_c()
    rhs_o, sc_o, vals_o = orc.assemble(o, ph_o, orc.default_numerics(ph_o), P, Pn, Pnm1, 1e-3)
    rhs_s = np.concatenate([rhs[s.part.first_owned_local:s.part.first_owned_local + s.part.n_owned].cpu().numpy()
                            for s, rhs, _ in out])
    vals_s = np.concatenate([v.cpu().numpy() for _, _, v in out])
    assert residual_error(rhs_s, rhs_o, sc_o) < RES_TOL
    assert jacobian_error_blocks(vals_s, vals_o, rp_g) < JAC_TOL


@pytest.mark.gpu
def test_sharded_assembly_at_config_4_size(W):
    """BASELINE config 4 (1M cells, RCM) cut into 8 ranks, emulated on one GPU: every owned row of every rank equals
    the single-GPU assembly bit for bit; each rank holds about an eighth of the Jacobian and a thin ghost layer."""
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    w = W.make_workload("c4b")
    g = api.Mesh.from_input(w.mesh)
    g.reorder("rcm")
    P = np.ascontiguousarray(w.state[g.get("perm")])
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ctx = api.Context(w.physics)
    rhs_g, vals_g = ctx.assemble(g, dev(P), dt=w.dt)
    rp_g = g.get("bsr_rowptr")
    out, _ = sharded_assembly(api, g, 8, P, P, P, w.dt)
    for s, rhs, vals in out:
        o0, n, c0 = s.part.first_owned_local, s.part.n_owned, s.part.first_owned_global
        assert torch.equal(rhs[o0:o0 + n], rhs_g[c0:c0 + n])
        assert torch.equal(vals, vals_g[int(rp_g[c0]):int(rp_g[c0 + n])])
        assert n == 125000 and s.part.n_local < 1.1 * n               # ghost layer below 10 % of the owned cells
