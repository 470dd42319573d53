"""tfa_face_states_static (include/tfa.h): step a2 with its scratch in the library's static device array, for
callers that cannot allocate.  Collected last on purpose (the file name): the suite runs with pytest -x.

What is checked: the face states equal those of the existing path (tfa_assemble_gradient + tfa_face_states) bit for
bit -- same kernels, same arithmetic, only the home of the least-squares coefficients differs -- on two calls in a
row that share the array (a larger mesh, then a smaller one with other stencils, then the first again: stale
coefficients of the previous call would show), that the device's free memory does not move across the calls, and
that a mesh beyond TFA_STATIC_MAX_STENCIL is refused with TFA_EINVAL."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_1809_02532_b200 import api, build, workloads as W
    build.build()
    torch.cuda.set_device(0)
    return torch, api, W


def _case(torch, api, W, mesh_input, seed, reorder=None):
    g = api.Mesh.from_input(mesh_input)
    if reorder:
        g.reorder(reorder)
    P = np.ascontiguousarray(W.wave_state(mesh_input.centroids(), seed=seed)[g.get("perm")])
    # noise on top of the wave so that the limiter is active in part of the cells
    P = P * (1.0 + 0.05 * np.random.default_rng(seed).uniform(-1.0, 1.0, P.shape))
    return g, torch.from_numpy(P).cuda()


def _existing(api, ctx, g, P):
    ctx.assemble_gradient(g, P)
    return ctx.face_states(g).clone()


@pytest.mark.gpu
def test_face_states_static_equals_the_existing_path_on_calls_in_a_row(env):
    torch, api, W = env
    tri = W.delaunay_mesh(41, 23, *W.GEM_DOMAIN, jitter=0.3, seed=5)            # 1760 triangles, ragged stencils
    quad = W.quad_mesh(24, 16, *W.GEM_DOMAIN, periodic_y=False, jitter=0.2, seed=6, tri_every=3)   # mixed, F = 4
    cases = [_case(torch, api, W, tri, 11, "rcm"), _case(torch, api, W, quad, 12)]
    ref_ctx = api.Context(W.Physics())
    refs = [_existing(api, ref_ctx, g, P) for g, P in cases]
    ctx = api.Context(W.Physics())           # a context that never built a workspace of its own
    outs = [torch.full((g.n_cells, g.max_faces, 18), float("nan"), dtype=torch.float64, device="cuda") for g, _ in cases]
    ctx.face_states_static(cases[0][0], cases[0][1], outs[0])                  # first call: address look-up
    for rnd in range(2):                     # large, small, large, small: back to back on one stream
        for (g, P), out, ref in zip(cases, outs, refs):
            out.fill_(float("nan"))
            ctx.face_states_static(g, P, out)
            assert g.get("stencil_ptr")[-1] <= api.STATIC_MAX_STENCIL
            assert not torch.isnan(out).any()
            assert torch.equal(out, ref), (rnd, g.n_cells, float((out - ref).abs().max()))
    # nothing is allocated on the device: free memory as the driver reports it, around calls with no torch operation
    # (hence no caching-allocator activity) in between
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        for (g, P), out in zip(cases, outs):
            ctx.face_states_static(g, P, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    for out, ref in zip(outs, refs):
        assert torch.equal(out, ref)
    ctx.check()
    # the existing path is untouched by the static one: same result again, and the context used above has no
    # face-state buffer of its own
    assert torch.equal(_existing(api, ref_ctx, *cases[0]), refs[0])
    assert ctx.face_states(cases[0][0]).numel() == 0


@pytest.mark.gpu
def test_face_states_static_refuses_a_mesh_beyond_its_scratch(env):
    torch, api, W = env
    big = W.split_quad_mesh(300, 300)                                           # 180 000 triangles, 12 entries each
    g = api.Mesh.from_input(big)
    assert g.get("stencil_ptr")[-1] > api.STATIC_MAX_STENCIL
    P = torch.zeros((g.n_cells, 18), dtype=torch.float64, device="cuda")
    out = torch.zeros((g.n_cells, 3, 18), dtype=torch.float64, device="cuda")
    ctx = api.Context(W.Physics())
    with pytest.raises(api.TfaError) as e:
        ctx.face_states_static(g, P, out)
    assert e.value.code == -1 and "TFA_STATIC_MAX_STENCIL" in str(e.value)
    assert float(out.abs().max()) == 0.0                                        # nothing was launched
    # empty mesh: nothing to do
    e0 = api.Mesh(np.zeros((0, 2)), np.zeros((0, 3), dtype=np.int32))
    ctx.face_states_static(e0, torch.zeros((0, 18), dtype=torch.float64, device="cuda"),
                           torch.zeros((0, 3, 18), dtype=torch.float64, device="cuda"))
