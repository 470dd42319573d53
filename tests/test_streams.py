"""Streams and CUDA graphs: tfa_assemble is asynchronous on the caller's stream and does nothing a graph capture
forbids (no synchronisation, no allocation after the first call on a mesh), so a Newton loop at small sizes can be
replayed as a CUDA graph instead of paying two launches per assembly; two contexts on two streams do not interfere."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_assemble_on_side_streams_and_in_a_cuda_graph(W):
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    w = W.make_workload("c1")
    g = api.Mesh.from_input(w.mesh)
    P = torch.from_numpy(w.state).cuda()
    ctx = api.Context(w.physics)
    rhs0, vals0 = ctx.assemble(g, P, dt=w.dt)                      # reference result, default stream
    torch.cuda.synchronize()

    # two contexts on two side streams at once, different states: each gets its own result
    P2 = P + 1e-3
    ctx2 = api.Context(w.physics)
    ref2 = ctx2.assemble(g, P2, dt=w.dt)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    out = {}
    for _ in range(3):
        with torch.cuda.stream(s1):
            out[1] = ctx.assemble(g, P, dt=w.dt)
        with torch.cuda.stream(s2):
            out[2] = ctx2.assemble(g, P2, dt=w.dt)
    torch.cuda.synchronize()
    assert torch.equal(out[1][0], rhs0) and torch.equal(out[1][1], vals0)
    assert torch.equal(out[2][0], ref2[0]) and torch.equal(out[2][1], ref2[1])

    # capture one assembly into a CUDA graph and replay it on new input values
    rhs = torch.empty_like(rhs0)
    vals = torch.empty_like(vals0)
    Pin = P.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        ctx.assemble(g, Pin, dt=w.dt, rhs=rhs, vals=vals)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(rhs, rhs0) and torch.equal(vals, vals0)
    Pin.copy_(P2)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(rhs, ref2[0]) and torch.equal(vals, ref2[1])
    # replay is cheaper than two launches through the binding (not asserted as a number: launch-bound sizes only)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(50):
        graph.replay()
    b.record()
    torch.cuda.synchronize()
    t_graph = a.elapsed_time(b) / 50
    a.record()
    for _ in range(50):
        ctx.assemble(g, Pin, dt=w.dt, rhs=rhs, vals=vals)
    b.record()
    torch.cuda.synchronize()
    t_calls = a.elapsed_time(b) / 50
    print(f"c1 assembly: {t_calls * 1e3:.1f} us per call through the binding, {t_graph * 1e3:.1f} us per graph replay")
    assert t_graph < 1.5 * t_calls
    ctx.check()
    ctx2.check()
