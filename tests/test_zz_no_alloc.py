"""dgswem_nodal_static -- nodal output for callers that cannot allocate device memory -- against dgswem_get_nodal.

Who needs it: code that wants element-averaged nodal fields at a moment when it may not call cudaMalloc
and so cannot create a Dgswem handle (which allocates its node -> element table and everything else at creation): an
output hook that runs while a stream capture is open, a solver inside an application whose memory pool already owns the
GPU, a time loop that must not take cudaMalloc's device-wide synchronisation.  The entry point keeps the table in a fixed
20 MiB array inside the library instead, which is what this file tests: same bits as the handle's path (the tolerance
the nodal-output parity tests use, np.array_equal), on calls made back to back so that what one call leaves behind in
the shared array is seen not to leak into the next, and a clear refusal beyond the array's size limit.

The file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides nothing else.  It holds
no state of its own and passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

from workloads import c2, c4, c5, perturbed

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_21208_b200 import build
    build.build()
    import paper_2508_21208_b200 as pk
    return pk


def _case(G, w):
    """Handle path: load the workload's state, read it back (set_state may have run a wet/dry pass) together with the
    nodal output of dgswem_get_nodal.  Returns what a handle-less caller would hold on the device, plus the expectation."""
    import torch
    g = G.Dgswem.from_workload(w, reorder=1)
    _, ze, qx, qy = g.get_state()
    want = [np.array(a) for a in g.get_nodal()]
    g.close()
    dev = torch.device("cuda", 0)
    tri = torch.from_numpy(np.ascontiguousarray(w.mesh.tri, dtype=np.int32)).to(dev)
    state = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev) for a in (ze, qx, qy)]
    out = [torch.full((w.mesh.n_nodes,), float("nan"), dtype=torch.float64, device=dev) for _ in range(3)]
    return int(w.params["p"]), tri, state, out, want


def test_nodal_static_matches_get_nodal_on_consecutive_calls(G):
    """Three meshes of different size and degree (p = 2 with 12,800 elements: several sort stages in global memory;
    p = 1 with wet/dry and 576 elements: a single shared-memory sort, far fewer nodes than the call before, so stale
    table entries of the larger mesh lie behind it; p = 3), called one after the other on one stream without any
    synchronisation in between, then the first one again.  Every output must equal dgswem_get_nodal's bit for bit."""
    import torch
    cases = [_case(G, perturbed(c2(nq=80, p=2, state="hump", nsteps=1), amp_z=0.2)),
             _case(G, perturbed(c4(nqx=24, nqy=12, nsteps=1), amp_z=0.2)),
             _case(G, perturbed(c5(nn=40, nsteps=1, p=3), amp_z=0.2))]
    order = [0, 1, 2, 0]
    got = []
    for i in order:                       # back to back: enqueue only
        p, tri, state, out, _ = cases[i]
        for o in out:
            o.fill_(float("nan"))
        G.nodal_static(p, tri, *state, *out)
        got.append([o.clone() for o in out])
    torch.cuda.synchronize()
    for i, res in zip(order, got):
        want = cases[i][4]
        for name, a, b in zip(("zeta", "qx", "qy"), res, want):
            a = a.cpu().numpy()
            assert np.isfinite(a).all(), (i, name)
            assert np.array_equal(a, b), (i, name, float(np.abs(a - b).max()))
    assert np.abs(cases[0][4][0]).max() > 1e-3 and np.abs(cases[0][4][1]).max() > 1e-3   # not a comparison of zeros


def test_nodal_static_ignores_unreferenced_nodes_and_refuses_oversize(G):
    """A node that no triangle references gets 0 (as in dgswem_get_nodal); sizes beyond the fixed array are refused
    with DGSWEM_E_ARG and a message naming the limit, before anything is launched (the outputs stay untouched)."""
    import torch
    from paper_2508_21208_b200.binding import STATIC_MAX_ELEM, STATIC_MAX_NODES
    dev = torch.device("cuda", 0)
    tri = torch.tensor([[0, 1, 2], [2, 1, 4]], dtype=torch.int32, device=dev)       # node 3 is referenced by nobody
    st = [torch.tensor([[1.0, 3.0], [0.5, -0.25], [0.125, 2.0]], dtype=torch.float64, device=dev) * s for s in (1.0, 2.0, -1.0)]
    out = [torch.full((5,), 7.0, dtype=torch.float64, device=dev) for _ in range(3)]
    G.nodal_static(1, tri, *st, *out)
    torch.cuda.synchronize()
    z = out[0].cpu().numpy()
    # p = 1 vertex values (a - b - c, a - b + c, a + 2b) of modes (a, b, c): element 0 = (1, .5, .125), element 1 = (3, -.25, 2)
    e0 = (1 - .5 - .125, 1 - .5 + .125, 1 + 2 * .5)
    e1 = (3 + .25 - 2, 3 + .25 + 2, 3 - 2 * .25)
    assert np.array_equal(z, np.array([e0[0], (e0[1] + e1[1]) / 2, (e0[2] + e1[0]) / 2, 0.0, e1[2]]))
    assert np.array_equal(out[1].cpu().numpy(), 2.0 * z) and np.array_equal(out[2].cpu().numpy(), -z)

    for kw, word in ((dict(n_elem=STATIC_MAX_ELEM + 1, n_nodes=5), "DGSWEM_STATIC_MAX_ELEM"),
                     (dict(n_elem=2, n_nodes=STATIC_MAX_NODES + 1), "DGSWEM_STATIC_MAX_NODES")):
        for o in out:
            o.fill_(7.0)
        with pytest.raises(G.DgswemError, match=word) as ei:
            G.nodal_static(1, tri, *st, *out, **kw)
        assert ei.value.code == -1
        torch.cuda.synchronize()
        assert all(bool((o == 7.0).all()) for o in out)
    with pytest.raises(G.DgswemError, match="p must be"):
        G.nodal_static(4, tri, *st, *out, n_elem=2, n_nodes=5)


def test_nodal_static_at_the_size_limit(G):
    """BASELINE configs[1] (C2: 524,288 elements = DGSWEM_STATIC_MAX_ELEM exactly, 2^21 padded sort keys, every merge
    stage of the network): accepted, and equal to dgswem_get_nodal bit for bit; called twice, second result checked."""
    import torch
    from paper_2508_21208_b200.binding import STATIC_MAX_ELEM
    w = perturbed(c2(p=1, state="hump", nsteps=1), amp_z=0.2)
    assert w.mesh.n_elem == STATIC_MAX_ELEM
    p, tri, state, out, want = _case(G, w)
    G.nodal_static(p, tri, *state, *out)
    for o in out:
        o.fill_(float("nan"))
    G.nodal_static(p, tri, *state, *out)
    torch.cuda.synchronize()
    for a, b in zip(out, want):
        assert np.array_equal(a.cpu().numpy(), b)
