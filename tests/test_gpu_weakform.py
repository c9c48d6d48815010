"""The CUDA path against the weak form itself, not against the oracle's text (GPU and oracle evaluate the
same expression trees by design, so their bitwise agreement cannot catch a formula both got wrong).

`helpers.brute_force_rhs` is an independent numpy statement of eq. (3) with the volume sign of eq. (6):
x-y-frame local Lax-Friedrichs flux, every integral by a 12 x 12 collapsed Gauss rule / 10-point edge rule, DENSE mass
matrix solve; it takes only the basis VALUES from the oracle's (separately pinned) `orc_basis`.  Where the method's own
quadrature is exact the GPU's `dgswem_eval_rhs` must equal it to round-off; for a generic discontinuous state with
friction, Coriolis and an ocean boundary, to the method's quadrature error."""
import numpy as np
import pytest

from helpers import brute_force_rhs, small_mesh, two_element_mesh
from test_oracle_rhs import _smooth_state
from workloads import default_params

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


def _gpu_rhs(G, mesh, bathy, W, tide=None, **kw):
    g = G.Dgswem(default_params(**kw), mesh.xy, bathy, mesh.tri, mesh.edge_elem, mesh.edge_local, mesh.edge_bc, mesh.elem_edge)
    if tide is not None:
        g.set_tide(*tide)
    g.set_state(0.0, *W)
    r = np.stack(g.eval_rhs())
    g.close()
    return r


@pytest.mark.parametrize("form", ["0", "1", "2", "3"], ids=["edge+elem", "stage", "stage-tile", "stage-staged"])
@pytest.mark.parametrize("p", [1, 2, 3])
@pytest.mark.parametrize("which", ["two", "eight"])
def test_gpu_rhs_equals_the_exactly_integrated_weak_form(O, G, monkeypatch, p, which, form):
    monkeypatch.setenv("DGSWEM_FUSED", form)
    mesh = two_element_mesh() if which == "two" else small_mesh(nq=2, L=1000.0)
    rng = np.random.default_rng(4)
    bathy = 10.0 + 2.0 * rng.uniform(-1, 1, mesh.n_nodes)
    W = _smooth_state(O, mesh, p, "poly_exact")
    r = _gpu_rhs(G, mesh, bathy, W, p=p)
    bf = brute_force_rhs(O, mesh, bathy, p, *W)
    assert np.abs(bf[1:]).max() > 1e-4
    assert np.abs(r - bf).max() < 1e-11 * max(1.0, np.abs(bf).max())
    # continuity row with momentum of full degree p (cubic modes at p = 3)
    flat = np.full(mesh.n_nodes, 10.0)
    W = _smooth_state(O, mesh, p, "continuity_exact")
    r = _gpu_rhs(G, mesh, flat, W, p=p)
    bf = brute_force_rhs(O, mesh, flat, p, *W)
    assert np.abs(bf[0]).max() > 1e-4
    assert np.abs(r[0] - bf[0]).max() < 1e-11 * max(1.0, np.abs(bf[0]).max())


@pytest.mark.parametrize("p", [1, 2, 3])
def test_gpu_rhs_generic_state_within_quadrature_error(O, G, p):
    """Discontinuous state, friction (strong enough that dropping it misses the tolerance), Coriolis, tidal boundary."""
    mesh = small_mesh(nq=2, L=1000.0, ocean=True)
    rng = np.random.default_rng(8)
    bathy = 10.0 + 2.0 * rng.uniform(-1, 1, mesh.n_nodes)
    W = _smooth_state(O, mesh, p, "generic")
    kw = dict(p=p, cf=0.25, coriolis_f=1e-2)
    r = _gpu_rhs(G, mesh, bathy, W, tide=(0.1, 0.0, np.pi / 2), **kw)
    bf = brute_force_rhs(O, mesh, bathy, p, *W, cf=0.25, fcor=1e-2, zeta_b=0.1)
    nofric = brute_force_rhs(O, mesh, bathy, p, *W, cf=0.0, fcor=1e-2, zeta_b=0.1)
    for c in range(3):
        sc = np.abs(bf[c]).max()
        tol = {1: 2e-3, 2: 1e-3, 3: 3e-4}[p] * sc          # the method's quadrature error on this state: 7e-4, 3e-4, 8e-5
        assert np.abs(r[c] - bf[c]).max() < tol
    # the friction term is worth more than ten times the tolerance: a dropped or mis-scaled term fails above
    assert min(np.abs(nofric[c] - bf[c]).max() / np.abs(bf[c]).max() for c in (1, 2)) > 1.2e-2
