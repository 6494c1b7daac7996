"""pn_dissipation_noalloc (include/pn.h): the entry point that allocates nothing -- its scratch is a file-scope
__device__ array -- against the existing handle-based pn_dissipation on the same solved networks, two calls in a row.
Collected last on purpose (the name): the suite runs with -x.  Tolerance as in test_gpu_parity.py: 1e-9 relative."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

G_TOL = 1e-9


@pytest.fixture(scope="module")
def pn():
    from paper_1908_03301_b200 import build, pn as _pn
    build.build()
    _pn.load_library()
    return _pn


def _solved(pn, net, direction, periodic=False, tol=1e-11):
    """Solve on a handle; return (device conductances in the caller's layout, pressures, pn_dissipation, g_eff)."""
    import torch
    h = pn.Network(net.nx, net.ny, net.nz)
    if periodic:
        h.set_option(pn.PN_OPT_LATERAL, 1)
    h.set_conductances(net.gx, net.gy, net.gz)
    h.solve(direction, tol, accept=(pn.PN_OK,))
    P = h.pressures().clone()
    g_e, g_eff = h.dissipation(), h.flux()[2]
    h.close()
    dev = [None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda().reshape(P.shape)
           for a in (net.gx, net.gy, net.gz)]
    return dev, P, g_e, g_eff


def _noalloc(pn, dev, P, out, mask=0):
    import torch
    pn.dissipation_noalloc(dev[0], dev[1], dev[2], P, out, periodic_mask=mask)
    torch.cuda.synchronize()
    return float(out[0].item())


def test_two_calls_in_a_row_match_the_handle_path(pn):
    """A larger network first, a smaller one second (the scratch array keeps the first call's chunk sums), then the
    first again: every result within 1e-9 of pn_dissipation's and of G_eff; repeated calls bit-identical."""
    import torch
    from paper_1908_03301_b200 import inputs
    big = inputs.cfg4_fbm_cut_3d(96, 80, 72)            # 67.5 chunks of 8192 nodes, ragged tail; 40 % closed bonds
    small = inputs.cfg3_percolation_3d(40, 36, 33, p=0.40)  # pinned and floating clusters
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    a_dev, a_P, a_ge, a_geff = _solved(pn, big, 0)
    b_dev, b_P, b_ge, b_geff = _solved(pn, small, 2)
    first = _noalloc(pn, a_dev, a_P, out)
    second = _noalloc(pn, b_dev, b_P, out)
    third = _noalloc(pn, a_dev, a_P, out)
    fourth = _noalloc(pn, b_dev, b_P, out)
    assert abs(first - a_ge) <= G_TOL * abs(a_ge)
    assert abs(second - b_ge) <= G_TOL * abs(b_ge)
    assert abs(first - a_geff) <= G_TOL * abs(a_geff)
    assert abs(second - b_geff) <= G_TOL * abs(b_geff)
    assert third == first and fourth == second          # fixed summation order, nothing left over from the call before
    free1 = torch.cuda.mem_get_info()[0]                # (the very first use may have loaded the module: measured after it)
    _noalloc(pn, a_dev, a_P, out)
    assert torch.cuda.mem_get_info()[0] == free1        # no device memory taken by a call


@pytest.mark.parametrize("direction", [0, 1])
def test_periodic_faces_and_2d(pn, direction):
    """Periodic lateral faces (the mask names the wrapping axes) in 3D, and a 2D lattice (gz = None)."""
    import torch
    from paper_1908_03301_b200 import inputs
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    net = inputs.cfg4_fbm_cut_3d(48, 40, 36)
    dev, P, g_e, g_eff = _solved(pn, net, direction, periodic=True)
    mask = 7 & ~(1 << direction)
    got = _noalloc(pn, dev, P, out, mask)
    assert abs(got - g_e) <= G_TOL * abs(g_e)
    assert abs(got - g_eff) <= G_TOL * abs(g_eff)
    assert abs(_noalloc(pn, dev, P, out, 0) - g_e) > 1e-6 * abs(g_e)      # the wrap bonds do carry flow
    flat = inputs.iid_diluted(300, 220, 1, seed=3, p=0.7)
    dev2, P2, g_e2, _ = _solved(pn, flat, direction)
    got2 = _noalloc(pn, dev2, P2, out)
    assert abs(got2 - g_e2) <= G_TOL * abs(g_e2)
    assert _noalloc(pn, dev2, P2, out) == got2


def test_callable_under_stream_capture(pn):
    """What the entry point is for: after one direct call (which asks for the symbol address), two calls are
    captured into a CUDA graph -- a capture fails on any allocation or synchronisation -- and replayed."""
    import torch
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(64, 64, 64)
    dev, P, g_e, _ = _solved(pn, net, 0)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    direct = _noalloc(pn, dev, P, out)
    half = P * 0.5                                       # pressures scaled by 1/2: the sum is exactly a quarter
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        pn.dissipation_noalloc(dev[0], dev[1], dev[2], P, out[0:1])
        pn.dissipation_noalloc(dev[0], dev[1], dev[2], half, out[1:2])
    out.zero_()
    for _ in range(2):
        graph.replay()
        torch.cuda.synchronize()
        assert float(out[0].item()) == direct
        assert float(out[1].item()) == direct * 0.25
        assert abs(float(out[0].item()) - g_e) <= G_TOL * abs(g_e)


def test_size_limit_is_reported(pn):
    import ctypes
    lib = pn.load_library()
    p = ctypes.c_void_p(256)
    assert lib.pn_dissipation_noalloc(1024, 1024, 257, p, p, p, p, 0, p, 0, None) == pn.PN_ERR_TOO_LARGE
    assert "PN_NOALLOC_MAX_NODES" in pn.strerror(pn.PN_ERR_TOO_LARGE)
