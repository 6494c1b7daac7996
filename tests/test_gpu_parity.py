"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 CPU oracle,
element by element on the same seeded inputs.

Tolerances are BASELINE.json's north_star: relative L_inf error 1e-8 in node pressures (max |P| = 1,
so absolute), 1e-9 in effective conductance.  Node classes (integer work) must match bit for bit.
Parity solves use tol = 1e-12 (1e-13 from 128^3 up): a 1e-10 residual does not imply 1e-8 in
pressure on the diluted networks (SURVEY.md 8(c) consequence (ii)); timing runs use 1e-10.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

P_TOL = 1e-8
G_TOL = 1e-9


@pytest.fixture(scope="module")
def pn():
    from paper_1908_03301_b200 import build, pn as _pn
    build.build()
    _pn.load_library()
    return _pn


@pytest.fixture(scope="module")
def oracle():
    from oracle import c_oracle
    c_oracle.build()
    return c_oracle


def gpu_solve(pn, net, direction, tol, opts=None):
    h = pn.Network(net.nx, net.ny, net.nz)
    for k, v in (opts or {}).items():
        h.set_option(k, v)
    h.set_conductances(net.gx, net.gy, net.gz)
    info = h.solve(direction, tol, accept=(pn.PN_OK, pn.PN_NO_SPANNING_CLUSTER, pn.PN_MAX_ITERS))
    P = h.pressures().cpu().numpy()
    cls = h.classes().cpu().numpy()
    fl = h.flux()
    n_launch = h.launch_count()
    h.close()
    return info, P, cls, fl, n_launch


def compare(pn, oracle, net, direction, tol=1e-12, opts=None, periodic=False):
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13, periodic=periodic)
    if periodic:
        opts = dict(opts or {})
        opts[pn.PN_OPT_LATERAL] = 1
    info, P, cls, fl, n_launch = gpu_solve(pn, net, direction, tol, opts)
    assert n_launch > 0
    # integer work: classes bit-exact, counts equal
    assert np.array_equal(cls, ref.classes), "node classes differ from the oracle's serial BFS"
    assert (info.n_solved, info.n_inlet_only, info.n_outlet_only, info.n_floating) == \
        (ref.n_solved, ref.n_inlet_only, ref.n_outlet_only, ref.n_floating)
    if ref.status == "no_spanning_cluster":
        assert info.status == pn.PN_NO_SPANNING_CLUSTER
        assert fl[0] == 0.0 and fl[1] == 0.0 and fl[2] == 0.0
        assert np.array_equal(P, ref.P)
        return info, P, fl, ref
    assert info.status == pn.PN_OK, f"status {info.status}, residual {info.rel_residual}"
    assert info.rel_residual <= tol
    assert ref.rel_residual <= 2e-13
    err = float(np.max(np.abs(P - ref.P)))
    assert err <= P_TOL, f"pressure L_inf error {err:.3e}"
    gerr = abs(fl[2] - ref.g_eff) / abs(ref.g_eff)
    assert gerr <= G_TOL, f"G_eff relative error {gerr:.3e}"
    assert abs(fl[0] - ref.q_in) <= 1e-8 * abs(ref.q_in)
    assert abs(fl[1] - ref.q_out) <= 1e-8 * abs(ref.q_out)
    n_a = (net.nx, net.ny, net.nz)[direction]
    s_perp = net.n_nodes // n_a
    assert fl[3] == pytest.approx(fl[2] * (n_a - 1) / s_perp, rel=1e-14)
    return info, P, fl, ref


# ---- the five configs (CFG1 full size; scaled-down siblings of CFG2..5) ---------------------------
def test_cfg1_full(pn, oracle):
    from paper_1908_03301_b200 import inputs
    info, *_ = compare(pn, oracle, inputs.cfg1_iid_2d(), 0)
    assert info.inner_iters > 0 and info.outer_cycles >= 2


def test_cfg2_sibling(pn, oracle):
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.cfg2_fbm_2d(256, 256), 0)


def test_cfg3_sibling(pn, oracle):
    from paper_1908_03301_b200 import inputs
    info, *_ = compare(pn, oracle, inputs.cfg3_percolation_3d(48, 48, 48), 0)
    assert info.n_floating > 0 and info.n_solved > 0


def test_cfg4_sibling(pn, oracle):
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.cfg4_fbm_cut_3d(64, 64, 64), 0)


@pytest.mark.parametrize("direction", [0, 2])
def test_cfg5_sibling(pn, oracle, direction):
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.cfg5_stratified_3d(48, 48, 48), direction)


def test_cfg4_sibling_128(pn, oracle):
    """2^21 nodes, tol 1e-13: several tiles in x and y and several z chunks with default options."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(128, 128, 128)
    auto, *_ = compare(pn, oracle, net, 0, tol=1e-13)
    tma, *_ = compare(pn, oracle, net, 0, tol=1e-13, opts={pn.PN_OPT_KERNEL: 3})
    assert auto.kernel_scheme == 8 and tma.kernel_scheme == 3


# ---- ragged shapes, every direction, 2D and 3D, with and without dilution ------------------------
@pytest.mark.parametrize("shape", [(17, 9, 5), (5, 17, 9), (9, 5, 17), (33, 31, 7), (130, 6, 3)])
@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("p", [1.0, 0.6])
@pytest.mark.parametrize("kernel", [1, 3, 8])
def test_ragged_3d(pn, oracle, shape, direction, p, kernel):
    """kernel 1 = reference two-kernel iteration, 3 = single fused TMA kernel per iteration (forced, whatever the size)."""
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(*shape, seed=7 + direction, p=p)
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: kernel})


@pytest.mark.parametrize("shape", [(19, 13), (13, 19), (64, 3), (3, 64), (257, 31)])
@pytest.mark.parametrize("direction", [0, 1])
@pytest.mark.parametrize("p", [1.0, 0.7])
@pytest.mark.parametrize("kernel", [1, 3, 6, 8])
def test_ragged_2d(pn, oracle, shape, direction, p, kernel):
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(shape[0], shape[1], 1, seed=11 + direction, p=p)
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: kernel})


@pytest.mark.parametrize("tile", [0, 1, 2, 3])
@pytest.mark.parametrize("shape,direction", [((300, 20, 70), 2), ((520, 9, 12), 1), ((260, 17, 40), 0), ((256, 33, 9), 0),
                                             ((130, 40, 21), 1), ((192, 70, 33), 2), ((66, 5, 40), 0)])
def test_tma_kernel_multi_tile(pn, oracle, shape, direction, tile):
    """Lattices wider than one TMA box and taller than one tile: x and y halos between tiles, several z chunks, ragged
    tails in all three directions.  All three 3D tiles (PN_OPT_TILE: 256 x 8, 128 x 16 and 64 x 32 nodes -- the last with two
    lattice rows per warp; 0 = automatic); widths that do not fill their last tile are cut into EQUAL narrower tiles
    (260 -> 2 x 132, 3 x 88 or 5 x 52; 300 -> 2 x 152, 3 x 100 or 5 x 60; 520 -> 3 x 176, 5 x 104 or 9 x 60; 130 -> 1 x 132,
    2 x 68 or 3 x 44; 66 -> 1 x 68 or 2 x 36), 256 and 192 = 3 x 64 are exact fits."""
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(*shape, seed=5, p=0.75)
    info, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_TILE: tile})
    assert info.kernel_scheme == 3
    one, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_TILE: tile, pn.PN_OPT_GRAPH: 0})
    assert one.kernel_scheme == 3                       # the same tiles, one launch per iteration


@pytest.mark.parametrize("kernel", [3, 6])
def test_tma_kernel_2d_wide(pn, oracle, kernel):
    """2D lattice wider than the 2048-node tile of the 2D configuration (x halo between tiles)."""
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(2100, 40, 1, seed=9, p=1.0)
    compare(pn, oracle, net, 1, opts={pn.PN_OPT_KERNEL: kernel})


@pytest.mark.parametrize("kernel", [1, 3, 8])
def test_kernel_variants(pn, oracle, kernel):
    """Both S4 kernels must pass the same parity bar (0 = automatic choice is what the other tests use)."""
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.cfg4_fbm_cut_3d(40, 36, 33), 0, opts={pn.PN_OPT_KERNEL: kernel})
    compare(pn, oracle, inputs.cfg1_iid_2d(), 0, opts={pn.PN_OPT_KERNEL: kernel})
    compare(pn, oracle, inputs.cfg3_percolation_3d(64, 64, 64), 0, opts={pn.PN_OPT_KERNEL: kernel})


def test_zero_start_and_restart_options(pn, oracle):
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(32, 32, 32)
    compare(pn, oracle, net, 0, opts={pn.PN_OPT_X0: 0})
    compare(pn, oracle, net, 0, opts={pn.PN_OPT_DELTA: 0.01, pn.PN_OPT_CHUNK: 7})
    compare(pn, oracle, net, 0, opts={pn.PN_OPT_X0: 0, pn.PN_OPT_KERNEL: 3})
    compare(pn, oracle, net, 0, opts={pn.PN_OPT_DELTA: 0.01, pn.PN_OPT_CHUNK: 7, pn.PN_OPT_KERNEL: 3})


# ---- closed forms straight on the GPU path (also pins of the oracle, see test_oracle_pins.py) ----
@pytest.mark.parametrize("direction", [0, 1, 2])
def test_uniform_closed_form(pn, direction):
    from paper_1908_03301_b200 import inputs
    net = inputs.uniform(9, 6, 5, 0.37)
    info, P, cls, fl, _ = gpu_solve(pn, net, direction, 1e-12)
    n_a = (9, 6, 5)[direction]
    s_perp = 9 * 6 * 5 // n_a
    assert fl[2] == pytest.approx(np.float64(np.float32(0.37)) * s_perp / (n_a - 1), rel=1e-12)
    assert fl[3] == pytest.approx(np.float64(np.float32(0.37)), rel=1e-12)
    c = np.arange(n_a) / (n_a - 1.0)
    shape = [1, 1, 1]
    shape[2 - direction] = n_a
    assert np.max(np.abs(P - (1.0 - c).reshape(shape))) < 1e-12


def test_layered_closed_form(pn):
    from paper_1908_03301_b200 import inputs
    rng = np.random.default_rng(5)
    nx, ny, nz = 12, 7, 9
    c = rng.uniform(0.2, 2.0, nz).astype(np.float32)
    e = rng.uniform(0.2, 2.0, nz).astype(np.float32)
    net = inputs.layered_exact(nx, ny, nz, c, e)
    _, _, _, flx, _ = gpu_solve(pn, net, 0, 1e-13)
    assert flx[2] == pytest.approx(ny * float(np.sum(c.astype(np.float64))) / (nx - 1), rel=1e-11)
    _, _, _, flz, _ = gpu_solve(pn, net, 2, 1e-13)
    assert flz[2] == pytest.approx(nx * ny / float(np.sum(1.0 / e[:-1].astype(np.float64))), rel=1e-11)


def test_worked_example_3x2(pn):
    """SURVEY.md 8(c) hand-worked example: P(1,0) = 27/71, P(1,1) = 29/71, G_eff = 170/71."""
    gx = np.array([[[1, 2, 99], [3, 4, 99]]], dtype=np.float32)
    gy = np.array([[[77, 5, 77], [88, 88, 88]]], dtype=np.float32)
    h = pn.Network(3, 2, 1)
    h.set_conductances(gx, gy, None)
    info = h.solve(0, 1e-13)
    P = h.pressures().cpu().numpy()
    fl = h.flux()
    h.close()
    assert info.status == pn.PN_OK
    assert P[0, 0, 1] == pytest.approx(27 / 71, abs=1e-13)
    assert P[0, 1, 1] == pytest.approx(29 / 71, abs=1e-13)
    assert fl[0] == pytest.approx(170 / 71, rel=1e-12)
    assert fl[1] == pytest.approx(170 / 71, rel=1e-12)


# ---- degenerate cases -----------------------------------------------------------------------------
def test_no_spanning_cluster(pn, oracle):
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(20, 18, 16, seed=3, p=0.08)
    info, P, fl, ref = compare(pn, oracle, net, 0)
    assert info.status == pn.PN_NO_SPANNING_CLUSTER and info.inner_iters == 0


def test_all_closed(pn, oracle):
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(8, 8, 8, seed=3, p=0.0)
    info, P, fl, ref = compare(pn, oracle, net, 2)
    assert info.n_floating == 8 * 8 * 6


def test_series_chain(pn):
    g = np.array([0.5, 2.0, 0.25, 4.0, 1.0, 9.0], dtype=np.float32)
    h = pn.Network(6, 1, 1)
    h.set_conductances(g, np.zeros(6, dtype=np.float32), None)
    info = h.solve(0, 1e-13)
    fl = h.flux()
    h.close()
    assert fl[2] == pytest.approx(1.0 / float(np.sum(1.0 / g[:5].astype(np.float64))), rel=1e-12)


def test_thin_axis(pn, oracle):
    """Three node planes along the solve axis: every unknown touches both Dirichlet planes."""
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.iid_diluted(3, 21, 10, seed=1, p=0.8), 0)
    compare(pn, oracle, inputs.iid_diluted(21, 10, 3, seed=1, p=0.8), 2)


def test_resolve_and_direction_switch(pn, oracle):
    """One handle, several solves: directions and networks can change between calls."""
    from paper_1908_03301_b200 import inputs
    a = inputs.iid_diluted(18, 14, 11, seed=21, p=0.7)
    b = inputs.iid_diluted(18, 14, 11, seed=22, p=1.0)
    h = pn.Network(18, 14, 11)
    for net, d in ((a, 0), (a, 2), (b, 1), (a, 0)):
        h.set_conductances(net.gx, net.gy, net.gz)
        info = h.solve(d, 1e-12)
        ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, d, 1e-13)
        assert np.max(np.abs(h.pressures().cpu().numpy() - ref.P)) <= P_TOL
        assert np.max(np.abs(h.pressures_host() - ref.P)) <= P_TOL
        assert abs(h.flux()[2] - ref.g_eff) <= G_TOL * abs(ref.g_eff)
    h.close()


def test_device_pointer_inputs(pn, oracle):
    import torch
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(24, 20, 16)
    h = pn.Network(net.nx, net.ny, net.nz)
    h.set_conductances(*(torch.from_numpy(g).cuda() for g in (net.gx, net.gy, net.gz)))
    h.solve(0, 1e-12)
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, 0, 1e-13)
    assert np.max(np.abs(h.pressures().cpu().numpy() - ref.P)) <= P_TOL
    h.close()


def test_error_paths(pn):
    h = pn.Network(8, 6, 4)
    with pytest.raises(pn.PnError) as e:
        h.solve(0, 1e-10)
    assert e.value.code == pn.PN_ERR_STATE
    g = np.ones((4, 6, 8), dtype=np.float32)
    bad = g.copy()
    bad[1, 2, 3] = -1.0
    with pytest.raises(pn.PnError) as e:
        h.set_conductances(bad, g, g)
    assert e.value.code == pn.PN_ERR_VALUE
    bad[1, 2, 3] = np.nan
    with pytest.raises(pn.PnError) as e:
        h.set_conductances(g, bad, g)
    assert e.value.code == pn.PN_ERR_VALUE
    # a bad value on an entry that is NOT a bond (forward neighbour off-lattice) is ignored
    edge = g.copy()
    edge[:, :, 7] = np.nan
    h.set_conductances(edge, g, g)
    with pytest.raises(pn.PnError) as e:
        h.set_conductances(g, g, None)
    assert e.value.code == pn.PN_ERR_ARG
    h.set_conductances(g, g, g)
    for d, tol in ((3, 1e-10), (-1, 1e-10), (0, 0.0), (0, 2.0)):
        with pytest.raises(pn.PnError) as e:
            h.solve(d, tol)
        assert e.value.code == pn.PN_ERR_ARG
    with pytest.raises(pn.PnError) as e:
        h.flux()
    assert e.value.code == pn.PN_ERR_STATE
    h.solve(1, 1e-10)
    h.flux()
    h.close()
    h2 = pn.Network(8, 2, 1)
    h2.set_conductances(np.ones(16, dtype=np.float32), np.ones(16, dtype=np.float32), None)
    with pytest.raises(pn.PnError) as e:
        h2.solve(1, 1e-10)          # only 2 node planes along y
    assert e.value.code == pn.PN_ERR_ARG
    h2.close()


def test_max_iters_status(pn):
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg2_fbm_2d(128, 128)
    for kernel in (1, 3, 8):
        info, *_ = gpu_solve(pn, net, 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 40, pn.PN_OPT_KERNEL: kernel})
        assert info.status == pn.PN_MAX_ITERS
        assert 40 <= info.inner_iters <= 40 + 64
        assert info.rel_residual > 1e-12


def test_deterministic(pn):
    """Fixed-order grid reductions: two solves of the same input agree bit for bit."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(40, 40, 40)
    for kernel in (1, 3, 8):
        a = gpu_solve(pn, net, 0, 1e-10, opts={pn.PN_OPT_KERNEL: kernel})
        b = gpu_solve(pn, net, 0, 1e-10, opts={pn.PN_OPT_KERNEL: kernel})
        assert a[0].inner_iters == b[0].inner_iters
        assert np.array_equal(a[1], b[1])
        assert a[3] == b[3]


# ---- dead-end peeling: integer work bit-exact, pressures of ALL nodes unchanged ----
def _oracle_dangling(net, classes):
    from oracle import pn_oracle as po
    g64 = po.widen(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz)
    return po.dangling_ends(net.nx, net.ny, net.nz, g64, classes)


@pytest.mark.parametrize("maker,direction", [
    (lambda i: i.cfg3_percolation_3d(64, 64, 64), 0), (lambda i: i.cfg3_percolation_3d(40, 33, 50), 2),
    (lambda i: i.cfg4_fbm_cut_3d(48, 40, 36), 1), (lambda i: i.iid_diluted(150, 120, 1, seed=4, p=0.62), 0),
    (lambda i: i.iid_diluted(150, 120, 1, seed=4, p=0.62), 1)])
def test_peeling_count_and_parity(pn, oracle, maker, direction):
    """The number of peeled nodes equals the oracle's serial leaf stripping (the 2-core is unique, so the
    asynchronous GPU peeling must remove exactly the same set); pressures and G_eff pass the same parity bar with
    and without peeling (peeled nodes are back-filled).  The iteration count is NOT guaranteed to fall (measured at
    512^3 on CFG4: 3.8 % peeled, +1.8 % iterations); only a gross regression is checked here."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    on, P_on, fl_on, ref = compare(pn, oracle, net, direction, opts={pn.PN_OPT_PEEL: 1})
    off, P_off, fl_off, _ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_PEEL: 0})
    mask = _oracle_dangling(net, ref.classes)
    assert on.n_peeled == int(mask.sum()) > 0
    assert off.n_peeled == 0
    assert on.n_solved == off.n_solved == ref.n_solved
    assert on.inner_iters <= 1.1 * off.inner_iters
    # a peeled node sits exactly at the pressure of some neighbour (the one it hangs from)
    P = P_on
    nb = np.full(P.shape, np.inf)
    for ax in range(3):
        for sh in (1, -1):
            d = np.abs(P - np.roll(P, sh, axis=ax))
            sl = [slice(None)] * 3
            sl[ax] = 0 if sh == 1 else -1
            d[tuple(sl)] = np.inf            # no wrap-around neighbours
            nb = np.minimum(nb, d)
    assert float(np.max(nb[mask])) == 0.0


def test_peeling_long_chain(pn, oracle):
    """A dangling chain of 300 nodes hanging from a uniform backbone: one asynchronous walk peels all of it."""
    nx, ny = 304, 3
    gx = np.zeros((1, ny, nx), dtype=np.float32)
    gy = np.zeros((1, ny, nx), dtype=np.float32)
    gx[0, 0, :nx - 1] = 1.0                  # backbone along the bottom row
    gy[0, 0, 1] = 0.5                        # stub up from (1,0) ...
    gy[0, 1, 1] = 0.5
    gx[0, 2, 1:301] = 2.0                    # ... then 300 nodes along the top row
    from paper_1908_03301_b200.inputs import Network
    net = Network(nx, ny, 1, gx, gy, None, name="chain")
    info, P, fl, ref = compare(pn, oracle, net, 0)
    assert info.n_peeled == 302
    assert np.all(P[0, 2, 1:302] == P[0, 0, 1])
    assert fl[2] == pytest.approx(1.0 / (nx - 1), rel=1e-12)


def test_warm_start(pn, oracle):
    """PN_OPT_X0 = 2: re-solve after a small change of the conductances starting from the
    previous pressures -- same parity bar, far fewer iterations than a cold solve."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(64, 64, 64)
    rng = np.random.default_rng(8)
    bump = lambda g: (g * (1.0 + 1e-5 * rng.standard_normal(g.shape))).astype(np.float32)   # zeros stay zero
    gx2, gy2, gz2 = bump(net.gx), bump(net.gy), bump(net.gz)
    ref = oracle.solve(net.nx, net.ny, net.nz, gx2, gy2, gz2, 0, 1e-13)
    h = pn.Network(net.nx, net.ny, net.nz)
    h.set_option(pn.PN_OPT_X0, 2)
    h.set_conductances(net.gx, net.gy, net.gz)
    first = h.solve(0, 1e-12)                          # nothing to start from: linear profile
    h.set_conductances(gx2, gy2, gz2)
    warm = h.solve(0, 1e-12)
    P = h.pressures().cpu().numpy()
    g_eff = h.flux()[2]
    h.set_option(pn.PN_OPT_X0, 1)
    cold = h.solve(0, 1e-12)
    h.close()
    assert np.max(np.abs(P - ref.P)) <= P_TOL
    assert abs(g_eff - ref.g_eff) <= G_TOL * abs(ref.g_eff)
    assert warm.inner_iters < 0.85 * cold.inner_iters
    assert first.inner_iters == pytest.approx(cold.inner_iters, rel=0.1)


def test_peeling_automatic_policy(pn, oracle):
    """PN_OPT_PEEL = 2 (the default): the peeling is kept when it removes >= 10 % of the solved nodes (CFG3-like,
    52 %) and undone below that (CFG4-like, 6 %) -- k_unpeel must restore the solve copy exactly, so the solve is
    bit-identical to one that never peeled."""
    from paper_1908_03301_b200 import inputs
    near = inputs.cfg3_percolation_3d(64, 64, 64)
    info, P, fl, ref = compare(pn, oracle, near, 0)                      # default options
    assert info.n_peeled == int(_oracle_dangling(near, ref.classes).sum()) >= 0.1 * info.n_solved
    far = inputs.cfg4_fbm_cut_3d(64, 64, 64)
    auto, P_auto, fl_auto, ref = compare(pn, oracle, far, 0)
    mask = _oracle_dangling(far, ref.classes)
    assert 0 < int(mask.sum()) < 0.1 * auto.n_solved and auto.n_peeled == 0
    never, P_never, fl_never, _ = compare(pn, oracle, far, 0, opts={pn.PN_OPT_PEEL: 0})
    assert auto.inner_iters == never.inner_iters
    assert np.array_equal(P_auto, P_never) and fl_auto == fl_never


# ---- periodic lateral faces: PN_OPT_LATERAL = 1 against the oracle's periodic=True ----
@pytest.mark.parametrize("shape", [(17, 9, 5), (5, 17, 9), (9, 5, 17), (33, 2, 7), (12, 6, 2)])
@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("p", [1.0, 0.6])
@pytest.mark.parametrize("kernel", [1, 3, 8])
def test_periodic_ragged_3d(pn, oracle, shape, direction, p, kernel):
    """All three kernel schemes; lateral axes of length 2 (a doubled bond) included."""
    from paper_1908_03301_b200 import inputs
    if shape[direction] < 3:
        pytest.skip("solve axis needs 3 node planes")
    net = inputs.iid_diluted(*shape, seed=17 + direction, p=p)
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: kernel}, periodic=True)


@pytest.mark.parametrize("shape", [(19, 13), (13, 19), (64, 3), (257, 31)])
@pytest.mark.parametrize("direction", [0, 1])
@pytest.mark.parametrize("kernel", [1, 3, 8])
def test_periodic_ragged_2d(pn, oracle, shape, direction, kernel):
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(shape[0], shape[1], 1, seed=13 + direction, p=0.75)
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: kernel}, periodic=True)


@pytest.mark.parametrize("kernel,tile", [(3, 1), (3, 2), (3, 3), (8, 0)])
@pytest.mark.parametrize("shape,direction", [((300, 20, 70), 2), ((520, 9, 12), 1), ((260, 17, 40), 0)])
def test_periodic_multi_tile(pn, oracle, shape, direction, kernel, tile):
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(*shape, seed=6, p=0.75)
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: kernel, pn.PN_OPT_TILE: tile}, periodic=True)


def test_periodic_config_siblings(pn, oracle):
    from paper_1908_03301_b200 import inputs
    compare(pn, oracle, inputs.cfg2_fbm_2d(256, 256), 0, periodic=True)
    compare(pn, oracle, inputs.cfg4_fbm_cut_3d(128, 128, 128), 0, tol=1e-13, periodic=True)    # automatic: persistent kernel, WRAP form
    compare(pn, oracle, inputs.cfg4_fbm_cut_3d(96, 80, 72), 1, periodic=True, opts={pn.PN_OPT_KERNEL: 3})   # fused TMA kernel + k_wrap_fix
    info, P, fl, ref = compare(pn, oracle, inputs.cfg3_percolation_3d(64, 64, 64), 0, periodic=True)
    from oracle import pn_oracle as po
    net = inputs.cfg3_percolation_3d(64, 64, 64)
    wrap = po.wrap_axes(64, 64, 64, 0, True)
    g64 = po.widen(64, 64, 64, net.gx, net.gy, net.gz, wrap)
    assert info.n_peeled == int(po.dangling_ends(64, 64, 64, g64, ref.classes, wrap).sum()) > 0


def test_periodic_closed_forms(pn):
    """Hand-worked golden example (tests/golden/worked_3x2_periodic.txt) and the uniform network."""
    gx = np.array([[[1, 2, 99], [3, 4, 99]]], dtype=np.float32)
    gy = np.array([[[77, 5, 77], [88, 7, 88]]], dtype=np.float32)
    h = pn.Network(3, 2, 1)
    h.set_option(pn.PN_OPT_LATERAL, 1)
    h.set_conductances(gx, gy, None)
    h.solve(0, 1e-13)
    P = h.pressures().cpu().numpy()
    fl = h.flux()
    h.close()
    assert P[0, 0, 1] == pytest.approx(55 / 141, abs=1e-13)
    assert P[0, 1, 1] == pytest.approx(57 / 141, abs=1e-13)
    assert fl[0] == pytest.approx(338 / 141, rel=1e-12) and fl[1] == pytest.approx(338 / 141, rel=1e-12)
    from paper_1908_03301_b200 import inputs
    net = inputs.uniform(9, 6, 5, 0.37)
    for d in range(3):
        info, P, cls, fl, _ = gpu_solve(pn, net, d, 1e-12, opts={pn.PN_OPT_LATERAL: 1})
        n_a = (9, 6, 5)[d]
        assert fl[2] == pytest.approx(np.float64(np.float32(0.37)) * (270 // n_a) / (n_a - 1), rel=1e-12)


def test_periodic_validates_wrap_entries(pn):
    """With wrapping axes the forward entry of a last node is a bond: a NaN there is PN_ERR_VALUE at pn_solve, and
    is still ignored with no-flux faces."""
    g = np.ones((4, 6, 8), dtype=np.float32)
    bad = g.copy()
    bad[2, 5, 3] = np.nan                      # gy of the last row: off-lattice unless y wraps
    h = pn.Network(8, 6, 4)
    h.set_conductances(g, bad, g)
    h.solve(0, 1e-10)
    h.set_option(pn.PN_OPT_LATERAL, 1)
    with pytest.raises(pn.PnError) as e:
        h.solve(0, 1e-10)
    assert e.value.code == pn.PN_ERR_VALUE
    h.solve(1, 1e-10)                          # y is the solve axis: it does not wrap, the entry is ignored again
    h.close()


def test_anisotropic_fbm_both_directions(pn, oracle):
    """Eq.(2) input (S8(f) item 3), periodic faces, x and y solves on one handle: parity in both directions, and
    layers parallel to x (beta_x / beta_y = 16) conduct better along x than across."""
    from paper_1908_03301_b200 import inputs
    net = inputs.aniso_fbm_2d(160, 128, 3, 0.75, 4.0, 0.25)
    k = []
    for d in net.directions:
        info, P, fl, ref = compare(pn, oracle, net, d, periodic=True)
        k.append(fl[3])
        assert fl[3] == pytest.approx(ref.k_eff, rel=1e-9)
    assert k[0] > k[1]


@pytest.mark.parametrize("kernel", [1, 3])
def test_graph_replay_is_bit_identical(pn, kernel):
    """PN_OPT_GRAPH: replaying chunks from a CUDA graph launches the same kernels on the same data -- pressures,
    fluxes and iteration counts are identical to direct launches; the graph is reused across solves of one handle.
    (The fused TMA kernel is replayed from a graph only with periodic faces -- otherwise PN_OPT_GRAPH = 1 means its
    persistent cooperative form, whose sums are grouped differently: test_persistent_launch_of_the_tma_kernel.)"""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(48, 48, 48)
    base = {pn.PN_OPT_KERNEL: kernel, pn.PN_OPT_LATERAL: 1 if kernel == 3 else 0}
    a = gpu_solve(pn, net, 0, 1e-10, opts={**base, pn.PN_OPT_GRAPH: 1})
    b = gpu_solve(pn, net, 0, 1e-10, opts={**base, pn.PN_OPT_GRAPH: 0})
    assert a[0].inner_iters == b[0].inner_iters and a[0].outer_cycles == b[0].outer_cycles
    assert np.array_equal(a[1], b[1]) and a[3] == b[3]
    assert a[4] == b[4]                                   # same launch count
    h = pn.Network(net.nx, net.ny, net.nz)
    for k, v in base.items():
        h.set_option(k, v)
    h.set_conductances(net.gx, net.gy, net.gz)
    for d in (0, 1, 0, 2):                                # direction changes force a re-capture
        h.solve(d, 1e-10)
        P = h.pressures().cpu().numpy()
        ref = gpu_solve(pn, net, d, 1e-10, opts={**base, pn.PN_OPT_GRAPH: 0})
        assert np.array_equal(P, ref[1])
    h.close()


def test_persistent_launch_of_the_tma_kernel(pn, oracle):
    """PN_OPT_KERNEL = 3 with PN_OPT_GRAPH = 1 (default) and no periodic faces: the fused TMA kernel runs as ONE cooperative
    launch per residual replacement.  Same parity bar, the iteration count of the launch-per-iteration form to a few per
    cent (the dot products are grouped per CTA instead of per block), far fewer launches, and bit-reproducible."""
    from paper_1908_03301_b200 import inputs
    for net, d in ((inputs.cfg4_fbm_cut_3d(64, 64, 64), 0), (inputs.iid_diluted(300, 20, 70, seed=5, p=0.75), 2),
                   (inputs.iid_diluted(130, 40, 21, seed=9, p=1.0), 1)):
        on, *_ = compare(pn, oracle, net, d, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0})
        off, *_ = compare(pn, oracle, net, d, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0, pn.PN_OPT_GRAPH: 0})
        assert on.kernel_scheme == off.kernel_scheme == 3
        assert on.residual_recovered == 1 and off.residual_recovered == 1   # no fp32 residual is stored, in either launch form
        assert abs(on.inner_iters - off.inner_iters) <= 0.05 * off.inner_iters + 5
        for chunk in (1, 2, 3, 7):    # launch boundaries at every phase of the three rotating direction slots
            cut, *_ = compare(pn, oracle, net, d, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0, pn.PN_OPT_CHUNK: chunk})
            assert cut.residual_recovered == 1 and abs(cut.inner_iters - on.inner_iters) <= 0.05 * on.inner_iters + 5
        nodefer, *_ = compare(pn, oracle, net, d, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0, pn.PN_OPT_XDEFER: 0})
        assert nodefer.residual_recovered == 1 and nodefer.n_xskip == 0
        a = gpu_solve(pn, net, d, 1e-10, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0})
        b = gpu_solve(pn, net, d, 1e-10, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0})
        c = gpu_solve(pn, net, d, 1e-10, opts={pn.PN_OPT_KERNEL: 3, pn.PN_OPT_COMPACT: 0, pn.PN_OPT_GRAPH: 0})
        assert a[0].inner_iters == b[0].inner_iters and np.array_equal(a[1], b[1]) and a[3] == b[3]
        assert a[4] < c[4] / 5                            # launches
    info, *_ = gpu_solve(pn, inputs.cfg2_fbm_2d(300, 200), 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 40, pn.PN_OPT_KERNEL: 3})
    assert info.status == pn.PN_MAX_ITERS and info.inner_iters == 40
    info, *_ = gpu_solve(pn, inputs.cfg4_fbm_cut_3d(40, 36, 33), 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 40, pn.PN_OPT_KERNEL: 3})
    assert info.status == pn.PN_MAX_ITERS and info.inner_iters == 40 and info.residual_recovered == 1
    flat, _, _, _, n_launch = gpu_solve(pn, inputs.iid_diluted(2100, 40, 1, seed=9, p=1.0), 1, 1e-12, opts={pn.PN_OPT_KERNEL: 3})
    assert flat.kernel_scheme == 3 and flat.residual_recovered == 1
    assert n_launch > flat.inner_iters                  # the 2D tile keeps one launch per iteration (measured faster)


@pytest.mark.parametrize("maker,direction,periodic", [
    (lambda i: i.cfg4_fbm_cut_3d(64, 64, 64), 0, False), (lambda i: i.cfg3_percolation_3d(40, 33, 50), 2, True),
    (lambda i: i.cfg2_fbm_2d(300, 200), 1, False), (lambda i: i.iid_diluted(17, 9, 5, seed=3, p=0.7), 0, True)])
def test_deferred_solution_update(pn, oracle, maker, direction, periodic):
    """PN_OPT_XDEFER: the single-kernel scheme folds two search directions into x_hat every other iteration (the earlier
    one recovered as (p - r) / beta).  Same parity bar with it on (default) and off, for odd and even iteration counts
    at the flush (several residual replacements per solve hit both), and a comparable iteration count."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    on, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_XDEFER: 1, pn.PN_OPT_KERNEL: 3}, periodic=periodic)
    off, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_XDEFER: 0, pn.PN_OPT_KERNEL: 3}, periodic=periodic)
    assert on.inner_iters <= 1.05 * off.inner_iters + 5
    for chunk in (1, 5):        # host polls at other iteration parities
        compare(pn, oracle, net, direction, opts={pn.PN_OPT_CHUNK: chunk, pn.PN_OPT_KERNEL: 3}, periodic=periodic)


def test_residual_history(pn):
    """pn_residual_history: one true fp64 residual per evaluation, strictly falling from the initial guess to the exit
    value reported in pn_info (reliable updates: every replacement sees a residual at least ~10x smaller)."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(48, 40, 36)
    h = pn.Network(net.nx, net.ny, net.nz)
    assert h.residual_history() == []
    h.set_conductances(net.gx, net.gy, net.gz)
    info = h.solve(0, 1e-11)
    hist = h.residual_history()
    h.close()
    assert len(hist) == info.outer_cycles >= 3
    assert hist[-1] == info.rel_residual <= 1e-11
    assert all(b < a for a, b in zip(hist, hist[1:]))
    assert 1e-3 < hist[0] < 10.0


def test_option_changes_between_solves_on_one_handle(pn, oracle):
    """The cached CUDA graph, the face arrays and the peeling state must follow every option change: each solve on a
    long-lived handle equals, bit for bit, the same solve on a fresh handle."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(40, 36, 33)
    steps = [({}, 0), ({pn.PN_OPT_CHUNK: 5}, 0), ({pn.PN_OPT_LATERAL: 1}, 0), ({pn.PN_OPT_LATERAL: 1}, 2),
             ({pn.PN_OPT_LATERAL: 0, pn.PN_OPT_KERNEL: 1}, 1), ({pn.PN_OPT_KERNEL: 3, pn.PN_OPT_PEEL: 0}, 1),
             ({pn.PN_OPT_KERNEL: 0, pn.PN_OPT_PEEL: 2, pn.PN_OPT_XDEFER: 0, pn.PN_OPT_CHUNK: 32}, 0)]
    h = pn.Network(net.nx, net.ny, net.nz)
    h.set_conductances(net.gx, net.gy, net.gz)
    sticky = {}
    for opts, d in steps:
        sticky.update(opts)
        for k, v in opts.items():
            h.set_option(k, v)
        info = h.solve(d, 1e-11)
        P = h.pressures().cpu().numpy()
        fl = h.flux()
        fresh = gpu_solve(pn, net, d, 1e-11, opts=sticky)
        assert info.inner_iters == fresh[0].inner_iters and info.n_peeled == fresh[0].n_peeled
        assert np.array_equal(P, fresh[1]) and fl == fresh[3]
    h.close()
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, 0, 1e-13)
    assert np.max(np.abs(P - ref.P)) <= 1e-7          # tol 1e-11 here; the parity bar proper is tested at 1e-12


@pytest.mark.parametrize("maker,direction,periodic", [
    (lambda i: i.cfg3_percolation_3d(64, 64, 64), 0, False), (lambda i: i.cfg4_fbm_cut_3d(64, 64, 64), 2, True),
    (lambda i: i.cfg2_fbm_2d(256, 256), 0, False)])
def test_dissipation_estimate_meets_1e9_at_the_timing_tolerance(pn, oracle, maker, direction, periodic):
    """pn_dissipation: G_E = sum_bonds g dP^2 has an error quadratic in that of the pressures (SURVEY.md 8(c) consequence
    (iv)), so it meets north_star's 1e-9 on the effective conductance already at tol = 1e-10 -- the tolerance bench.py
    times -- where the boundary-flux G_eff is only good to a few 1e-9."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13, periodic=periodic)
    h = pn.Network(net.nx, net.ny, net.nz)
    h.set_option(pn.PN_OPT_LATERAL, 1 if periodic else 0)
    with pytest.raises(pn.PnError) as e:
        h.dissipation()
    assert e.value.code == pn.PN_ERR_STATE
    h.set_conductances(net.gx, net.gy, net.gz)
    h.solve(direction, 1e-10)
    g_e, g_eff = h.dissipation(), h.flux()[2]
    h.close()
    assert abs(g_e - ref.g_eff) <= 1e-10 * ref.g_eff
    assert abs(g_eff - ref.g_eff) <= 1e-7 * ref.g_eff


@pytest.mark.parametrize("maker,direction,bound", [
    (lambda i: i.cfg4_fbm_cut_3d(96, 96, 96), 0, 1.35), (lambda i: i.cfg3_percolation_3d(64, 64, 64), 0, 1.35),
    (lambda i: i.cfg5_stratified_3d(64, 64, 64), 2, 1.35), (lambda i: i.cfg2_fbm_2d(512, 512), 0, 1.35)])
def test_iteration_count_close_to_fp64_cg(pn, oracle, maker, direction, bound):
    """DESIGN.md reading 4: the never-restarted fp32 CG with fp64 residual replacements ("reliable updates") stays within
    SURVEY.md 8(c)'s 1.0 - 1.35x of the iterations the oracle's fp64 Jacobi-PCG needs to the same 1e-10 residual, compared
    like for like (zero start, no peeling).  Measured on B200: +1.3 % (CFG4 160^3), +5.8 % (CFG4 256^3), +16 % (CFG4 96^3),
    +1 % (CFG3 128^3), +0.8 % (CFG5 128^3), +23 % (CFG2 1024^2); restarted refinement would cost 1.3 - 2x."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-10)
    info, *_ = gpu_solve(pn, net, direction, 1e-10, opts={pn.PN_OPT_X0: 0, pn.PN_OPT_PEEL: 0})
    assert info.status == pn.PN_OK and info.rel_residual <= 1e-10
    assert info.inner_iters <= bound * ref.iterations
    assert info.inner_iters >= 0.8 * ref.iterations


# ---- lattices that fit one SM's shared memory: the whole inner loop in one launch (pn_onchip.cu, scheme 5) ----
@pytest.mark.parametrize("maker,direction", [
    (lambda i: i.cfg1_iid_2d(), 0), (lambda i: i.cfg1_iid_2d(), 1), (lambda i: i.iid_diluted(17, 9, 5, seed=7, p=0.6), 0),
    (lambda i: i.iid_diluted(5, 17, 9, seed=8, p=1.0), 1), (lambda i: i.iid_diluted(9, 5, 17, seed=9, p=0.6), 2),
    (lambda i: i.iid_diluted(19, 13, 1, seed=11, p=0.7), 1), (lambda i: i.iid_diluted(64, 3, 1, seed=11, p=1.0), 0),
    (lambda i: i.cfg3_percolation_3d(16, 16, 16, p=0.4), 0), (lambda i: i.cfg4_fbm_cut_3d(18, 16, 14), 2),
    (lambda i: i.cfg5_stratified_3d(16, 16, 16), 2)])
def test_onchip_scheme(pn, oracle, maker, direction):
    """Scheme 5 is the automatic choice on these sizes; same parity bar, iteration count that of the reference
    two-kernel scheme to within ~10 % (same arithmetic, other summation order; a replacement more or less)."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    auto, P5, fl5, ref = compare(pn, oracle, net, direction)
    assert auto.kernel_scheme == 5
    k1, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 1})
    assert k1.kernel_scheme == 1
    assert abs(auto.inner_iters - k1.inner_iters) <= 0.15 * k1.inner_iters + 8
    # the launch count shows the point: one launch per residual replacement instead of two per iteration
    _, _, _, _, n5 = gpu_solve(pn, net, direction, 1e-12)
    _, _, _, _, n1 = gpu_solve(pn, net, direction, 1e-12, opts={pn.PN_OPT_KERNEL: 1})
    assert n5 < n1


def test_onchip_scheme_options(pn, oracle):
    """Budget, zero start, warm start, peeling and the fall-back for periodic faces / large lattices."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(16, 16, 16, p=0.4)
    info, *_ = gpu_solve(pn, net, 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 10})
    assert info.status == pn.PN_MAX_ITERS and info.kernel_scheme == 5 and info.inner_iters == 10
    compare(pn, oracle, net, 0, opts={pn.PN_OPT_X0: 0, pn.PN_OPT_DELTA: 0.01})
    on, *_ = compare(pn, oracle, net, 0, opts={pn.PN_OPT_PEEL: 1})
    assert on.n_peeled > 0 and on.kernel_scheme == 5
    per, *_ = compare(pn, oracle, net, 0, periodic=True)
    assert per.kernel_scheme == 8                       # periodic faces on a small lattice: the persistent kernel's WRAP form
    big, *_ = compare(pn, oracle, inputs.cfg3_percolation_3d(24, 24, 24, p=0.4), 0, opts={pn.PN_OPT_KERNEL: 5})
    assert big.kernel_scheme == 3                       # 24^3 does not fit: falls back
    a = gpu_solve(pn, net, 0, 1e-10)
    b = gpu_solve(pn, net, 0, 1e-10)
    assert np.array_equal(a[1], b[1]) and a[0].inner_iters == b[0].inner_iters      # deterministic


# ---- handles are independent: no process-global state behind the per-handle API (include/pn.h "Ownership") ----
def test_handles_on_streams_and_recreate(pn, oracle):
    """create / solve / destroy / create again on the same device with another stream; two live handles interleaved."""
    import torch
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(40, 36, 33)
    ref = oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, 0, 1e-13)
    first = gpu_solve(pn, net, 0, 1e-12)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    a = pn.Network(net.nx, net.ny, net.nz, stream=s1)
    b = pn.Network(net.nx, net.ny, net.nz, stream=s2)
    a.set_conductances(net.gx, net.gy, net.gz)
    b.set_conductances(net.gx, net.gy, net.gz)
    ia = a.solve(0, 1e-12)
    ib = b.solve(0, 1e-12)
    Pa, Pb = a.pressures().cpu().numpy(), b.pressures().cpu().numpy()
    a.close()
    ib2 = b.solve(0, 1e-12)                         # the surviving handle is unaffected by the other's destruction
    Pb2 = b.pressures().cpu().numpy()
    b.close()
    assert ia.inner_iters == ib.inner_iters == ib2.inner_iters == first[0].inner_iters
    assert np.array_equal(Pa, Pb) and np.array_equal(Pb, Pb2) and np.array_equal(Pa, first[1])
    assert float(np.max(np.abs(Pa - ref.P))) <= P_TOL


def test_two_devices_in_one_process(pn, oracle):
    """Handles on two GPUs in ONE process (the large-shared-memory opt-in and the SM count are per device)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(40, 36, 33)
    out = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            h = pn.Network(net.nx, net.ny, net.nz, device=dev)
            h.set_conductances(net.gx, net.gy, net.gz)
            info = h.solve(0, 1e-12)
            out.append((info.inner_iters, h.pressures().cpu().numpy()))
            h.close()
    assert out[0][0] == out[1][0] and np.array_equal(out[0][1], out[1][1])


def test_removed_kernel_schemes_are_refused(pn):
    h = pn.Network(8, 8, 1)
    for k in (2, 4, 7):
        with pytest.raises(pn.PnError) as e:
            h.set_option(pn.PN_OPT_KERNEL, k)
        assert e.value.code == pn.PN_ERR_ARG
    h.close()


# ---- persistent in-place kernel for 2D lattices (pn_resident.cu, scheme 6) ----
@pytest.mark.parametrize("shape,direction,p", [
    ((1024, 300), 0, 1.0), ((2048, 160), 1, 1.0), ((600, 1000), 0, 0.7), ((513, 149), 1, 0.8), ((260, 400), 0, 1.0),
    ((100, 2), 0, 1.0), ((7, 500), 1, 1.0)])
def test_resident_scheme(pn, oracle, shape, direction, p):
    """All four row widths (1, 2, 4, 8 TMA boxes), more rows than CTAs and fewer, one row per CTA, ragged widths; the
    automatic choice for every 2D lattice up to 2048 wide that does not fit one SM.  Iteration counts stay those of the
    one-launch-per-iteration kernel (same arithmetic per node; only the summation order of the dot products differs)."""
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(shape[0], shape[1], 1, seed=21, p=p)
    auto, *_ = compare(pn, oracle, net, direction)
    assert auto.kernel_scheme == (5 if shape[0] * shape[1] < 6000 else 6)
    k6, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 6})
    k3, *_ = compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 3})
    assert k6.kernel_scheme == 6 and k3.kernel_scheme == 3
    assert abs(k6.inner_iters - k3.inner_iters) <= 0.05 * k3.inner_iters + 5
    compare(pn, oracle, net, direction, opts={pn.PN_OPT_KERNEL: 6, pn.PN_OPT_XDEFER: 0, pn.PN_OPT_DELTA: 0.01})


def test_resident_scheme_fallbacks_and_budget(pn, oracle):
    from paper_1908_03301_b200 import inputs
    wide, *_ = compare(pn, oracle, inputs.iid_diluted(2100, 40, 1, seed=9, p=1.0), 1, opts={pn.PN_OPT_KERNEL: 6})
    assert wide.kernel_scheme == 3                       # wider than 2048: the tiled kernel
    cube, *_ = compare(pn, oracle, inputs.cfg4_fbm_cut_3d(40, 36, 33), 0, opts={pn.PN_OPT_KERNEL: 6})
    assert cube.kernel_scheme == 3                       # 3D
    per, *_ = compare(pn, oracle, inputs.cfg2_fbm_2d(300, 200), 0, opts={pn.PN_OPT_KERNEL: 6}, periodic=True)
    assert per.kernel_scheme == 3                        # periodic faces
    net = inputs.cfg2_fbm_2d(300, 200)
    info, *_ = gpu_solve(pn, net, 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 40, pn.PN_OPT_KERNEL: 6})
    assert info.status == pn.PN_MAX_ITERS and info.kernel_scheme == 6 and info.inner_iters == 40
    a = gpu_solve(pn, net, 0, 1e-10, opts={pn.PN_OPT_KERNEL: 6})
    b = gpu_solve(pn, net, 0, 1e-10, opts={pn.PN_OPT_KERNEL: 6})
    assert a[0].inner_iters == b[0].inner_iters and np.array_equal(a[1], b[1]) and a[3] == b[3]   # bit-reproducible


# ---- active-node compaction (pn_compact.cu, kernel_scheme 7) ----
@pytest.mark.parametrize("maker,direction", [
    (lambda i: i.cfg3_percolation_3d(64, 64, 64), 0), (lambda i: i.cfg3_percolation_3d(40, 36, 33, p=0.32), 2),
    (lambda i: i.cfg3_percolation_3d(66, 35, 33, p=0.29), 1), (lambda i: i.cfg3_percolation_3d(130, 30, 27, p=0.31), 0),
    (lambda i: i.iid_diluted(257, 131, 1, seed=6, p=0.515), 1), (lambda i: i.iid_diluted(300, 520, 1, seed=8, p=0.51), 0)])
def test_compacted_unknowns(pn, oracle, maker, direction):
    """PN_OPT_COMPACT = 1 forces the CSR form wherever its table fits the workspace (at most one entry per padded lattice
    node: networks near their threshold, 2D and 3D, ragged shapes, with and without peeling): pressures of ALL nodes,
    classes and G_eff keep the parity bar; iteration counts stay those of the structured kernel to a few per cent (same
    recurrences; the operator's sum is ordered differently)."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    # tol 1e-13: on these small near-threshold networks G_eff is carried by a few paths (1e-12 leaves ~2e-9 in it)
    on, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={pn.PN_OPT_COMPACT: 1, pn.PN_OPT_KERNEL: 3, pn.PN_OPT_CONTRACT: 0})
    off, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={pn.PN_OPT_COMPACT: 0, pn.PN_OPT_KERNEL: 3})
    assert on.kernel_scheme == 7 and off.kernel_scheme == 3
    assert on.n_unknowns == off.n_unknowns == on.n_solved - on.n_peeled
    assert abs(on.inner_iters - off.inner_iters) <= 0.05 * off.inner_iters + 5
    compare(pn, oracle, net, direction, tol=1e-13, opts={pn.PN_OPT_COMPACT: 1, pn.PN_OPT_KERNEL: 3, pn.PN_OPT_PEEL: 0,
                                                         pn.PN_OPT_GRAPH: 0, pn.PN_OPT_CHUNK: 7, pn.PN_OPT_X0: 0,
                                                         pn.PN_OPT_CONTRACT: 0})


def test_compaction_policy_and_determinism(pn, oracle):
    from paper_1908_03301_b200 import inputs
    near = inputs.cfg3_percolation_3d(64, 64, 64)             # p = 0.30: a third of the nodes are unknowns after peeling
    auto, *_ = compare(pn, oracle, near, 0)
    assert auto.kernel_scheme == 7 and auto.n_unknowns < 0.45 * near.n_nodes
    dense = inputs.cfg5_stratified_3d(32, 32, 32)
    d, *_ = compare(pn, oracle, dense, 0)
    assert d.kernel_scheme == 8                                # nothing to skip: a structured kernel (small lattice: persistent)
    per, *_ = compare(pn, oracle, near, 0, periodic=True)
    assert per.kernel_scheme == 8                              # periodic faces: a structured kernel (wrap bonds inside it)
    forced, *_ = compare(pn, oracle, near, 0, opts={pn.PN_OPT_KERNEL: 3})
    assert forced.kernel_scheme == 3                           # an explicit kernel choice is honoured
    full, *_ = compare(pn, oracle, inputs.cfg4_fbm_cut_3d(48, 40, 36), 1, opts={pn.PN_OPT_COMPACT: 1})
    assert full.kernel_scheme == 8                             # table larger than the workspace arrays: structured kernel
    a = gpu_solve(pn, near, 0, 1e-10)
    b = gpu_solve(pn, near, 0, 1e-10)
    assert a[0].inner_iters == b[0].inner_iters and np.array_equal(a[1], b[1]) and a[3] == b[3]
    info, *_ = gpu_solve(pn, near, 0, 1e-12, opts={pn.PN_OPT_MAX_ITERS: 40})
    assert info.status == pn.PN_MAX_ITERS and info.kernel_scheme == 7 and 40 <= info.inner_iters <= 40 + 64


def test_automatic_kernel_choice_by_size(pn, oracle):
    """0 = automatic: one CTA (5) / resident 2D slabs (6) / the persistent structured kernel up to 5 000 000 padded nodes (8; periodic
    faces included) / the fused TMA kernel above (3: tests/test_gpu_fullsize.py) -- all through the
    same parity bar."""
    from paper_1908_03301_b200 import inputs
    for net, d, want in ((inputs.cfg5_stratified_3d(16, 16, 16), 0, 5), (inputs.cfg2_fbm_2d(300, 200), 0, 6),
                         (inputs.cfg5_stratified_3d(64, 64, 64), 2, 8), (inputs.cfg5_stratified_3d(96, 96, 80), 0, 8)):
        info, *_ = compare(pn, oracle, net, d)
        assert info.kernel_scheme == want, (net.name, info.kernel_scheme)


# ---- degree-2 chain elimination on top of the compacted unknowns (pn_chain.cu, PN_OPT_CONTRACT) ----
@pytest.mark.parametrize("maker,direction", [
    (lambda i: i.cfg3_percolation_3d(64, 64, 64), 0), (lambda i: i.cfg3_percolation_3d(40, 36, 33, p=0.32), 2),
    (lambda i: i.cfg3_percolation_3d(66, 35, 33, p=0.29), 1), (lambda i: i.cfg3_percolation_3d(130, 30, 27, p=0.31), 0),
    (lambda i: i.iid_diluted(257, 131, 1, seed=6, p=0.515), 1), (lambda i: i.iid_diluted(300, 520, 1, seed=8, p=0.51), 0),
    (lambda i: i.iid_diluted(300, 520, 1, seed=9, p=0.52), 1)])
def test_chain_elimination(pn, oracle, maker, direction):
    """Links (solved nodes with two open bonds, both to solved nodes) are eliminated as series resistors and back-filled by
    interpolation: pressures of ALL nodes, classes and G_eff keep the parity bar, with and without peeling (without it
    dangling trees hang from chain nodes), from a zero start, and bit-reproducibly."""
    from paper_1908_03301_b200 import inputs
    net = maker(inputs)
    base = {pn.PN_OPT_COMPACT: 1, pn.PN_OPT_KERNEL: 3}
    on, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={**base, pn.PN_OPT_CONTRACT: 1})
    off, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={**base, pn.PN_OPT_CONTRACT: 0})
    assert on.kernel_scheme == 7 and off.kernel_scheme == 7
    assert on.n_chain > 0 and off.n_chain == 0
    assert on.n_unknowns == on.n_solved - on.n_peeled - on.n_chain and off.n_unknowns == on.n_unknowns + on.n_chain
    assert on.inner_iters <= off.inner_iters
    nopeel, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={**base, pn.PN_OPT_PEEL: 0, pn.PN_OPT_X0: 0, pn.PN_OPT_GRAPH: 0})
    # (without peeling the table may outgrow the workspace arrays: then the marks are undone and the structured kernel runs)
    assert nopeel.n_peeled == 0 and (nopeel.n_chain > 0 if nopeel.kernel_scheme == 7 else nopeel.n_chain == 0)
    a = gpu_solve(pn, net, direction, 1e-10, opts=base)
    b = gpu_solve(pn, net, direction, 1e-10, opts=base)
    assert a[0].inner_iters == b[0].inner_iters and np.array_equal(a[1], b[1]) and a[3] == b[3]


def test_chain_elimination_hand_built(pn, oracle):
    """A ladder whose rungs are mostly closed: long chains, a loop hanging from one node (closed ring of links), two chains
    between the same pair of nodes (parallel entries), a chain next to a direct bond."""
    nx, ny = 40, 6
    gx = np.zeros((1, ny, nx), np.float32)
    gy = np.zeros((1, ny, nx), np.float32)
    rng = np.random.default_rng(1)
    gx[0, 0, :] = rng.uniform(0.2, 2.0, nx)          # rail 0
    gx[0, 1, :] = rng.uniform(0.2, 2.0, nx)          # rail 1
    for i in (5, 6, 20, 33):                          # rungs between the rails (5, 6 adjacent: a 4-node loop of two chains)
        gy[0, 0, i] = rng.uniform(0.2, 2.0)
    # a ring hanging from rail 1 at i = 12: up along y to row 3, across to i = 15, back down
    for j in (1, 2):
        gy[0, j, 12] = 0.7
        gy[0, j, 15] = 0.9
    gx[0, 3, 12:15] = 1.1
    # a stem from rail 1 at i = 25 up to (25, 3), which carries a closed ring of three links: a chain that loops back to its
    # own end node (no current; all its nodes sit at that node's pressure)
    gy[0, 1, 25] = 0.6
    gy[0, 2, 25] = 1.3
    gx[0, 3, 25] = 0.8
    gy[0, 3, 26] = 1.7
    gx[0, 4, 25] = 0.5
    gy[0, 3, 25] = 1.2
    net = type("N", (), dict(nx=nx, ny=ny, nz=1, gx=gx, gy=gy, gz=None, n_nodes=nx * ny, name="ladder"))()
    for peel in (0, 1):
        info, *_ = compare(pn, oracle, net, 0, tol=1e-13, opts={pn.PN_OPT_COMPACT: 1, pn.PN_OPT_KERNEL: 3, pn.PN_OPT_PEEL: peel})
        assert info.kernel_scheme == 7 and info.n_chain > 40


# ---- seeded random configurations: shapes, dilution, direction, faces, kernels, tiles and launch cuts drawn together ----
@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_configurations(pn, oracle, seed):
    """40 cases per seed through the same element-by-element comparison as everything above: 2D and 3D shapes up to
    ~530 wide (several TMA tiles, both 3D tile shapes, equal narrow tiles), p from 1 down to 0.4, all solve axes,
    periodic faces, every kernel scheme, persistent launches cut after 1 .. 5 iterations, with and without the deferred
    solution update, peeling, graph replay and the zero start."""
    from paper_1908_03301_b200 import inputs
    rng = np.random.default_rng(seed)
    done = 0
    while done < 40:
        if rng.random() < 0.7:
            shape = [int(rng.integers(3, 90)), int(rng.integers(1, 40)), int(rng.integers(1, 40))]
            if rng.random() < 0.25:
                shape[0] = int(rng.integers(250, 530))
            if rng.random() < 0.3:
                rng.shuffle(shape)
        else:
            shape = [int(rng.integers(3, 400)), int(rng.integers(3, 120)), 1]
            if rng.random() < 0.2:
                shape[0] = int(rng.integers(2040, 2200))
        nx, ny, nz = shape
        axes = [d for d in range(3 if nz > 1 else 2) if shape[d] >= 3]
        if not axes:
            continue
        direction = int(rng.choice(axes))
        p = float(rng.choice([1.0, 0.85, 0.6, 0.4]))
        periodic = bool(rng.random() < 0.35)
        kernel = int(rng.choice([0, 1, 3, 3, 8, 8]))
        opts = {pn.PN_OPT_KERNEL: kernel}
        if kernel == 3:
            opts[pn.PN_OPT_TILE] = int(rng.choice([0, 1, 2, 3]))
        if rng.random() < 0.3:
            opts[pn.PN_OPT_CHUNK] = int(rng.choice([1, 2, 3, 5, 64]))
        for key, values in ((pn.PN_OPT_GRAPH, [0]), (pn.PN_OPT_XDEFER, [0]), (pn.PN_OPT_PEEL, [0, 1]), (pn.PN_OPT_X0, [0])):
            if rng.random() < 0.2:
                opts[key] = int(rng.choice(values))
        net = inputs.iid_diluted(nx, ny, nz, seed=int(rng.integers(1 << 30)), p=p)
        compare(pn, oracle, net, direction, tol=1e-13, opts=opts, periodic=periodic)
        done += 1


def test_link_elimination_safety_net(pn, oracle):
    """tests/golden/chain_case_53x22x7.npz: a near-threshold network (p = 0.35, every open bond drifted by 1 %) found by a
    random stress run of the update path: the SECOND solve on a handle whose first solve had eliminated the links broke
    down (-6) or stagnated, whatever the second network's path.  Cause: the compacted scheme and the chain records borrow
    lattice arrays and left garbage in their halo planes, which the iteration kernels read as zeros; pn_solve now zeroes
    the halos at every solve (and repeats a solve that fails with the links eliminated on the plain lattice kernels).
    The network alone, and sequences on one handle through set / replace, must meet the full parity bar."""
    import os
    from types import SimpleNamespace
    d = np.load(os.path.join(os.path.dirname(__file__), "golden", "chain_case_53x22x7.npz"))
    net = SimpleNamespace(nx=53, ny=22, nz=7, gx=d["gx"], gy=d["gy"], gz=d["gz"], name="chain_case_53x22x7", n_nodes=53 * 22 * 7)
    direction = int(d["direction"])
    info, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={pn.PN_OPT_PEEL: 1})
    assert info.status == pn.PN_OK
    plain, *_ = compare(pn, oracle, net, direction, tol=1e-13, opts={pn.PN_OPT_PEEL: 1, pn.PN_OPT_CONTRACT: 0})
    assert plain.status == pn.PN_OK and plain.n_chain == 0
    # on one handle: a good network, the bad one through pn_replace_conductances (label reuse, warm start), a good one again
    from paper_1908_03301_b200 import inputs
    h = pn.Network(53, 22, 7)
    h.set_option(pn.PN_OPT_PEEL, 1)
    good = inputs.iid_diluted(53, 22, 7, seed=4, p=0.35)
    for arrays in ((good.gx, good.gy, good.gz), (d["gx"], d["gy"], d["gz"]), (good.gx, good.gy, good.gz)):
        h.set_conductances(*arrays) if arrays[0] is good.gx else h.replace_conductances(*arrays)
        got = h.solve(direction, 1e-13, accept=(pn.PN_OK, pn.PN_NO_SPANNING_CLUSTER))
        if got.status != pn.PN_OK:
            continue
        ref = oracle.solve(53, 22, 7, arrays[0], arrays[1], arrays[2], direction, 1e-13)
        assert np.max(np.abs(h.pressures().cpu().numpy() - ref.P)) <= 1e-8
        assert abs(h.flux()[2] - ref.g_eff) <= 1e-9 * abs(ref.g_eff)
    h.close()
