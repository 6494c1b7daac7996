"""Pins for the CPU oracle: what the paper and the mathematics fix (SURVEY.md 8(c) "What pins the
oracle").  None of these compares the oracle with itself through the same formula: closed forms,
a hand-worked example, dense LAPACK on an independently assembled matrix, brute-force labelling,
conservation invariants and symmetry transformations."""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components

from oracle import pn_oracle as po
from paper_1908_03301_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def run(net, direction=0, tol=1e-13, **kw):
    return po.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, tol, **kw)


# ---------------------------------------------------------------- closed forms -------------------
@pytest.mark.parametrize("shape,direction", [((9, 6, 5), 0), ((9, 6, 5), 1), ((9, 6, 5), 2),
                                             ((7, 4, 1), 0), ((7, 4, 1), 1), ((3, 3, 3), 2)])
def test_uniform_gives_linear_profile_and_gA_over_L(shape, direction):
    """Uniform g: P linear along a; G_eff = g * S_perp / (n_a - 1) exactly; K = g (north_star)."""
    nx, ny, nz = shape
    g = 0.37
    net = inputs.uniform(nx, ny, nz, g)
    res = run(net, direction)
    n_a = shape[direction]
    # P has shape (nz, ny, nx): the coordinate along lattice axis `direction` runs along array axis 2 - direction
    shp = [1, 1, 1]
    shp[2 - direction] = n_a
    expect = np.broadcast_to(1.0 - np.arange(n_a, dtype=np.float64).reshape(shp) / (n_a - 1), (nz, ny, nx))
    assert np.max(np.abs(res.P - expect)) < 1e-12
    g32 = float(np.float32(g))
    s_perp = nx * ny * nz // n_a
    assert res.g_eff == pytest.approx(g32 * s_perp / (n_a - 1), rel=1e-12)
    assert res.k_eff == pytest.approx(g32, rel=1e-12)
    assert res.q_in == pytest.approx(res.q_out, rel=1e-12)
    if shape == (9, 6, 5) and direction == 0:
        assert res.g_eff == pytest.approx(g32 * 30 / 8, rel=1e-12)      # SURVEY probe: 1.3875


def test_layered_arithmetic_and_harmonic_means():
    """Noise-free layers along z: arithmetic mean parallel (x), harmonic mean across (z)."""
    nx, ny, nz = 6, 5, 7
    rng = np.random.default_rng(11)
    c = rng.uniform(0.2, 3.0, nz).astype(np.float32)
    e = rng.uniform(0.2, 3.0, nz).astype(np.float32)
    net = inputs.layered_exact(nx, ny, nz, c, e)
    rx = run(net, 0)
    rz = run(net, 2)
    c64, e64 = c.astype(np.float64), e.astype(np.float64)
    assert rx.g_eff == pytest.approx(ny * c64.sum() / (nx - 1), rel=1e-12)
    assert rz.g_eff == pytest.approx(nx * ny / np.sum(1.0 / e64[:nz - 1]), rel=1e-12)
    # y is also parallel to the layers
    ry = run(net, 1)
    assert ry.g_eff == pytest.approx(nx * c64.sum() / (ny - 1), rel=1e-12)


def test_series_chain():
    """ny = nz = 1: resistors in series, G = 1 / sum(1/g)."""
    rng = np.random.default_rng(5)
    g = rng.uniform(0.1, 2.0, 12).astype(np.float32)
    net = inputs.Network(12, 1, 1, g.reshape(1, 1, 12), np.ones((1, 1, 12), np.float32), None)
    res = run(net, 0)
    g64 = g.astype(np.float64)[:11]
    assert res.g_eff == pytest.approx(1.0 / np.sum(1.0 / g64), rel=1e-12)
    # pressure drops are proportional to the resistances
    drops = res.P.ravel()[:-1] - res.P.ravel()[1:]
    assert np.allclose(drops, (1.0 / g64) / np.sum(1.0 / g64), rtol=1e-11)


def test_parallel_chains_lower_bound_is_attained_without_cross_bonds():
    """gy = 0: independent series chains; G = sum_chains 1/sum(1/g)."""
    rng = np.random.default_rng(6)
    nx, ny = 8, 5
    gx = rng.uniform(0.1, 2.0, (1, ny, nx)).astype(np.float32)
    net = inputs.Network(nx, ny, 1, gx, np.zeros((1, ny, nx), np.float32), None)
    res = run(net, 0)
    g64 = gx.astype(np.float64)[0, :, :nx - 1]
    assert res.g_eff == pytest.approx(np.sum(1.0 / np.sum(1.0 / g64, axis=1)), rel=1e-12)


def test_hand_worked_3x2_example():
    """tests/golden/worked_3x2.txt (derivation in the file)."""
    vals = {}
    with open(os.path.join(GOLDEN, "worked_3x2.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, num, den = line.split()
            vals[name] = float(Fraction(int(num), int(den)))
    gx = np.zeros((1, 2, 3), np.float32)
    gy = np.zeros((1, 2, 3), np.float32)
    gx[0, 0, 0], gx[0, 0, 1], gx[0, 1, 0], gx[0, 1, 1] = 1, 2, 3, 4
    gy[0, 0, 1] = 5
    gx[0, :, 2] = 99.0          # not bonds: must be ignored
    gy[0, 1, :] = 77.0
    gy[0, 0, 0] = 55.0          # bond inside the inlet column: carries no current
    net = inputs.Network(3, 2, 1, gx, gy, None)
    for dense in (False, True):
        res = run(net, 0, dense=dense)
        assert res.P[0, 0, 1] == pytest.approx(vals["P_1_0"], rel=1e-13)
        assert res.P[0, 1, 1] == pytest.approx(vals["P_1_1"], rel=1e-13)
        assert res.q_in == pytest.approx(vals["Q_in"], rel=1e-13)
        assert res.q_out == pytest.approx(vals["Q_out"], rel=1e-13)
        assert res.g_eff == pytest.approx(vals["G_eff"], rel=1e-13)
        assert res.g_eff == pytest.approx(2.394366197183099, rel=1e-12)


# ---------------------------------------------------------------- dense cross-check ----------------
def brute_force_dense(net, direction, periodic=False):
    """Independent statement of the problem: full N x N graph Laplacian built bond by bond in Python
    loops, Dirichlet rows replaced by identity, nodes with no path to a Dirichlet plane... are
    handled by least-norm-free elimination: we solve only on nodes connected to a Dirichlet node."""
    nx, ny, nz = net.nx, net.ny, net.nz
    N = nx * ny * nz
    L = np.zeros((N, N))
    gs = (net.gx, net.gy, net.gz)
    dims = (nx, ny, nz)
    stride = (1, nx, nx * ny)
    for k, j, i in itertools.product(range(nz), range(ny), range(nx)):
        n = i + nx * (j + ny * k)
        c = (i, j, k)
        for a in range(3):
            if gs[a] is None:
                continue
            if c[a] + 1 < dims[a]:
                m = n + stride[a]
            elif periodic and a != direction and dims[a] >= 2:
                m = n - (dims[a] - 1) * stride[a]          # lateral faces wrap
            else:
                continue
            g = float(gs[a][k, j, i])
            L[n, n] += g
            L[m, m] += g
            L[n, m] -= g
            L[m, n] -= g
    coord = [(n % nx, (n // nx) % ny, n // (nx * ny))[direction] for n in range(N)]
    n_a = dims[direction]
    fixed = {n: 1.0 for n in range(N) if coord[n] == 0}
    fixed.update({n: 0.0 for n in range(N) if coord[n] == n_a - 1})
    # connectivity to any Dirichlet node through open bonds, by boolean closure
    adj = (L < 0)
    reach = np.zeros(N, bool)
    reach[list(fixed)] = True
    # interior-only propagation: a path may not pass THROUGH a Dirichlet node
    frontier = set()
    for d in fixed:
        for m in np.flatnonzero(adj[d]):
            if m not in fixed:
                frontier.add(int(m))
    seen = set(frontier)
    while frontier:
        n = frontier.pop()
        for m in np.flatnonzero(adj[n]):
            m = int(m)
            if m not in fixed and m not in seen:
                seen.add(m)
                frontier.add(m)
    free = sorted(seen)
    P = np.zeros(N)
    for n, v in fixed.items():
        P[n] = v
    if free:
        fl = list(fixed)
        Aff = L[np.ix_(free, free)]
        rhs = -L[np.ix_(free, fl)] @ np.array([fixed[n] for n in fl])
        P[free] = np.linalg.solve(Aff, rhs)
    return P.reshape(nz, ny, nx), set(free)


@pytest.mark.parametrize("shape,p,seed,direction", [
    ((6, 5, 1), 1.0, 1, 0), ((6, 5, 1), 0.7, 2, 1), ((5, 4, 3), 1.0, 3, 2), ((5, 4, 3), 0.6, 4, 0),
    ((4, 5, 4), 0.5, 5, 1), ((8, 8, 1), 0.6, 6, 0), ((16, 16, 1), 0.65, 7, 0), ((7, 6, 5), 0.45, 8, 2),
])
def test_against_dense_lapack_on_bruteforce_laplacian(shape, p, seed, direction):
    """Networks of <= 16 nodes per side: dense direct solve of an independently built system must
    agree (north_star).  Pressures on nodes connected to a Dirichlet plane are unique."""
    net = inputs.iid_diluted(*shape, seed=seed, p=p)
    res = run(net, direction)
    Pd, connected = brute_force_dense(net, direction)
    # every node class that has a defined pressure: Dirichlet, solved, inlet-only, outlet-only
    defined = res.classes != po.FLOATING
    assert np.max(np.abs(res.P[defined] - Pd[defined])) < 1e-11
    # floating nodes are exactly those not connected to any Dirichlet node; convention P = 0
    flat_float = set(np.flatnonzero(res.classes.ravel() == po.FLOATING).tolist())
    interior = set(np.flatnonzero((res.classes.ravel() != po.INLET)
                                  & (res.classes.ravel() != po.OUTLET)).tolist())
    assert flat_float == interior - connected
    assert np.all(res.P[res.classes == po.FLOATING] == 0.0)
    # the oracle's own dense path agrees too
    rd = run(net, direction, dense=True)
    assert np.max(np.abs(rd.P - res.P)) < 1e-11
    assert rd.g_eff == pytest.approx(res.g_eff, rel=1e-11, abs=1e-14)


# ---------------------------------------------------------------- invariants ----------------------
@pytest.mark.parametrize("maker,direction", [
    (lambda: inputs.cfg1_iid_2d(24, 20, seed=0), 0),
    (lambda: inputs.cfg3_percolation_3d(12, 11, 10, seed=2, p=0.45), 0),
    (lambda: inputs.cfg4_fbm_cut_3d(12, 12, 12, seed=3), 1),
    (lambda: inputs.cfg5_stratified_3d(10, 9, 12, seed=4), 2),
])
def test_conservation_invariants(maker, direction):
    net = maker()
    res = run(net, direction)
    g64 = po.widen(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz)
    # Kirchhoff's law at every solved node
    kr = po.kirchhoff_residual(net.nx, net.ny, net.nz, g64, res.P)
    scale = max(res.q_in, 1e-30)
    assert np.max(np.abs(kr[res.classes == po.SOLVED])) < 1e-11 * max(scale, 1.0)
    # pinned interior nodes carry no current either
    for c in (po.INLET_ONLY, po.OUTLET_ONLY, po.FLOATING):
        if np.any(res.classes == c):
            assert np.max(np.abs(kr[res.classes == c])) == 0.0
    # same total flow through every cross-section; inflow = outflow (eq.(4) is section-independent)
    pf = po.plane_fluxes(net.nx, net.ny, net.nz, g64, res.P, direction)
    assert np.max(np.abs(pf - pf[0])) < 1e-11 * max(abs(pf[0]), 1.0)
    assert res.q_in == pytest.approx(res.q_out, rel=1e-10, abs=1e-13)
    # energy identity Q dP = sum_bonds g dP_bond^2 (bonds inside Dirichlet planes contribute 0)
    assert po.dissipation(net.nx, net.ny, net.nz, g64, res.P) == pytest.approx(res.g_eff, rel=1e-10,
                                                                               abs=1e-13)
    assert res.rel_residual <= 1e-13


def test_variational_bounds():
    """Linear trial field: G <= sum_{a-bonds} g / (n_a-1)^2; independent chains: G >= sum 1/sum(1/g)."""
    net = inputs.iid_diluted(12, 12, 12, seed=9, p=1.0)
    res = run(net, 0)
    g = net.gx.astype(np.float64)[:, :, :11]
    upper = g.sum() / 11 ** 2
    lower = np.sum(1.0 / np.sum(1.0 / g, axis=2))
    assert lower < res.g_eff < upper


# ---------------------------------------------------------------- symmetry transformations --------
def test_axis_relabelling_reversal_and_scaling():
    net = inputs.iid_diluted(7, 6, 5, seed=21, p=0.8)
    base = run(net, 0)
    # relabel axes: new x = old y, new y = old z, new z = old x; old x-solve is the new z-solve
    perm = (1, 2, 0)
    tn = inputs.transpose_axes(net, perm)
    assert (tn.nx, tn.ny, tn.nz) == (net.ny, net.nz, net.nx)
    rt = run(tn, 2)
    assert rt.g_eff == pytest.approx(base.g_eff, rel=1e-11)
    # P_new[z', y', x'] with z' = old x, y' = old z, x' = old y
    assert np.max(np.abs(rt.P - np.transpose(base.P, (2, 0, 1)))) < 1e-11
    # reverse the solve axis: P -> 1 - P on every node connected to a Dirichlet plane
    gxr = np.zeros_like(net.gx)
    gxr[:, :, :-1] = net.gx[:, :, -2::-1]
    rnet = inputs.Network(net.nx, net.ny, net.nz, gxr, net.gy[:, :, ::-1].copy(),
                          net.gz[:, :, ::-1].copy())
    rr = run(rnet, 0)
    defined = base.classes != po.FLOATING
    assert rr.g_eff == pytest.approx(base.g_eff, rel=1e-11)
    assert np.max(np.abs((1.0 - rr.P[:, :, ::-1])[defined] - base.P[defined])) < 1e-11
    # scale g -> 4 g (exact in fp32): P unchanged, G -> 4 G
    snet = inputs.Network(net.nx, net.ny, net.nz, net.gx * 4, net.gy * 4, net.gz * 4)
    rs = run(snet, 0)
    assert np.max(np.abs(rs.P - base.P)) < 1e-11
    assert rs.g_eff == pytest.approx(4 * base.g_eff, rel=1e-11)


# ---------------------------------------------------------------- labelling -----------------------
def independent_classes(net, direction):
    """Second labeller: scipy connected components on interior-interior open bonds."""
    nx, ny, nz = net.nx, net.ny, net.nz
    N = nx * ny * nz
    flat = np.arange(N)
    coord = (flat % nx, (flat // nx) % ny, flat // (nx * ny))
    n_a = (nx, ny, nz)[direction]
    inlet = coord[direction] == 0
    outlet = coord[direction] == n_a - 1
    interior = ~(inlet | outlet)
    rows, cols = [], []
    t_in = np.zeros(N, bool)
    t_out = np.zeros(N, bool)
    for a, g in enumerate((net.gx, net.gy, net.gz)):
        if g is None:
            continue
        ok = (coord[a] + 1 < (nx, ny, nz)[a]) & (g.ravel() > 0)
        n0 = flat[ok]
        n1 = n0 + (1, nx, nx * ny)[a]
        both = interior[n0] & interior[n1]
        rows.append(n0[both])
        cols.append(n1[both])
        for u, v in ((n0, n1), (n1, n0)):
            t_in[u[interior[u] & inlet[v]]] = True
            t_out[u[interior[u] & outlet[v]]] = True
    rows, cols = np.concatenate(rows), np.concatenate(cols)
    G = sp.coo_matrix((np.ones(rows.size), (rows, cols)), shape=(N, N))
    _, lab = connected_components(G, directed=False)
    cin = np.zeros(lab.max() + 1, bool)
    cout = np.zeros(lab.max() + 1, bool)
    np.logical_or.at(cin, lab, t_in)
    np.logical_or.at(cout, lab, t_out)
    cls = np.where(cin[lab] & cout[lab], po.SOLVED,
                   np.where(cin[lab], po.INLET_ONLY, np.where(cout[lab], po.OUTLET_ONLY, po.FLOATING)))
    cls[inlet] = po.INLET
    cls[outlet] = po.OUTLET
    return cls.reshape(nz, ny, nx).astype(np.int8)


def test_labelling_all_bond_masks_on_4x2():
    """Every one of the 2^10 open/closed patterns of a 4x2 lattice against the second labeller."""
    nx, ny = 4, 2
    slots = [("x", j, i) for j in range(ny) for i in range(nx - 1)] + [("y", 0, i) for i in range(nx)]
    assert len(slots) == 10
    for mask in range(1 << len(slots)):
        gx = np.zeros((1, ny, nx), np.float32)
        gy = np.zeros((1, ny, nx), np.float32)
        for b, (d, j, i) in enumerate(slots):
            if mask >> b & 1:
                (gx if d == "x" else gy)[0, j, i] = 1.0
        net = inputs.Network(nx, ny, 1, gx, gy, None)
        g64 = po.widen(nx, ny, 1, gx, gy, None)
        assert np.array_equal(po.classify(nx, ny, 1, g64, 0), independent_classes(net, 0))


@pytest.mark.parametrize("shape,p,direction,seed", [
    ((9, 8, 7), 0.25, 0, 1), ((9, 8, 7), 0.3, 1, 2), ((9, 8, 7), 0.35, 2, 3), ((20, 17, 1), 0.5, 0, 4),
    ((20, 17, 1), 0.55, 1, 5), ((13, 5, 9), 0.2, 2, 6), ((6, 6, 6), 0.0, 0, 7), ((6, 6, 6), 1.0, 0, 8),
])
def test_labelling_random_lattices(shape, p, direction, seed):
    net = inputs.iid_diluted(*shape, seed=seed, p=p)
    g64 = po.widen(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz)
    cls = po.classify(net.nx, net.ny, net.nz, g64, direction)
    assert np.array_equal(cls, independent_classes(net, direction))
    if p == 0.0:
        res = run(net, direction)
        assert res.status == "no_spanning_cluster" and res.g_eff == 0.0 and res.n_solved == 0
        assert res.n_floating == (shape[direction] - 2) * np.prod(shape) // shape[direction]
    if p == 1.0:
        assert np.all((cls == po.SOLVED) | (cls == po.INLET) | (cls == po.OUTLET))


def test_below_threshold_has_no_spanning_cluster_2d():
    """2D square bond percolation threshold is 1/2: far below it, Q = 0."""
    net = inputs.iid_diluted(40, 40, 1, seed=3, p=0.25)
    res = run(net, 0)
    assert res.status == "no_spanning_cluster"
    assert res.q_in == 0.0 and res.q_out == 0.0 and res.g_eff == 0.0
    assert set(np.unique(res.P)) <= {0.0, 1.0}


def test_inlet_only_cluster_sits_at_inlet_pressure():
    """A dead-end cluster hanging off the inlet is at P = 1 exactly (no current)."""
    nx, ny = 6, 3
    gx = np.zeros((1, ny, nx), np.float32)
    gy = np.zeros((1, ny, nx), np.float32)
    gx[0, 0, :5] = 1.0              # row 0 spans
    gx[0, 2, 0] = 2.0               # row 2: stub from the inlet to (1,2),(2,2)
    gx[0, 2, 1] = 2.0
    gx[0, 2, 3] = 3.0               # outlet-side stub: (3,2)-(4,2)-(5,2)
    gx[0, 2, 4] = 3.0
    net = inputs.Network(nx, ny, 1, gx, gy, None)
    res = run(net, 0)
    assert res.classes[0, 2, 1] == po.INLET_ONLY and res.P[0, 2, 2] == 1.0
    assert res.classes[0, 2, 3] == po.OUTLET_ONLY and res.P[0, 2, 4] == 0.0
    assert res.classes[0, 1, 2] == po.FLOATING and res.P[0, 1, 2] == 0.0
    assert res.g_eff == pytest.approx(1.0 / 5.0, rel=1e-13)
    assert (res.n_solved, res.n_inlet_only, res.n_outlet_only, res.n_floating) == (4, 2, 2, 4)


def test_rejects_bad_input():
    net = inputs.uniform(4, 4, 1, 1.0)
    bad = net.gx.copy()
    bad[0, 1, 1] = -1.0
    with pytest.raises(ValueError):
        po.solve(4, 4, 1, bad, net.gy, None, 0)
    bad[0, 1, 1] = np.nan
    with pytest.raises(ValueError):
        po.solve(4, 4, 1, bad, net.gy, None, 0)
    with pytest.raises(ValueError):
        po.solve(2, 4, 1, net.gx[:, :, :2], net.gy[:, :, :2], None, 0)


def test_residual_certificate_detects_a_wrong_field():
    net = inputs.cfg3_percolation_3d(10, 10, 10, seed=2, p=0.5)
    res = run(net, 0)
    rel, pin = po.residual_certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, res.P, 0)
    assert rel <= 1e-13 and pin == 0.0
    bad = res.P.copy()
    idx = np.argwhere(res.classes == po.SOLVED)[3]
    bad[tuple(idx)] += 1e-6
    rel2, _ = po.residual_certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, bad, 0)
    assert rel2 > 1e-8


# ---------------------------------------------------------------- dangling ends (S8c reading 7) ---
def _open_nbrs(nx, ny, nz, g64, n, wrap=(False, False, False)):
    """Open-bond neighbours of node n, written independently of the oracle (coordinate loops)."""
    i, j, k = n % nx, (n // nx) % ny, n // (nx * ny)
    out = []
    for (di, dj, dk) in ((1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
        a, b, c = i + di, j + dj, k + dk
        arr = g64[0] if di else (g64[1] if dj else g64[2])
        if not (0 <= a < nx and 0 <= b < ny and 0 <= c < nz):
            ax = 0 if di else (1 if dj else 2)
            if not wrap[ax]:
                continue
            a, b, c = a % nx, b % ny, c % nz
            # the wrap bond is stored at the LAST node along the axis
            g = arr[max(k, c), max(j, b), max(i, a)]
            if g > 0.0:
                out.append(a + nx * (b + ny * c))
            continue
        g = arr[min(k, c), min(j, b), min(i, a)]        # the forward bond lives on the lower-index end
        if g > 0.0:
            out.append(a + nx * (b + ny * c))
    return out


@pytest.mark.parametrize("shape,direction,p,seed", [((5, 4, 1), 0, 0.7, s) for s in range(6)] +
                         [((4, 5, 1), 1, 0.75, s) for s in range(4)] + [((4, 3, 3), 0, 0.6, s) for s in range(6)])
def test_dangling_ends_equal_complement_of_bruteforce_2core(shape, direction, p, seed, periodic=False):
    """The nodes left after stripping are the 2-core (Dirichlet nodes kept): the UNION of all node subsets in
    which every member keeps >= 2 open neighbours inside (subset + Dirichlet planes).  Enumerated outright."""
    nx, ny, nz = shape
    net = inputs.iid_diluted(nx, ny, nz, seed=100 + seed, p=p)
    wrap = po.wrap_axes(nx, ny, nz, direction, periodic)
    g64 = po.widen(nx, ny, nz, net.gx, net.gy, net.gz, wrap)
    cls = po.classify(nx, ny, nz, g64, direction, wrap)
    mask = po.dangling_ends(nx, ny, nz, g64, cls, wrap)
    flat = cls.ravel()
    solved = [n for n in range(nx * ny * nz) if flat[n] == po.SOLVED]
    assert len(solved) <= 18
    dirichlet = {n for n in range(nx * ny * nz) if flat[n] in (po.INLET, po.OUTLET)}
    nbrs = {n: _open_nbrs(nx, ny, nz, g64, n, wrap) for n in solved}
    core = set()
    for bits in range(1 << len(solved)):
        sub = {solved[t] for t in range(len(solved)) if bits >> t & 1}
        keep = sub | dirichlet
        if all(sum(m in keep for m in nbrs[n]) >= 2 for n in sub):
            core |= sub
    expect = np.zeros(nx * ny * nz, dtype=bool)
    expect[[n for n in solved if n not in core]] = True
    assert np.array_equal(mask.ravel(), expect)
    assert not mask.ravel()[[n for n in range(nx * ny * nz) if flat[n] != po.SOLVED]].any()


def test_dangling_ends_hand_built_stub():
    """5 x 3 lattice, x direction: the middle row is the backbone; a two-node stub (2,2) -- (3,2) hangs from
    (2,1).  Exactly those two nodes are dangling; they sit at the pressure of (2,1) = 1/2."""
    nx, ny = 5, 3
    gx = np.zeros((1, ny, nx), dtype=np.float32)
    gy = np.zeros((1, ny, nx), dtype=np.float32)
    gx[0, 1, :4] = 1.0           # backbone
    gy[0, 1, 2] = 2.0            # (2,1) -- (2,2)
    gx[0, 2, 2] = 3.0            # (2,2) -- (3,2)
    g64 = po.widen(nx, ny, 1, gx, gy, None)
    cls = po.classify(nx, ny, 1, g64, 0)
    mask = po.dangling_ends(nx, ny, 1, g64, cls)
    expect = np.zeros((1, ny, nx), dtype=bool)
    expect[0, 2, 2] = expect[0, 2, 3] = True
    assert np.array_equal(mask, expect)
    res = po.solve(nx, ny, 1, gx, gy, None, 0, 1e-14)
    assert res.P[0, 2, 2] == pytest.approx(0.5, abs=1e-13) and res.P[0, 2, 3] == pytest.approx(0.5, abs=1e-13)


@pytest.mark.parametrize("direction", [0, 2])
def test_dangling_ends_carry_no_current(direction):
    """Physics pin: in the solution of the FULL system every bond at a dangling node carries zero current."""
    net = inputs.iid_diluted(14, 12, 10, seed=41, p=0.36)
    nx, ny, nz = net.nx, net.ny, net.nz
    res = run(net, direction, tol=1e-14)
    assert res.status == "ok"
    g64 = po.widen(nx, ny, nz, net.gx, net.gy, net.gz)
    mask = po.dangling_ends(nx, ny, nz, g64, res.classes)
    assert 0 < mask.sum() < res.n_solved
    P = res.P
    cur = [np.zeros(P.shape) for _ in range(3)]
    cur[0][:, :, :-1] = g64[0][:, :, :-1] * (P[:, :, 1:] - P[:, :, :-1])
    cur[1][:, :-1, :] = g64[1][:, :-1, :] * (P[:, 1:, :] - P[:, :-1, :])
    cur[2][:-1, :, :] = g64[2][:-1, :, :] * (P[1:, :, :] - P[:-1, :, :])
    # only bonds between nodes of the solved system matter (pinned clusters are not connected to it)
    worst = 0.0
    for a, (sl_lo, sl_hi) in enumerate((((slice(None), slice(None), slice(0, -1)), (slice(None), slice(None), slice(1, None))),
                                        ((slice(None), slice(0, -1), slice(None)), (slice(None), slice(1, None), slice(None))),
                                        ((slice(0, -1), slice(None), slice(None)), (slice(1, None), slice(None), slice(None))))):
        touched = mask[sl_lo] | mask[sl_hi]
        worst = max(worst, float(np.max(np.abs(cur[a][sl_lo][touched]), initial=0.0)))
    assert worst < 1e-11
    # and some bond that is NOT at a dangling node does carry current
    assert max(float(np.max(np.abs(c))) for c in cur) > 1e-3


# ---------------------------------------------------------------- periodic lateral faces ---
def test_periodic_hand_worked_3x2_example():
    """tests/golden/worked_3x2_periodic.txt: the wrap bond doubles the a-b connection; 55/141, 57/141, 338/141."""
    vals = {}
    for line in open(os.path.join(GOLDEN, "worked_3x2_periodic.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        vals[k] = Fraction(v)
    gx = np.array([[[1, 2, 99], [3, 4, 99]]], dtype=np.float32)
    gy = np.array([[[77, 5, 77], [88, 7, 88]]], dtype=np.float32)   # 77/88: bonds inside the Dirichlet columns
    res = po.solve(3, 2, 1, gx, gy, None, 0, 1e-15, periodic=True)
    assert res.P[0, 0, 1] == pytest.approx(float(vals["Pa"]), abs=1e-14)
    assert res.P[0, 1, 1] == pytest.approx(float(vals["Pb"]), abs=1e-14)
    assert res.g_eff == pytest.approx(float(vals["G_eff"]), rel=1e-13)
    assert res.q_in == pytest.approx(res.q_out, rel=1e-13)
    # without the flag the wrap entry is not a bond: the no-flux golden values (27/71, 29/71)
    res0 = po.solve(3, 2, 1, gx, gy, None, 0, 1e-15)
    assert res0.P[0, 0, 1] == pytest.approx(27 / 71, abs=1e-14)


@pytest.mark.parametrize("shape,direction", [((9, 6, 5), 0), ((9, 6, 5), 1), ((9, 6, 5), 2), ((7, 4, 1), 0), ((7, 4, 1), 1)])
def test_periodic_uniform_closed_form(shape, direction):
    nx, ny, nz = shape
    net = inputs.uniform(nx, ny, nz, 0.37)
    res = run(net, direction, periodic=True)
    n_a = shape[direction]
    coord = po._coord_along(nx, ny, nz, direction)[0]
    assert np.max(np.abs(res.P - (1.0 - coord / (n_a - 1)))) < 1e-12
    assert res.g_eff == pytest.approx(float(np.float32(0.37)) * (nx * ny * nz // n_a) / (n_a - 1), rel=1e-12)


@pytest.mark.parametrize("shape,p,seed,direction", [
    ((6, 5, 1), 1.0, 1, 0), ((6, 5, 1), 0.7, 2, 1), ((5, 4, 3), 1.0, 3, 2), ((5, 4, 3), 0.6, 4, 0),
    ((4, 5, 4), 0.5, 5, 1), ((8, 8, 1), 0.6, 6, 0), ((7, 2, 5), 0.7, 8, 2), ((5, 2, 1), 0.9, 9, 0)])
def test_periodic_against_dense_lapack_on_bruteforce_laplacian(shape, p, seed, direction):
    """Same independent dense statement as the no-flux case, with the wrap bonds added bond by bond (lengths 2 and
    1 along a lateral axis included: a doubled bond, resp. no wrap bond at all)."""
    net = inputs.iid_diluted(*shape, seed=seed, p=p)
    res = run(net, direction, periodic=True)
    Pd, connected = brute_force_dense(net, direction, periodic=True)
    defined = res.classes != po.FLOATING
    assert np.max(np.abs(res.P[defined] - Pd[defined])) < 1e-11
    interior = set(np.flatnonzero((res.classes.ravel() != po.INLET) & (res.classes.ravel() != po.OUTLET)).tolist())
    assert set(np.flatnonzero(res.classes.ravel() == po.FLOATING).tolist()) == interior - connected
    # and the flag matters on these inputs (the wrap bonds carry current)
    if p == 1.0:
        assert abs(run(net, direction).g_eff - res.g_eff) > 1e-6 * res.g_eff


@pytest.mark.parametrize("direction,axis,shift", [(0, 1, 3), (0, 2, 2), (2, 0, 5), (1, 2, 1)])
def test_periodic_translation_invariance(direction, axis, shift):
    """A cyclic shift of the network along a lateral axis shifts the solution and leaves G_eff alone -- true for
    periodic faces only (with no-flux faces the shifted network is a different problem)."""
    net = inputs.iid_diluted(8, 7, 6, seed=12, p=0.8)
    ax = 2 - axis                                    # numpy axis of lattice axis `axis`
    roll = lambda a: np.roll(a, shift, axis=ax)
    a = run(net, direction, periodic=True)
    b = po.solve(net.nx, net.ny, net.nz, roll(net.gx), roll(net.gy), roll(net.gz), direction, 1e-13, periodic=True)
    assert np.max(np.abs(roll(a.P) - b.P)) < 1e-11
    assert b.g_eff == pytest.approx(a.g_eff, rel=1e-11)
    assert np.array_equal(roll(a.classes), b.classes)
    c = run(net, direction)
    d = po.solve(net.nx, net.ny, net.nz, roll(net.gx), roll(net.gy), roll(net.gz), direction, 1e-13)
    assert abs(c.g_eff - d.g_eff) > 1e-6 * c.g_eff


@pytest.mark.parametrize("maker,direction", [
    (lambda: inputs.cfg3_percolation_3d(12, 11, 10, seed=2, p=0.45), 0),
    (lambda: inputs.cfg4_fbm_cut_3d(12, 12, 12, seed=3), 1),
    (lambda: inputs.iid_diluted(20, 17, 1, seed=3, p=0.7), 1)])
def test_periodic_conservation_invariants(maker, direction):
    net = maker()
    res = run(net, direction, periodic=True)
    wrap = po.wrap_axes(net.nx, net.ny, net.nz, direction, True)
    g64 = po.widen(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, wrap)
    kr = po.kirchhoff_residual(net.nx, net.ny, net.nz, g64, res.P, wrap)
    assert np.max(np.abs(kr[res.classes == po.SOLVED])) < 1e-11 * max(res.q_in, 1.0)
    pf = po.plane_fluxes(net.nx, net.ny, net.nz, g64, res.P, direction)
    assert np.max(np.abs(pf - pf[0])) < 1e-11 * max(abs(pf[0]), 1.0)
    assert po.dissipation(net.nx, net.ny, net.nz, g64, res.P, wrap) == pytest.approx(res.g_eff, rel=1e-10, abs=1e-13)
    rel, pin_err = po.residual_certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, res.P, direction, periodic=True)
    assert rel <= 1e-13 and pin_err == 0.0
    # the certificate of the OTHER boundary condition rejects this field
    rel0, _ = po.residual_certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, res.P, direction)
    assert rel0 > 1e-6


@pytest.mark.parametrize("shape,direction,p,seed", [((5, 4, 1), 0, 0.6, s) for s in range(4)] + [((4, 3, 3), 0, 0.5, s) for s in range(4)])
def test_periodic_dangling_ends_bruteforce_2core(shape, direction, p, seed):
    test_dangling_ends_equal_complement_of_bruteforce_2core(shape, direction, p, seed, periodic=True)
