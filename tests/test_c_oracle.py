"""The plain-C oracle (oracle/pn_oracle.c) against the same pins as the Python one, and against it."""
import numpy as np
import pytest

from oracle import c_oracle, pn_oracle as po
from paper_1908_03301_b200 import inputs
from test_oracle_pins import brute_force_dense, independent_classes


def crun(net, direction=0, tol=1e-13, **kw):
    return c_oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, tol, **kw)


@pytest.mark.parametrize("shape,direction", [((9, 6, 5), 0), ((9, 6, 5), 1), ((9, 6, 5), 2), ((7, 4, 1), 1)])
def test_c_oracle_uniform(shape, direction):
    nx, ny, nz = shape
    res = crun(inputs.uniform(nx, ny, nz, 0.37), direction)
    n_a = shape[direction]
    coord = po._coord_along(nx, ny, nz, direction)[0]
    assert np.max(np.abs(res.P - (1.0 - coord / (n_a - 1)))) < 1e-12
    g32 = float(np.float32(0.37))
    assert res.g_eff == pytest.approx(g32 * (nx * ny * nz // n_a) / (n_a - 1), rel=1e-12)
    assert res.k_eff == pytest.approx(g32, rel=1e-12)


def test_c_oracle_layered_means():
    nx, ny, nz = 6, 5, 7
    rng = np.random.default_rng(11)
    c = rng.uniform(0.2, 3.0, nz).astype(np.float32)
    e = rng.uniform(0.2, 3.0, nz).astype(np.float32)
    net = inputs.layered_exact(nx, ny, nz, c, e)
    assert crun(net, 0).g_eff == pytest.approx(ny * c.astype(float).sum() / (nx - 1), rel=1e-12)
    assert crun(net, 2).g_eff == pytest.approx(nx * ny / np.sum(1.0 / e.astype(float)[:nz - 1]), rel=1e-12)


def test_c_oracle_worked_example():
    gx = np.zeros((1, 2, 3), np.float32)
    gy = np.zeros((1, 2, 3), np.float32)
    gx[0, 0, 0], gx[0, 0, 1], gx[0, 1, 0], gx[0, 1, 1] = 1, 2, 3, 4
    gy[0, 0, 1] = 5
    gx[0, :, 2] = 99.0
    gy[0, 1, :] = 77.0
    res = crun(inputs.Network(3, 2, 1, gx, gy, None), 0)
    assert res.P[0, 0, 1] == pytest.approx(27 / 71, rel=1e-13)
    assert res.P[0, 1, 1] == pytest.approx(29 / 71, rel=1e-13)
    assert res.q_in == pytest.approx(170 / 71, rel=1e-13)
    assert res.q_out == pytest.approx(170 / 71, rel=1e-13)


@pytest.mark.parametrize("shape,p,seed,direction", [
    ((6, 5, 1), 0.7, 2, 1), ((5, 4, 3), 0.6, 4, 0), ((4, 5, 4), 0.5, 5, 1), ((16, 16, 1), 0.65, 7, 0),
    ((7, 6, 5), 0.45, 8, 2)])
def test_c_oracle_dense_bruteforce_and_labels(shape, p, seed, direction):
    net = inputs.iid_diluted(*shape, seed=seed, p=p)
    res = crun(net, direction)
    Pd, _ = brute_force_dense(net, direction)
    defined = res.classes != po.FLOATING
    assert np.max(np.abs(res.P[defined] - Pd[defined])) < 1e-11
    assert np.array_equal(res.classes, independent_classes(net, direction))


@pytest.mark.parametrize("maker,direction", [
    (lambda: inputs.cfg1_iid_2d(64, 64, seed=0), 0),
    (lambda: inputs.cfg2_fbm_2d(48, 40, seed=1), 0),
    (lambda: inputs.cfg3_percolation_3d(20, 18, 16, seed=2, p=0.35), 0),
    (lambda: inputs.cfg4_fbm_cut_3d(20, 20, 20, seed=3), 1),
    (lambda: inputs.cfg5_stratified_3d(16, 14, 18, seed=4), 2),
])
def test_c_oracle_matches_python_oracle(maker, direction):
    net = maker()
    a = po.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13)
    b = crun(net, direction)
    assert np.array_equal(a.classes, b.classes)
    assert (a.n_solved, a.n_inlet_only, a.n_outlet_only, a.n_floating) == \
           (b.n_solved, b.n_inlet_only, b.n_outlet_only, b.n_floating)
    assert np.max(np.abs(a.P - b.P)) < 1e-11
    assert b.g_eff == pytest.approx(a.g_eff, rel=1e-11)
    assert b.q_in == pytest.approx(a.q_in, rel=1e-11) and b.q_out == pytest.approx(a.q_out, rel=1e-11)
    assert b.rel_residual <= 1e-13 and b.status == "ok"
    rel, pin = c_oracle.certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, a.P, direction)
    assert rel <= 1e-13 and pin == 0.0
    relp, _ = po.residual_certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, b.P, direction)
    assert relp <= 1e-13


def test_c_oracle_no_spanning_cluster_and_errors():
    net = inputs.iid_diluted(30, 30, 1, seed=3, p=0.2)
    res = crun(net, 0)
    assert res.status == "no_spanning_cluster" and res.g_eff == 0.0
    bad = inputs.uniform(4, 4, 1, 1.0)
    bad.gx[0, 1, 1] = -2.0
    with pytest.raises(ValueError):
        crun(bad, 0)
    with pytest.raises(ValueError):
        crun(inputs.uniform(2, 4, 1, 1.0), 0)
    # max_iter is honoured and reported
    net = inputs.cfg1_iid_2d(32, 32, seed=0)
    r = crun(net, 0, tol=1e-13, max_iter=5)
    assert r.status == "max_iters" and r.iterations == 5 and r.rel_residual > 1e-13


# ---------------------------------------------------------------- periodic lateral faces ---
def test_c_oracle_periodic_hand_worked_example():
    """tests/golden/worked_3x2_periodic.txt: 55/141, 57/141, 338/141."""
    gx = np.array([[[1, 2, 99], [3, 4, 99]]], dtype=np.float32)
    gy = np.array([[[77, 5, 77], [88, 7, 88]]], dtype=np.float32)
    r = c_oracle.solve(3, 2, 1, gx, gy, None, 0, 1e-15, periodic=True)
    assert r.P[0, 0, 1] == pytest.approx(55 / 141, abs=1e-14)
    assert r.P[0, 1, 1] == pytest.approx(57 / 141, abs=1e-14)
    assert r.g_eff == pytest.approx(338 / 141, rel=1e-13)


@pytest.mark.parametrize("maker,direction", [
    (lambda: inputs.cfg1_iid_2d(40, 33, seed=0), 0),
    (lambda: inputs.cfg3_percolation_3d(20, 18, 16, seed=2, p=0.35), 0),
    (lambda: inputs.cfg4_fbm_cut_3d(20, 20, 20, seed=3), 1),
    (lambda: inputs.iid_diluted(9, 2, 7, seed=5, p=0.8), 2),
])
def test_c_oracle_periodic_matches_python_oracle(maker, direction):
    net = maker()
    a = po.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13, periodic=True)
    b = c_oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13, periodic=True)
    assert np.array_equal(a.classes, b.classes)
    assert np.max(np.abs(a.P - b.P)) < 1e-11
    assert b.g_eff == pytest.approx(a.g_eff, rel=1e-11)
    rel, pin = c_oracle.certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, a.P, direction, periodic=True)
    assert rel <= 1e-13 and pin == 0.0
    rel0, _ = c_oracle.certificate(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, a.P, direction)
    assert rel0 > 1e-6          # the no-flux operator rejects the periodic solution


def test_starting_iterate_and_decade_log():
    """`P_start` (used by tests/golden/make_digest.py to carry a tol-1e-12 solution on to the floor) changes only x0: the
    continued solve lands on the zero-start solution; the per-decade iteration log is a record (monotone, ends at the
    last decade reached) and does not touch the iteration."""
    from oracle import c_oracle
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg4_fbm_cut_3d(40, 36, 33)
    args = (net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, 0)
    zero = c_oracle.solve(*args, 1e-13)
    a = c_oracle.solve(*args, 1e-12)
    b = c_oracle.solve(*args, 1e-13, P_start=a.P)
    assert a.status == b.status == zero.status == "ok"
    assert 0 < b.iterations < 0.5 * zero.iterations
    assert np.max(np.abs(b.P - zero.P)) <= 1e-9 and abs(b.g_eff - zero.g_eff) <= 1e-11 * abs(zero.g_eff)
    assert np.array_equal(b.classes, zero.classes)
    dec = [d for d in a.it_decade if d > 0]
    assert dec == sorted(dec) and len(dec) == 13 and dec[-1] <= a.iterations    # decades 1e-0 .. 1e-12 reached
    assert a.it_decade[13] == -1
    c = c_oracle.solve(*args, 1e-12)
    assert c.iterations == a.iterations and np.max(np.abs(c.P - a.P)) <= 1e-12      # (OpenMP sums: not bit-identical)


def test_digest_script_on_a_small_sibling(tmp_path):
    """tests/golden/make_digest.py end to end at 24^3: the stored numbers are the oracle's."""
    import json
    import os
    import subprocess
    import sys
    from oracle import c_oracle
    from paper_1908_03301_b200 import inputs
    script = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_digest.py")
    subprocess.check_call([sys.executable, script, "cfg4", "--n", "24", "--out", str(tmp_path)], stdout=subprocess.DEVNULL)
    d = json.load(open(tmp_path / "cfg4_24_x_digest.json"))
    sub = np.load(tmp_path / "cfg4_24_x_P_sub8.npy")
    net = inputs.cfg4_fbm_cut_3d(24, 24, 24)
    ref = c_oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, 0, 1e-13)
    assert d["input_sha256"] == net.sha256() and d["n_solved"] == ref.n_solved
    assert abs(d["g_eff"] - ref.g_eff) <= 1e-11 * abs(ref.g_eff)
    assert np.max(np.abs(sub - ref.P[4::8, 4::8, 4::8])) <= 1e-9
    assert len(d["plane_fluxes"]) == 23 and max(abs(f - d["g_eff"]) for f in d["plane_fluxes"]) <= 1e-9 * abs(d["g_eff"])
