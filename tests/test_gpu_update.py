"""GPU parity of pn_update_conductances / pn_replace_conductances ("thousands of time
steps"): a sequence of networks, each a small change of the one before, solved on ONE handle (labels reused, warm
start) and compared at EVERY step, element by element, with the oracle solving that step's network from scratch.
Tolerances as in test_gpu_parity.py (north_star): 1e-8 L_inf on pressures, 1e-9 relative on G_eff."""
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


def _check(pn, oracle, h, arrays, shape, direction, tol, periodic=False):
    nx, ny, nz = shape
    info = h.solve(direction, tol, accept=(pn.PN_OK,))
    P = h.pressures().cpu().numpy()
    cls = h.classes().cpu().numpy()
    fl = h.flux()
    ref = oracle.solve(nx, ny, nz, arrays[0], arrays[1], arrays[2], direction, 1e-13, periodic=periodic)
    assert np.array_equal(cls, ref.classes)
    assert (info.n_solved, info.n_floating) == (ref.n_solved, ref.n_floating)
    err = float(np.max(np.abs(P - ref.P)))
    assert err <= P_TOL, f"pressure L_inf error {err:.3e}"
    assert abs(fl[2] - ref.g_eff) <= G_TOL * abs(ref.g_eff)
    return info


def _perturb_open(rng, arrays, frac, eps):
    """A random subset of the OPEN bonds changes by a factor exp(eps * N(0,1)): none crosses zero.  Returns the lists."""
    axis, node, value = [], [], []
    for a, g in enumerate(arrays):
        if g is None:
            continue
        flat = g.reshape(-1)
        idx = np.flatnonzero(flat > 0)
        pick = rng.choice(idx, size=max(1, int(frac * idx.size)), replace=False)
        new = (flat[pick].astype(np.float64) * np.exp(eps * rng.standard_normal(pick.size))).astype(np.float32)
        new = np.maximum(new, np.float32(1e-6))
        flat[pick] = new
        axis.append(np.full(pick.size, a, dtype=np.int32))
        node.append(pick.astype(np.int64))
        value.append(new)
    return np.concatenate(axis), np.concatenate(node), np.concatenate(value)


def test_time_stepping_sequence_128(pn, oracle):
    """Ten steps at 128^3 (CFG4's recipe, 40 % of the bonds closed): sparse updates from host and device lists, one
    full replacement, one step that opens and closes bonds (labels must be redone there and only there)."""
    import torch
    from paper_1908_03301_b200 import inputs
    n = 128
    net = inputs.cfg4_fbm_cut_3d(n, n, n)
    arrays = [net.gx.copy(), net.gy.copy(), net.gz.copy()]
    rng = np.random.default_rng(5)
    h = pn.Network(n, n, n)
    h.set_conductances(*arrays)
    cold = _check(pn, oracle, h, arrays, (n, n, n), 0, 1e-13)
    assert cold.labels_reused == 0
    iters = []
    for step in range(10):
        if step == 4:          # full replacement, every open bond drifts by ~0.1 %
            for g in arrays:
                flat = g.reshape(-1)
                openb = flat > 0
                flat[openb] = (flat[openb].astype(np.float64) * np.exp(1e-3 * rng.standard_normal(int(openb.sum())))).astype(np.float32)
            h.replace_conductances(*(torch.from_numpy(g).cuda() for g in arrays))
            expect_reuse = 1
        elif step == 7:        # topology change: close some open bonds, open some closed ones
            axis, node, value = [], [], []
            for a, g in enumerate(arrays):
                flat = g.reshape(-1)
                op = rng.choice(np.flatnonzero(flat > 0), size=200, replace=False)
                cl = rng.choice(np.flatnonzero(flat == 0), size=200, replace=False)
                flat[op] = 0.0
                flat[cl] = 0.5
                axis += [np.full(400, a, dtype=np.int32)]
                node += [np.concatenate([op, cl]).astype(np.int64)]
                value += [np.concatenate([np.zeros(200, np.float32), np.full(200, 0.5, np.float32)])]
            h.update_conductances(np.concatenate(axis), np.concatenate(node), np.concatenate(value))
            expect_reuse = 0
        else:
            axis, node, value = _perturb_open(rng, arrays, 0.01, 0.05)
            if step % 2:
                h.update_conductances(torch.from_numpy(axis).cuda(), torch.from_numpy(node).cuda(), torch.from_numpy(value).cuda())
            else:
                h.update_conductances(axis, node, value)
            expect_reuse = 1
        info = _check(pn, oracle, h, arrays, (n, n, n), 0, 1e-13)
        assert info.labels_reused == expect_reuse, f"step {step}"
        iters.append(info.inner_iters)
    h.close()
    # a warm start never costs more than the cold solve; how much it saves depends on the size of the change
    assert max(iters) <= cold.inner_iters * 1.02


@pytest.mark.parametrize("periodic", [False, True])
def test_update_with_peeling_and_direction_change(pn, oracle, periodic):
    """Near the threshold with dead-end peeling forced on: the peeled set is topology, so it is reused with the labels;
    a change of direction voids them."""
    from paper_1908_03301_b200 import inputs
    net = inputs.cfg3_percolation_3d(40, 36, 33, p=0.32)
    arrays = [net.gx.copy(), net.gy.copy(), net.gz.copy()]
    rng = np.random.default_rng(8)
    h = pn.Network(net.nx, net.ny, net.nz)
    h.set_option(pn.PN_OPT_PEEL, 1)
    if periodic:
        h.set_option(pn.PN_OPT_LATERAL, 1)
    h.set_conductances(*arrays)
    shape = (net.nx, net.ny, net.nz)
    first = _check(pn, oracle, h, arrays, shape, 0, 1e-12, periodic)
    assert first.n_peeled > 0 and first.labels_reused == 0
    h.update_conductances(*_perturb_open(rng, arrays, 0.2, 0.3))
    second = _check(pn, oracle, h, arrays, shape, 0, 1e-12, periodic)
    assert second.labels_reused == 1 and second.n_peeled == first.n_peeled
    third = _check(pn, oracle, h, arrays, shape, 2, 1e-12, periodic)      # other direction: labels redone
    assert third.labels_reused == 0
    h.update_conductances(*_perturb_open(rng, arrays, 0.2, 0.3))
    h.set_option(pn.PN_OPT_X0, 0)                                         # explicit zero start with reused labels
    fourth = _check(pn, oracle, h, arrays, shape, 2, 1e-12, periodic)
    assert fourth.labels_reused == 1
    h.set_option(pn.PN_OPT_REUSE_LABELS, 0)
    fifth = _check(pn, oracle, h, arrays, shape, 2, 1e-12, periodic)
    assert fifth.labels_reused == 0
    h.close()


def test_update_2d_and_repeat_solve(pn, oracle):
    """2D (caller axis 1 = the internal row-to-row bonds); a second solve without any change reuses the labels too."""
    from paper_1908_03301_b200 import inputs
    net = inputs.iid_diluted(300, 220, 1, seed=3, p=0.7)
    arrays = [net.gx.copy(), net.gy.copy(), None]
    rng = np.random.default_rng(2)
    h = pn.Network(300, 220, 1)
    h.set_conductances(arrays[0], arrays[1], None)
    _check(pn, oracle, h, arrays, (300, 220, 1), 1, 1e-12)
    again = _check(pn, oracle, h, arrays, (300, 220, 1), 1, 1e-12)
    assert again.labels_reused == 1
    h.update_conductances(*_perturb_open(rng, arrays, 0.3, 0.2))
    upd = _check(pn, oracle, h, arrays, (300, 220, 1), 1, 1e-12)
    assert upd.labels_reused == 1
    h.close()


def test_update_error_paths(pn):
    from paper_1908_03301_b200 import inputs
    net = inputs.uniform(8, 6, 5, 1.0)
    h = pn.Network(8, 6, 5)
    one = (np.array([0], np.int32), np.array([3], np.int64), np.array([2.0], np.float32))
    with pytest.raises(pn.PnError) as e:
        h.update_conductances(*one)
    assert e.value.code == pn.PN_ERR_STATE                      # no network yet
    h.set_conductances(net.gx, net.gy, net.gz)
    h.solve(0, 1e-10)
    h.update_conductances(*one)
    with pytest.raises(pn.PnError) as e:
        h.flux()                                                # the previous solve's results are gone
    assert e.value.code == pn.PN_ERR_STATE
    h.solve(0, 1e-10)
    for bad, code in (((np.array([3], np.int32), np.array([3], np.int64), np.array([1.0], np.float32)), pn.PN_ERR_ARG),
                      ((np.array([0], np.int32), np.array([240], np.int64), np.array([1.0], np.float32)), pn.PN_ERR_ARG),
                      ((np.array([0], np.int32), np.array([3], np.int64), np.array([-1.0], np.float32)), pn.PN_ERR_VALUE),
                      ((np.array([1], np.int32), np.array([3], np.int64), np.array([np.nan], np.float32)), pn.PN_ERR_VALUE)):
        h.set_conductances(net.gx, net.gy, net.gz)
        with pytest.raises(pn.PnError) as e:
            h.update_conductances(*bad)
        assert e.value.code == code
        with pytest.raises(pn.PnError) as e:
            h.solve(0, 1e-10)                                   # the handle keeps no network after a failed update
        assert e.value.code == pn.PN_ERR_STATE
    h.set_conductances(net.gx, net.gy, net.gz)
    bad = net.gx.copy()
    bad.reshape(-1)[5] = -2.0
    with pytest.raises(pn.PnError) as e:
        h.replace_conductances(bad, net.gy, net.gz)
    assert e.value.code == pn.PN_ERR_VALUE
    h.close()
