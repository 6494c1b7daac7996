"""DESIGN.md reading 19, checked on the CPU: an fp32 conjugate-gradient loop with reliable updates (the arithmetic of the
single-kernel schemes, written out plainly in numpy) needs the same number of iterations whether the recursive residual is
STORED or RECOVERED from the last two search directions, r_t = p_t - beta_t p_{t-1}.  This is the experiment that was run
before the kernels stopped storing the residual; the kernels themselves are compared with the oracle in the GPU tests.
The operator comes from the oracle's assembly (test infrastructure); nothing here touches the CUDA path."""
import numpy as np
import pytest
import scipy.sparse as sp

f32 = np.float32


def _dot(a, c):
    return float(np.dot(a.astype(np.float64), c.astype(np.float64)))   # fp32 values, fp64 accumulation (S8c reading 19)


def _solve(A, b, diag, recover, delta=0.3, tol=1e-10, maxit=20000):
    """Jacobi-scaled fp32 CG, never restarted; fp64 true residual whenever the recursive one has fallen by `delta`."""
    m = A.shape[0]
    s = 1.0 / np.sqrt(diag)
    S = sp.diags(s)
    Ah32 = (S @ A @ S).tocsr().astype(f32)
    x64 = np.zeros(m)
    bn = np.linalg.norm(b)
    r = (s * b).astype(f32)
    rr = _dot(r, r)
    rr_max, rr_target = rr, (0.7 * tol) ** 2 * rr
    p, pold, xh = r.copy(), np.zeros(m, f32), np.zeros(m, f32)
    beta, explicit, its, outer = 0.0, True, 0, 1
    while its < maxit:
        q = (Ah32 @ p).astype(f32)
        alpha = rr / _dot(p, q)
        xh = (xh + f32(alpha) * p).astype(f32)
        if recover and not explicit:
            r = (p - f32(beta) * pold).astype(f32)          # r_t from p_t = r_t + beta_t p_{t-1}
        r = (r - f32(alpha) * q).astype(f32)
        explicit = False
        rr_new = _dot(r, r)
        its += 1
        if rr_new < delta * delta * rr_max or rr_new <= rr_target:
            x64 += s * xh.astype(np.float64)
            xh[:] = 0
            r64 = b - A @ x64
            outer += 1
            rel = np.linalg.norm(r64) / bn
            if rel <= tol:
                return its, outer, rel
            r = (s * r64).astype(f32)                        # the explicit residual of the replacement
            rr_true = _dot(r, r)
            beta, rr, rr_max, explicit = rr_true / rr, rr_true, rr_true, True
        else:
            beta, rr = rr_new / rr, rr_new
            rr_max = max(rr_max, rr)
        pold = p
        p = (r + f32(beta) * p).astype(f32)
    return its, outer, None


@pytest.mark.parametrize("maker,n", [("cfg4_fbm_cut_3d", 40), ("cfg5_stratified_3d", 32), ("cfg3_percolation_3d", 40)])
def test_recovered_residual_needs_the_same_iterations(maker, n):
    from oracle import pn_oracle as po
    from paper_1908_03301_b200 import inputs
    net = getattr(inputs, maker)(n, n, n)
    g64 = po.widen(n, n, n, net.gx, net.gy, net.gz)
    cls = po.classify(n, n, n, g64, 0)
    cls = cls[0] if isinstance(cls, tuple) else cls
    A, b, diag, _ = po.assemble(n, n, n, g64, cls)
    if A.shape[0] == 0:
        pytest.skip("no spanning cluster")
    stored = _solve(A, b, diag, recover=False)
    recovered = _solve(A, b, diag, recover=True)
    assert stored[2] is not None and recovered[2] is not None            # both reach the true fp64 residual 1e-10
    assert abs(recovered[0] - stored[0]) <= 0.08 * stored[0] + 3, (stored, recovered)
    assert abs(recovered[1] - stored[1]) <= 2
