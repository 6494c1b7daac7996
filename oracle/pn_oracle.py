"""CPU ORACLE (test infrastructure, NOT the product) for the bond-network pressure solve.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this file.  It shares no code with the CUDA path (`paper_1908_03301_b200/`) and imports nothing
from it; inputs arrive as plain numpy arrays.

What it computes (citations: /root/reference/PAPER.md = `P:<line>`, SURVEY.md 8(c) = `S8c`):

  * bond law and node balance:  q_ij = g_ij (P_j - P_i),  sum_{j in i} q_ij = 0  at every
    interior node  ->  G P = b, eq.(3) P:55;
  * boundary conditions, P:57 + S8c readings 1-2: fixed pressure drop along axis `a`, imposed as
    P = 1 on the node plane coord_a = 0 and P = 0 on coord_a = n_a - 1; NO-FLUX on every other face
    (BASELINE.json north_star / configs[0] bind this); `periodic=True` gives the paper's own side condition,
    lateral axes wrapping around (S8(f) item 2);
  * isolated / dead-end clusters, S8c step 3 (the paper is silent; north_star mandates it): serial
    breadth-first labelling of interior nodes through open (g > 0) bonds; a component that touches
    both Dirichlet planes is SOLVED, inlet-only is pinned to 1, outlet-only to 0, floating to 0;
  * the solve, P:63 / P:79 / ref [57] P:218: assembled sparse Laplacian over the solved nodes,
    textbook Jacobi-preconditioned conjugate gradient (Barrett et al. "Templates" form) in fp64,
    true residual recomputed and the iteration restarted from it until ||b - A x||2 <= tol ||b||2;
  * effective conductance / permeability, eq.(4) P:59-61 + S8c readings 16-17:
    Q_in, Q_out through the bonds leaving the inlet plane / entering the outlet plane,
    G_eff = (Q_in + Q_out) / 2 (dP = 1),  K = G_eff (n_a - 1) / S_perp  (mu = l = 1).

The float32 input conductances are widened to fp64 exactly: they ARE the problem (S8c reading 14).
Array layout: shape (nz, ny, nx), x fastest, forward-bond convention (see the inputs module).

Parity pins: every function here is pinned by tests/test_oracle_pins.py (closed forms, the hand-worked
3x2 example of S8c, dense LAPACK solves, brute-force labelling, conservation invariants).
"""
from __future__ import annotations

from collections import deque
from dataclasses import dataclass

import numpy as np
import scipy.sparse as sp

# node classes (S8c steps 2-3)
INLET, OUTLET, SOLVED, INLET_ONLY, OUTLET_ONLY, FLOATING = 0, 1, 2, 3, 4, 5


@dataclass
class OracleResult:
    P: np.ndarray                 # (nz, ny, nx) fp64 pressures on ALL nodes
    classes: np.ndarray           # (nz, ny, nx) int8 node class
    q_in: float
    q_out: float
    g_eff: float
    k_eff: float
    iterations: int
    restarts: int
    rel_residual: float           # true ||b - A x||2 / ||b||2 over solved nodes
    n_solved: int
    n_inlet_only: int
    n_outlet_only: int
    n_floating: int
    status: str                   # "ok" | "no_spanning_cluster" | "max_iters"


# --------------------------------------------------------------------------------------------------
# step 1: inputs
# --------------------------------------------------------------------------------------------------
def wrap_axes(nx, ny, nz, direction, periodic):
    """Which lattice axes wrap around.  P:57: "periodic boundary conditions in the second direction" -- with
    `periodic` every LATERAL axis (not the axis of the pressure drop) of length >= 2 wraps: the forward-bond
    entry of the last node along that axis is then a real bond to the first node.  (Length 1: the wrap bond
    would join a node to itself and carries nothing.)  Without `periodic`: no-flux faces, nothing wraps."""
    dims = (nx, ny, nz)
    return tuple(bool(periodic) and a != direction and dims[a] >= 2 for a in range(3))


def widen(nx, ny, nz, gx, gy, gz, wrap=(False, False, False)):
    """fp32 -> fp64 exactly; zero the entries that are not bonds (forward neighbour off-lattice and the axis
    does not wrap)."""
    shp = (nz, ny, nx)
    out = []
    for a, g in enumerate((gx, gy, gz)):
        if g is None:
            if a == 2 and nz == 1:
                out.append(np.zeros(shp, dtype=np.float64))
                continue
            raise ValueError("missing conductance array")
        g = np.asarray(g)
        if g.shape != shp:
            g = g.reshape(shp)
        g64 = g.astype(np.float32).astype(np.float64)
        g64 = g64.copy()
        if wrap[a]:
            pass                              # the last entry along a is the bond back to index 0
        elif a == 0:
            g64[:, :, nx - 1] = 0.0
        elif a == 1:
            g64[:, ny - 1, :] = 0.0
        else:
            g64[nz - 1, :, :] = 0.0
        if not np.all(np.isfinite(g64)) or np.any(g64 < 0.0):
            raise ValueError("conductances must be finite and >= 0")
        out.append(g64)
    return out


def _coord_along(nx, ny, nz, direction):
    """Integer coordinate along the solve axis for every node, and the axis length."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    c = (i, j, k)[direction]
    return c, (nx, ny, nz)[direction]


# --------------------------------------------------------------------------------------------------
# steps 2-3: node classes by serial breadth-first labelling
# --------------------------------------------------------------------------------------------------
def classify(nx, ny, nz, g64, direction, wrap=(False, False, False)):
    """Class of every node (S8c steps 2-3).  Plain serial BFS with an explicit queue.

    Edges of the search: interior-interior bonds with g > 0.  `touches_in` / `touches_out` of a
    component: some member has an open bond to an inlet- / outlet-plane node.
    """
    gx, gy, gz = g64
    N = nx * ny * nz
    n_a = (nx, ny, nz)[direction]
    if n_a < 3:
        raise ValueError("axis along the pressure drop needs >= 3 node planes")
    fx, fy, fz = gx.ravel(), gy.ravel(), gz.ravel()
    stride = (1, nx, nx * ny)
    dims = (nx, ny, nz)
    fwd = (fx, fy, fz)

    def coords(n):
        return (n % nx, (n // nx) % ny, n // (nx * ny))

    cls = np.full(N, -1, dtype=np.int8)
    ca = _coord_along(nx, ny, nz, direction)[0].ravel()
    cls[ca == 0] = INLET
    cls[ca == n_a - 1] = OUTLET

    fxl, fyl, fzl = fx.tolist(), fy.tolist(), fz.tolist()
    fl = (fxl, fyl, fzl)
    clsl = cls.tolist()

    def neighbours(n):
        c = coords(n)
        for a in range(3):
            if c[a] + 1 < dims[a]:
                g = fl[a][n]
                if g > 0.0:
                    yield n + stride[a]
            elif wrap[a]:
                if fl[a][n] > 0.0:
                    yield n - (dims[a] - 1) * stride[a]
            if c[a] > 0:
                m = n - stride[a]
                g = fl[a][m]
                if g > 0.0:
                    yield m
            elif wrap[a]:
                m = n + (dims[a] - 1) * stride[a]
                if fl[a][m] > 0.0:
                    yield m

    for seed in range(N):
        if clsl[seed] != -1:
            continue
        comp = [seed]
        clsl[seed] = SOLVED            # provisional mark = "visited"
        queue = deque([seed])
        t_in = t_out = False
        while queue:
            n = queue.popleft()
            for m in neighbours(n):
                cm = clsl[m]
                if cm == INLET:
                    t_in = True
                elif cm == OUTLET:
                    t_out = True
                elif cm == -1:
                    clsl[m] = SOLVED
                    comp.append(m)
                    queue.append(m)
        if t_in and t_out:
            c = SOLVED
        elif t_in:
            c = INLET_ONLY
        elif t_out:
            c = OUTLET_ONLY
        else:
            c = FLOATING
        if c != SOLVED:
            for n in comp:
                clsl[n] = c
    return np.asarray(clsl, dtype=np.int8).reshape(nz, ny, nx)


# --------------------------------------------------------------------------------------------------
# dead ends inside the spanning clusters (S8c reading 7, S8(f) item 1)
# --------------------------------------------------------------------------------------------------
def dangling_ends(nx, ny, nz, g64, classes, wrap=(False, False, False)):
    """Boolean mask (nz, ny, nx) of the SOLVED nodes that are dangling (tree-like dead) ends.

    Definition (S8c reading 7: "dangling branches inside a spanning cluster have well-defined pressures
    ... tree ends carrying no flow"): strip, one at a time and until none is left, any SOLVED node that has
    exactly ONE open bond to a node that is still present (present = SOLVED and not yet stripped, or on a
    Dirichlet plane).  What remains is the 2-core of the spanning clusters with the Dirichlet nodes kept;
    the stripped nodes carry no current and sit at the pressure of the node their tree hangs from.
    These nodes STAY unknowns of the oracle's linear system; this mask only says which ones a solver may
    remove and back-fill.  Serial work-list implementation."""
    gx, gy, gz = g64
    N = nx * ny * nz
    cls = classes.ravel().tolist()
    fl = (gx.ravel().tolist(), gy.ravel().tolist(), gz.ravel().tolist())
    stride = (1, nx, nx * ny)
    dims = (nx, ny, nz)
    present = [c in (INLET, OUTLET, SOLVED) for c in cls]

    def open_neighbours(n):
        c = (n % nx, (n // nx) % ny, n // (nx * ny))
        out = []
        for a in range(3):
            up = n + stride[a] if c[a] + 1 < dims[a] else (n - (dims[a] - 1) * stride[a] if wrap[a] else -1)
            if up >= 0 and fl[a][n] > 0.0 and present[up]:
                out.append(up)
            dn = n - stride[a] if c[a] > 0 else (n + (dims[a] - 1) * stride[a] if wrap[a] else -1)
            if dn >= 0 and fl[a][dn] > 0.0 and present[dn]:
                out.append(dn)
        return out

    stripped = [False] * N
    work = deque(n for n in range(N) if cls[n] == SOLVED)
    while work:
        n = work.popleft()
        if stripped[n] or cls[n] != SOLVED:
            continue
        nb = open_neighbours(n)
        if len(nb) == 1 and cls[nb[0]] == SOLVED:
            stripped[n] = True
            present[n] = False
            work.append(nb[0])
    return np.asarray(stripped, dtype=bool).reshape(nz, ny, nx)


# --------------------------------------------------------------------------------------------------
# step 4: assembled sparse Laplacian over the solved nodes
# --------------------------------------------------------------------------------------------------
def assemble(nx, ny, nz, g64, classes, wrap=(False, False, False)):
    """CSR `A` (fp64) and `b` over SOLVED nodes (S8c step 4).

    A_ii = sum of g over ALL open incident bonds (bonds to Dirichlet nodes included),
    A_ij = -g_ij for solved-solved bonds, b_i = sum_{j in inlet plane} g_ij * 1.
    Returns (A, b, diag, idx) with idx = flat lattice index of every unknown.
    """
    N = nx * ny * nz
    cls = classes.ravel()
    solved = cls == SOLVED
    idx = np.flatnonzero(solved)
    m = idx.size
    unk = np.full(N, -1, dtype=np.int64)
    unk[idx] = np.arange(m)
    diag = np.zeros(m)
    b = np.zeros(m)
    rows, cols, vals = [], [], []
    stride = (1, nx, nx * ny)
    flat = np.arange(N)
    coord = (flat % nx, (flat // nx) % ny, flat // (nx * ny))
    dims = (nx, ny, nz)
    for a in range(3):
        g = g64[a].ravel()
        inside = coord[a] + 1 < dims[a]
        has = (inside | wrap[a]) & (g > 0.0)
        n0 = flat[has]                       # the end that stores the bond (forward-bond convention)
        n1 = np.where(inside[has], n0 + stride[a], n0 - (dims[a] - 1) * stride[a])   # other end (wrapped at the face)
        gb = g[has]
        for me, other in ((n0, n1), (n1, n0)):
            mine = solved[me]
            u = unk[me[mine]]
            o = other[mine]
            gg = gb[mine]
            np.add.at(diag, u, gg)
            oc = cls[o]
            np.add.at(b, u[oc == INLET], gg[oc == INLET])
            ss = oc == SOLVED
            rows.append(u[ss])
            cols.append(unk[o[ss]])
            vals.append(-gg[ss])
    rows.append(np.arange(m))
    cols.append(np.arange(m))
    vals.append(diag)
    A = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                      shape=(m, m))
    return A, b, diag, idx


# --------------------------------------------------------------------------------------------------
# step 5: textbook Jacobi-PCG (Barrett et al., "Templates", fig. 2.5), fp64
# --------------------------------------------------------------------------------------------------
def pcg(A, b, diag, x0, target, max_iter):
    """Preconditioned CG with M = diag(A).  Stops when the RECURSIVE residual 2-norm <= target.

    x0 = start; r = b - A x0; z = r / diag; p = z; rho = r.z
    loop: q = A p; alpha = rho / (p.q); x += alpha p; r -= alpha q; test; z = r / diag;
          rho' = r.z; beta = rho' / rho; p = z + beta p; rho = rho'
    """
    x = x0.copy()
    r = b - A @ x
    it = 0
    if np.sqrt(r @ r) <= target:
        return x, it
    z = r / diag
    p = z.copy()
    rho = r @ z
    while it < max_iter:
        q = A @ p
        alpha = rho / (p @ q)
        x += alpha * p
        r -= alpha * q
        it += 1
        if np.sqrt(r @ r) <= target:
            break
        z = r / diag
        rho_new = r @ z
        beta = rho_new / rho
        p = z + beta * p
        rho = rho_new
    return x, it


def solve_spd(A, b, diag, tol, max_iter=200000, max_restarts=20):
    """Run `pcg` from zero; recompute the TRUE residual; restart from it while it misses `tol`
    (recursive and true residual part ways near the fp64 floor, S8c consequence (iii))."""
    nb = np.sqrt(b @ b)
    x = np.zeros_like(b)
    total = 0
    restarts = 0
    rel = 0.0
    if nb == 0.0:
        return x, 0, 0, 0.0
    best = None
    for restarts in range(max_restarts):
        x, it = pcg(A, b, diag, x, 0.7 * tol * nb if restarts else tol * nb, max_iter - total)
        total += it
        rel = np.sqrt(np.sum((b - A @ x) ** 2)) / nb
        if best is None or rel < best[1]:
            best = (x.copy(), rel)
        if rel <= tol or total >= max_iter or it == 0:
            break
    x, rel = best
    return x, total, restarts, rel


# --------------------------------------------------------------------------------------------------
# steps 6-7: scatter and flux
# --------------------------------------------------------------------------------------------------
def pin_values(classes):
    P = np.zeros(classes.shape, dtype=np.float64)
    P[classes == INLET] = 1.0
    P[classes == INLET_ONLY] = 1.0
    return P


def flux(nx, ny, nz, g64, P, direction):
    """Q_in, Q_out, G_eff, K (S8c step 7; eq.(4) P:61 with mu = l = 1, dP = 1, L = n_a - 1)."""
    g = g64[direction]
    n_a = (nx, ny, nz)[direction]
    ax = 2 - direction                       # array axis of lattice axis `direction`
    Pm = np.moveaxis(P, ax, 0)
    gm = np.moveaxis(g, ax, 0)
    q_in = float(np.sum(gm[0] * (Pm[0] - Pm[1])))
    q_out = float(np.sum(gm[n_a - 2] * (Pm[n_a - 2] - Pm[n_a - 1])))
    g_eff = 0.5 * (q_in + q_out)
    s_perp = (nx * ny * nz) // n_a
    return q_in, q_out, g_eff, g_eff * (n_a - 1) / s_perp


def plane_fluxes(nx, ny, nz, g64, P, direction):
    """Total flow through every plane of bonds perpendicular to the solve axis (n_a - 1 values)."""
    g = g64[direction]
    ax = 2 - direction
    Pm = np.moveaxis(P, ax, 0)
    gm = np.moveaxis(g, ax, 0)
    n_a = Pm.shape[0]
    return np.array([np.sum(gm[c] * (Pm[c] - Pm[c + 1])) for c in range(n_a - 1)])


def dissipation(nx, ny, nz, g64, P, wrap=(False, False, False)):
    """sum over all bonds of g (dP_bond)^2  (= Q * dP at the exact solution; energy identity)."""
    e = 0.0
    if wrap[0]:
        e += float(np.sum(g64[0][:, :, -1] * (P[:, :, 0] - P[:, :, -1]) ** 2))
    if wrap[1]:
        e += float(np.sum(g64[1][:, -1, :] * (P[:, 0, :] - P[:, -1, :]) ** 2))
    if wrap[2]:
        e += float(np.sum(g64[2][-1, :, :] * (P[0, :, :] - P[-1, :, :]) ** 2))
    e += float(np.sum(g64[0][:, :, :-1] * (P[:, :, 1:] - P[:, :, :-1]) ** 2))
    e += float(np.sum(g64[1][:, :-1, :] * (P[:, 1:, :] - P[:, :-1, :]) ** 2))
    e += float(np.sum(g64[2][:-1, :, :] * (P[1:, :, :] - P[:-1, :, :]) ** 2))
    return e


def kirchhoff_residual(nx, ny, nz, g64, P, wrap=(False, False, False)):
    """Net current into every node, sum_j g_ij (P_j - P_i), on the whole lattice."""
    r = np.zeros((nz, ny, nx))
    if wrap[0]:
        f = g64[0][:, :, -1] * (P[:, :, 0] - P[:, :, -1])
        r[:, :, -1] += f
        r[:, :, 0] -= f
    if wrap[1]:
        f = g64[1][:, -1, :] * (P[:, 0, :] - P[:, -1, :])
        r[:, -1, :] += f
        r[:, 0, :] -= f
    if wrap[2]:
        f = g64[2][-1, :, :] * (P[0, :, :] - P[-1, :, :])
        r[-1, :, :] += f
        r[0, :, :] -= f
    fx = g64[0][:, :, :-1] * (P[:, :, 1:] - P[:, :, :-1])
    r[:, :, :-1] += fx
    r[:, :, 1:] -= fx
    fy = g64[1][:, :-1, :] * (P[:, 1:, :] - P[:, :-1, :])
    r[:, :-1, :] += fy
    r[:, 1:, :] -= fy
    fz = g64[2][:-1, :, :] * (P[1:, :, :] - P[:-1, :, :])
    r[:-1, :, :] += fz
    r[1:, :, :] -= fz
    return r


# --------------------------------------------------------------------------------------------------
# the whole path
# --------------------------------------------------------------------------------------------------
def solve(nx, ny, nz, gx, gy, gz, direction=0, tol=1e-13, max_iter=200000, dense=False, periodic=False):
    """Pressures on all nodes + effective conductance (S8c steps 1-8).  `periodic`: lateral faces wrap (the
    paper's own side condition) instead of the default no-flux faces (north_star)."""
    wrap = wrap_axes(nx, ny, nz, direction, periodic)
    g64 = widen(nx, ny, nz, gx, gy, gz, wrap)
    classes = classify(nx, ny, nz, g64, direction, wrap)
    P = pin_values(classes)
    counts = [int(np.sum(classes == c)) for c in (SOLVED, INLET_ONLY, OUTLET_ONLY, FLOATING)]
    if counts[0] == 0:
        q_in, q_out, g_eff, k_eff = flux(nx, ny, nz, g64, P, direction)
        return OracleResult(P, classes, q_in, q_out, g_eff, k_eff, 0, 0, 0.0, *counts,
                            "no_spanning_cluster")
    A, b, diag, idx = assemble(nx, ny, nz, g64, classes, wrap)
    if dense:
        x = np.linalg.solve(A.toarray(), b)
        it, restarts = 0, 0
        rel = float(np.sqrt(np.sum((b - A @ x) ** 2)) / np.sqrt(b @ b))
    else:
        x, it, restarts, rel = solve_spd(A, b, diag, tol, max_iter)
    P.ravel()[idx] = x
    q_in, q_out, g_eff, k_eff = flux(nx, ny, nz, g64, P, direction)
    status = "ok" if (dense or rel <= tol) else "max_iters"
    return OracleResult(P, classes, q_in, q_out, g_eff, k_eff, it, restarts, float(rel), *counts,
                        status)


def residual_certificate(nx, ny, nz, gx, gy, gz, P, direction, classes=None, periodic=False):
    """Independent check of ANY pressure field: ||b - A P_S||2 / ||b||2 with the oracle's own
    assembled operator (S8c last pin row: one CPU SpMV, usable at sizes where a second solve is
    too slow).  Returns (rel_residual, max |P - pin| over pinned and Dirichlet nodes)."""
    wrap = wrap_axes(nx, ny, nz, direction, periodic)
    g64 = widen(nx, ny, nz, gx, gy, gz, wrap)
    if classes is None:
        classes = classify(nx, ny, nz, g64, direction, wrap)
    A, b, diag, idx = assemble(nx, ny, nz, g64, classes, wrap)
    P = np.asarray(P, dtype=np.float64).reshape(nz, ny, nx)
    pins = pin_values(classes)
    not_solved = classes != SOLVED
    pin_err = float(np.max(np.abs(P[not_solved] - pins[not_solved]))) if not_solved.any() else 0.0
    if idx.size == 0:
        return 0.0, pin_err
    x = P.ravel()[idx]
    rel = float(np.sqrt(np.sum((b - A @ x) ** 2)) / np.sqrt(b @ b))
    return rel, pin_err
