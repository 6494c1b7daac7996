/* CPU ORACLE in plain C (test infrastructure, NOT the product).
 *
 * Same steps as oracle/pn_oracle.py, written out in C so that 256^3 and 512^3 networks finish and
 * so that bench.py can time "the oracle as it stands" on the host cores.  Shares no code with the
 * CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.  Pinned by tests/test_oracle_pins.py::test_c_oracle_* (same closed forms and
 * dense checks as the Python oracle, plus agreement with it on seeded inputs).
 *
 * Citations (/root/reference/PAPER.md = P:<line>; SURVEY.md 8(c) = S8c):
 *   node balance  sum_j g_ij (P_i - P_j) = 0,  q_ij = g_ij dP_ij            P:53, eq.(3)
 *   fixed pressure drop along one axis; side faces no-flux                  P:57, S8c readings 1-2
 *   cluster classes S / inlet-only / outlet-only / floating, serial BFS     S8c step 3
 *   assembled CSR Laplacian over the solved nodes                           S8c step 4
 *   textbook Jacobi-PCG, "Templates" form                                   P:63, ref[57] P:218
 *   flux and Darcy permeability                                             eq.(4), S8c step 7
 *
 * Layout: node n = i + nx*(j + ny*k); gx[n] = bond n -- n+1, gy[n] = bond n -- n+nx,
 * gz[n] = bond n -- n+nx*ny; entries whose forward neighbour is off-lattice are not bonds.
 * All arithmetic fp64; the fp32 inputs are widened exactly (S8c reading 14).
 * OpenMP only on SpMV / axpy / dot.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { C_INLET = 0, C_OUTLET = 1, C_SOLVED = 2, C_INLET_ONLY = 3, C_OUTLET_ONLY = 4, C_FLOATING = 5 };

typedef struct {
    long long n_solved, n_inlet_only, n_outlet_only, n_floating, nnz;
    int iterations, restarts, status; /* status: 0 ok, 1 no spanning cluster, 2 max iterations */
    int threads;
    double rel_residual, q_in, q_out, g_eff, k_eff;
    double t_label, t_assemble, t_pcg;
    int it_decade[16]; /* record only: first iteration at which the recursive ||r||2/||b||2 <= 1e-k (k = index), -1 if never */
} pno_info;

static double now(void) {
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return ts.tv_sec + 1e-9 * ts.tv_nsec;
}

typedef struct {
    int nx, ny, nz, dir;
    long long N, stride[3];
    int dims[3];
    int wrap[3]; /* lateral axis wraps around (periodic side faces); never the solve axis */
    const float *g[3];
} lattice;

static inline int coord(const lattice *L, long long n, int a) {
    if (a == 0) return (int)(n % L->nx);
    if (a == 1) return (int)((n / L->nx) % L->ny);
    return (int)(n / ((long long)L->nx * L->ny));
}

/* conductance of the bond between n and its forward neighbour along a (0 if not a bond) */
static inline double bond(const lattice *L, long long n, int a) {
    if (!L->g[a]) return 0.0;
    if (coord(L, n, a) + 1 >= L->dims[a]) return 0.0;
    return (double)L->g[a][n];
}

/* Neighbour of n along axis a (side 0: forward, 1: backward) and the conductance of the bond between them.
 * Returns 0 when there is none: a lattice face that does not wrap.  On a wrapping axis the forward entry of
 * the LAST node is the bond back to the first node (forward-bond convention carried around the ring). */
static inline int nbr(const lattice *L, long long n, int a, int side, long long *m, double *g) {
    if (!L->g[a]) return 0;
    const int c = coord(L, n, a), d = L->dims[a];
    if (side == 0) {
        if (c + 1 < d) *m = n + L->stride[a];
        else if (L->wrap[a]) *m = n - (long long)(d - 1) * L->stride[a];
        else return 0;
        *g = (double)L->g[a][n];
    } else {
        if (c > 0) *m = n - L->stride[a];
        else if (L->wrap[a]) *m = n + (long long)(d - 1) * L->stride[a];
        else return 0;
        *g = (double)L->g[a][*m];
    }
    return 1;
}

/* ---- S8c steps 2-3: serial breadth-first labelling ------------------------------------------- */
static int classify(const lattice *L, signed char *cls, pno_info *info) {
    const long long N = L->N;
    const int n_a = L->dims[L->dir];
    long long *queue = (long long *)malloc(sizeof(long long) * (size_t)N);
    if (!queue) return -1;
    for (long long n = 0; n < N; ++n) {
        int c = coord(L, n, L->dir);
        cls[n] = c == 0 ? C_INLET : (c == n_a - 1 ? C_OUTLET : -1);
    }
    info->n_solved = info->n_inlet_only = info->n_outlet_only = info->n_floating = 0;
    for (long long seed = 0; seed < N; ++seed) {
        if (cls[seed] != -1) continue;
        long long head = 0, tail = 0;
        int t_in = 0, t_out = 0;
        queue[tail++] = seed;
        cls[seed] = C_SOLVED; /* provisional = visited */
        while (head < tail) {
            long long n = queue[head++];
            for (int a = 0; a < 3; ++a) {
                for (int side = 0; side < 2; ++side) {
                    long long m;
                    double g;
                    if (!nbr(L, n, a, side, &m, &g)) continue;
                    if (!(g > 0.0)) continue;
                    if (cls[m] == C_INLET) t_in = 1;
                    else if (cls[m] == C_OUTLET) t_out = 1;
                    else if (cls[m] == -1) { cls[m] = C_SOLVED; queue[tail++] = m; }
                }
            }
        }
        signed char c = (t_in && t_out) ? C_SOLVED : t_in ? C_INLET_ONLY : t_out ? C_OUTLET_ONLY : C_FLOATING;
        if (c != C_SOLVED) for (long long q = 0; q < tail; ++q) cls[queue[q]] = c;
        if (c == C_SOLVED) info->n_solved += tail;
        else if (c == C_INLET_ONLY) info->n_inlet_only += tail;
        else if (c == C_OUTLET_ONLY) info->n_outlet_only += tail;
        else info->n_floating += tail;
    }
    free(queue);
    return 0;
}

/* ---- S8c step 4: CSR over solved nodes -------------------------------------------------------- */
typedef struct {
    long long m, nnz;
    long long *rowptr;
    int *col;
    double *val, *diag, *b;
    long long *idx; /* unknown -> lattice node */
} csr;

static void csr_free(csr *A) {
    free(A->rowptr); free(A->col); free(A->val); free(A->diag); free(A->b); free(A->idx);
    memset(A, 0, sizeof(*A));
}

static int assemble(const lattice *L, const signed char *cls, csr *A) {
    const long long N = L->N;
    long long m = 0;
    int *unk = (int *)malloc(sizeof(int) * (size_t)N);
    if (!unk) return -1;
    for (long long n = 0; n < N; ++n) unk[n] = cls[n] == C_SOLVED ? (int)m++ : -1;
    A->m = m;
    A->rowptr = (long long *)calloc((size_t)m + 1, sizeof(long long));
    A->diag = (double *)calloc((size_t)m, sizeof(double));
    A->b = (double *)calloc((size_t)m, sizeof(double));
    A->idx = (long long *)malloc(sizeof(long long) * (size_t)(m ? m : 1));
    if (!A->rowptr || !A->diag || !A->b || !A->idx) { free(unk); return -1; }
    /* pass 1: count entries per row (diagonal + solved neighbours) */
    for (long long n = 0; n < N; ++n) {
        if (unk[n] < 0) continue;
        long long cnt = 1;
        A->idx[unk[n]] = n;
        for (int a = 0; a < 3; ++a)
            for (int side = 0; side < 2; ++side) {
                long long mn;
                double g;
                if (nbr(L, n, a, side, &mn, &g) && g > 0.0 && cls[mn] == C_SOLVED) ++cnt;
            }
        A->rowptr[unk[n] + 1] = cnt;
    }
    for (long long u = 0; u < m; ++u) A->rowptr[u + 1] += A->rowptr[u];
    A->nnz = A->rowptr[m];
    A->col = (int *)malloc(sizeof(int) * (size_t)(A->nnz ? A->nnz : 1));
    A->val = (double *)malloc(sizeof(double) * (size_t)(A->nnz ? A->nnz : 1));
    if (!A->col || !A->val) { free(unk); return -1; }
    /* pass 2: fill (backward z, y, x, diagonal, forward x, y, z: columns ascending unless an axis wraps) */
    for (long long n = 0; n < N; ++n) {
        int u = unk[n];
        if (u < 0) continue;
        long long p = A->rowptr[u];
        double d = 0.0, bi = 0.0;
        long long dpos = -1;
        for (int pass = 0; pass < 2; ++pass) {
            for (int aa = 0; aa < 3; ++aa) {
                int a = pass == 0 ? 2 - aa : aa; /* backward: z,y,x ; forward: x,y,z */
                long long mnode;
                double g;
                if (!nbr(L, n, a, pass == 0 ? 1 : 0, &mnode, &g)) continue;
                if (!(g > 0.0)) continue;
                d += g;
                if (cls[mnode] == C_INLET) bi += g;
                if (cls[mnode] == C_SOLVED) { A->col[p] = unk[mnode]; A->val[p] = -g; ++p; }
            }
            if (pass == 0) { dpos = p; A->col[p] = u; ++p; }
        }
        A->val[dpos] = d;
        A->diag[u] = d;
        A->b[u] = bi;
    }
    free(unk);
    return 0;
}

/* ---- BLAS-1 and SpMV (the only OpenMP-parallel parts) ------------------------------------------ */
static void spmv(const csr *A, const double *x, double *y) {
    const long long m = A->m;
#pragma omp parallel for schedule(static)
    for (long long u = 0; u < m; ++u) {
        double s = 0.0;
        for (long long p = A->rowptr[u]; p < A->rowptr[u + 1]; ++p) s += A->val[p] * x[A->col[p]];
        y[u] = s;
    }
}
static double dot(long long m, const double *a, const double *b) {
    double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long long u = 0; u < m; ++u) s += a[u] * b[u];
    return s;
}
static void axpy(long long m, double alpha, const double *x, double *y) {
#pragma omp parallel for schedule(static)
    for (long long u = 0; u < m; ++u) y[u] += alpha * x[u];
}

/* ---- S8c step 5: textbook Jacobi-PCG ---------------------------------------------------------- */
/* x: start and result.  Stops when the recursive residual 2-norm <= target.  Returns iterations. */
static int pcg(const csr *A, double *x, double target, int max_iter, double *r, double *z, double *p, double *q,
               double nb, int it_base, int *it_decade) {
    const long long m = A->m;
    int it = 0;
    spmv(A, x, q);
#pragma omp parallel for schedule(static)
    for (long long u = 0; u < m; ++u) r[u] = A->b[u] - q[u];
    if (sqrt(dot(m, r, r)) <= target) return 0;
#pragma omp parallel for schedule(static)
    for (long long u = 0; u < m; ++u) { z[u] = r[u] / A->diag[u]; p[u] = z[u]; }
    double rho = dot(m, r, z);
    while (it < max_iter) {
        spmv(A, p, q);
        double alpha = rho / dot(m, p, q);
        axpy(m, alpha, p, x);
        axpy(m, -alpha, q, r);
        ++it;
        const double rn = sqrt(dot(m, r, r));
        for (int k = 0; k < 16; ++k) /* record only (tests/golden/make_digest.py): no effect on the iteration */
            if (it_decade[k] < 0 && rn <= pow(10.0, -k) * nb) it_decade[k] = it_base + it;
        if (rn <= target) break;
#pragma omp parallel for schedule(static)
        for (long long u = 0; u < m; ++u) z[u] = r[u] / A->diag[u];
        double rho_new = dot(m, r, z);
        double beta = rho_new / rho;
#pragma omp parallel for schedule(static)
        for (long long u = 0; u < m; ++u) p[u] = z[u] + beta * p[u];
        rho = rho_new;
    }
    return it;
}

static double true_rel_residual(const csr *A, const double *x, double *tmp, double nb) {
    spmv(A, x, tmp);
    double s = 0.0;
    const long long m = A->m;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long long u = 0; u < m; ++u) { double e = A->b[u] - tmp[u]; s += e * e; }
    return sqrt(s) / nb;
}

/* ---- S8c step 7: flux -------------------------------------------------------------------------- */
static void flux(const lattice *L, const double *P, pno_info *info) {
    const int a = L->dir, n_a = L->dims[a];
    double qi = 0.0, qo = 0.0;
    for (long long n = 0; n < L->N; ++n) {
        int c = coord(L, n, a);
        if (c == 0) qi += bond(L, n, a) * (P[n] - P[n + L->stride[a]]);
        if (c == n_a - 2) qo += bond(L, n, a) * (P[n] - P[n + L->stride[a]]);
    }
    info->q_in = qi;
    info->q_out = qo;
    info->g_eff = 0.5 * (qi + qo);
    info->k_eff = info->g_eff * (n_a - 1) / (double)(L->N / n_a);
}

static int setup(lattice *L, int nx, int ny, int nz, const float *gx, const float *gy, const float *gz, int dir,
                 int periodic) {
    if (nx < 1 || ny < 1 || nz < 1 || dir < 0 || dir > 2 || !gx || !gy || (nz > 1 && !gz)) return -1;
    L->nx = nx; L->ny = ny; L->nz = nz; L->dir = dir;
    L->dims[0] = nx; L->dims[1] = ny; L->dims[2] = nz;
    L->N = (long long)nx * ny * nz;
    L->stride[0] = 1; L->stride[1] = nx; L->stride[2] = (long long)nx * ny;
    L->g[0] = gx; L->g[1] = gy; L->g[2] = nz > 1 ? gz : NULL;
    if (L->dims[dir] < 3) return -1;
    for (int a = 0; a < 3; ++a) L->wrap[a] = periodic && a != dir && L->dims[a] >= 2;
    for (int a = 0; a < 3; ++a) {
        if (!L->g[a]) continue;
        for (long long n = 0; n < L->N; ++n) {
            if (coord(L, n, a) + 1 >= L->dims[a] && !L->wrap[a]) continue;
            float g = L->g[a][n];
            if (!(g >= 0.0f) || isinf(g)) return -2;
        }
    }
    return 0;
}

/* Whole path.  P_out: N doubles.  classes_out: N bytes or NULL.  max_threads <= 0: all cores.
 * P_start: NULL = the textbook zero start (S8c step 5); else N doubles whose values on the solved nodes are the
 * starting iterate (used by tests/golden/make_digest.py to carry a converged tol-1e-12 solution on to the fp64 floor
 * without repeating its iterations; same loop, same restarts, only x0 differs).
 * Returns 0 ok / 1 no spanning cluster / 2 max iterations / <0 error. */
int pno_solve_from(int nx, int ny, int nz, const float *gx, const float *gy, const float *gz, int direction,
                   int periodic, double tol, int max_iter, int max_threads, const double *P_start, double *P_out,
                   signed char *classes_out, pno_info *info) {
    lattice L;
    pno_info local;
    if (!info) info = &local;
    memset(info, 0, sizeof(*info));
    for (int k = 0; k < 16; ++k) info->it_decade[k] = -1;
    int rc = setup(&L, nx, ny, nz, gx, gy, gz, direction, periodic);
    if (rc) return rc;
#ifdef _OPENMP
    if (max_threads > 0) omp_set_num_threads(max_threads);
    info->threads = omp_get_max_threads();
#else
    info->threads = 1;
#endif
    signed char *cls = classes_out ? classes_out : (signed char *)malloc((size_t)L.N);
    if (!cls) return -3;
    double t0 = now();
    if (classify(&L, cls, info)) return -3;
    info->t_label = now() - t0;
    for (long long n = 0; n < L.N; ++n) P_out[n] = (cls[n] == C_INLET || cls[n] == C_INLET_ONLY) ? 1.0 : 0.0;
    if (info->n_solved == 0) {
        flux(&L, P_out, info);
        info->status = 1;
        if (!classes_out) free(cls);
        return 1;
    }
    csr A;
    memset(&A, 0, sizeof(A));
    t0 = now();
    if (assemble(&L, cls, &A)) { csr_free(&A); return -3; }
    info->t_assemble = now() - t0;
    info->nnz = A.nnz;
    const long long m = A.m;
    double *x = (double *)calloc((size_t)m, sizeof(double));
    double *w = (double *)malloc(sizeof(double) * (size_t)m * 4);
    double *best = (double *)malloc(sizeof(double) * (size_t)m);
    if (!x || !w || !best) return -3;
    if (P_start) for (long long u = 0; u < m; ++u) x[u] = P_start[A.idx[u]];
    double nb = sqrt(dot(m, A.b, A.b));
    t0 = now();
    double best_rel = INFINITY, rel = 0.0;
    int total = 0, restarts = 0;
    if (nb > 0.0) {
        for (restarts = 0; restarts < 20; ++restarts) {
            int it = pcg(&A, x, (restarts ? 0.7 : 1.0) * tol * nb, max_iter - total, w, w + m, w + 2 * m, w + 3 * m, nb,
                         total, info->it_decade);
            total += it;
            rel = true_rel_residual(&A, x, w, nb);
            if (rel < best_rel) { best_rel = rel; memcpy(best, x, sizeof(double) * (size_t)m); }
            if (rel <= tol || total >= max_iter || it == 0) break;
        }
    } else best_rel = 0.0, memcpy(best, x, sizeof(double) * (size_t)m);
    info->t_pcg = now() - t0;
    info->iterations = total;
    info->restarts = restarts;
    info->rel_residual = best_rel;
    for (long long u = 0; u < m; ++u) P_out[A.idx[u]] = best[u];
    flux(&L, P_out, info);
    info->status = best_rel <= tol ? 0 : 2;
    free(x); free(w); free(best);
    csr_free(&A);
    if (!classes_out) free(cls);
    return info->status;
}

int pno_solve(int nx, int ny, int nz, const float *gx, const float *gy, const float *gz, int direction, int periodic,
              double tol, int max_iter, int max_threads, double *P_out, signed char *classes_out, pno_info *info) {
    return pno_solve_from(nx, ny, nz, gx, gy, gz, direction, periodic, tol, max_iter, max_threads, NULL, P_out,
                          classes_out, info);
}

/* Independent residual certificate of ANY pressure field (S8c last pin row): ||b - A P_S||2/||b||2 with
 * this file's assembled operator, and max |P - pin| over Dirichlet and pinned nodes.  classes_out (N bytes,
 * may be NULL) receives the node classes of the serial labelling. */
int pno_certificate(int nx, int ny, int nz, const float *gx, const float *gy, const float *gz, int direction,
                    int periodic, const double *P, double *rel_residual, double *pin_err, signed char *classes_out) {
    lattice L;
    pno_info info;
    memset(&info, 0, sizeof(info));
    int rc = setup(&L, nx, ny, nz, gx, gy, gz, direction, periodic);
    if (rc) return rc;
    signed char *cls = classes_out ? classes_out : (signed char *)malloc((size_t)L.N);
    if (!cls || classify(&L, cls, &info)) return -3;
    double pe = 0.0;
    for (long long n = 0; n < L.N; ++n) {
        if (cls[n] == C_SOLVED) continue;
        double pin = (cls[n] == C_INLET || cls[n] == C_INLET_ONLY) ? 1.0 : 0.0;
        double e = fabs(P[n] - pin);
        if (e > pe || e != e) pe = e;
    }
    *pin_err = pe;
    *rel_residual = 0.0;
    if (info.n_solved) {
        csr A;
        memset(&A, 0, sizeof(A));
        if (assemble(&L, cls, &A)) return -3;
        double *x = (double *)malloc(sizeof(double) * (size_t)A.m * 2);
        if (!x) return -3;
        for (long long u = 0; u < A.m; ++u) x[u] = P[A.idx[u]];
        *rel_residual = true_rel_residual(&A, x, x + A.m, sqrt(dot(A.m, A.b, A.b)));
        free(x);
        csr_free(&A);
    }
    if (!classes_out) free(cls);
    return 0;
}
