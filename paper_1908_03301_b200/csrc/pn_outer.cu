// pn_outer.cu -- the double-precision outer loop, the boundary flux (S8) and
// the export kernels.
//
// "...iterations with the DP are used to converge to the final solution within the allowed
// error of the outer loop".  Here (north_star (c)): fp64 true residual r = b - A x with A applied
// matrix-free from the fp32 conductances widened exactly, the diagonal summed on the fly in fp64;
// the residual is handed to the fp32 inner CG in the symmetric-Jacobi-scaled variables
// (r_hat = s r, s = diag^-1/2), and the fp32 correction comes back as x += s * x_hat.
#include "pn_internal.cuh"

namespace {

constexpr int TPB = 256;

int grid_for(long long work_items, int sms) {
    long long nb = (work_items + TPB - 1) / TPB;
    long long cap = (long long)sms * 8;
    if (cap > PN_MAX_BLOCKS) cap = PN_MAX_BLOCKS;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    return (int)nb;
}

// ---- S3: r = b - A x in fp64 on solved nodes, written as r_hat = (float)(s r) -------------------
// x64 carries the Dirichlet and pin values on the nodes that are not unknowns, so
// (b - A x)_i = sum_j g_ij (x_j - x_i) over all six neighbours.  acc[0] = ||r||^2, acc[1] = ||r_hat||^2
// (of the rounded fp32 values, i.e. exactly what the inner recurrence starts from).
// `bufmode` 1: the single-kernel iteration double-buffers r; the next kernel reads buffer (iters & 1).
// 8 blocks per SM (32 registers, ~60 bytes of spills): the kernel is bound by the latency of its scattered fp64 loads, not by
// registers -- ncu at 512^3 (profiles/r02_ncu.md): 72 registers gave 34 % of the warps and 2192 us (24 % of the DRAM rate),
// 64 registers 1150 us, 32 registers 1020 us; 256^3: 299 -> 138 us
__global__ void __launch_bounds__(TPB, 8) k_residual64(pn_geom g, pn_ptrs P, int bufmode) {
    __shared__ double sm[32];
    __shared__ double tot[2];
    double a0 = 0.0, a1 = 0.0;
    // `bufmode` 3: no stored residual (persistent fused TMA kernel): three direction slots {p, p2, r} rotate with the
    // iteration count; the explicit residual goes where the direction before the last one lay (k_flush is done with it)
    float* __restrict__ rdst = (bufmode == 1 && (P.st->iters & 1)) ? P.r2 : P.r;
    if (bufmode == 3) { const int sl = (P.st->iters + 2) % 3; rdst = sl == 0 ? P.p : (sl == 1 ? P.p2 : P.r); }
    const bool wrap = g.wrap[0] || g.wrap[1] || g.wrap[2];
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const float s = P.s[n];
        float rh = 0.f;
        if (s != 0.f) {
            const double xc = P.x64[n];
            double r = (double)P.gs[0][n] * (P.x64[n + 1] - xc);
            r += (double)P.gs[0][n - 1] * (P.x64[n - 1] - xc);
            r += (double)P.gs[1][n] * (P.x64[n + g.px] - xc);
            r += (double)P.gs[1][n - g.px] * (P.x64[n - g.px] - xc);
            r += (double)P.gs[2][n] * (P.x64[n + g.plane] - xc);
            r += (double)P.gs[2][n - g.plane] * (P.x64[n - g.plane] - xc);
            if (wrap) {   // periodic lateral faces: the wrap bonds of a node on such a face
                const int ci = (int)(n % g.px), cj = (int)((n / g.px) % g.ny), ck = (int)(n / g.plane);
                for (int b = 0; b < 3; ++b) {
                    if (!g.wrap[b]) continue;
                    const int cb = b == 0 ? ci : (b == 1 ? cj : ck), db = b == 0 ? g.nx : (b == 1 ? g.ny : g.nz);
                    if (cb != 0 && cb != db - 1) continue;
                    const double gw = (double)P.gsw[b][pn_face_index(g, b, ci, cj, ck)];
                    const long long span = pn_wrap_span(g, b);
                    if (cb == 0) r += gw * (P.x64[n + span] - xc);
                    if (cb == db - 1) r += gw * (P.x64[n - span] - xc);
                }
            }
            rh = (float)((double)s * r);
            a0 += r * r;
            a1 += (double)rh * (double)rh;
        }
        rdst[n] = rh;
    }
    a0 = pn_block_sum(a0, sm);
    a1 = pn_block_sum(a1, sm);
    const double v[2] = {a0, a1};
    if (pn_grid_sum<2>(v, P.slots, &P.st->ticket, sm, tot)) {
        if (threadIdx.x == 0) { P.st->acc[0] = tot[0]; P.st->acc[1] = tot[1]; }
    }
}

// ---- S7: x64 += s * (x_hat + alpha_x p)  (the pending deferred update included); x_hat = 0 ------
// Single-kernel scheme with a skipped x_hat update pending (state.xpend): the direction before the last one is
// recovered as p_{T-1} = (p_T - r_T) / beta_T from the last kernel's p and r, exactly as the next kernel would have.
__global__ void k_flush(pn_geom g, pn_ptrs P, int bufmode) {
    const double ax = P.st->alpha_x;
    const bool odd = bufmode != 2 && (P.st->iters & 1);     // in-place scheme: one buffer each
    const float* __restrict__ p = odd ? P.p2 : P.p;   // the direction of the last iteration
    const float* __restrict__ r = odd ? P.r2 : P.r;   // single-kernel schemes: the residual it was built from
    const bool pend = P.st->xpend != 0;
    double c2 = pend ? P.st->alpha2 / P.st->beta_prev : 0.0;
    double c1 = 1.0;                                        // dx = x_hat + ax p + c2 (c1 p - r)
    if (bufmode == 3) {   // direction slots {p, p2, r}: p_T in slot T % 3, p_{T-1} -- what a skipped update is owed on -- in (T + 2) % 3
        const int s1 = P.st->iters % 3, s2 = (P.st->iters + 2) % 3;
        p = s1 == 0 ? P.p : (s1 == 1 ? P.p2 : P.r);
        r = s2 == 0 ? P.p : (s2 == 1 ? P.p2 : P.r);
        c2 = pend ? -P.st->alpha2 : 0.0;
        c1 = 0.0;
    }
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const float s = P.s[n];
        if (s != 0.f) {
            double dx = (double)P.xh[n] + ax * (double)p[n];
            if (pend) dx += c2 * (c1 * (double)p[n] - (double)r[n]);
            P.x64[n] += (double)s * dx;
        }
        P.xh[n] = 0.f;
    }
}

__global__ void k_set_state(pn_state* st, double rr, double beta, double rr_max, double rr_target, double delta2,
                            int max_iters, int reset_iters, double xskip_min) {
    st->alpha2 = 0.0;
    st->beta_prev = 0.0;
    st->xskip_min = xskip_min;
    st->xpend = 0;
    st->beta_last = 0.0;
    st->rexp = 1;               // the residual k_residual64 has just written is explicit (not recoverable from directions)
    st->rr = rr;
    st->rr_old = rr;
    st->beta = beta;
    st->alpha = 0.0;
    st->alpha_x = 0.0;
    st->pq = 0.0;
    st->rr_max = rr_max;
    st->rr_target = rr_target;
    st->delta2 = delta2;
    st->max_iters = max_iters;
    if (reset_iters) { st->iters = 0; st->n_xskip = 0; }
    st->flag = PN_FLAG_RUN;
    st->ticket = 0u;
}

// ---- S8: boundary fluxes, eq.(4) P:61.  acc[0] = Q_in, acc[1] = Q_out ---------------------------
// One thread per node of a plane normal to the solve axis; the solve copy of g has every bond of a
// pinned node zeroed, so summing over ALL boundary bonds is exact (SURVEY.md 8(a) note on S1/S8).
__global__ void k_flux(pn_geom g, pn_ptrs P) {
    __shared__ double sm[32];
    __shared__ double tot[2];
    const int d0 = g.dir == 0 ? g.ny : g.nx;                       // fast in-plane extent
    const int d1 = g.dir == 2 ? g.ny : g.nz;                       // slow in-plane extent
    const long long s0 = g.dir == 0 ? g.px : 1;                    // their element strides
    const long long s1 = g.dir == 2 ? g.px : g.plane;
    const long long m = (long long)d0 * d1;
    double qi = 0.0, qo = 0.0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < m; t += (long long)gridDim.x * blockDim.x) {
        const long long base = (t % d0) * s0 + (t / d0) * s1;
        const long long n_in = base;                                // node on the inlet plane
        const long long n_out = base + (long long)(g.n_a - 2) * g.stride_a;  // node next to the outlet plane
        qi += (double)P.gs[g.dir][n_in] * (P.x64[n_in] - P.x64[n_in + g.stride_a]);
        qo += (double)P.gs[g.dir][n_out] * (P.x64[n_out] - P.x64[n_out + g.stride_a]);
    }
    qi = pn_block_sum(qi, sm);
    qo = pn_block_sum(qo, sm);
    const double v[2] = {qi, qo};
    if (pn_grid_sum<2>(v, P.slots, &P.st->ticket, sm, tot)) {
        if (threadIdx.x == 0) { P.st->acc[0] = tot[0]; P.st->acc[1] = tot[1]; }
    }
}

// ---- dissipation estimate of the effective conductance:  G_E = sum over all bonds g (dP_bond)^2 / dP^2 ----------
// (dP = 1; energy identity Q dP = sum g dP_bond^2, P:59-61 with P:53).  Its error is QUADRATIC in the error of the
// pressures, where the boundary fluxes of S8 are linear (SURVEY.md 8(c) consequence (iv)): at the 1e-10 residual of
// the timing runs it is good to ~1e-12, the boundary-flux G_eff to a few 1e-9.  acc[3] = G_E.
__global__ void k_dissipation(pn_geom g, pn_ptrs P) {
    __shared__ double sm[32];
    __shared__ double tot[1];
    double e = 0.0;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const double xc = P.x64[n];
        const float g0 = P.gs[0][n], g1 = P.gs[1][n], g2 = P.gs[2][n];
        if (g0 != 0.f) { const double d = P.x64[n + 1] - xc; e += (double)g0 * d * d; }
        if (g1 != 0.f) { const double d = P.x64[n + g.px] - xc; e += (double)g1 * d * d; }
        if (g2 != 0.f) { const double d = P.x64[n + g.plane] - xc; e += (double)g2 * d * d; }
    }
    for (int b = 0; b < 3; ++b) {   // wrap bonds of periodic lateral faces
        if (!g.wrap[b]) continue;
        const long long nf = pn_face_count(g, b), span = pn_wrap_span(g, b);
        for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
            const float gw = P.gsw[b][f];
            if (gw == 0.f) continue;
            const long long lo = b == 0 ? (f % g.ny) * (long long)g.px + (f / g.ny) * g.plane
                                        : (b == 1 ? (f % g.px) + (f / g.px) * g.plane : f);
            const double d = P.x64[lo + span] - P.x64[lo];
            e += (double)gw * d * d;
        }
    }
    e = pn_block_sum(e, sm);
    const double v[1] = {e};
    if (pn_grid_sum<1>(v, P.slots, &P.st->ticket, sm, tot)) {
        if (threadIdx.x == 0) P.st->acc[3] = tot[0];
    }
}

// ---- padded -> user layout ----------------------------------------------------------------------
__global__ void k_export_x(pn_geom g, const double* __restrict__ x64, double* __restrict__ out) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.n; n += (long long)gridDim.x * blockDim.x) {
        const long long row = n / g.nx;
        out[n] = x64[row * g.px + (n - row * g.nx)];
    }
}
__global__ void k_export_cls(pn_geom g, const signed char* __restrict__ cls, signed char* __restrict__ out) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.n; n += (long long)gridDim.x * blockDim.x) {
        const long long row = n / g.nx;
        const signed char c = cls[row * g.px + (n - row * g.nx)];
        out[n] = c >= PN_CLASS_PEELED ? (signed char)PN_CLASS_SOLVED : c;   // peeled dangling ends are solved nodes
    }
}

}  // namespace

cudaError_t pn_launch_residual64(const pn_geom& g, const pn_ptrs& P, int bufmode, cudaStream_t st, int* launches) {
    k_residual64<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P, bufmode);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_flush(const pn_geom& g, const pn_ptrs& P, int bufmode, cudaStream_t st, int* launches) {
    k_flush<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P, bufmode);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_set_state(const pn_ptrs& P, double rr, double beta, double rr_max, double rr_target,
                                double delta2, int max_iters, int reset_iters, double xskip_min, cudaStream_t st,
                                int* launches) {
    k_set_state<<<1, 1, 0, st>>>(P.st, rr, beta, rr_max, rr_target, delta2, max_iters, reset_iters, xskip_min);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_flux(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    const long long m = g.n / g.n_a;
    k_flux<<<grid_for(m, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_export_x(const pn_geom& g, const pn_ptrs& P, double* out, cudaStream_t st, int* launches) {
    k_export_x<<<grid_for(g.n, g.sms), TPB, 0, st>>>(g, P.x64, out);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_export_cls(const pn_geom& g, const pn_ptrs& P, signed char* out, int, cudaStream_t st,
                                 int* launches) {
    k_export_cls<<<grid_for(g.n, g.sms), TPB, 0, st>>>(g, P.cls, out);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_dissipation(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_dissipation<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
