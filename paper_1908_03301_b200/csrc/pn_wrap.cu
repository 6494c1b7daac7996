// pn_wrap.cu -- periodic lateral faces in the inner iteration.
//
// Paper: "a fixed pressure gradient is applied to the network in one direction ... periodic boundary
// conditions in the second direction".  BASELINE.json's north_star fixes no-flux side faces for the headline
// path, so the lattice-shaped arrays and the three S4 kernels know nothing about wrap-around: their flat-index
// stencil sees a zero bond at every face.  With PN_OPT_LATERAL = 1 the operator is
//        A_hat = I - W - W_wrap,
// W_wrap holding the (scaled) bonds that join the last and the first node along every lateral axis.  Those
// bonds touch only the face nodes, O(N^(2/3)) of them, so their part of q = A_hat p is added by this small
// kernel after the main one:
//        q_n -= sum over the wrap bonds at n of  ww * p_partner          (face nodes only)
// and the dot products the main kernel accumulated (stored unfinished in state.part) are corrected by
//        p.q += sum p_n dq_n     q.q += sum (2 q_n dq_n + dq_n^2)     r.q += sum r_n dq_n
// before the last block of THIS kernel computes alpha (and the predicted beta of the single-kernel scheme).
// One thread per face node; a node lying on several faces (edges, corners) is handled once, by the first
// wrapping axis it belongs to, and gathers all its wrap bonds in a fixed order: bit-reproducible.
#include "pn_internal.cuh"

namespace {

constexpr int TPB = 256;

// fused != 0: single-kernel scheme (r, q double-buffered, four sums); 0: two-kernel schemes (q in P.q, p.q only)
__global__ void __launch_bounds__(TPB) k_wrap_fix(pn_geom g, pn_ptrs P, int fused) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    __shared__ double sm[32];
    __shared__ double tot[3];
    const int par = st->iters & 1;                       // same parity the main kernel of this iteration used
    const float* __restrict__ p = par ? P.p : P.p2;      // p_t, written by the main kernel
    float* __restrict__ q = fused ? (par ? P.q : P.q2) : P.q;
    // single-kernel scheme: no stored residual; directions in three rotating slots {p, p2, r} (pn_fused_tma.cu):
    // p_t in slot (iters + 1) % 3, p_{t-1} in slot iters % 3, and r_t = p_t - beta_t p_{t-1}
    const float* __restrict__ pm = nullptr;
    const float beta_t = (float)st->beta;
    if (fused) {
        const int s0 = (st->iters + 1) % 3, s1 = st->iters % 3;
        p = s0 == 0 ? P.p : (s0 == 1 ? P.p2 : P.r);
        pm = s1 == 0 ? P.p : (s1 == 1 ? P.p2 : P.r);
    }
    const int dims[3] = {g.nx, g.ny, g.nz};
    double d_pq = 0.0, d_qq = 0.0, d_rq = 0.0;
    for (int b = 0; b < 3; ++b) {
        if (!g.wrap[b]) continue;
        const long long nf = pn_face_count(g, b), span = pn_wrap_span(g, b);
        for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < 2 * nf; t += (long long)gridDim.x * blockDim.x) {
            const int hi = t >= nf;
            const long long f = hi ? t - nf : t;
            int c[3];
            if (b == 0) { c[0] = 0; c[1] = (int)(f % g.ny); c[2] = (int)(f / g.ny); }
            else if (b == 1) { c[0] = (int)(f % g.px); c[1] = 0; c[2] = (int)(f / g.px); }
            else { c[0] = (int)(f % g.px); c[1] = (int)(f / g.px); c[2] = 0; }
            if (hi) c[b] = dims[b] - 1;
            if (c[0] >= g.nx) continue;                                    // pad column
            bool primary = true;
            for (int e = 0; e < b; ++e)
                if (g.wrap[e] && (c[e] == 0 || c[e] == dims[e] - 1)) primary = false;
            if (!primary) continue;
            const long long n = c[0] + (long long)g.px * c[1] + g.plane * c[2];
            float dq = 0.f;
            for (int e = b; e < 3; ++e) {
                if (!g.wrap[e] || !(c[e] == 0 || c[e] == dims[e] - 1)) continue;
                const float w = P.ww[e][pn_face_index(g, e, c[0], c[1], c[2])];
                const long long sp = pn_wrap_span(g, e);
                dq -= w * p[c[e] == 0 ? n + sp : n - sp];
            }
            (void)span;
            const float qo = q[n];
            q[n] = qo + dq;
            d_pq += (double)(p[n] * dq);
            if (fused) {
                d_qq += (double)(2.f * qo * dq + dq * dq);
                d_rq += (double)(fmaf(-beta_t, pm[n], p[n]) * dq);
            }
        }
    }
    d_pq = pn_block_sum(d_pq, sm);
    d_qq = pn_block_sum(d_qq, sm);
    d_rq = pn_block_sum(d_rq, sm);
    const double v3[3] = {d_pq, d_qq, d_rq};
    if (pn_grid_sum<3>(v3, P.slots, &st->ticket, sm, tot)) {
        if (threadIdx.x == 0) {
            if (fused) pn_finish_F(st, st->part[0], st->part[1] + tot[0], st->part[2] + tot[2], st->part[3] + tot[1]);
            else pn_finish_A(st, st->part[0] + tot[0]);
        }
    }
}

}  // namespace

cudaError_t pn_launch_wrap_fix(const pn_geom& g, const pn_ptrs& P, int fused, cudaStream_t st) {
    long long items = 0;
    for (int b = 0; b < 3; ++b)
        if (g.wrap[b] && 2 * pn_face_count(g, b) > items) items = 2 * pn_face_count(g, b);
    long long nb = (items + TPB - 1) / TPB;
    const long long cap = (long long)g.sms * 4;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    k_wrap_fix<<<(int)nb, TPB, 0, st>>>(g, P, fused);
    return cudaGetLastError();
}
