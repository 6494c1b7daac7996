// pn_onchip.cu -- the fp32 inner CG loop (SURVEY.md 8(a) S4 + S5 + S6) for lattices that fit ONE SM's shared
// memory: the whole loop between two fp64 residual replacements runs in a single kernel launch of one CTA.
//
// SURVEY.md section 7 ("Small problems"): BASELINE.json configs[0] (64 x 64 nodes) is about 100 KB of working set;
// launched kernel by kernel it is bound by launch latency (about 20 us per iteration through a CUDA graph), not by
// memory or arithmetic.  Here the three weight arrays and r, p, q, x_hat live in shared memory in the library's
// padded layout (zero halo plane before and after, so the same flat-index 7-point stencil applies), the two dot
// products of an iteration are block reductions, and alpha, beta and the triggers stay in registers / shared
// memory: an iteration costs three block-wide passes and no launch.  Arithmetic and stopping rules are those of the
// two-kernel scheme (pn_inner.cu): fp32 products, fp64 accumulation, alpha = rr / p.Ap, beta = rr' / rr, the same
// flags (proxy exit, reliable-update threshold, budget, breakdown).  The paper's K2 / K3 with its host
// round trip per dot product is the opposite extreme.
// Not for periodic lateral faces (those lattices fall back to the TMA kernel + k_wrap_fix).
#include "pn_internal.cuh"

namespace {

constexpr int TPB = 1024;
constexpr int PN_ONCHIP_MAX_FLOATS = 7168;   // padded nodes + two halo planes, per array; 7 arrays -> 196 KB

__global__ void __launch_bounds__(TPB, 1) k_cg_onchip(pn_geom g, pn_ptrs P, int max_launch_iters) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    extern __shared__ __align__(16) float sh[];
    __shared__ double red[32];
    __shared__ double bc[2];                       // broadcast of a reduced sum
    const int halo = (int)g.plane, npad = (int)g.npad, len = npad + 2 * halo;
    float* wx = sh + halo;                          // every array: [halo | npad | halo], index 0 = node 0
    float* wy = wx + len;
    float* wz = wy + len;
    float* r = wz + len;
    float* p = r + len;
    float* q = p + len;
    float* xh = q + len;
    const int tid = threadIdx.x;
    const int px = g.px, plane = (int)g.plane;
    // the direction of the last iteration lives in the buffer of parity (iters & 1), as in the two-kernel scheme
    float* __restrict__ pg = (st->iters & 1) ? P.p2 : P.p;
    for (int i = tid - halo; i < npad + halo; i += TPB) {
        const bool in = i >= 0 && i < npad;
        wx[i] = in ? P.w[0][i] : 0.f;
        wy[i] = in ? P.w[1][i] : 0.f;
        wz[i] = in ? P.w[2][i] : 0.f;
        r[i] = in ? P.r[i] : 0.f;
        p[i] = in ? pg[i] : 0.f;
        q[i] = 0.f;
        xh[i] = in ? P.xh[i] : 0.f;
    }
    double rr = st->rr, rr_old = st->rr_old, rr_max = st->rr_max, pq = 0.0;
    const double rr_target = st->rr_target, delta2 = st->delta2;
    float beta = (float)st->beta;
    int it = st->iters, flag = PN_FLAG_RUN;
    const int max_iters = st->max_iters;
    __syncthreads();
    for (int k = 0; k < max_launch_iters && flag == PN_FLAG_RUN; ++k) {
        // pass 1: p = r + beta p
        for (int i = tid; i < npad; i += TPB) p[i] = fmaf(beta, p[i], r[i]);
        __syncthreads();
        // pass 2: q = p - W p ; p.q
        double acc = 0.0;
        for (int i = tid; i < npad; i += TPB) {
            const float pc = p[i];
            float s = wx[i - 1] * p[i - 1];
            s = fmaf(wx[i], p[i + 1], s);
            s = fmaf(wy[i - px], p[i - px], s);
            s = fmaf(wy[i], p[i + px], s);
            s = fmaf(wz[i - plane], p[i - plane], s);
            s = fmaf(wz[i], p[i + plane], s);
            const float qv = pc - s;
            q[i] = qv;
            acc += (double)(pc * qv);
        }
        acc = pn_block_sum(acc, red);
        if (tid == 0) bc[0] = acc;
        __syncthreads();
        pq = bc[0];
        if (rr == 0.0) { flag = PN_FLAG_CONVERGED; break; }
        if (!(pq > 0.0) || isinf(pq)) { flag = PN_FLAG_BREAKDOWN; break; }
        const float alpha = (float)(rr / pq);
        // pass 3: x_hat += alpha p ; r -= alpha q ; r.r
        acc = 0.0;
        for (int i = tid; i < npad; i += TPB) {
            xh[i] = fmaf(alpha, p[i], xh[i]);
            const float rv = fmaf(-alpha, q[i], r[i]);
            r[i] = rv;
            acc += (double)(rv * rv);
        }
        acc = pn_block_sum(acc, red);
        if (tid == 0) bc[1] = acc;
        __syncthreads();
        const double rr_new = bc[1];
        rr_old = rr;
        rr = rr_new;
        ++it;
        if (rr_new > rr_max) rr_max = rr_new;
        if (!(rr_new >= 0.0) || isinf(rr_new)) flag = PN_FLAG_BREAKDOWN;
        else if (rr_new <= rr_target) flag = PN_FLAG_CONVERGED;
        else if (rr_new < delta2 * rr_max) flag = PN_FLAG_UPDATE;
        else if (it >= max_iters) flag = PN_FLAG_BUDGET;
        beta = (float)(rr_new / rr_old);
    }
    __syncthreads();
    // back to HBM for S7 / S3; nothing is owed on x_hat (alpha_x = 0)
    float* __restrict__ pout = (it & 1) ? P.p2 : P.p;
    for (int i = tid; i < npad; i += TPB) {
        P.r[i] = r[i];
        pout[i] = p[i];
        P.xh[i] = xh[i];
    }
    if (tid == 0) {
        st->rr = rr; st->rr_old = rr_old; st->rr_max = rr_max; st->pq = pq;
        st->beta = rr_old > 0.0 ? rr / rr_old : 0.0;
        st->alpha = 0.0; st->alpha_x = 0.0; st->xpend = 0;
        st->iters = it;
        st->flag = flag;
    }
}

}  // namespace

bool pn_onchip_supported(const pn_geom& g) {
    return !(g.wrap[0] | g.wrap[1] | g.wrap[2]) && g.npad + 2 * g.plane <= PN_ONCHIP_MAX_FLOATS;
}

cudaError_t pn_onchip_init_device() {
    return cudaFuncSetAttribute(k_cg_onchip, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                7 * PN_ONCHIP_MAX_FLOATS * (int)sizeof(float));
}

cudaError_t pn_launch_cg_onchip(const pn_geom& g, const pn_ptrs& P, int max_launch_iters, cudaStream_t st) {
    const size_t smem = (size_t)7 * (size_t)(g.npad + 2 * g.plane) * sizeof(float);
    k_cg_onchip<<<1, TPB, smem, st>>>(g, P, max_launch_iters);
    return cudaGetLastError();
}
