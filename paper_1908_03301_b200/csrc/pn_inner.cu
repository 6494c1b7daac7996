// pn_inner.cu -- the fp32 inner conjugate-gradient iteration: two fused
// kernels per iteration, all scalars device-resident.
//
// Paper: K2 "sparse matrix-vector multiplication ... each Z_i multiplied by its P_i, block reduction"
// (P:89), K3 "a thread is assigned for the calculation of each element of U, R and Z ... partial
// result of dot products", "Merging the calculations of the vectors' entries into a single
// kernel ... decreasing the number of times that the global memory must be accessed", final
// sums of the 2^6 block partials on the CPU.  Here: matrix-free 7-point operator, the final
// sums stay on the device (last-block-done), and the Jacobi preconditioner (north_star (b)) is
// applied as the symmetric scaling A_hat = D^-1/2 A D^-1/2 folded into one fp32 weight per bond,
//     w_ij = g_ij / sqrt(d_i d_j),   A_hat = I - W,
// so that Jacobi-PCG on A is plain CG on A_hat (same iterates in exact arithmetic) and the unit
// diagonal costs no memory traffic.  Nodes that are not unknowns (Dirichlet planes, pinned clusters,
// pad columns) have all their weights zero and r = p = 0, so they need no mask.
//
// Iteration t (state.iters == t), p double-buffered because kernel A reads neighbours' old p:
//   kernel A:  p_new = r + beta p_old          (at the node AND its six neighbours, recomputed)
//              x_hat += alpha_x p_old          (the solution update of iteration t-1, deferred)
//              q = p_new - W p_new ;  pq = p_new . q     -> alpha = rr / pq       (last block)
//   kernel B:  r -= alpha q ;  rr' = r . r     -> beta = rr'/rr, alpha_x = alpha, flags (last block)
// Bytes per node-iteration (3D): A reads r, p, x_hat, wx, wy, wz (24) writes p, q, x_hat (12);
// B reads r, q (8) writes r (4): 48 B.
#include "pn_internal.cuh"

namespace {

constexpr int TPB = 256;

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4& v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 fma4(float a, const float4& x, const float4& y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}

// Last-block epilogue of kernel B: beta, bookkeeping, and the triggers the host polls for.
__device__ __forceinline__ void finish_B(pn_state* st, double rr_new) {
    const double rr_old = st->rr;
    st->rr_old = rr_old;
    st->rr = rr_new;
    st->beta = rr_new / rr_old;
    st->alpha_x = st->alpha;
    const int it = st->iters + 1;
    st->iters = it;
    double rr_max = st->rr_max;
    if (rr_new > rr_max) { rr_max = rr_new; st->rr_max = rr_max; }
    if (!(rr_new >= 0.0) || isinf(rr_new)) st->flag = PN_FLAG_BREAKDOWN;
    else if (rr_new <= st->rr_target) st->flag = PN_FLAG_CONVERGED;
    else if (rr_new < st->delta2 * rr_max) st->flag = PN_FLAG_UPDATE;
    else if (it >= st->max_iters) st->flag = PN_FLAG_BUDGET;
}

// ---- kernel A, reference variant: one thread per 4 consecutive nodes, neighbours through L1/L2 ---
__global__ void __launch_bounds__(TPB) k_stencil_simple(int nvec, int px, int plane, pn_ptrs P, float* p0, float* p1, int defer) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    __shared__ double sm[32];
    __shared__ double tot[1];
    const float beta = (float)st->beta;
    const float ax = (float)st->alpha_x;
    const int par = st->iters & 1;
    const float* __restrict__ pin = par ? p1 : p0;
    float* __restrict__ pout = par ? p0 : p1;
    const float* __restrict__ r = P.r;
    const float* __restrict__ wx = P.w[0];
    const float* __restrict__ wy = P.w[1];
    const float* __restrict__ wz = P.w[2];
    double acc = 0.0;
    for (int v = blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += gridDim.x * blockDim.x) {
        const long long n = 4ll * v;
        const float4 pc = ld4(pin + n);
        const float4 pn = fma4(beta, pc, ld4(r + n));
        st4(P.xh + n, fma4(ax, pc, ld4(P.xh + n)));
        const float pl = fmaf(beta, pin[n - 1], r[n - 1]);
        const float pr = fmaf(beta, pin[n + 4], r[n + 4]);
        const float4 pym = fma4(beta, ld4(pin + n - px), ld4(r + n - px));
        const float4 pyp = fma4(beta, ld4(pin + n + px), ld4(r + n + px));
        const float4 pzm = fma4(beta, ld4(pin + n - plane), ld4(r + n - plane));
        const float4 pzp = fma4(beta, ld4(pin + n + plane), ld4(r + n + plane));
        const float4 gx = ld4(wx + n), gy = ld4(wy + n), gz = ld4(wz + n);
        const float gxl = wx[n - 1];
        const float4 gym = ld4(wy + n - px), gzm = ld4(wz + n - plane);
        float4 q;
        q.x = pn.x - (gxl * pl + gx.x * pn.y + gym.x * pym.x + gy.x * pyp.x + gzm.x * pzm.x + gz.x * pzp.x);
        q.y = pn.y - (gx.x * pn.x + gx.y * pn.z + gym.y * pym.y + gy.y * pyp.y + gzm.y * pzm.y + gz.y * pzp.y);
        q.z = pn.z - (gx.y * pn.y + gx.z * pn.w + gym.z * pym.z + gy.z * pyp.z + gzm.z * pzm.z + gz.z * pzp.z);
        q.w = pn.w - (gx.z * pn.z + gx.w * pr + gym.w * pym.w + gy.w * pyp.w + gzm.w * pzm.w + gz.w * pzp.w);
        st4(pout + n, pn);
        st4(P.q + n, q);
        acc += (double)(pn.x * q.x + pn.y * q.y + pn.z * q.z + pn.w * q.w);
    }
    acc = pn_block_sum(acc, sm);
    const double v1[1] = {acc};
    if (pn_grid_sum<1>(v1, P.slots, &st->ticket, sm, tot)) {
        if (threadIdx.x == 0) {
            if (defer) st->part[0] = tot[0];   // periodic faces: k_wrap_fix finishes
            else pn_finish_A(st, tot[0]);
        }
    }
}

// ---- kernel B: r -= alpha q, rr = r.r  (a pure stream: 12 B per node) ---------------------------
__global__ void __launch_bounds__(TPB) k_update(int nvec, pn_ptrs P) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    __shared__ double sm[32];
    __shared__ double tot[1];
    const float nalpha = -(float)st->alpha;
    float* __restrict__ r = P.r;
    const float* __restrict__ q = P.q;
    double acc = 0.0;
    const int stride = gridDim.x * blockDim.x;
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    for (; v + 3 * stride < nvec; v += 4 * stride) {   // four independent 16-byte loads per array in flight
        float4 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = ld4(r + 4ll * (v + u * stride)); b[u] = __ldcs(reinterpret_cast<const float4*>(q + 4ll * (v + u * stride))); }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 t = fma4(nalpha, b[u], a[u]);
            st4(r + 4ll * (v + u * stride), t);
            acc += (double)(t.x * t.x + t.y * t.y + t.z * t.z + t.w * t.w);
        }
    }
    for (; v < nvec; v += stride) {
        const float4 t = fma4(nalpha, ld4(q + 4ll * v), ld4(r + 4ll * v));
        st4(r + 4ll * v, t);
        acc += (double)(t.x * t.x + t.y * t.y + t.z * t.z + t.w * t.w);
    }
    acc = pn_block_sum(acc, sm);
    const double v1[1] = {acc};
    if (pn_grid_sum<1>(v1, P.slots, &st->ticket, sm, tot)) {
        if (threadIdx.x == 0) finish_B(st, tot[0]);
    }
}

// ---- the single-kernel iteration as ONE persistent cooperative launch per residual replacement, cache-fed -----------------
// Below a few million nodes an iteration is bound by launch boundaries, not by memory (the pair above: 12 us at 64^3; the
// fused TMA kernel: ~16 us of ring ramp + reduction tail per launch; profiles/r02_small_lattices.md).  Here every CTA owns a
// fixed range of the lattice for the whole launch and runs the recurrences of k_cg_fused_tma (pn_fused_tma.cu) on it:
//   r_t = r - alpha q ;  p_t = r_t + beta p  at the node AND, recomputed from their r, q, p, at its six neighbours (through
//   L1 / L2: no shared-memory tiles) ;  x_hat every other iteration ;  q_t = p_t - W p_t ;  r.r, p.q, r.q, q.q
//   ONE grid barrier; then every CTA adds the slots in the same fixed order and runs pn_finish_F on its own copy of the state
// (k_cg_resident2d and k_cpersist work the same way).  r, q, p are double-buffered by iteration parity as in k_cg_fused_tma.
// A two-phase form (update, barrier, stencil, barrier; single buffers) was measured first: 7.8 / 16.7 / 34.0 us at 64^3 /
// 128^3 / 2048^2 against 6.5 / 16.1 / 28.5 us for this one.
// Threads per CTA (template parameter ST): 1024 (64 registers: a few spills since the residual is recovered from two
// directions) streams best on the larger lattices, 768 (80 registers) is faster where latency counts -- measured per iteration,
// 1024 / 768: 64^3 5.7 / 5.4 us, 128^3 15.2 / 14.2, 160^3 31.9 / 34.9, 2048^2 26.7 / 28.7, 3072^2 56.5 / 60.8; periodic 128^3
// 21.6 / 17.1.  Chosen by the launcher: 768 with periodic faces and up to 3 M padded nodes.

__device__ __forceinline__ void sp_grid_barrier(unsigned int* bar, unsigned int target) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(bar), "r"(1u) : "memory");
    unsigned int v;
    do { asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory"); } while (v < target);
    __threadfence();   // acquire; also drops the SM's L1 lines, so that the plain loads that follow see the other CTAs' stores
}

// No residual is stored (as in k_cg_fused_tma, pn_fused_tma.cu): the directions live in three rotating slots {P.p, P.p2, P.r},
// p_{t-1} in `p`, p_{t-2} in `p2`, and r_{t-1} = ca p_{t-1} + cb p_{t-2} with (ca, cb) = (1, -beta_{t-1}), or (0, 1) right after a
// residual replacement, when the slot of p_{t-2} holds the explicit residual k_residual64 wrote.
struct sp_rec { float ca, cb, nal, beta; };
__device__ __forceinline__ float4 rec4(const sp_rec& c, const float4& p1, const float4& p2) {
    return make_float4(fmaf(c.cb, p2.x, c.ca * p1.x), fmaf(c.cb, p2.y, c.ca * p1.y), fmaf(c.cb, p2.z, c.ca * p1.z), fmaf(c.cb, p2.w, c.ca * p1.w));
}
// p_t at a node from the previous iteration's p_{t-2}, q, p_{t-1} there: the deferred residual update, recomputed wherever needed
__device__ __forceinline__ float4 pnew4(const float* __restrict__ p2, const float* __restrict__ q, const float* __restrict__ p,
                                        long long n, const sp_rec& c) {
    const float4 p1 = ld4(p + n);
    return fma4(c.beta, p1, fma4(c.nal, ld4(q + n), rec4(c, p1, ld4(p2 + n))));
}
__device__ __forceinline__ float pnew1(const float* __restrict__ p2, const float* __restrict__ q, const float* __restrict__ p,
                                       long long n, const sp_rec& c) {
    const float p1 = p[n];
    return fmaf(c.beta, p1, fmaf(c.nal, q[n], fmaf(c.cb, p2[n], c.ca * p1)));
}

// WRAP: periodic lateral faces.  A node on a wrapping face has one more bond, to the node on the
// opposite face, weight in the face array ww (pn_setup.cu k_wrap_weights; zero on pad columns); its p_t is recomputed from
// r, q, p there like any other neighbour's: no second kernel (k_wrap_fix, pn_wrap.cu) and no second barrier.
template <bool WRAP, int ST>
__global__ void __launch_bounds__(ST, 1) k_cg_persist(pn_geom g, pn_ptrs P, int max_launch_iters) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;   // same value in every CTA: nobody enters the barrier alone
    __shared__ double red[4 * 32 + 8];
    __shared__ pn_state ls;                 // this CTA's copy of the iteration state
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;
    if (tid == 0) ls = *st;
    __syncthreads();
    const long long nvec = g.npad >> 2;
    const long long per = (nvec + G - 1) / G;
    const long long v0 = min(per * c, nvec), v1 = min(v0 + per, nvec);
    const int px = g.px;
    const long long plane = g.plane;
    const bool has_y = g.ny > 1;            // 2D lattices are held as nx x 1 x rows: no y bonds
    const float* __restrict__ wx = P.w[0];
    const float* __restrict__ wy = P.w[1];
    const float* __restrict__ wz = P.w[2];
    unsigned int* bar = P.gbar;
    unsigned int bar_target = 0;

    for (int li = 0; li < max_launch_iters; ++li) {
        const int pin = li & 1;
        const int par = ls.iters & 1;                               // buffer holding q_{t-1}
        const int s1 = ls.iters % 3, s2 = (ls.iters + 2) % 3, s0 = (ls.iters + 1) % 3;   // slots of p_{t-1}, p_{t-2}, p_t
        const float* __restrict__ r = s2 == 0 ? P.p : (s2 == 1 ? P.p2 : P.r);   // p_{t-2} (or the explicit residual): r_{t-1} is recovered
        const float* __restrict__ q = par ? P.q2 : P.q;
        const float* __restrict__ p = s1 == 0 ? P.p : (s1 == 1 ? P.p2 : P.r);
        float* __restrict__ q_out = par ? P.q : P.q2;
        float* __restrict__ p_out = s0 == 0 ? P.p : (s0 == 1 ? P.p2 : P.r);
        const float al = (float)ls.alpha, nal = -al, beta = (float)ls.beta, a2 = (float)ls.alpha2;
        const sp_rec rc{ls.rexp ? 0.f : 1.f, ls.rexp ? 1.f : -(float)ls.beta_last, nal, beta};
        // x_hat every other iteration, exactly as in k_cg_fused_tma
        const int xmode = ls.xpend ? 2 : ((ls.xskip_min > 0.0 && ls.beta >= ls.xskip_min) ? 0 : 1);
        double a_rr = 0.0, a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;
        for (long long v = v0 + tid; v < v1; v += ST) {
            const long long n = 4 * v;
            const float4 p2o = ld4(r + n), po = ld4(p + n);
            const float4 rn = fma4(nal, ld4(q + n), rec4(rc, po, p2o));
            const float4 pn = fma4(beta, po, rn);
            const float pl = pnew1(r, q, p, n - 1, rc), pr = pnew1(r, q, p, n + 4, rc);
            const float4 pzm = pnew4(r, q, p, n - plane, rc), pzp = pnew4(r, q, p, n + plane, rc);
            const float4 gx = ld4(wx + n), gz = ld4(wz + n), gzm = ld4(wz + n - plane);
            const float gxl = wx[n - 1];
            float4 s;
            s.x = gxl * pl + gx.x * pn.y + gzm.x * pzm.x + gz.x * pzp.x;
            s.y = gx.x * pn.x + gx.y * pn.z + gzm.y * pzm.y + gz.y * pzp.y;
            s.z = gx.y * pn.y + gx.z * pn.w + gzm.z * pzm.z + gz.z * pzp.z;
            s.w = gx.z * pn.z + gx.w * pr + gzm.w * pzm.w + gz.w * pzp.w;
            if (has_y) {
                const float4 pym = pnew4(r, q, p, n - px, rc), pyp = pnew4(r, q, p, n + px, rc);
                const float4 gy = ld4(wy + n), gym = ld4(wy + n - px);
                s.x += gym.x * pym.x + gy.x * pyp.x;
                s.y += gym.y * pym.y + gy.y * pyp.y;
                s.z += gym.z * pym.z + gy.z * pyp.z;
                s.w += gym.w * pym.w + gy.w * pyp.w;
            }
            if (WRAP) {
                const long long row = n / px;
                const int i0 = (int)(n - row * px), j = (int)(row % g.ny), k = (int)(row / g.ny);
                if (g.wrap[0]) {
                    const int last = g.nx - 1, e = last - i0;
                    const float w0 = P.ww[0][j + (long long)g.ny * k];
                    if (i0 == 0) s.x += w0 * pnew1(r, q, p, n + last, rc);
                    if (e >= 0 && e < 4) {
                        const float t = w0 * pnew1(r, q, p, n + e - last, rc);
                        if (e == 0) s.x += t; else if (e == 1) s.y += t; else if (e == 2) s.z += t; else s.w += t;
                    }
                }
                if (g.wrap[1] && (j == 0 || j == g.ny - 1)) {
                    const long long sp = (long long)(g.ny - 1) * px;
                    const float4 w1 = ld4(P.ww[1] + i0 + (long long)px * k);
                    const float4 pp = pnew4(r, q, p, j == 0 ? n + sp : n - sp, rc);
                    s.x += w1.x * pp.x; s.y += w1.y * pp.y; s.z += w1.z * pp.z; s.w += w1.w * pp.w;
                }
                if (g.wrap[2] && (k == 0 || k == g.nz - 1)) {
                    const long long sp = (long long)(g.nz - 1) * plane;
                    const float4 w2 = ld4(P.ww[2] + i0 + (long long)px * j);
                    const float4 pp = pnew4(r, q, p, k == 0 ? n + sp : n - sp, rc);
                    s.x += w2.x * pp.x; s.y += w2.y * pp.y; s.z += w2.z * pp.z; s.w += w2.w * pp.w;
                }
            }
            const float4 qv = make_float4(pn.x - s.x, pn.y - s.y, pn.z - s.z, pn.w - s.w);
            st4(p_out + n, pn);
            st4(q_out + n, qv);
            if (xmode) {
                float4 xn = fma4(al, po, ld4(P.xh + n));
                if (xmode == 2) xn = fma4(a2, p2o, xn);       // the owed alpha_{t-2} p_{t-2}
                st4(P.xh + n, xn);
            }
            a_rr += (double)(rn.x * rn.x + rn.y * rn.y + rn.z * rn.z + rn.w * rn.w);
            a_pq += (double)(pn.x * qv.x + pn.y * qv.y + pn.z * qv.z + pn.w * qv.w);
            a_rq += (double)(rn.x * qv.x + rn.y * qv.y + rn.z * qv.z + rn.w * qv.w);
            a_qq += (double)(qv.x * qv.x + qv.y * qv.y + qv.z * qv.z + qv.w * qv.w);
        }
        a_rr = pn_warp_sum(a_rr); a_pq = pn_warp_sum(a_pq); a_rq = pn_warp_sum(a_rq); a_qq = pn_warp_sum(a_qq);
        if (lane == 0) { red[wid] = a_rr; red[32 + wid] = a_pq; red[64 + wid] = a_rq; red[96 + wid] = a_qq; }
        __syncthreads();
        if (wid == 0) {
            double* my = P.slots + ((size_t)pin * PN_MAX_BLOCKS + c) * 4;     // [parity][CTA][4]: one 32-byte sector per CTA
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double v = pn_warp_sum(lane < ST / 32 ? red[32 * k + lane] : 0.0);
                if (lane == 0) my[k] = v;
            }
            if (lane == 0) { bar_target += G; sp_grid_barrier(bar, bar_target); }
            __syncwarp();
            double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
            const double2* sl = reinterpret_cast<const double2*>(P.slots + (size_t)pin * PN_MAX_BLOCKS * 4);
            double2 va[(PN_RESIDENT_MAX_CTAS + 31) / 32], vb[(PN_RESIDENT_MAX_CTAS + 31) / 32];
#pragma unroll
            for (int u = 0; u < (PN_RESIDENT_MAX_CTAS + 31) / 32; ++u) {
                const int b = lane + 32 * u;
                va[u] = b < G ? __ldcg(sl + 2 * b) : make_double2(0.0, 0.0);
                vb[u] = b < G ? __ldcg(sl + 2 * b + 1) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < (PN_RESIDENT_MAX_CTAS + 31) / 32; ++u) { t0 += va[u].x; t1 += va[u].y; t2 += vb[u].x; t3 += vb[u].y; }
            t0 = pn_warp_sum(t0); t1 = pn_warp_sum(t1); t2 = pn_warp_sum(t2); t3 = pn_warp_sum(t3);
            if (lane == 0) pn_finish_F(&ls, t0, t1, t2, t3);
        }
        __syncthreads();
        if (ls.flag != PN_FLAG_RUN) break;
    }
    if (c == 0 && tid == 0) *st = ls;
}

int grid_for(long long work_items, int sms) {
    long long nb = (work_items + TPB - 1) / TPB;
    long long cap = (long long)sms * 8;
    if (cap > PN_MAX_BLOCKS) cap = PN_MAX_BLOCKS;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    return (int)nb;
}

}  // namespace

// PN_OPT_KERNEL: 0 = automatic: the whole loop in one CTA when the lattice fits one SM's shared memory (5); the persistent
// shared-memory-resident kernel for 2D lattices whose slabs fit all SMs (6); the persistent structured kernel above (8)
// for the other lattices of at most PN_SMALL_LATTICE (3D) / PN_SMALL_LATTICE_2D padded nodes (periodic faces included:
// its WRAP instantiation; without cooperative launch: the cache-fed pair, 1); else the single fused TMA kernel (3).  Measured on B200 (profiles/r02_small_lattices.md), per
// iteration, persistent / fused TMA: 6.5 / 15.3 us at 64^3, 9.6 / 19.1 at 96^3, 16.1 / 26.0 at 128^3, 34.2 / 43.1 at 160^3,
// 71.1 / 61.0 at 192^3; 2D: 12.0 / 27.1 at 1448^2, 28.5 / 34.3 at 2048^2, 61.9 / 75.2 at 3072^2, 109.1 / 107.9 at 4096^2.
// The TMA kernel pays ~16 us of ring ramp and reduction tail per launch but fetches every value from L2 / HBM once per
// tile; the persistent kernel re-reads the neighbours' r, q, p through L1 / L2, which is free while the lattice's planes
// sit there and costs bandwidth beyond.
// 1 = the pair on any lattice (independently written cross-check).  The two superseded schemes of round 1 (2: TMA S4
// kernel + S5 kernel, 4: q recomputed) are gone; their write-ups remain in profiles/r01_tma_kernel.md and
// profiles/r01_q_recompute_experiment.md.
constexpr long long PN_SMALL_LATTICE = 5000000;      // 3D
constexpr long long PN_SMALL_LATTICE_2D = 12000000;  // 2D lattices (held as nx x 1 x rows)
int pn_resolve_variant(const pn_geom& g, const pn_ptrs& P, int variant) {
    const int big = pn_tma_supported() ? 3 : 1;
    if (variant == 0) {
        if (pn_onchip_supported(g)) return 5;
        if (pn_resident_supported(g, P)) return 6;
        if (g.npad <= (g.ny == 1 ? PN_SMALL_LATTICE_2D : PN_SMALL_LATTICE)) return g.coop ? 8 : 1;
        return big;
    }
    if (variant == 8 && !g.coop) return 1;   // no cooperative launch on this device
    if (variant == 5 && !pn_onchip_supported(g)) return big;   // too large for one SM, or periodic faces
    if (variant == 6 && !pn_resident_supported(g, P)) return big;   // 3D, wider than 2048, or periodic faces
    return variant;
}

// `scheme` is a resolved variant (1, 3 or 5).  ev (optional, 2*iterations+1 events): kernel boundaries, for
// the per-kernel timing of PN_OPT_PROFILE (scheme 3: the second interval of every iteration is empty).
cudaError_t pn_launch_inner(const pn_geom& g, const pn_ptrs& P, int iterations, int scheme, cudaStream_t st,
                            int* launches, cudaEvent_t* ev, const pn_cptrs* compact) {
    const int nvec = (int)(g.npad / 4);
    const int nb = grid_for(nvec, g.sms);
    pn_fused_plan* fplan = nullptr;
    if ((scheme == 3 || scheme == 10) && !(pn_tma_supported() && pn_fused_plan_build(&fplan, g, P))) return cudaErrorNotSupported;
    if (scheme == 10) {   // the fused TMA kernel as one persistent cooperative launch up to the next trigger (internal code)
        if (ev) cudaEventRecord(ev[0], st);
        cudaError_t e10 = pn_launch_cg_fused(fplan, g, P, st, iterations);
        if (ev) { cudaEventRecord(ev[1], st); cudaEventRecord(ev[2], st); }
        pn_fused_plan_free(fplan);
        *launches += 1;
        return e10;
    }
    if (scheme == 5 || scheme == 6 || scheme == 8) {   // the whole loop up to the next trigger (or `iterations`) in ONE launch (pn_onchip.cu, pn_resident.cu, k_cg_persist)
        if (ev) cudaEventRecord(ev[0], st);
        cudaError_t e5;
        if (scheme == 5) e5 = pn_launch_cg_onchip(g, P, iterations, st);
        else if (scheme == 6) e5 = pn_launch_cg_resident(g, P, iterations, st);
        else {
            e5 = cudaMemsetAsync(P.gbar, 0, sizeof(unsigned int), st);
            int G = g.sms < PN_RESIDENT_MAX_CTAS ? g.sms : PN_RESIDENT_MAX_CTAS, mi = iterations;
            pn_geom gg = g;
            pn_ptrs PP = P;
            void* args[] = {(void*)&gg, (void*)&PP, (void*)&mi};
            const bool wrap8 = (g.wrap[0] | g.wrap[1] | g.wrap[2]) != 0, few = wrap8 || g.npad <= 3000000;
            const void* fn = wrap8 ? (const void*)k_cg_persist<true, 768>
                                   : (few ? (const void*)k_cg_persist<false, 768> : (const void*)k_cg_persist<false, 1024>);
            if (e5 == cudaSuccess) e5 = cudaLaunchCooperativeKernel(fn, dim3(G), dim3(few ? 768 : 1024), args, 0, st);
        }
        if (ev) { cudaEventRecord(ev[1], st); cudaEventRecord(ev[2], st); }
        *launches += 1;
        return e5;
    }
    if (scheme == 7 || scheme == 9) {   // compacted unknowns (pn_compact.cu): two kernels per iteration (7) / one persistent launch (9, internal)
        if (!compact) return cudaErrorInvalidValue;
        if (scheme == 7) return pn_launch_compact_inner(g, P, *compact, iterations, st, launches, ev);
        if (ev) cudaEventRecord(ev[0], st);
        cudaError_t e9 = pn_launch_compact_persist(g, P, *compact, iterations, st);
        if (ev) { cudaEventRecord(ev[1], st); cudaEventRecord(ev[2], st); }
        *launches += 1;
        return e9;
    }
    const bool wrap = g.wrap[0] || g.wrap[1] || g.wrap[2];   // periodic lateral faces: k_wrap_fix finishes kernel A
    cudaError_t e = cudaSuccess;
    if (ev) cudaEventRecord(ev[0], st);
    for (int it = 0; it < iterations && e == cudaSuccess; ++it) {
        if (scheme == 3) e = pn_launch_cg_fused(fplan, g, P, st);
        else k_stencil_simple<<<nb, TPB, 0, st>>>(nvec, g.px, (int)g.plane, P, P.p, P.p2, wrap ? 1 : 0);
        if (wrap && e == cudaSuccess) e = pn_launch_wrap_fix(g, P, scheme == 3, st);
        if (ev) cudaEventRecord(ev[2 * it + 1], st);
        if (scheme < 3) k_update<<<nb, TPB, 0, st>>>(nvec, P);
        if (ev) cudaEventRecord(ev[2 * it + 2], st);
    }
    pn_fused_plan_free(fplan);
    *launches += ((scheme == 3 ? 1 : 2) + (wrap ? 1 : 0)) * iterations;
    return e != cudaSuccess ? e : cudaGetLastError();
}
