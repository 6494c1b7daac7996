// pn_compact.cu -- active-node compaction (second half): the fp32 inner CG iteration on the
// UNKNOWNS only, stored contiguously with an ELL-3 + overflow neighbour table, for diluted networks in which most lattice nodes are
// not unknowns (pinned clusters, Dirichlet planes, peeled dangling ends).
//
// Why a gather form and not bricks (profiles/r02_compaction.md): near the threshold (configs[2],
// p = 0.30) one third of the lattice nodes are unknowns after peeling (the critical slow-down case), but
// they are spread uniformly: 12.7 % of the 8-node x-segments and 0.1 % of the 32-node ones hold no unknown, so dropping
// empty segments or tiles of the structured kernel would skip next to nothing.  The 2-core that remains has mean
// degree 2.37 (69 % of its nodes have two bonds, 25 % three), so the table is ELL of width 3 -- three (index, weight)
// slots per row, structure of arrays, unused slots pointing at the row itself with weight 0 -- and the 6 % of rows with
// more bonds keep entries 3..6 in an overflow record their third slot points to: 24 bytes per row + 32 per long row, no
// row-pointer indirection (a CSR version measured 136 us per iteration on configs[2] against 117 us structured: its
// rowptr -> col -> p chain of dependent loads was latency-bound).
//
// Iteration t (same recurrences as k_cg_fused_tma: deferred residual update, beta predicted from r.r, r.q, q.q, so that
// both kernels know their scalars at launch; all sums fp32 products -> fp64, fixed-order grid reduction):
//   k_cupdate:  r_t = r - alpha_{t-1} q ;  x_hat += alpha_{t-1} p ;  p_t = r_t + beta_t p ;  r_t.r_t      (pure stream, 28 B)
//   k_cspmv:    q_t = p_t - sum_k val_k p_t[col_k] ;  p.q, r.q, q.q  -> alpha_t, beta_{t+1}, flags        (36 B + gathers)
// = 64 bytes per UNKNOWN and iteration, against 40 bytes per LATTICE NODE for the structured kernel: pays when fewer
// than ~0.45 of the padded lattice nodes are unknowns.  Unknowns are numbered in lattice order, so x-neighbours are
// adjacent and y / z neighbours a fixed few thousand entries away: the gathers are served by L1 / L2.
// The fp64 outer steps stay on the lattice (k_residual64 writes r_hat there); k_cgather / k_cflush move r_hat and the
// correction between the two numberings.  No periodic faces (those lattices keep the structured kernels).
// With PN_OPT_CONTRACT the degree-2 link nodes are eliminated first (pn_chain.cu): a bond towards a chain becomes a table
// entry to the chain's far end.  By default the two kernels run as the two phases of ONE persistent cooperative launch
// per residual replacement (k_cpersist, below); kernel by kernel with PN_OPT_GRAPH = 0.
#include "pn_chain.cuh"

namespace {

constexpr int TPB = 256;
constexpr int SCAN_T = 1024;                 // threads of the scan kernels

int grid_for(long long work_items, int sms) {
    long long nb = (work_items + TPB - 1) / TPB;
    long long cap = (long long)sms * 8;
    if (cap > PN_MAX_BLOCKS) cap = PN_MAX_BLOCKS;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    return (int)nb;
}

// one scan over (unknown count, long-row count) numbers the unknowns AND the overflow records
struct scan2 { unsigned long long n, e; };
__device__ __forceinline__ scan2 operator+(const scan2& a, const scan2& b) { return scan2{a.n + b.n, a.e + b.e}; }

// scaled weight of the bond of padded node n in direction code c (0:+x 1:-x 2:+y 3:-y 4:+z 5:-z)
__device__ __forceinline__ float weight_dir(const pn_geom& g, const pn_ptrs& P, long long n, int c) {
    const int b = c >> 1;
    const long long sb = b == 0 ? 1 : (b == 1 ? (long long)g.px : g.plane);
    return P.w[b][(c & 1) ? n - sb : n];
}
// does direction c of unknown n give a table entry?  A non-zero scaled weight (weights towards Dirichlet, pinned and
// peeled nodes are zero: they live in the diagonal and in b), or -- with degree-2 chains eliminated (pn_chain.cu) -- an
// open bond towards a chain node: the entry then points at the chain's far end
__device__ __forceinline__ bool has_entry(const pn_geom& g, const pn_ptrs& P, long long n, int c, int chains) {
    if (weight_dir(g, P, n, c) != 0.f) return true;
    if (!chains) return false;
    long long m;
    return pn_bond_dir(g, P, n, c, &m) != 0.f && P.cls[m] == PN_CLASS_CHAIN;
}

// (is unknown, is a long row) of lattice node n: an unknown has a non-zero Jacobi scale; long = more than three entries
__device__ __forceinline__ scan2 node_counts(const pn_geom& g, const pn_ptrs& P, long long n, int chains) {
    scan2 v{0ull, 0ull};
    if (P.s[n] != 0.f) {
        v.n = 1ull;
        int deg = 0;
#pragma unroll
        for (int c = 0; c < 6; ++c) deg += has_entry(g, P, n, c, chains) ? 1 : 0;
        v.e = deg > 3 ? 1ull : 0ull;
    }
    return v;
}

__device__ __forceinline__ scan2 warp_sum2(scan2 v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.n += __shfl_down_sync(0xffffffffu, v.n, o);
        v.e += __shfl_down_sync(0xffffffffu, v.e, o);
    }
    return v;
}

// pass 1: totals of every block's contiguous chunk [b * chunk, (b + 1) * chunk)
__global__ void __launch_bounds__(SCAN_T) k_cscan_totals(pn_geom g, pn_ptrs P, int chains, long long chunk, scan2* part) {
    __shared__ scan2 sm[32];
    const long long lo = blockIdx.x * chunk, hi = min(lo + chunk, g.npad);
    scan2 v{0ull, 0ull};
    for (long long n = lo + threadIdx.x; n < hi; n += SCAN_T) v = v + node_counts(g, P, n, chains);
    v = warp_sum2(v);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = sm[threadIdx.x];
        v = warp_sum2(v);
        if (threadIdx.x == 0) part[blockIdx.x] = v;
    }
}

// pass 2 (one block): exclusive scan of the block totals in place; grand totals -> state
__global__ void __launch_bounds__(SCAN_T) k_cscan_partials(int nblocks, scan2* part, pn_state* st) {
    if (threadIdx.x == 0) {
        scan2 run{0ull, 0ull};
        for (int b = 0; b < nblocks; ++b) { const scan2 t = part[b]; part[b] = run; run = run + t; }
        st->cm = run.n;
        st->clong = run.e;
    }
}

// pass 3: lattice -> compact index (cidx, -1 on nodes that are not unknowns), compact -> lattice (lat); a long row's
// third slot gets the code of its overflow record (-1 - record)
__global__ void __launch_bounds__(SCAN_T) k_cscan_write(pn_geom g, pn_ptrs P, int chains, long long chunk, const scan2* part,
                                                         int* cidx, int* lat, int* c2) {
    __shared__ scan2 wsum[32];
    __shared__ scan2 carry;
    const long long lo = blockIdx.x * chunk, hi = min(lo + chunk, g.npad);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = part[blockIdx.x];
    __syncthreads();
    for (long long base = lo; base < hi; base += SCAN_T) {
        const long long n = base + threadIdx.x;
        const scan2 mine = n < hi ? node_counts(g, P, n, chains) : scan2{0ull, 0ull};
        scan2 inc = mine;                                   // inclusive scan inside the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long an = __shfl_up_sync(0xffffffffu, inc.n, o), ae = __shfl_up_sync(0xffffffffu, inc.e, o);
            if (lane >= o) { inc.n += an; inc.e += ae; }
        }
        if (lane == 31) wsum[wid] = inc;
        __syncthreads();
        if (wid == 0) {                                     // exclusive scan of the 32 warp totals
            const scan2 t = wsum[lane];
            scan2 s = t;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned long long an = __shfl_up_sync(0xffffffffu, s.n, o), ae = __shfl_up_sync(0xffffffffu, s.e, o);
                if (lane >= o) { s.n += an; s.e += ae; }
            }
            wsum[lane] = scan2{s.n - t.n, s.e - t.e};
        }
        __syncthreads();
        const scan2 c0 = carry, w0 = wsum[wid];
        if (n < hi) {
            const unsigned long long my_n = c0.n + w0.n + inc.n - mine.n, my_e = c0.e + w0.e + inc.e - mine.e;
            if (mine.n) {
                cidx[n] = (int)my_n;
                lat[my_n] = (int)n;
                c2[my_n] = mine.e ? -1 - (int)my_e : 0;
            } else cidx[n] = -1;
        }
        __syncthreads();
        if (threadIdx.x == SCAN_T - 1) carry = scan2{c0.n + w0.n + inc.n, c0.e + w0.e + inc.e};
        __syncthreads();
    }
}

// pass 4: the rows, directions in the order -z, -y, -x, +x, +y, +z (ascending compact index without chains).  With
// chains eliminated a bond towards a chain node becomes the entry (far end of the chain, series conductance x the two
// Jacobi scales), rounded once from fp64 like every weight; a chain that loops back to the row itself carries no current
// and leaves an empty slot.  Parallel entries (two chains, or a chain and a bond, to the same node) stay separate.
__global__ void k_cfill(pn_geom g, pn_ptrs P, pn_cptrs C, int chains) {
    const long long m = (long long)P.st->cm;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < m; i += (long long)gridDim.x * blockDim.x) {
        const long long n = C.lat[i];
        int ec[6];
        float ev[6];
        int k = 0;
        const int order[6] = {5, 3, 1, 0, 2, 4};
#pragma unroll 1
        for (int o = 0; o < 6; ++o) {
            const int c = order[o];
            const float w = weight_dir(g, P, n, c);
            long long mnode;
            const float gv = pn_bond_dir(g, P, n, c, &mnode);
            if (w != 0.f) { ec[k] = C.cidx[mnode]; ev[k] = w; ++k; }
            else if (chains && gv != 0.f && P.cls[mnode] == PN_CLASS_CHAIN) {
                const pn_walk wk = pn_chain_canonical(g, P, n, c);
                if (wk.end == n) { ec[k] = (int)i; ev[k] = 0.f; }
                else { ec[k] = C.cidx[wk.end]; ev[k] = (float)((1.0 / wk.R) * (double)P.s[n] * (double)P.s[wk.end]); }
                ++k;
            }
        }
        for (int u = k; u < 6; ++u) { ec[u] = (int)i; ev[u] = 0.f; }   // unused slots: the row itself, weight 0
        C.c[0][i] = ec[0]; C.v[0][i] = ev[0];
        C.c[1][i] = ec[1]; C.v[1][i] = ev[1];
        if (k <= 3) { C.c[2][i] = ec[2]; C.v[2][i] = ev[2]; }
        else {
            const int rec = -1 - C.c[2][i];               // written by k_cscan_write
            C.v[2][i] = 0.f;
            reinterpret_cast<int4*>(C.ovc)[rec] = make_int4(ec[2], ec[3], ec[4], ec[5]);
            reinterpret_cast<float4*>(C.ovv)[rec] = make_float4(ev[2], ev[3], ev[4], ev[5]);
        }
    }
}

// ---- between the two numberings (once per fp64 residual replacement) -----------------------------------------------
__global__ void k_cgather(pn_ptrs P, pn_cptrs C) {
    const long long m = (long long)P.st->cm;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < m; i += (long long)gridDim.x * blockDim.x)
        C.r[i] = P.r[C.lat[i]];
}

// S7 in the compact numbering: x64 += s (x_hat + alpha_x p) on the unknowns; x_hat = 0
__global__ void k_cflush(pn_ptrs P, pn_cptrs C) {
    const long long m = (long long)P.st->cm;
    const double ax = P.st->alpha_x;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < m; i += (long long)gridDim.x * blockDim.x) {
        const long long n = C.lat[i];
        P.x64[n] += (double)P.s[n] * ((double)C.x[i] + ax * (double)C.p[i]);
        C.x[i] = 0.f;
    }
}

// ---- the iteration ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4& v) { *reinterpret_cast<float4*>(p) = v; }

// r_t = r - alpha q ; x_hat += alpha p ; p_t = r_t + beta p ; r_t.r_t -> state.part[0]   (alpha = alpha_{t-1}, 0 right
// after a residual replacement; beta = beta_t, predicted by the previous k_cspmv or set from the true residual)
__global__ void __launch_bounds__(TPB) k_cupdate(pn_ptrs P, pn_cptrs C) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    __shared__ double sm[32];
    __shared__ double tot[1];
    const long long m = (long long)st->cm, m4 = m >> 2;
    const float al = (float)st->alpha, nal = -al, beta = (float)st->beta;
    double acc = 0.0;
    for (long long v = blockIdx.x * (long long)blockDim.x + threadIdx.x; v < m4; v += (long long)gridDim.x * blockDim.x) {
        const long long i = 4 * v;
        float4 r = ld4(C.r + i);
        const float4 q = __ldcs(reinterpret_cast<const float4*>(C.q + i));
        float4 p = ld4(C.p + i), x = ld4(C.x + i);
        r.x = fmaf(nal, q.x, r.x); r.y = fmaf(nal, q.y, r.y); r.z = fmaf(nal, q.z, r.z); r.w = fmaf(nal, q.w, r.w);
        x.x = fmaf(al, p.x, x.x); x.y = fmaf(al, p.y, x.y); x.z = fmaf(al, p.z, x.z); x.w = fmaf(al, p.w, x.w);
        p.x = fmaf(beta, p.x, r.x); p.y = fmaf(beta, p.y, r.y); p.z = fmaf(beta, p.z, r.z); p.w = fmaf(beta, p.w, r.w);
        st4(C.r + i, r); st4(C.x + i, x); st4(C.p + i, p);
        acc += (double)(r.x * r.x + r.y * r.y + r.z * r.z + r.w * r.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(m - 4 * m4)) {   // the last 0..3 unknowns
        const long long i = 4 * m4 + threadIdx.x;
        const float r = fmaf(nal, C.q[i], C.r[i]);
        const float p = C.p[i];
        C.x[i] = fmaf(al, p, C.x[i]);
        C.r[i] = r;
        C.p[i] = fmaf(beta, p, r);
        acc += (double)(r * r);
    }
    acc = pn_block_sum(acc, sm);
    const double v1[1] = {acc};
    if (pn_grid_sum<1>(v1, P.slots, &st->ticket, sm, tot)) {
        if (threadIdx.x == 0) st->part[0] = tot[0];
    }
}

// q_t = p_t - W p_t over the table rows ; p.q, r.q, q.q ; last block: alpha_t, predicted beta_{t+1}, flags (pn_finish_F)
__global__ void __launch_bounds__(TPB) k_cspmv(pn_ptrs P, pn_cptrs C) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    __shared__ double sm[32];
    __shared__ double tot[3];
    const long long m = (long long)st->cm, m4 = m >> 2;
    const float* __restrict__ p = C.p;
    double a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;
    // one row: two dependent rounds of loads (slots, then the gathered p); FOUR consecutive rows per thread put four
    // times as many of them in flight (measured on configs[2]: one row per thread ran at 2.4 TB/s, latency-bound)
    for (long long v = blockIdx.x * (long long)blockDim.x + threadIdx.x; v < m4; v += (long long)gridDim.x * blockDim.x) {
        const long long i = 4 * v;
        const int4 c0 = *reinterpret_cast<const int4*>(C.c[0] + i), c1 = *reinterpret_cast<const int4*>(C.c[1] + i),
                   c2 = *reinterpret_cast<const int4*>(C.c[2] + i);
        const float4 v0 = ld4(C.v[0] + i), v1 = ld4(C.v[1] + i), v2 = ld4(C.v[2] + i);
        const float4 pi = ld4(p + i), ri = ld4(C.r + i);
        const int cc0[4] = {c0.x, c0.y, c0.z, c0.w}, cc1[4] = {c1.x, c1.y, c1.z, c1.w}, cc2[4] = {c2.x, c2.y, c2.z, c2.w};
        const float w0[4] = {v0.x, v0.y, v0.z, v0.w}, w1[4] = {v1.x, v1.y, v1.z, v1.w}, w2[4] = {v2.x, v2.y, v2.z, v2.w};
        const float pp[4] = {pi.x, pi.y, pi.z, pi.w};
        float g0[4], g1[4], g2[4], qq[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            g0[u] = p[cc0[u]];
            g1[u] = p[cc1[u]];
            g2[u] = cc2[u] >= 0 ? p[cc2[u]] : 0.f;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float acc = w0[u] * g0[u];
            acc = fmaf(w1[u], g1[u], acc);
            if (cc2[u] >= 0) acc = fmaf(w2[u], g2[u], acc);
            else {                                          // long row: entries 3..6 from its overflow record
                const int4 oc = reinterpret_cast<const int4*>(C.ovc)[-1 - cc2[u]];
                const float4 ov = reinterpret_cast<const float4*>(C.ovv)[-1 - cc2[u]];
                acc = fmaf(ov.x, p[oc.x], acc);
                acc = fmaf(ov.y, p[oc.y], acc);
                acc = fmaf(ov.z, p[oc.z], acc);
                acc = fmaf(ov.w, p[oc.w], acc);
            }
            qq[u] = pp[u] - acc;
        }
        const float4 q = make_float4(qq[0], qq[1], qq[2], qq[3]);
        st4(C.q + i, q);
        a_pq += (double)(pi.x * q.x + pi.y * q.y + pi.z * q.z + pi.w * q.w);
        a_rq += (double)(ri.x * q.x + ri.y * q.y + ri.z * q.z + ri.w * q.w);
        a_qq += (double)(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(m - 4 * m4)) {   // the last 0..3 rows
        const long long i = 4 * m4 + threadIdx.x;
        const int c2 = C.c[2][i];
        const float pi = p[i];
        float acc = C.v[0][i] * p[C.c[0][i]];
        acc = fmaf(C.v[1][i], p[C.c[1][i]], acc);
        if (c2 >= 0) acc = fmaf(C.v[2][i], p[c2], acc);
        else {
            const int4 oc = reinterpret_cast<const int4*>(C.ovc)[-1 - c2];
            const float4 ov = reinterpret_cast<const float4*>(C.ovv)[-1 - c2];
            acc = fmaf(ov.x, p[oc.x], acc);
            acc = fmaf(ov.y, p[oc.y], acc);
            acc = fmaf(ov.z, p[oc.z], acc);
            acc = fmaf(ov.w, p[oc.w], acc);
        }
        const float q = pi - acc;
        C.q[i] = q;
        a_pq += (double)(pi * q);
        a_rq += (double)(C.r[i] * q);
        a_qq += (double)(q * q);
    }
    a_pq = pn_block_sum(a_pq, sm);
    a_rq = pn_block_sum(a_rq, sm);
    a_qq = pn_block_sum(a_qq, sm);
    const double v3[3] = {a_pq, a_rq, a_qq};
    if (pn_grid_sum<3>(v3, P.slots, &st->ticket, sm, tot)) {
        if (threadIdx.x == 0) pn_finish_F(st, st->part[0], tot[0], tot[1], tot[2]);
    }
}

// ---- the same iteration as ONE persistent cooperative launch per residual replacement ------------------------------------
// With the links eliminated configs[2] has 1.7 M unknowns: the two kernels of an iteration take 21 us and their two
// boundaries (launch gap, last-block reduction tail, start-up of 1184 CTAs) another 14 (profiles/r02_ncu.md).  Here every CTA
// owns a fixed range of rows for the whole launch and the boundaries become two grid barriers per iteration: one after
// the vector updates (the gathers read other CTAs' p_t), one after the operator (alpha, beta need the four sums).  As in
// k_cg_resident2d, after the second barrier EVERY CTA adds the slots in the same fixed order and runs pn_finish_F on its
// own copy of the state.  Same arithmetic per row as k_cupdate / k_cspmv; the partial sums are grouped per CTA range.
constexpr int PT = 1024;

__device__ __forceinline__ void cp_red_release_add(unsigned int* p, unsigned int v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned int cp_ld_relaxed(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// one thread per CTA, between two CTA barriers; __threadfence after the spin also drops the SM's L1 lines, so that the
// plain loads that follow see what the other CTAs wrote
__device__ __forceinline__ void cp_grid_barrier(unsigned int* bar, unsigned int target) {
    cp_red_release_add(bar, 1u);
    while (cp_ld_relaxed(bar) < target) { }
    __threadfence();
}

// one table row (shared by the persistent kernel's operator phase)
__device__ __forceinline__ float row_sum(const pn_cptrs& C, const float* __restrict__ p, int c0, int c1, int c2, float v0, float v1,
                                         float v2) {
    float acc = v0 * p[c0];
    acc = fmaf(v1, p[c1], acc);
    if (c2 >= 0) acc = fmaf(v2, p[c2], acc);
    else {
        const int4 oc = reinterpret_cast<const int4*>(C.ovc)[-1 - c2];
        const float4 ov = reinterpret_cast<const float4*>(C.ovv)[-1 - c2];
        acc = fmaf(ov.x, p[oc.x], acc);
        acc = fmaf(ov.y, p[oc.y], acc);
        acc = fmaf(ov.z, p[oc.z], acc);
        acc = fmaf(ov.w, p[oc.w], acc);
    }
    return acc;
}

__global__ void __launch_bounds__(PT, 1) k_cpersist(pn_ptrs P, pn_cptrs C, int max_launch_iters) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;   // same value in every CTA: nobody enters the barriers alone
    __shared__ double red[4 * 32 + 8];
    __shared__ pn_state ls;                 // this CTA's copy of the iteration state
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;
    if (tid == 0) ls = *st;
    __syncthreads();
    const long long m = (long long)ls.cm;
    const long long per = ((m + 4ll * G - 1) / (4ll * G)) * 4;             // rows per CTA, a multiple of 4
    const long long i0 = min(per * c, m), i1 = min(i0 + per, m);
    const long long v0i = i0 >> 2, v1i = i1 >> 2;                           // whole groups of 4 rows in [i0, i1)
    const long long t0i = max(4 * v1i, i0);                                 // the range's last 0..3 rows (an empty range has none)
    const float* __restrict__ p = C.p;
    unsigned int* bar = P.gbar;
    unsigned int bar_target = 0;

    for (int li = 0; li < max_launch_iters; ++li) {
        const int pin = li & 1;
        const float al = (float)ls.alpha, nal = -al, beta = (float)ls.beta;
        double a_rr = 0.0, a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;
        // ---- r_t = r - alpha q ; x_hat += alpha p ; p_t = r_t + beta p ; r_t.r_t (own rows) ----
        for (long long v = v0i + tid; v < v1i; v += PT) {
            const long long i = 4 * v;
            float4 r = ld4(C.r + i);
            const float4 q = ld4(C.q + i);
            float4 pp = ld4(C.p + i), x = ld4(C.x + i);
            r.x = fmaf(nal, q.x, r.x); r.y = fmaf(nal, q.y, r.y); r.z = fmaf(nal, q.z, r.z); r.w = fmaf(nal, q.w, r.w);
            x.x = fmaf(al, pp.x, x.x); x.y = fmaf(al, pp.y, x.y); x.z = fmaf(al, pp.z, x.z); x.w = fmaf(al, pp.w, x.w);
            pp.x = fmaf(beta, pp.x, r.x); pp.y = fmaf(beta, pp.y, r.y); pp.z = fmaf(beta, pp.z, r.z); pp.w = fmaf(beta, pp.w, r.w);
            st4(C.r + i, r); st4(C.x + i, x); st4(C.p + i, pp);
            a_rr += (double)(r.x * r.x + r.y * r.y + r.z * r.z + r.w * r.w);
        }
        for (long long i = t0i + tid; i < i1; i += PT) {
            const float r = fmaf(nal, C.q[i], C.r[i]);
            const float pp = C.p[i];
            C.x[i] = fmaf(al, pp, C.x[i]);
            C.r[i] = r;
            C.p[i] = fmaf(beta, pp, r);
            a_rr += (double)(r * r);
        }
        __syncthreads();
        if (tid == 0) { bar_target += G; cp_grid_barrier(bar, bar_target); }
        __syncthreads();
        // ---- q_t = p_t - W p_t over the table rows (own rows; the gathers reach any row) ; p.q, r.q, q.q ----
        for (long long v = v0i + tid; v < v1i; v += PT) {
            const long long i = 4 * v;
            const int4 c0 = *reinterpret_cast<const int4*>(C.c[0] + i), c1 = *reinterpret_cast<const int4*>(C.c[1] + i),
                       c2 = *reinterpret_cast<const int4*>(C.c[2] + i);
            const float4 w0 = ld4(C.v[0] + i), w1 = ld4(C.v[1] + i), w2 = ld4(C.v[2] + i);
            const float4 pi = ld4(p + i), ri = ld4(C.r + i);
            float4 q;
            q.x = pi.x - row_sum(C, p, c0.x, c1.x, c2.x, w0.x, w1.x, w2.x);
            q.y = pi.y - row_sum(C, p, c0.y, c1.y, c2.y, w0.y, w1.y, w2.y);
            q.z = pi.z - row_sum(C, p, c0.z, c1.z, c2.z, w0.z, w1.z, w2.z);
            q.w = pi.w - row_sum(C, p, c0.w, c1.w, c2.w, w0.w, w1.w, w2.w);
            st4(C.q + i, q);
            a_pq += (double)(pi.x * q.x + pi.y * q.y + pi.z * q.z + pi.w * q.w);
            a_rq += (double)(ri.x * q.x + ri.y * q.y + ri.z * q.z + ri.w * q.w);
            a_qq += (double)(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
        }
        for (long long i = t0i + tid; i < i1; i += PT) {
            const float pi = p[i];
            const float q = pi - row_sum(C, p, C.c[0][i], C.c[1][i], C.c[2][i], C.v[0][i], C.v[1][i], C.v[2][i]);
            C.q[i] = q;
            a_pq += (double)(pi * q);
            a_rq += (double)(C.r[i] * q);
            a_qq += (double)(q * q);
        }
        // ---- the four sums: warp -> CTA -> slots -> grid barrier -> every CTA adds the slots in the same order ----
        a_rr = pn_warp_sum(a_rr); a_pq = pn_warp_sum(a_pq); a_rq = pn_warp_sum(a_rq); a_qq = pn_warp_sum(a_qq);
        if (lane == 0) { red[wid] = a_rr; red[32 + wid] = a_pq; red[64 + wid] = a_rq; red[96 + wid] = a_qq; }
        __syncthreads();
        if (wid == 0) {
            double* my = P.slots + ((size_t)pin * PN_MAX_BLOCKS + c) * 4;     // [parity][CTA][4]: one 32-byte sector per CTA
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double v = pn_warp_sum(red[32 * k + lane]);
                if (lane == 0) my[k] = v;
            }
            if (lane == 0) { bar_target += G; cp_grid_barrier(bar, bar_target); }
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

}  // namespace

// Where the compact arrays live: in lattice-shaped arrays the structured kernels do not need during a compact solve.
// Each holds npad floats; with `off` = cm rounded up to 64 entries and 2 * off <= npad, two row-indexed arrays share
// one: p2 = c0 | c1, r2 = c2 | v0, q = v1 | v2, q2 = lat | overflow records (8 words per long row).  cidx is scratch of
// the build only (P.r is rewritten by the first k_residual64 afterwards); the vectors q and r take the place of the
// scaled weights, which the build has consumed by the time they are first written.
bool pn_compact_fits(const pn_geom& g, long long m, long long n_long) {
    const long long off = (m + 63) & ~63ll;
    return m >= 1 && 2 * off <= g.npad && off + 8 * n_long + 8 <= g.npad;
}

pn_cptrs pn_compact_ptrs(const pn_geom& g, const pn_ptrs& P, long long m, long long n_long) {
    const long long off = (m + 63) & ~63ll;
    pn_cptrs C;
    C.cidx = (int*)P.r;
    C.lat = (int*)P.q2;
    C.ovc = (int*)P.q2 + off;
    C.ovv = (float*)(C.ovc + 4 * ((n_long + 3) & ~3ll));
    C.c[0] = (int*)P.p2; C.c[1] = (int*)P.p2 + off;
    C.c[2] = (int*)P.r2; C.v[0] = P.r2 + off;
    C.v[1] = P.q;        C.v[2] = P.q + off;
    C.p = P.p;
    C.x = P.xh;
    C.q = P.w[0];
    C.r = P.w[1];
    // back-fill records of the chain nodes: the node list in the unused upper half of w[0]; (a, b) and t in the upper half
    // of w[1] and all of w[2] (consecutive in the workspace; the weights are dead once the table is built)
    C.chv = (int*)P.w[0] + off;
    char* lo = (char*)(P.w[1] + off);
    long long cap = (long long)((char*)(P.w[2] + g.npad) - lo) / 16;
    if (cap > g.npad - off) cap = g.npad - off;
    if (cap < 0) cap = 0;
    C.chab = reinterpret_cast<int2*>(lo);
    C.cht = reinterpret_cast<double*>(lo + 8 * cap);
    C.chcap = cap;
    return C;
}

static int scan_blocks(const pn_geom& g) {
    int nb = g.sms * 8;
    if (nb > PN_MAX_BLOCKS) nb = PN_MAX_BLOCKS;
    const long long need = (g.npad + SCAN_T - 1) / SCAN_T;
    if (nb > need) nb = (int)need;
    return nb < 1 ? 1 : nb;
}

// passes 1-2: how many unknowns and long rows -> state.cm, state.clong (the host decides whether to compact)
cudaError_t pn_launch_compact_count(const pn_geom& g, const pn_ptrs& P, int chains, cudaStream_t st, int* launches) {
    const int nb = scan_blocks(g);
    const long long chunk = ((g.npad + nb - 1) / nb + SCAN_T - 1) / SCAN_T * SCAN_T;
    scan2* part = reinterpret_cast<scan2*>(P.slots);
    k_cscan_totals<<<nb, SCAN_T, 0, st>>>(g, P, chains, chunk, part);
    k_cscan_partials<<<1, SCAN_T, 0, st>>>(nb, part, P.st);
    *launches += 2;
    return cudaGetLastError();
}

// passes 3-4 (after pn_launch_compact_count, same scaled weights): numbering, table, zeroed q
cudaError_t pn_launch_compact_build(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, int chains,
                                    cudaStream_t st, int* launches) {
    const int nb = scan_blocks(g);
    const long long chunk = ((g.npad + nb - 1) / nb + SCAN_T - 1) / SCAN_T * SCAN_T;
    k_cscan_write<<<nb, SCAN_T, 0, st>>>(g, P, chains, chunk, reinterpret_cast<const scan2*>(P.slots), C.cidx, C.lat, C.c[2]);
    k_cfill<<<grid_for(m, g.sms), TPB, 0, st>>>(g, P, C, chains);
    *launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaMemsetAsync(C.q, 0, (size_t)m * 4, st);   // the weights' array becomes q (finite before its first use)
}

cudaError_t pn_launch_compact_gather(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, cudaStream_t st,
                                     int* launches) {
    k_cgather<<<grid_for(m, g.sms), TPB, 0, st>>>(P, C);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_compact_flush(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, cudaStream_t st,
                                    int* launches) {
    k_cflush<<<grid_for(m, g.sms), TPB, 0, st>>>(P, C);
    ++*launches;
    return cudaGetLastError();
}

// All iterations up to the next trigger in ONE cooperative launch (k_cpersist)
cudaError_t pn_launch_compact_persist(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, int max_launch_iters, cudaStream_t st) {
    int G = g.sms < PN_RESIDENT_MAX_CTAS ? g.sms : PN_RESIDENT_MAX_CTAS;
    cudaError_t e = cudaMemsetAsync(P.gbar, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    pn_ptrs PP = P;
    pn_cptrs CC = C;
    void* args[] = {(void*)&PP, (void*)&CC, (void*)&max_launch_iters};
    return cudaLaunchCooperativeKernel((const void*)k_cpersist, dim3(G), dim3(PT), args, 0, st);
}

// `iterations` iterations of the compact scheme: two launches each
cudaError_t pn_launch_compact_inner(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, int iterations, cudaStream_t st,
                                    int* launches, cudaEvent_t* ev) {
    int nb = g.sms * 8;
    if (nb > PN_MAX_BLOCKS) nb = PN_MAX_BLOCKS;
    if (ev) cudaEventRecord(ev[0], st);
    for (int it = 0; it < iterations; ++it) {
        k_cupdate<<<nb, TPB, 0, st>>>(P, C);
        if (ev) cudaEventRecord(ev[2 * it + 1], st);
        k_cspmv<<<nb, TPB, 0, st>>>(P, C);
        if (ev) cudaEventRecord(ev[2 * it + 2], st);
    }
    *launches += 2 * iterations;
    return cudaGetLastError();
}
