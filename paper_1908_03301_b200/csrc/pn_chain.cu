// pn_chain.cu -- exact elimination of the degree-2 "link" nodes of the spanning clusters (series resistors) before the
// inner iteration, and their back-fill (PN_OPT_CONTRACT; used together with the compacted unknowns, pn_compact.cu).
// See pn_chain.cuh.  The paper never says how it treats the near-threshold structure that makes its CG slow (P:111,
// P:132); SURVEY.md 8(c) reading 7 allows a solver to remove nodes it can back-fill exactly, so that the pressures of
// ALL nodes stay those of the full system -- the rule dead-end peeling already follows (degree 1; this is degree 2).
#include "pn_chain.cuh"

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

// A solved node with exactly two open bonds (after pruning and peeling), both to solved nodes, becomes a chain node.
// Neighbours are tested for "solved or already marked": marking is a monotone 2 -> 14 change, so the races are benign.
__global__ void k_chain_mark(pn_geom g, pn_ptrs P) {
    unsigned long long cnt = 0;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        if (P.cls[n] != PN_CLASS_SOLVED) continue;
        int deg = 0;
        bool ok = true;
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            long long m;
            if (pn_bond_dir(g, P, n, d, &m) != 0.f) {
                ++deg;
                const int c = P.cls[m];
                ok &= (c == PN_CLASS_SOLVED || c == PN_CLASS_CHAIN);
            }
        }
        if (deg == 2 && ok) { P.cls[n] = (signed char)PN_CLASS_CHAIN; ++cnt; }
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&P.st->n_chain, cnt);
}

__global__ void k_chain_unmark(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x)
        if (P.cls[n] == PN_CLASS_CHAIN) P.cls[n] = (signed char)PN_CLASS_SOLVED;
}

// Jacobi scale of the reduced system on the nodes that keep a chain as a neighbour: the chain's bond counts with its
// series conductance (a loop back to the node itself with nothing); chain nodes are no unknowns (s = 0).
__global__ void k_chain_scale(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const int c = P.cls[n];
        if (c == PN_CLASS_CHAIN) { P.s[n] = 0.f; continue; }
        if (c != PN_CLASS_SOLVED) continue;
        double d = 0.0;
        bool any = false;
#pragma unroll 1
        for (int dir = 0; dir < 6; ++dir) {
            long long m;
            const float gv = pn_bond_dir(g, P, n, dir, &m);
            if (gv == 0.f) continue;
            if (P.cls[m] == PN_CLASS_CHAIN) {
                any = true;
                const pn_walk w = pn_chain_canonical(g, P, n, dir);
                if (w.end != n) d += 1.0 / w.R;
            } else d += (double)gv;
        }
        if (any) P.s[n] = d > 0.0 ? (float)(1.0 / sqrt(d)) : 0.f;
    }
}

// Back-fill: every chain node takes the resistance-weighted interpolation of the pressures at the two ends of its chain
// (all nodes of a loop: the pressure of the node the loop hangs from).  One walk per chain, from its smaller end.
__global__ void k_chain_fill(pn_geom g, pn_ptrs P) {
    for (long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x; a < g.npad; a += (long long)gridDim.x * blockDim.x) {
        if (P.cls[a] != PN_CLASS_SOLVED) continue;
#pragma unroll 1
        for (int dir = 0; dir < 6; ++dir) {
            long long first;
            const float g0 = pn_bond_dir(g, P, a, dir, &first);
            if (g0 == 0.f || P.cls[first] != PN_CLASS_CHAIN) continue;
            const pn_walk w = pn_walk_chain(g, P, a, dir);
            if (w.end < a || (w.end == a && w.last < first)) continue;   // the other end (or the other way round the loop) does it
            const double xa = P.x64[a];
            const double slope = w.end == a ? 0.0 : (P.x64[w.end] - xa) / w.R;
            long long prev = a, cur = first;
            double R = 1.0 / (double)g0;
            while (P.cls[cur] == PN_CLASS_CHAIN) {
                P.x64[cur] = xa + slope * R;
                long long nxt = -1;
                float gn = 0.f;
#pragma unroll
                for (int d = 0; d < 6; ++d) {
                    long long m;
                    const float gv = pn_bond_dir(g, P, cur, d, &m);
                    if (gv != 0.f && m != prev) { nxt = m; gn = gv; }
                }
                if (nxt < 0) break;
                R += 1.0 / (double)gn;
                prev = cur;
                cur = nxt;
            }
        }
    }
}

// The same walk, once per solve: instead of pressures it leaves one record per chain node -- (node, a, b, t) with
// t = R(a -> node) / R(a -> b) -- so that every later back-fill is a flat gather (k_chain_fill_rec) instead of 3.9 M
// dependent-load walks (configs[2]: 1.8 ms per walk-based fill, ~20 of them per solve, against 0.05 ms).  Record slots
// are handed out by an atomic counter: their order varies from run to run, what each holds does not.
__global__ void k_chain_record(pn_geom g, pn_ptrs P, pn_cptrs C) {
    for (long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x; a < g.npad; a += (long long)gridDim.x * blockDim.x) {
        if (P.cls[a] != PN_CLASS_SOLVED) continue;
#pragma unroll 1
        for (int dir = 0; dir < 6; ++dir) {
            long long first;
            const float g0 = pn_bond_dir(g, P, a, dir, &first);
            if (g0 == 0.f || P.cls[first] != PN_CLASS_CHAIN) continue;
            const pn_walk w = pn_walk_chain(g, P, a, dir);
            if (w.end < a || (w.end == a && w.last < first)) continue;   // the other end (or the other way round the loop) does it
            const double inv = w.end == a ? 0.0 : 1.0 / w.R;
            long long prev = a, cur = first;
            double R = 1.0 / (double)g0;
            while (P.cls[cur] == PN_CLASS_CHAIN) {
                const unsigned long long slot = atomicAdd(&P.st->n_rec, 1ull);
                if ((long long)slot < C.chcap) {
                    C.chv[slot] = (int)cur;
                    C.chab[slot] = make_int2((int)a, (int)w.end);
                    C.cht[slot] = R * inv;
                }
                long long nxt = -1;
                float gn = 0.f;
#pragma unroll
                for (int d = 0; d < 6; ++d) {
                    long long m;
                    const float gv = pn_bond_dir(g, P, cur, d, &m);
                    if (gv != 0.f && m != prev) { nxt = m; gn = gv; }
                }
                if (nxt < 0) break;
                R += 1.0 / (double)gn;
                prev = cur;
                cur = nxt;
            }
        }
    }
}

__global__ void k_chain_fill_rec(pn_ptrs P, pn_cptrs C, long long n) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        const int2 ab = C.chab[j];
        const double xa = P.x64[ab.x];
        P.x64[C.chv[j]] = xa + C.cht[j] * (P.x64[ab.y] - xa);
    }
}

}  // namespace

cudaError_t pn_launch_chain_record(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, cudaStream_t st, int* launches) {
    cudaError_t e = cudaMemsetAsync(&P.st->n_rec, 0, sizeof(P.st->n_rec), st);
    if (e != cudaSuccess) return e;
    k_chain_record<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P, C);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_chain_fill_rec(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long n_chain, cudaStream_t st,
                                     int* launches) {
    k_chain_fill_rec<<<grid_for(n_chain, g.sms), TPB, 0, st>>>(P, C, n_chain);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_chain_mark(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_chain_mark<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_chain_unmark(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_chain_unmark<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_chain_scale(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_chain_scale<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_chain_fill(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_chain_fill<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
