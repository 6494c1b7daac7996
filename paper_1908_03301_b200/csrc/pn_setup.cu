// pn_setup.cu -- S0 validation and S1 "classify & prune", plus the per-direction
// set-up of the scaled inner system.  Integer / fp64 work done once per solve; not the hot loop.
//
// S1 is not in the paper (it never says how isolated clusters are handled, P:111, P:132 only note the
// critical slow-down); BASELINE.json's north_star mandates it: "Dead-end and isolated clusters ... are
// removed before the solve by a connectivity labelling pass, and their rows are pinned."  Classes
// follow SURVEY.md 8(c) steps 2-3.  The labelling is a lock-free union-find over the interior nodes
// (hook the larger root under the smaller with atomicCAS, path halving on find); the oracle uses a
// serial BFS, so the two share nothing but the definition of a component.
#include "pn_chain.cuh"

namespace {

constexpr int TPB = 256;

__host__ __device__ inline long long cdiv(long long a, long long b) { return (a + b - 1) / b; }

int grid_for(long long work_items, int sms) {
    long long nb = cdiv(work_items, TPB);
    long long cap = (long long)sms * 8;
    if (cap > PN_MAX_BLOCKS) cap = PN_MAX_BLOCKS;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    return (int)nb;
}

// ---- S0: every in-lattice bond finite and >= 0; note whether any is closed ----------------------
__global__ void k_validate(pn_geom g, const float* __restrict__ r0, const float* __restrict__ r1,
                           const float* __restrict__ r2, pn_state* st) {
    int bad = 0, closed = 0;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.n; n += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(n % g.nx), j = (int)((n / g.nx) % g.ny), k = (int)(n / ((long long)g.nx * g.ny));
        if (i + 1 < g.nx) { const float v = r0[n]; bad |= !(v >= 0.0f) || isinf(v); closed |= (v == 0.0f); }
        if (r1 && j + 1 < g.ny) { const float v = r1[n]; bad |= !(v >= 0.0f) || isinf(v); closed |= (v == 0.0f); }
        if (r2 && k + 1 < g.nz) { const float v = r2[n]; bad |= !(v >= 0.0f) || isinf(v); closed |= (v == 0.0f); }
    }
    bad = __syncthreads_or(bad);
    closed = __syncthreads_or(closed);
    if (threadIdx.x == 0) {
        if (bad) atomicOr(&st->bad_value, 1);
        if (closed) atomicOr(&st->any_closed, 1);
    }
}

// ---- S8(f) item 4: conductances that change between solves ("thousands of time steps") ----------------------
// Sparse form: bond (axis[i], node[i]) of the CALLER's lattice (forward-bond convention) takes value[i].  Entries must be
// distinct.  2D lattices: caller axis 1 is the internal z-bond array (raw[2]).
__global__ void k_update_raw(int unx, int uny, int unz, float* r0, float* r1, float* r2, long long count,
                             const int* __restrict__ axis, const long long* __restrict__ node,
                             const float* __restrict__ value, pn_state* st) {
    const long long N = (long long)unx * uny * unz;
    const bool is2d = unz == 1;
    int bad = 0, closed = 0, topo = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < count; t += (long long)gridDim.x * blockDim.x) {
        const int a = axis[t];
        const long long n = node[t];
        if (a < 0 || a > (is2d ? 1 : 2) || n < 0 || n >= N) { bad |= 2; continue; }
        const float v = value[t];
        if (!(v >= 0.0f) || isinf(v)) { bad |= 1; continue; }
        float* arr = a == 0 ? r0 : (is2d ? r2 : (a == 1 ? r1 : r2));
        const float old = arr[n];
        topo |= (old == 0.0f) != (v == 0.0f);
        closed |= (v == 0.0f);
        arr[n] = v;
    }
    bad = __syncthreads_or(bad & 1) | (__syncthreads_or(bad & 2) ? 2 : 0);
    closed = __syncthreads_or(closed);
    topo = __syncthreads_or(topo);
    if (threadIdx.x == 0) {
        if (bad) atomicOr(&st->bad_value, bad);
        if (closed) atomicOr(&st->any_closed, 1);
        if (topo) atomicOr(&st->topo_changed, 1);
    }
}

// Full form, one array at a time: raw <- src with S0's validation of the in-lattice bonds (which entries are bonds
// depends on the INTERNAL axis b of this array) and the zero-crossing note.
__global__ void k_replace_raw(pn_geom g, float* __restrict__ raw, const float* __restrict__ src, int b, pn_state* st) {
    int bad = 0, closed = 0, topo = 0;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.n; n += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(n % g.nx), j = (int)((n / g.nx) % g.ny), k = (int)(n / ((long long)g.nx * g.ny));
        const float v = src[n], old = raw[n];
        const bool bond = b == 0 ? i + 1 < g.nx : (b == 1 ? j + 1 < g.ny : k + 1 < g.nz);
        if (bond) { bad |= !(v >= 0.0f) || isinf(v); closed |= (v == 0.0f); }
        // entries that are not bonds without periodic faces may become bonds with them: their crossings count too
        topo |= (old == 0.0f) != (v == 0.0f);
        raw[n] = v;
    }
    bad = __syncthreads_or(bad);
    closed = __syncthreads_or(closed);
    topo = __syncthreads_or(topo);
    if (threadIdx.x == 0) {
        if (bad) atomicOr(&st->bad_value, 1);
        if (closed) atomicOr(&st->any_closed, 1);
        if (topo) atomicOr(&st->topo_changed, 1);
    }
}

struct coords { int i, j, k; };
__device__ __forceinline__ coords coords_of(const pn_geom& g, long long n) {
    coords c;
    c.i = (int)(n % g.px);
    c.j = (int)((n / g.px) % g.ny);
    c.k = (int)(n / g.plane);
    return c;
}
__device__ __forceinline__ int along(const pn_geom& g, const coords& c) { return g.dir == 0 ? c.i : (g.dir == 1 ? c.j : c.k); }

// Neighbour of padded node n along axis b (side 0: forward, 1: backward) and the storage of the bond between
// them in the SOLVE COPY: the lattice-shaped array, or the face array when the step crosses a wrapping face
// (periodic lateral faces).  A step off a face that does not wrap lands on a pad / halo entry whose
// bond is 0, as everywhere in this layout.
struct pn_nb { long long m; float* slot; };
__device__ __forceinline__ pn_nb pn_nbr(const pn_geom& g, const pn_ptrs& P, long long n, const coords& c, int b, int side) {
    const long long sb = b == 0 ? 1 : (b == 1 ? (long long)g.px : g.plane);
    pn_nb r;
    if (g.wrap[b]) {
        const int cb = b == 0 ? c.i : (b == 1 ? c.j : c.k), db = b == 0 ? g.nx : (b == 1 ? g.ny : g.nz);
        if ((side == 0 && cb == db - 1) || (side == 1 && cb == 0)) {
            r.slot = P.gsw[b] + pn_face_index(g, b, c.i, c.j, c.k);
            r.m = side == 0 ? n - pn_wrap_span(g, b) : n + pn_wrap_span(g, b);
            return r;
        }
    }
    r.m = side == 0 ? n + sb : n - sb;
    r.slot = P.gs[b] + (side == 0 ? n : n - sb);
    return r;
}
__device__ __forceinline__ bool any_wrap(const pn_geom& g) { return g.wrap[0] | g.wrap[1] | g.wrap[2]; }

// ---- S1a: solve copy of g in the padded layout; union-find forest initialised -------------------
// Off-lattice forward entries and pad columns -> 0.  Bonds lying INSIDE a Dirichlet plane (both ends
// at the same fixed pressure, no current) -> 0.
__global__ void k_solve_copy(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const coords c = coords_of(g, n);
        float v[3] = {0.f, 0.f, 0.f};
        if (c.i < g.nx) {
            const long long nu = c.i + (long long)g.nx * (c.j + (long long)g.ny * c.k);
            const int ca = along(g, c);
            const bool dirichlet = (ca == 0) || (ca == g.n_a - 1);
            const bool in0 = c.i + 1 < g.nx, in1 = c.j + 1 < g.ny, in2 = c.k + 1 < g.nz;
            if (in0 && !(dirichlet && g.dir != 0)) v[0] = P.raw[0][nu];
            if (in1 && P.raw[1] && !(dirichlet && g.dir != 1)) v[1] = P.raw[1][nu];
            if (in2 && P.raw[2] && !(dirichlet && g.dir != 2)) v[2] = P.raw[2][nu];
        }
        P.gs[0][n] = v[0];
        P.gs[1][n] = v[1];
        P.gs[2][n] = v[2];
        P.parent[n] = (int)n;
        P.flags[n] = 0;
    }
}

// ---- periodic lateral faces: solve copy of the wrap bonds (face arrays) --------------------------------
// gsw[b][f] = the caller's forward entry of the LAST node along b (the bond back to the first node); 0 on pad
// columns and when both ends lie in a Dirichlet plane (no current, as for the in-plane bonds above).
__global__ void k_wrap_copy(pn_geom g, pn_ptrs P) {
    for (int b = 0; b < 3; ++b) {
        if (!g.wrap[b]) { continue; }
        const long long nf = pn_face_count(g, b);
        for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
            coords c;   // the hi node of this face entry
            if (b == 0) { c.i = g.nx - 1; c.j = (int)(f % g.ny); c.k = (int)(f / g.ny); }
            else if (b == 1) { c.i = (int)(f % g.px); c.j = g.ny - 1; c.k = (int)(f / g.px); }
            else { c.i = (int)(f % g.px); c.j = (int)(f / g.px); c.k = g.nz - 1; }
            float v = 0.f;
            const int ca = along(g, c);
            if (c.i < g.nx && P.raw[b]) {
                // with a wrapping axis this entry IS a bond: same validation as k_validate (S0), done here because
                // which axes wrap is known only once the solve direction is
                v = P.raw[b][c.i + (long long)g.nx * (c.j + (long long)g.ny * c.k)];
                if (!(v >= 0.0f) || isinf(v)) atomicOr(&P.st->bad_value, 1);
                if (v == 0.0f) atomicOr(&P.st->any_closed, 1);
                if (ca == 0 || ca == g.n_a - 1) v = 0.f;
            }
            P.gsw[b][f] = v;
        }
    }
}

// unite the two ends of every open wrap bond (both are interior: Dirichlet-plane entries were zeroed)
__global__ void k_wrap_union(pn_geom g, pn_ptrs P);

// ---- union-find primitives (parent[] read at L2: another SM may have just re-hooked a root) -----
__device__ __forceinline__ int uf_find(int* parent, int x) {
    int p = __ldcg(parent + x);
    while (p != x) {
        const int gp = __ldcg(parent + p);
        if (gp != p) parent[x] = gp;  // path halving; benign race: gp is an ancestor of x
        x = p;
        p = gp;
    }
    return x;
}
__device__ __forceinline__ void uf_union(int* parent, int a, int b) {
    while (true) {
        a = uf_find(parent, a);
        b = uf_find(parent, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }
        const int old = atomicCAS(parent + a, a, b);  // hook the larger root under the smaller
        if (old == a) return;
        a = old;  // a stopped being a root meanwhile: carry on from its new parent
    }
}

__global__ void k_wrap_union(pn_geom g, pn_ptrs P) {
    for (int b = 0; b < 3; ++b) {
        if (!g.wrap[b]) { continue; }
        const long long nf = pn_face_count(g, b), span = pn_wrap_span(g, b);
        for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
            if (!(P.gsw[b][f] > 0.f)) continue;
            const long long lo = b == 0 ? (f % g.ny) * (long long)g.px + (f / g.ny) * g.plane
                                        : (b == 1 ? (f % g.px) + (f / g.px) * g.plane : f);
            uf_union(P.parent, (int)lo, (int)(lo + span));
        }
    }
}

// prune the wrap bonds: zero every one that has a pinned end
__global__ void k_wrap_prune(pn_geom g, pn_ptrs P) {
    for (int b = 0; b < 3; ++b) {
        if (!g.wrap[b]) { continue; }
        const long long nf = pn_face_count(g, b), span = pn_wrap_span(g, b);
        for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
            if (P.gsw[b][f] == 0.f) continue;
            const long long lo = b == 0 ? (f % g.ny) * (long long)g.px + (f / g.ny) * g.plane
                                        : (b == 1 ? (f % g.px) + (f / g.px) * g.plane : f);
            if (!(P.cls[lo] <= PN_CLASS_SOLVED && P.cls[lo + span] <= PN_CLASS_SOLVED)) P.gsw[b][f] = 0.f;
        }
    }
}

// scaled weights of the wrap bonds: ww = g s_lo s_hi (fp64 product, rounded once), as k_weights
__global__ void k_wrap_weights(pn_geom g, pn_ptrs P) {
    for (int b = 0; b < 3; ++b) {
        if (!g.wrap[b]) { continue; }
        const long long nf = pn_face_count(g, b), span = pn_wrap_span(g, b);
        for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
            const long long lo = b == 0 ? (f % g.ny) * (long long)g.px + (f / g.ny) * g.plane
                                        : (b == 1 ? (f % g.px) + (f / g.px) * g.plane : f);
            const double v = (double)P.gsw[b][f];
            P.ww[b][f] = v != 0.0 ? (float)(v * (double)P.s[lo] * (double)P.s[lo + span]) : 0.f;
        }
    }
}

// ---- S1b: unite interior nodes joined by an open bond -------------------------------------------
__global__ void k_union(pn_geom g, pn_ptrs P) {
    const long long stride[3] = {1, g.px, g.plane};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const coords c = coords_of(g, n);
        if (c.i >= g.nx) continue;
        const int ca = along(g, c);
        if (ca == 0 || ca == g.n_a - 1) continue;  // Dirichlet nodes are not part of any cluster
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            if (!(P.gs[b][n] > 0.f)) continue;
            if (b == g.dir && ca + 1 == g.n_a - 1) continue;  // forward neighbour is an outlet node
            uf_union(P.parent, (int)n, (int)(n + stride[b]));
        }
    }
}

// ---- S1c: which clusters touch the inlet / outlet plane through an open bond --------------------
__global__ void k_touch(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const coords c = coords_of(g, n);
        if (c.i >= g.nx) continue;
        const int ca = along(g, c);
        if (ca == 0 || ca == g.n_a - 1) continue;
        const int root = uf_find(P.parent, (int)n);
        P.parent[n] = root;
        int t = 0;
        if (ca == 1 && P.gs[g.dir][n - g.stride_a] > 0.f) t |= 1;          // open bond to the inlet plane
        if (ca == g.n_a - 2 && P.gs[g.dir][n] > 0.f) t |= 2;               // open bond to the outlet plane
        if (t) atomicOr(P.flags + root, t);
    }
}

// ---- S1d: node classes, class counts, pin values and the initial guess --------------------------
// x0_linear: 0 = zero, 1 = linear profile along the solve axis, 2 = warm start (keep what x64 holds on the
// solved nodes: the previous solve's pressures)
template <bool LABEL>
__global__ void k_classify(pn_geom g, pn_ptrs P, int x0_linear) {
    unsigned long long cnt[4] = {0, 0, 0, 0};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const coords c = coords_of(g, n);
        int cls = PN_CLASS_PAD;
        double x = 0.0;
        if (c.i < g.nx) {
            const int ca = along(g, c);
            if (ca == 0) { cls = PN_CLASS_INLET; x = 1.0; }
            else if (ca == g.n_a - 1) { cls = PN_CLASS_OUTLET; }
            else {
                int f = 3;
                if (LABEL) f = __ldcg(P.flags + uf_find(P.parent, (int)n));
                if (f == 3) { cls = PN_CLASS_SOLVED; const double lin = 1.0 - (double)ca / (double)(g.n_a - 1);
                    x = x0_linear ? lin : 0.0;
                    if (x0_linear == 2) { const double old = P.x64[n]; if (isfinite(old)) x = old; }
                    cnt[0]++; }
                else if (f == 1) { cls = PN_CLASS_INLET_ONLY; x = 1.0; cnt[1]++; }
                else if (f == 2) { cls = PN_CLASS_OUTLET_ONLY; cnt[2]++; }
                else { cls = PN_CLASS_FLOATING; cnt[3]++; }
            }
        }
        P.cls[n] = (signed char)cls;
        P.x64[n] = x;
    }
    __shared__ unsigned long long sc[4];
    if (threadIdx.x < 4) sc[threadIdx.x] = 0;
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        unsigned long long v = cnt[q];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sc[q], v);
    }
    __syncthreads();
    if (threadIdx.x < 4 && sc[threadIdx.x]) atomicAdd(&P.st->count[threadIdx.x], sc[threadIdx.x]);
}

// Label reuse with PN_OPT_X0 = 0 / 1: the solved nodes (peeled ones included) go back to the zero / linear start
__global__ void k_reset_x0(pn_geom g, pn_ptrs P, int x0_linear) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const int c = P.cls[n];
        if (c == PN_CLASS_SOLVED || c >= PN_CLASS_PEELED) {
            const coords cc = coords_of(g, n);
            P.x64[n] = x0_linear ? 1.0 - (double)along(g, cc) / (double)(g.n_a - 1) : 0.0;
        }
    }
}

// ---- S1e: prune -- zero every bond that has a pinned end (pinned rows get a zero diagonal) ------
__global__ void k_prune(pn_geom g, pn_ptrs P) {
    const long long stride[3] = {1, g.px, g.plane};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const int c0 = P.cls[n];
        const bool keep0 = c0 <= PN_CLASS_SOLVED || c0 == PN_CLASS_CHAIN;   // (chain nodes: label reuse; they keep their bonds)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float v = P.gs[b][n];
            if (v == 0.f) continue;
            // v != 0 implies the forward neighbour is a real node (off-lattice entries were zeroed)
            const int c1 = P.cls[n + stride[b]];
            const bool keep1 = c1 <= PN_CLASS_SOLVED || c1 == PN_CLASS_CHAIN;
            if (!(keep0 && keep1)) P.gs[b][n] = 0.f;
        }
    }
}

// ---- S1f: dead-end (leaf) peeling inside the spanning clusters (SURVEY.md 8(f) item 1, 8(c) reading 7) ----
// A solved node with a single open bond carries no current: its pressure equals that of the node it hangs
// from, and so on up the dangling tree.  Such nodes are taken out of the linear system (their bond is
// zeroed in the solve copy, so the neighbour's diagonal no longer counts it) and back-filled after the
// solve (k_backfill), which keeps the pressures of ALL nodes those of the full system.  Near the
// percolation threshold about half of a spanning cluster is dangling ends; removing them is what shortens
// the critical slow-down -- fewer unknowns and a better-conditioned operator.
// Asynchronous peeling: live bond degrees in an int array; a thread that removes a leaf decrements the
// neighbour's degree and, if that made the neighbour a leaf, carries on with it (no rounds, so a long
// dangling chain costs one walk, not one launch per node).  A node is claimed with atomicCAS(deg, 1, 0).
__global__ void k_degree(pn_geom g, pn_ptrs P) {
    int* __restrict__ deg = P.flags;
    const bool wrap = any_wrap(g);
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        int d = 0;
        if (P.cls[n] == PN_CLASS_SOLVED) {
            if (!wrap) {
                d = (P.gs[0][n] != 0.f) + (P.gs[0][n - 1] != 0.f) + (P.gs[1][n] != 0.f) + (P.gs[1][n - g.px] != 0.f) +
                    (P.gs[2][n] != 0.f) + (P.gs[2][n - g.plane] != 0.f);
            } else {
                const coords c = coords_of(g, n);
                for (int b = 0; b < 3; ++b)
                    for (int side = 0; side < 2; ++side) d += (*pn_nbr(g, P, n, c, b, side).slot != 0.f);
            }
        }
        deg[n] = d;
    }
}

__global__ void k_peel(pn_geom g, pn_ptrs P) {
    int* deg = P.flags;
    unsigned long long cnt = 0;
    for (long long n0 = blockIdx.x * (long long)blockDim.x + threadIdx.x; n0 < g.npad; n0 += (long long)gridDim.x * blockDim.x) {
        long long n = n0;
        while (__ldcg(deg + n) == 1 && atomicCAS(deg + n, 1, 0) == 1) {
            // the one bond left (bonds zeroed by other threads are read at L2: their stores were fenced
            // before the degree decrement that made this node a leaf)
            const coords c = coords_of(g, n);
            int code = -1;
            pn_nb hit;
            hit.m = -1; hit.slot = nullptr;
            for (int b = 0; b < 3; ++b)
                for (int side = 0; side < 2; ++side) {
                    const pn_nb nb = pn_nbr(g, P, n, c, b, side);
                    if (__ldcg(nb.slot) != 0.f) { code = 2 * b + side; hit = nb; }
                }
            if (code < 0) break;
            if (P.cls[hit.m] != PN_CLASS_SOLVED) { deg[n] = 1; break; }   // hangs from a Dirichlet node: not a dead end
            P.cls[n] = (signed char)(PN_CLASS_PEELED + code);
            __stcg(hit.slot, 0.f);
            __threadfence();
            ++cnt;
            if (atomicSub(deg + hit.m, 1) != 2) break;                   // the neighbour did not become a leaf
            n = hit.m;
        }
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&P.st->n_peeled, cnt);
}

// Undo a peeling that removed too few nodes to pay (PN_OPT_PEEL = 2, see pn_api.cu): put every peeled node back
// as an unknown and restore its bond from the caller's conductances.
__global__ void k_unpeel(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const int c = P.cls[n];
        if (c < PN_CLASS_PEELED || c >= PN_CLASS_CHAIN) continue;
        const int code = c - PN_CLASS_PEELED, b = code >> 1, side = code & 1;
        const pn_nb nb = pn_nbr(g, P, n, coords_of(g, n), b, side);
        const coords cc = coords_of(g, side == 0 ? n : nb.m);      // the node whose FORWARD entry this bond is
        *nb.slot = P.raw[b][cc.i + (long long)g.nx * (cc.j + (long long)g.ny * cc.k)];
        P.cls[n] = PN_CLASS_SOLVED;
    }
}

// After the solve: every peeled node takes the pressure of the unpeeled node its dangling tree hangs from.
__global__ void k_backfill(pn_geom g, pn_ptrs P) {
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        int c = P.cls[n];
        if (c < PN_CLASS_PEELED || c >= PN_CLASS_CHAIN) continue;
        long long m = n;
        for (long long guard = 0; c >= PN_CLASS_PEELED && c < PN_CLASS_CHAIN && guard < g.npad; ++guard) {
            const int code = c - PN_CLASS_PEELED;
            m = pn_nbr(g, P, m, coords_of(g, m), code >> 1, code & 1).m;
            c = P.cls[m];
        }
        P.x64[n] = P.x64[m];
    }
}

// ---- diagonal (on the fly, fp64) -> symmetric Jacobi scale s = 1/sqrt(diag); ||b||^2 -----------
// b_i = sum over inlet-plane neighbours of g_ij * 1 ("b is a vector related to the external
// boundary conditions"); only nodes on the plane coord_a = 1 have one.
__global__ void k_scale(pn_geom g, pn_ptrs P) {
    __shared__ double sm[32];
    __shared__ double tot[1];
    double bb = 0.0;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        float s = 0.f;
        if (P.cls[n] == PN_CLASS_SOLVED) {
            const coords c = coords_of(g, n);
            double d = (double)P.gs[0][n] + (double)P.gs[0][n - 1] + (double)P.gs[1][n] + (double)P.gs[1][n - g.px] +
                       (double)P.gs[2][n] + (double)P.gs[2][n - g.plane];
            for (int b = 0; b < 3; ++b) {   // wrap bonds of a node on a periodic face (the lattice arrays hold 0 there)
                if (!g.wrap[b]) continue;
                const int cb = b == 0 ? c.i : (b == 1 ? c.j : c.k), db = b == 0 ? g.nx : (b == 1 ? g.ny : g.nz);
                if (cb == 0 || cb == db - 1) d += (double)P.gsw[b][pn_face_index(g, b, c.i, c.j, c.k)];
            }
            s = d > 0.0 ? (float)(1.0 / sqrt(d)) : 0.f;
            if (along(g, c) == 1) { const double b = (double)P.gs[g.dir][n - g.stride_a]; bb += b * b; }
        }
        P.s[n] = s;
    }
    bb = pn_block_sum(bb, sm);
    const double v[1] = {bb};
    if (pn_grid_sum<1>(v, P.slots, &P.st->ticket, sm, tot)) {
        if (threadIdx.x == 0) P.st->acc[2] = tot[0];
    }
}

// ---- scaled bond weights of the inner system: w_ij = g_ij s_i s_j (fp64 product, rounded once) --
__global__ void k_weights(pn_geom g, pn_ptrs P) {
    const long long stride[3] = {1, g.px, g.plane};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < g.npad; n += (long long)gridDim.x * blockDim.x) {
        const double s0 = (double)P.s[n];
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const double v = (double)P.gs[b][n];
            float w = 0.f;
            if (v != 0.0 && s0 != 0.0) w = (float)(v * s0 * (double)P.s[n + stride[b]]);
            P.w[b][n] = w;
        }
    }
}

}  // namespace

cudaError_t pn_launch_validate(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_validate<<<grid_for(g.n, g.sms), TPB, 0, st>>>(g, P.raw[0], P.raw[1], P.raw[2], P.st);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_label(const pn_geom& g, const pn_ptrs& P, bool do_label, bool do_peel, int x0_linear,
                            cudaStream_t st, int* launches) {
    const int nb = grid_for(g.npad, g.sms);
    const bool wrap = g.wrap[0] || g.wrap[1] || g.wrap[2];
    long long nface = 1;
    for (int b = 0; b < 3; ++b) if (g.wrap[b] && pn_face_count(g, b) > nface) nface = pn_face_count(g, b);
    const int nbf = grid_for(nface, g.sms);
    k_solve_copy<<<nb, TPB, 0, st>>>(g, P);
    ++*launches;
    if (do_label) {
        k_union<<<nb, TPB, 0, st>>>(g, P);
        if (wrap) { k_wrap_union<<<nbf, TPB, 0, st>>>(g, P); ++*launches; }
        k_touch<<<nb, TPB, 0, st>>>(g, P);
        k_classify<true><<<nb, TPB, 0, st>>>(g, P, x0_linear);
        k_prune<<<nb, TPB, 0, st>>>(g, P);
        if (wrap) { k_wrap_prune<<<nbf, TPB, 0, st>>>(g, P); ++*launches; }
        *launches += 4;
        if (do_peel) {
            k_degree<<<nb, TPB, 0, st>>>(g, P);
            k_peel<<<nb, TPB, 0, st>>>(g, P);
            *launches += 2;
        }
    } else {
        k_classify<false><<<nb, TPB, 0, st>>>(g, P, x0_linear);
        ++*launches;
    }
    return cudaGetLastError();
}

// S1 when no bond crossed zero since the classes were computed (same direction and options): the classes -- and with them
// the pins, the peeled set and the counts -- stand; only the values of the solve copy change.  A bond survives iff both
// ends are Dirichlet or solved nodes (k_prune's rule; peeled nodes have class codes above SOLVED, so their one bond goes).
cudaError_t pn_launch_label_reuse(const pn_geom& g, const pn_ptrs& P, int x0_mode, cudaStream_t st, int* launches) {
    const int nb = grid_for(g.npad, g.sms);
    k_solve_copy<<<nb, TPB, 0, st>>>(g, P);
    k_prune<<<nb, TPB, 0, st>>>(g, P);
    *launches += 2;
    if (g.wrap[0] || g.wrap[1] || g.wrap[2]) {
        long long nface = 1;
        for (int b = 0; b < 3; ++b) if (g.wrap[b] && pn_face_count(g, b) > nface) nface = pn_face_count(g, b);
        k_wrap_prune<<<grid_for(nface, g.sms), TPB, 0, st>>>(g, P);
        ++*launches;
    }
    if (x0_mode != 2) { k_reset_x0<<<nb, TPB, 0, st>>>(g, P, x0_mode); ++*launches; }
    return cudaGetLastError();
}

cudaError_t pn_launch_update_raw(int unx, int uny, int unz, const pn_ptrs& P, float* const raw[3], long long count,
                                 const int* axis, const long long* node, const float* value, int sms, cudaStream_t st,
                                 int* launches) {
    k_update_raw<<<grid_for(count, sms), TPB, 0, st>>>(unx, uny, unz, raw[0], raw[1], raw[2], count, axis, node, value, P.st);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_replace_raw(const pn_geom& g, float* raw, const float* src, int axis_internal, pn_state* state,
                                  cudaStream_t st, int* launches) {
    k_replace_raw<<<grid_for(g.n, g.sms), TPB, 0, st>>>(g, raw, src, axis_internal, state);
    ++*launches;
    return cudaGetLastError();
}

// Diagonal scale, ||b||^2 and the scaled weights of the inner system, from the final solve copy.
cudaError_t pn_launch_scale(const pn_geom& g, const pn_ptrs& P, int chains, cudaStream_t st, int* launches) {
    const int nb = grid_for(g.npad, g.sms);
    k_scale<<<nb, TPB, 0, st>>>(g, P);
    if (chains) {   // the nodes next to a chain take the reduced system's diagonal before the weights are formed
        cudaError_t e = pn_launch_chain_scale(g, P, st, launches);
        if (e != cudaSuccess) return e;
    }
    k_weights<<<nb, TPB, 0, st>>>(g, P);
    *launches += 2;
    if (g.wrap[0] || g.wrap[1] || g.wrap[2]) {
        long long nface = 1;
        for (int b = 0; b < 3; ++b) if (g.wrap[b] && pn_face_count(g, b) > nface) nface = pn_face_count(g, b);
        k_wrap_weights<<<grid_for(nface, g.sms), TPB, 0, st>>>(g, P);
        ++*launches;
    }
    return cudaGetLastError();
}

cudaError_t pn_launch_backfill(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_backfill<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_unpeel(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    k_unpeel<<<grid_for(g.npad, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}

// Periodic lateral faces: solve copy of the wrap bonds + their validation (sets state.bad_value / any_closed).
// Runs before pn_launch_label so that the host can read the two flags first.
cudaError_t pn_launch_wrap_copy(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches) {
    long long nface = 1;
    for (int b = 0; b < 3; ++b) if (g.wrap[b] && pn_face_count(g, b) > nface) nface = pn_face_count(g, b);
    k_wrap_copy<<<grid_for(nface, g.sms), TPB, 0, st>>>(g, P);
    ++*launches;
    return cudaGetLastError();
}
