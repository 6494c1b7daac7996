// pn_chain.cuh -- chains of degree-2 nodes inside the spanning clusters (shared by pn_chain.cu and pn_compact.cu).
//
// A solved node with exactly two open bonds, both to solved nodes, only passes current on: eliminating it is exact
// (series resistors; the Schur complement of the Kirchhoff system), and its pressure is the resistance-weighted
// interpolation of the two nodes its chain ends at.  Near the percolation threshold 69 % of the unknowns left after
// dead-end peeling are such nodes (the "links" of the links-nodes-blobs picture; profiles/r02_compaction.md), and they
// are what makes CG slow there (critical slow-down).  Nothing about a chain is stored: whoever needs one
// walks it from an end through the solve copy of the conductances.
#pragma once
#include "pn_internal.cuh"

#define PN_CLASS_CHAIN 14       // internal: solved node eliminated as a link of a chain (exported as SOLVED)

struct pn_walk {
    long long end;              // the non-chain node the chain arrives at (== start for a loop)
    long long last;             // the chain node next to it
    double R;                   // sum of 1 / g over the chain's bonds, in walking order
    int steps;                  // chain nodes passed
};

// bond value between padded node n and its neighbour in direction code c (0:+x 1:-x 2:+y 3:-y 4:+z 5:-z), and that neighbour
__device__ __forceinline__ float pn_bond_dir(const pn_geom& g, const pn_ptrs& P, long long n, int c, long long* m) {
    const int b = c >> 1;
    const long long sb = b == 0 ? 1 : (b == 1 ? (long long)g.px : g.plane);
    if (c & 1) { *m = n - sb; return P.gs[b][n - sb]; }
    *m = n + sb;
    return P.gs[b][n];
}

// From the non-chain node `a`, along its bond in direction `c` (which leads to a chain node), to the other end.
__device__ __forceinline__ pn_walk pn_walk_chain(const pn_geom& g, const pn_ptrs& P, long long a, int c) {
    pn_walk w;
    long long prev = a, cur;
    const float g0 = pn_bond_dir(g, P, a, c, &cur);
    w.R = 1.0 / (double)g0;
    w.steps = 0;
    while (P.cls[cur] == PN_CLASS_CHAIN && w.steps < (1 << 30)) {
        long long nxt = -1;
        float gn = 0.f;
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            long long m;
            const float gv = pn_bond_dir(g, P, cur, d, &m);
            if (gv != 0.f && m != prev) { nxt = m; gn = gv; }
        }
        if (nxt < 0) break;      // cannot happen on a marked chain node (two open bonds)
        w.R += 1.0 / (double)gn;
        prev = cur;
        cur = nxt;
        ++w.steps;
    }
    w.end = cur;
    w.last = prev;
    return w;
}

// direction code at `end` of the bond back to `last` (to walk the same chain the other way round)
__device__ __forceinline__ int pn_dir_between(const pn_geom& g, long long from, long long to) {
    const long long d = to - from;
    if (d == 1) return 0;
    if (d == -1) return 1;
    if (g.ny > 1) {             // (2D lattices are held as nx x 1 x rows: the row stride is the z stride there)
        if (d == g.px) return 2;
        if (d == -(long long)g.px) return 3;
    }
    return d > 0 ? 4 : 5;
}

// Series resistance of the chain leaving `a` in direction `c`, summed in the order that starts at the end with the SMALLER
// index, so that both ends obtain bit-identical values (a symmetric reduced operator).  end == a: a loop (carries no current).
__device__ __forceinline__ pn_walk pn_chain_canonical(const pn_geom& g, const pn_ptrs& P, long long a, int c) {
    pn_walk w = pn_walk_chain(g, P, a, c);
    if (w.end < a) {
        const pn_walk back = pn_walk_chain(g, P, w.end, pn_dir_between(g, w.end, w.last));
        w.R = back.R;
    }
    return w;
}
