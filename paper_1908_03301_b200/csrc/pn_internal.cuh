// pn_internal.cuh -- shared declarations of the libpn CUDA sources (not part of the C ABI).
//
// Internal lattice layout:
//   every lattice-shaped device array is stored x-fastest with a padded row pitch `px`
//   (px = nx rounded up to 4 floats, so every row starts 16-byte aligned), plane stride
//   `plane = px*ny`, `npad = plane*nz` elements, plus ONE zero plane before element 0 and one after
//   element npad-1.  Pad columns (i >= nx) and the two halo planes hold zeros in every array, and
//   forward-bond entries whose neighbour is off-lattice are zero, so the 7-point operator can be
//   written on flat indices (n-1, n+1, n-px, n+px, n-plane, n+plane) with no coordinate tests:
//   a neighbour that does not exist is always multiplied by a zero bond weight and is always finite.
//   A 2D lattice nx x ny is held as the 3D lattice nx x 1 x ny (identical node order), so there is
//   one code path: user gy plays the role of internal gz and the internal y-bond array is all zero.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pn.h"

#define PN_MAX_BLOCKS 2048      // upper bound on gridDim.x of every reducing kernel (partial slots)
#define PN_RESIDENT_MAX_CTAS 160 // upper bound on the cooperative grid of k_cg_resident2d (sizes its exchange array)
#define PN_CLASS_PAD 7          // internal: pad column (never exported)
#define PN_CLASS_PEELED 8       // internal: 8 + c = solved node peeled off as a dangling end, hanging from its
                                // neighbour in direction c (0:+x 1:-x 2:+y 3:-y 4:+z 5:-z); exported as SOLVED

struct pn_geom {
    int nx, ny, nz;             // INTERNAL lattice dims (2D user lattices: ny = 1, nz = user ny)
    int px;                     // padded row pitch in elements (multiple of 4)
    long long plane;            // px * ny
    long long npad;             // plane * nz
    long long n;                // nx * ny * nz (real nodes)
    int dir;                    // INTERNAL solve axis 0/1/2
    int n_a;                    // lattice length along dir
    long long stride_a;         // element stride along dir (1, px, plane)
    int wrap[3];                // INTERNAL axis wraps around (periodic lateral faces); never `dir`, never a length-1 axis
    int sms;                    // SM count of the handle's device (sizes the persistent grids); set by pn_create
    int coop;                   // the device launches cooperative kernels (pn_resident.cu)
    int tile;                   // PN_OPT_TILE: 3D tile of the fused TMA kernel (0 automatic, 1: 256 x 8, 2: 128 x 16, 3: 64 x 32)
};

// ---- periodic lateral faces: the wrap bonds live in small FACE arrays, not in the lattice-shaped ones ----
// (the flat-index stencil of the lattice arrays knows nothing about them; k_wrap_fix adds their part of q).
// Face of axis b = the nodes with coordinate 0 along b, indexed  b=0: j + ny*k,  b=1: i + px*k,  b=2: i + px*j.
// Entry f of a face array = the bond between the node at coordinate dims[b]-1 ("hi") and the node at 0 ("lo").
__host__ __device__ inline long long pn_face_count(const pn_geom& g, int b) {
    return b == 0 ? (long long)g.ny * g.nz : (b == 1 ? (long long)g.px * g.nz : g.plane);
}
__host__ __device__ inline long long pn_face_index(const pn_geom& g, int b, int i, int j, int k) {
    return b == 0 ? j + (long long)g.ny * k : (b == 1 ? i + (long long)g.px * k : i + (long long)g.px * j);
}
__host__ __device__ inline long long pn_wrap_span(const pn_geom& g, int b) {   // flat distance lo -> hi
    return b == 0 ? (long long)(g.nx - 1) : (b == 1 ? (long long)(g.ny - 1) * g.px : (long long)(g.nz - 1) * g.plane);
}

// Device-resident scalars of the inner iteration (S8(a) S6: alpha, beta never leave the device).
struct pn_state {
    double rr;                  // r.r of the current fp32 residual (scaled system)
    double rr_old;              // r.r one iteration earlier
    double pq;                  // p.Ap of the current iteration
    double alpha;               // rr / pq, written by kernel A's last block, read by kernel B
    double alpha_x;             // pending solution update x += alpha_x * p_old (applied by kernel A)
    double beta;                // rr_new / rr_old, written by kernel B's last block, read by kernel A
    double rr_max;              // largest rr since the last fp64 residual replacement
    double rr_target;           // proxy exit threshold on rr (set by the host from tol)
    double delta2;              // reliable-update threshold squared
    // single-kernel scheme: the x_hat update is applied every OTHER iteration (two search directions at once)
    double alpha2;              // alpha of the skipped update (pending on the direction before the current one)
    double beta_prev;           // beta that built the current direction from the skipped one
    double xskip_min;           // skip only while beta >= this (0: never skip)
    // persistent fused TMA kernel: the residual is not stored, r_{t-1} = p_{t-1} - beta_{t-1} p_{t-2} (pn_fused_tma.cu)
    double beta_last;           // the beta that built the last direction from the one before (beta_{t-1} for kernel t)
    int xpend;                  // 1: the previous kernel skipped its x_hat update
    int n_xskip;                // iterations of this solve that skipped it (36 instead of 44 B per node)
    int rexp;                   // 1: first iteration after a residual replacement: r_{t-1} is given explicitly (k_residual64)
    int pad_;
    double part[4];             // periodic faces: the main kernel's sums, finished by k_wrap_fix (rr, pq, rq, qq | pq)
    double acc[4];              // results of the fp64 reductions (residual norms, b norm, flux)
    unsigned long long count[4];// class counts (solved, inlet-only, outlet-only, floating)
    unsigned long long n_peeled;// solved nodes removed from the system as dangling ends (back-filled after the solve)
    unsigned long long n_chain; // solved nodes eliminated as links of degree-2 chains (pn_chain.cu; back-filled)
    unsigned long long n_rec;   // back-fill records written so far (k_chain_record)
    unsigned long long cm;      // active-node compaction (pn_compact.cu): unknowns of the inner system ...
    unsigned long long clong;   // ... and rows of its neighbour table with more than three entries
    int flag;                   // 0 run, 1 proxy-converged, 2 reliable update due, 3 breakdown, 4 budget
    int iters;                  // inner iterations done in this solve
    int max_iters;
    // bad_value, any_closed, topo_changed: cleared together (one memset of three ints), keep them adjacent
    int bad_value;              // set by the validation kernel
    int any_closed;             // some in-lattice bond has g == 0
    int topo_changed;           // pn_update_conductances / pn_replace_conductances: some bond went from closed to open or back
    unsigned int ticket;        // last-block-done counter (always 0 between kernels)
};

enum { PN_FLAG_RUN = 0, PN_FLAG_CONVERGED = 1, PN_FLAG_UPDATE = 2, PN_FLAG_BREAKDOWN = 3, PN_FLAG_BUDGET = 4 };

// ---- last-block epilogues of the inner iteration (shared by the main kernels and k_wrap_fix) ----
// Last-block epilogue of kernel A: alpha = rr / (p.Ap); breakdown guards.
__device__ __forceinline__ void pn_finish_A(pn_state* st, double pq) {
    st->pq = pq;
    // kernel A has just applied x_hat += alpha_x p_old: nothing is owed any more.  On the normal path finish_B sets
    // alpha_x again; on the two early exits below k_flush must not add the same direction a second time.
    st->alpha_x = 0.0;
    if (st->rr == 0.0) st->flag = PN_FLAG_CONVERGED;
    else if (!(pq > 0.0) || isinf(pq)) st->flag = PN_FLAG_BREAKDOWN;
    else st->alpha = st->rr / pq;
}

// Last-block epilogue: alpha_t, the predicted beta_{t+1}, bookkeeping and the triggers the host polls for.
__device__ __forceinline__ void pn_finish_F(pn_state* st, double rr, double pq, double rq, double qq) {
    st->rr_old = st->rr;
    st->rr = rr;
    st->pq = pq;
    const int it = st->iters + 1;
    st->iters = it;
    double rr_max = st->rr_max;
    if (rr > rr_max) { rr_max = rr; st->rr_max = rr_max; }
    int flag = PN_FLAG_RUN;
    double alpha = 0.0, beta = 0.0;
    if (!(rr >= 0.0) || isinf(rr)) flag = PN_FLAG_BREAKDOWN;
    else if (rr == 0.0) flag = PN_FLAG_CONVERGED;
    else if (!(pq > 0.0) || isinf(pq)) flag = PN_FLAG_BREAKDOWN;
    else {
        alpha = rr / pq;
        const double rr_next = rr - 2.0 * alpha * rq + alpha * alpha * qq;   // ||r_t - alpha_t q_t||^2
        if (rr <= st->rr_target) flag = PN_FLAG_CONVERGED;
        else if (rr < st->delta2 * rr_max) flag = PN_FLAG_UPDATE;
        else if (it >= st->max_iters) flag = PN_FLAG_BUDGET;
        else if (!(rr_next > 0.0) || isinf(rr_next)) flag = PN_FLAG_UPDATE;   // prediction lost: replace the residual
        else beta = rr_next / rr;
    }
    // the kernel that just ran skipped its x_hat update iff nothing was pending and its beta allowed the recovery
    // p_{t-1} = (p_t - r_t) / beta_t later (same test as in k_cg_fused_tma)
    if (!st->xpend && st->xskip_min > 0.0 && st->beta >= st->xskip_min) {
        st->xpend = 1;
        st->n_xskip += 1;
        st->alpha2 = st->alpha;       // alpha_{t-1}, still owed on p_{t-1}
        st->beta_prev = st->beta;     // beta_t
    } else {
        st->xpend = 0;
    }
    st->alpha = alpha;      // alpha_t: next kernel's residual and solution updates
    st->alpha_x = alpha;    // ... and what k_flush applies to the pending direction p_t
    st->beta_last = st->beta;   // beta_t built p_t, the direction the next kernel recovers r_t from
    st->rexp = 0;
    st->beta = beta;
    st->flag = flag;
}

// ---- reductions: warp shuffle -> block -> per-block slot -> last block sums slots in fixed order ----
__device__ __forceinline__ double pn_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in thread 0.  `sm` holds >= 32 doubles and may be reused by a
// following call (the leading barrier orders the reuse).
__device__ __forceinline__ double pn_block_sum(double v, double* sm) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    v = pn_warp_sum(v);
    __syncthreads();
    if (lane == 0) sm[wid] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? sm[threadIdx.x] : 0.0;
    if (wid == 0) v = pn_warp_sum(v);
    return v;
}

// Grid-wide deterministic sum of K doubles per block (values valid in thread 0 of each block).
// Every thread of every block must call it.  Returns true in ALL threads of the block that arrived
// last; in that block total[0..K) (shared memory) holds the sums over all blocks, added in slot order
// by a fixed tree, so the result does not depend on block scheduling.  The ticket is left at 0.
template <int K>
__device__ __forceinline__ bool pn_grid_sum(const double (&v0)[K], double* slots, unsigned int* ticket, double* sm,
                                            double* total) {
    __shared__ int s_last;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) slots[k * PN_MAX_BLOCKS + blockIdx.x] = v0[k];
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
#pragma unroll
    for (int k = 0; k < K; ++k) {
        double v = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) v += __ldcg(slots + k * PN_MAX_BLOCKS + b);
        v = pn_block_sum(v, sm);
        if (threadIdx.x == 0) total[k] = v;
    }
    if (threadIdx.x == 0) *ticket = 0u;
    __syncthreads();
    return true;
}

// ---- host-side launchers (one per S8(a) step); all enqueue on `st` and return cudaGetLastError ----
struct pn_ptrs {
    const float* raw[3];        // user-layout copies of the conductances (raw[1] == nullptr for 2D)
    float* gs[3];               // solve copy: pruned, off-lattice entries zeroed (padded layout)
    float* w[3];                // symmetric-Jacobi-scaled bond weights of the fp32 inner system
    float* gsw[3];              // face arrays: solve copy of the wrap bonds (periodic lateral faces)
    float* ww[3];               // face arrays: their scaled weights
    float* s;                   // s_i = 1/sqrt(diag_i) on solved nodes, 0 elsewhere
    double* x64;                // pressures (fp64), all nodes
    float *r, *p, *p2, *q, *xh; // fp32 CG vectors of the scaled system (p, p2: double-buffered search direction)
    float *r2, *q2;             // second buffers of r and q for the single-kernel iteration (pn_fused_tma.cu)
    signed char* cls;           // node classes
    int* parent;                // union-find forest (aliases q)
    int* flags;                 // per-root inlet/outlet contact bits (aliases xh); after S1d: live bond degree (peeling)
    double* slots;              // 8 x PN_MAX_BLOCKS partial sums (4 sums; double-buffered by the persistent kernel)
    float* xchg;                // 2D lattices up to 2048 wide: boundary rows of r, q, p exchanged between the CTAs of
                                // k_cg_resident2d, [2 parities][3 vectors][2 * PN_RESIDENT_MAX_CTAS rows][px]; else nullptr
    unsigned int* gbar;         // arrival counter of its grid barrier
    pn_state* st;
    void* scratch;              // export staging (aliases p, p2)
};

cudaError_t pn_launch_validate(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_label(const pn_geom& g, const pn_ptrs& P, bool do_label, bool do_peel, int x0_linear,
                            cudaStream_t st, int* launches);
// S1 with the node classes of the previous solve kept (no bond crossed zero since): solve copy + pruning only;
// x0_mode 0 / 1 re-initialise the solved nodes' pressures, 2 keeps them (warm start)
cudaError_t pn_launch_label_reuse(const pn_geom& g, const pn_ptrs& P, int x0_mode, cudaStream_t st, int* launches);
// sparse / full replacement of conductances in the caller-layout copy (pn_update_conductances, pn_replace_conductances):
// validates, notes closed bonds and zero crossings in the state (bad_value: 1 = value, 2 = index)
cudaError_t pn_launch_update_raw(int unx, int uny, int unz, const pn_ptrs& P, float* const raw[3], long long count,
                                 const int* axis, const long long* node, const float* value, int sms, cudaStream_t st,
                                 int* launches);
cudaError_t pn_launch_replace_raw(const pn_geom& g, float* raw, const float* src, int axis_internal, pn_state* state,
                                  cudaStream_t st, int* launches);
cudaError_t pn_launch_scale(const pn_geom& g, const pn_ptrs& P, int chains, cudaStream_t st, int* launches);
cudaError_t pn_launch_unpeel(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_backfill(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
// `bufmode`: which buffers hold the vectors of the inner iteration -- 0: two-kernel schemes (r single, p double-buffered
// by iteration parity), 1: k_cg_fused_tma (r, q, p double-buffered by parity), 2: in place (k_cg_resident2d: P.r, P.q, P.p)
cudaError_t pn_launch_residual64(const pn_geom& g, const pn_ptrs& P, int bufmode, cudaStream_t st, int* launches);
cudaError_t pn_launch_flush(const pn_geom& g, const pn_ptrs& P, int bufmode, cudaStream_t st, int* launches);
cudaError_t pn_launch_set_state(const pn_ptrs& P, double rr, double beta, double rr_max, double rr_target,
                                double delta2, int max_iters, int reset_iters, double xskip_min, cudaStream_t st,
                                int* launches);
struct pn_cptrs;
cudaError_t pn_launch_inner(const pn_geom& g, const pn_ptrs& P, int iterations, int variant, cudaStream_t st,
                            int* launches, cudaEvent_t* ev, const pn_cptrs* compact = nullptr);
cudaError_t pn_launch_flux(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_dissipation(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_export_x(const pn_geom& g, const pn_ptrs& P, double* out, cudaStream_t st, int* launches);
cudaError_t pn_launch_export_cls(const pn_geom& g, const pn_ptrs& P, signed char* out, int user_dir_is_2d,
                                 cudaStream_t st, int* launches);

// Single-kernel CG iteration, TMA-fed (pn_fused_tma.cu): S4 + S5 + S6 in one launch
struct pn_fused_plan;
bool pn_fused_plan_build(pn_fused_plan** out, const pn_geom& g, const pn_ptrs& P);
void pn_fused_plan_free(pn_fused_plan* pl);
cudaError_t pn_launch_cg_fused(const pn_fused_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int max_launch_iters = 0);

// periodic lateral faces (pn_wrap.cu): the wrap bonds' part of q and of the dot products; finishes alpha / beta
cudaError_t pn_launch_wrap_fix(const pn_geom& g, const pn_ptrs& P, int fused, cudaStream_t st);
cudaError_t pn_launch_wrap_copy(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);

// Whole inner loop in one CTA's shared memory (pn_onchip.cu): lattices of at most 7168 padded floats per array
bool pn_onchip_supported(const pn_geom& g);
// Per-DEVICE opt-in to large dynamic shared memory for the kernels that need it (cudaFuncSetAttribute is per device,
// not per process): called by pn_create with the handle's device current.
cudaError_t pn_fused_init_device();
cudaError_t pn_onchip_init_device();
cudaError_t pn_launch_cg_onchip(const pn_geom& g, const pn_ptrs& P, int max_launch_iters, cudaStream_t st);

// Degree-2 chain elimination (pn_chain.cu): mark / undo, reduced Jacobi scale, back-fill by interpolation
cudaError_t pn_launch_chain_mark(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_chain_unmark(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_chain_scale(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_chain_fill(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
struct pn_cptrs;
cudaError_t pn_launch_chain_record(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, cudaStream_t st, int* launches);
cudaError_t pn_launch_chain_fill_rec(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long n_chain, cudaStream_t st,
                                     int* launches);

// Active-node compaction (pn_compact.cu): the inner iteration on the unknowns only, ELL-3 + overflow neighbour table
struct pn_cptrs {
    int* cidx;                  // lattice -> compact index (build scratch)
    int* lat;                   // compact -> lattice index
    int* c[3];                  // three neighbour slots per row (compact numbering); c[2] < 0: -1 - overflow record
    float* v[3];                // their scaled weights
    int* ovc;                   // overflow records: entries 3..6 of the long rows, 4 indices ...
    float* ovv;                 // ... and 4 weights per record
    float *r, *q, *p, *x;       // cm entries each
    // degree-2 chains (pn_chain.cu): one back-fill record per chain node, written once per solve -- the node, the two ends
    // of its chain (lattice indices) and its share t of the chain's resistance: P_node = P_a + t (P_b - P_a)
    int* chv;
    int2* chab;
    double* cht;
    long long chcap;            // records these arrays hold (0: none -- the back-fill walks the chains every time)
};
bool pn_compact_fits(const pn_geom& g, long long m, long long n_long);
pn_cptrs pn_compact_ptrs(const pn_geom& g, const pn_ptrs& P, long long m, long long n_long);
// `chains`: degree-2 chain nodes are marked (pn_chain.cu): a bond towards one is a table entry to the chain's far end
cudaError_t pn_launch_compact_count(const pn_geom& g, const pn_ptrs& P, int chains, cudaStream_t st, int* launches);
cudaError_t pn_launch_compact_build(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, int chains,
                                    cudaStream_t st, int* launches);
cudaError_t pn_launch_compact_gather(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, cudaStream_t st,
                                     int* launches);
cudaError_t pn_launch_compact_flush(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, long long m, cudaStream_t st,
                                    int* launches);
cudaError_t pn_launch_compact_inner(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, int iterations, cudaStream_t st,
                                    int* launches, cudaEvent_t* ev);
cudaError_t pn_launch_compact_persist(const pn_geom& g, const pn_ptrs& P, const pn_cptrs& C, int max_launch_iters, cudaStream_t st);

// Persistent in-place iteration for 2D lattices (pn_resident.cu): all iterations up to the next trigger in ONE cooperative launch
bool pn_resident_supported(const pn_geom& g, const pn_ptrs& P);
cudaError_t pn_resident_init_device();
cudaError_t pn_launch_cg_resident(const pn_geom& g, const pn_ptrs& P, int max_launch_iters, cudaStream_t st);

// Which iteration scheme a PN_OPT_KERNEL value selects on this lattice: 1 = reference two-kernel,
// 3 = single fused TMA kernel, 5 = whole loop in one CTA's shared memory, 6 = persistent in-place 2D kernel
int pn_resolve_variant(const pn_geom& g, const pn_ptrs& P, int variant);

bool pn_tma_supported();   // the driver exports cuTensorMapEncodeTiled (pn_fused_tma.cu)
