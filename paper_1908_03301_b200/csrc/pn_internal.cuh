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
};

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
    double acc[4];              // results of the fp64 reductions (residual norms, b norm, flux)
    unsigned long long count[4];// class counts (solved, inlet-only, outlet-only, floating)
    unsigned long long n_peeled;// solved nodes removed from the system as dangling ends (back-filled after the solve)
    int flag;                   // 0 run, 1 proxy-converged, 2 reliable update due, 3 breakdown, 4 budget
    int iters;                  // inner iterations done in this solve
    int max_iters;
    int bad_value;              // set by the validation kernel
    int any_closed;             // some in-lattice bond has g == 0
    unsigned int ticket;        // last-block-done counter (always 0 between kernels)
};

enum { PN_FLAG_RUN = 0, PN_FLAG_CONVERGED = 1, PN_FLAG_UPDATE = 2, PN_FLAG_BREAKDOWN = 3, PN_FLAG_BUDGET = 4 };

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
    float* s;                   // s_i = 1/sqrt(diag_i) on solved nodes, 0 elsewhere
    double* x64;                // pressures (fp64), all nodes
    float *r, *p, *p2, *q, *xh; // fp32 CG vectors of the scaled system (p, p2: double-buffered search direction)
    float *r2, *q2;             // second buffers of r and q for the single-kernel iteration (pn_fused_tma.cu)
    signed char* cls;           // node classes
    int* parent;                // union-find forest (aliases q)
    int* flags;                 // per-root inlet/outlet contact bits (aliases xh); after S1d: live bond degree (peeling)
    double* slots;              // 4 x PN_MAX_BLOCKS partial sums
    pn_state* st;
    void* scratch;              // export staging (aliases p, p2)
};

int pn_sm_count();

cudaError_t pn_launch_validate(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_label(const pn_geom& g, const pn_ptrs& P, bool do_label, bool do_peel, int x0_linear,
                            cudaStream_t st, int* launches);
cudaError_t pn_launch_scale(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_unpeel(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_backfill(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_residual64(const pn_geom& g, const pn_ptrs& P, int fused, cudaStream_t st, int* launches);
cudaError_t pn_launch_flush(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_set_state(const pn_ptrs& P, double rr, double beta, double rr_max, double rr_target,
                                double delta2, int max_iters, int reset_iters, cudaStream_t st, int* launches);
cudaError_t pn_launch_inner(const pn_geom& g, const pn_ptrs& P, int iterations, int variant, cudaStream_t st,
                            int* launches, cudaEvent_t* ev);
cudaError_t pn_launch_flux(const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int* launches);
cudaError_t pn_launch_export_x(const pn_geom& g, const pn_ptrs& P, double* out, cudaStream_t st, int* launches);
cudaError_t pn_launch_export_cls(const pn_geom& g, const pn_ptrs& P, signed char* out, int user_dir_is_2d,
                                 cudaStream_t st, int* launches);

// Single-kernel CG iteration, TMA-fed (pn_fused_tma.cu): S4 + S5 + S6 in one launch
struct pn_fused_plan;
bool pn_fused_plan_build(pn_fused_plan** out, const pn_geom& g, const pn_ptrs& P);
void pn_fused_plan_free(pn_fused_plan* pl);
cudaError_t pn_launch_cg_fused(const pn_fused_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st);

// Which iteration scheme a PN_OPT_KERNEL value selects on this lattice: 1 = reference two-kernel,
// 2 = two-kernel with the TMA S4 kernel, 3 = single fused TMA kernel
int pn_resolve_variant(const pn_geom& g, int variant);

// TMA-fed S4 kernel (pn_stencil_tma.cu)
struct pn_tma_plan;
bool pn_tma_supported();
bool pn_tma_plan_build(pn_tma_plan** out, const pn_geom& g, const pn_ptrs& P);
void pn_tma_plan_free(pn_tma_plan* pl);
cudaError_t pn_launch_stencil_tma(const pn_tma_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st);
