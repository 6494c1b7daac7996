/* pn.h -- C ABI of libpn: mixed-precision conjugate-gradient solve of bond-network Kirchhoff systems
 * on one NVIDIA B200 (sm_100a).
 *
 * The problem (citations: /root/reference/PAPER.md = P:<line>; SURVEY.md section 8 = S8):
 *   nodes of a square (nz == 1) or simple-cubic lattice nx x ny x nz, node n = i + nx*(j + ny*k);
 *   bonds with conductance g_ij >= 0 (g == 0: closed bond); flow in a bond q_ij = g_ij (P_j - P_i)
 *   mass balance at every interior node  sum_j g_ij (P_i - P_j) = 0  ->  G P = b, eq.(3)
 *   a fixed macroscopic pressure drop along one lattice axis `a`: P = 1 on the node plane coord_a = 0,
 *   P = 0 on the plane coord_a = n_a - 1; every other face is a no-flux face                        P:57, S8(c) 1-2
 *   (the paper's lateral faces are periodic; BASELINE.json's north_star and configs[0] fix no-flux)
 *   solved by conjugate gradients, single precision inside, double precision outside
 *   then total flow Q through a cross-section and Darcy permeability K = (Q/S)(mu L/dP), eq.(4)
 *
 * Conductance arrays (S8(a)): three (two in 2D) float arrays of nx*ny*nz entries each, x fastest,
 * FORWARD-BOND convention:  gx[n] = bond (i,j,k)--(i+1,j,k),  gy[n] = bond (i,j,k)--(i,j+1,k),
 * gz[n] = bond (i,j,k)--(i,j,k+1).  Entries whose forward neighbour is outside the lattice are not
 * bonds; they are ignored whatever they hold.  The float values ARE the problem: the double
 * precision steps widen exactly these values (S8(c) reading 14).
 *
 * Ownership: the caller owns every device buffer (workspace, inputs, outputs).  The library owns
 * the host-side handle and a few hundred bytes of pinned host memory.  All device work is enqueued
 * on the stream given to pn_create.  A handle is not thread-safe; distinct handles are independent.
 * No call prints, aborts or throws.  There is no CPU fallback: without a CUDA device every call
 * that needs one returns PN_ERR_CUDA.
 */
#ifndef PN_H
#define PN_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pn_ctx pn_ctx; /* opaque handle: one network on one device / stream */

/* return codes: 0 ok, > 0 valid non-error outcomes, < 0 errors */
enum {
    PN_OK = 0,
    PN_NO_SPANNING_CLUSTER = 1, /* no cluster joins inlet and outlet: Q = 0, pressures = pin values */
    PN_MAX_ITERS = 2,           /* iteration budget spent or residual stagnated; the LAST iterate is
                                   kept (pn_info.rel_residual is its true residual)                 */
    PN_ERR_ARG = -1,            /* null pointer, bad shape / direction / tol, axis shorter than 3   */
    PN_ERR_STATE = -2,          /* solve before set_conductances, flux / pressures before solve     */
    PN_ERR_VALUE = -3,          /* negative, NaN or Inf conductance on an in-lattice bond           */
    PN_ERR_WORKSPACE = -4,      /* workspace missing, misaligned (256 B) or too small               */
    PN_ERR_CUDA = -5,           /* a CUDA call failed (sticky; pn_last_error has the text)          */
    PN_ERR_BREAKDOWN = -6,      /* CG breakdown: p.Ap <= 0 or non-finite                            */
    PN_ERR_TOO_LARGE = -7       /* pn_dissipation_noalloc: more than PN_NOALLOC_MAX_NODES nodes     */
};

/* node classes written by pn_get_classes (S8(c) steps 2-3) */
enum {
    PN_CLASS_INLET = 0,       /* Dirichlet plane coord_a = 0,        P = 1                          */
    PN_CLASS_OUTLET = 1,      /* Dirichlet plane coord_a = n_a - 1,  P = 0                          */
    PN_CLASS_SOLVED = 2,      /* interior node of a cluster that reaches both planes: unknown       */
    PN_CLASS_INLET_ONLY = 3,  /* cluster reaches only the inlet:  no flow, P = 1 exactly (pinned)   */
    PN_CLASS_OUTLET_ONLY = 4, /* cluster reaches only the outlet: no flow, P = 0 exactly (pinned)   */
    PN_CLASS_FLOATING = 5     /* cluster reaches neither: P undefined, pinned to 0 by convention    */
};

typedef struct {
    int status;            /* the code pn_solve returned                                            */
    int outer_cycles;      /* fp64 true-residual evaluations  r = b - A x  (S8(a) S3)                */
    int inner_iters;       /* fp32 CG iterations (S8(a) S4+S5), summed over the solve               */
    int kernel_scheme;     /* inner-iteration kernels used: the resolved PN_OPT_KERNEL value (1, 3, 5, 6 or 8), or 7 = compacted unknowns (PN_OPT_COMPACT) */
    double rel_residual;   /* true fp64 ||b - A x||_2 / ||b||_2 over the solved nodes at exit       */
    double b_norm;         /* ||b||_2 of the zero-initial-guess system (S8(c) reading 5)            */
    long long n_solved, n_inlet_only, n_outlet_only, n_floating; /* interior node counts by class    */
    double t_label_ms;     /* S1 + set-up (labelling, pruning, scaling), device time                */
    double t_solve_ms;     /* S3..S7 loop, device time                                              */
    double t_stencil_ms;   /* with PN_OPT_PROFILE: summed device time of the S4 kernel launches (scheme 3:
                              of the single fused S4+S5+S6 kernel; t_update_ms is then 0) ...       */
    double t_update_ms;    /* ... and of the S5 kernel launches (CUDA events on the handle's stream) */
    int n_timed_iters;     /* ... over this many inner iterations                                   */
    int n_xskip;           /* single-kernel scheme: inner iterations that skipped the x_hat update (PN_OPT_XDEFER):
                              they move 8 bytes per node less than the others                        */
    long long n_peeled;    /* solved nodes taken out of the system as dangling ends (PN_OPT_PEEL) and
                              back-filled after the solve; they are counted in n_solved too           */
    long long n_unknowns;  /* unknowns of the inner linear system: n_solved - n_peeled - n_chain           */
    long long n_chain;     /* solved nodes eliminated as links of degree-2 chains (PN_OPT_CONTRACT) and back-filled
                              by interpolation between the ends of their chain; counted in n_solved too   */
    long long n_long_rows; /* compacted unknowns (kernel_scheme 7): rows of the neighbour table with more than three
                              entries (they carry a 32-byte overflow record)                               */
    int labels_reused;     /* 1: S1's labelling and peeling were skipped, the classes of the previous solve
                              still hold (pn_update_conductances / pn_replace_conductances, no bond crossed zero) */
    int residual_recovered;/* 1: the fused kernel ran as persistent launches that store no fp32 residual (it is recovered
                              from the last two search directions): 36 instead of 40 bytes per node and iteration */
} pn_info;

/* options for pn_set_option */
enum {
    PN_OPT_MAX_ITERS = 0,   /* inner-iteration budget per solve            (default 200000)         */
    PN_OPT_DELTA = 1,       /* reliable-update threshold: fp64 residual replacement when the fp32
                               recursive residual has fallen by this factor since the last one
                               (default 0.3; S8(c) reading 4)                                       */
    PN_OPT_X0 = 2,          /* initial guess on solved nodes: 0 = zero, 1 = linear profile along the
                               solve axis (default 1; S8(c) reading 6), 2 = warm start: the pressures
                               this handle's previous solve left (S8(f) item 4: re-solves after a
                               change of conductances or direction; first solve: same as 1)         */
    PN_OPT_CHUNK = 3,       /* inner iterations enqueued between host polls (default 32); the persistent
                               launches (schemes 5, 6, 7, 8 and 3 with PN_OPT_GRAPH = 1) run to the next residual
                               replacement, or for this many iterations once the caller has set it  */
    PN_OPT_SKIP_LABEL = 4,  /* 1: skip S1 when the caller guarantees all bonds are open (default 0;
                               S1 is always skipped automatically when no in-lattice g == 0 exists) */
    PN_OPT_KERNEL = 5,      /* inner-iteration kernels: 0 = automatic (5 when the lattice fits one SM's shared
                               memory -- at most 7168 padded floats per array, no periodic faces --, 6 where it
                               applies, 8 on other lattices of at most 5 000 000 (3D) / 12 000 000 (2D) padded nodes, else 3),
                               1 = reference pair: S4 kernel reading neighbours through the caches + S5
                               kernel (kept as an independently written cross-check),
                               3 = ONE TMA-fed kernel per iteration (S4 + S5 + S6 fused),
                               5 = the whole inner loop in ONE launch of one CTA, vectors in shared memory,
                               6 = 2D lattices whose rows / SMs slabs fit the SMs' shared memory (about 1.2 M nodes,
                               at most 2048 wide, no periodic faces): ONE persistent cooperative launch per residual
                               replacement, every CTA keeping its slab on chip, grid barrier per iteration; else 3,
                               8 = any lattice, periodic faces included: ONE persistent cooperative launch per residual
                               replacement, neighbours through L1 / L2, one grid barrier per iteration (for lattices
                               whose planes sit in the L2, where launch boundaries cost more than the re-reads).
                               (2 and 4 were round-1 experiments, since removed: PN_ERR_ARG)                   */
    PN_OPT_PROFILE = 6,     /* 1: record CUDA events around every S4 / S5 launch and report the
                               summed kernel times in pn_info (default 0)                           */
    PN_OPT_PEEL = 7,        /* dead-end peeling: solved nodes left with one open bond carry no current
                               (S8(c) reading 7, S8(f) item 1); they are removed from the system,
                               recursively, and take the pressure of the node they hang from after the
                               solve.  Pressures of all nodes stay those of the full system.
                               0: never (all solved nodes are unknowns), 1: always, 2 (default): only if
                               at least 10 % of the solved nodes can be removed (below that -- 3.8 % on
                               configs[3] -- no gain was measured, and the peeling is undone)       */
    PN_OPT_LATERAL = 8,     /* lateral (side) faces: 0 (default) = no-flux (north_star, configs[0]); 1 = periodic,
                               the paper's own condition ("periodic boundary conditions in the second
                               direction"; S8(f) item 2): every axis other than the solve axis wraps around, and
                               the forward entry of the LAST node along such an axis is the bond back to the
                               first node (validated at pn_solve: PN_ERR_VALUE).  An axis of one node does
                               not wrap                                                             */
    PN_OPT_GRAPH = 9,       /* 1 (default): a chunk of inner iterations is replayed from a CUDA graph (captured
                               once per geometry / direction / scheme); with the compacted unknowns (scheme 7): ONE
                               persistent cooperative launch runs all iterations up to the next residual
                               replacement.  0: every kernel launched directly, one by one.  2: as 1, and the 2D tile of
                               scheme 3 runs as a persistent launch too (it measured slower than graph replay and is
                               not chosen automatically; kept for measurements)                              */
    PN_OPT_REUSE_LABELS = 11, /* 1 (default): a solve that follows pn_update_conductances / pn_replace_conductances (or simply
                               repeats the previous one) keeps the node classes, pins and peeled set of the previous solve
                               when no bond went from closed to open or back and direction, PN_OPT_LATERAL, PN_OPT_PEEL
                               and PN_OPT_SKIP_LABEL are unchanged; 0: S1 is always redone                    */
    PN_OPT_COMPACT = 12,    /* active-node compaction (S8(f) item 1; the paper's critical slow-down case): the
                               inner iteration runs on the UNKNOWNS only, stored contiguously with a neighbour
                               table (kernel_scheme 7; 64 bytes per unknown and iteration instead of 40 per lattice
                               node).  0: never, 1: whenever it applies, 2 (default): when at most 0.45 of the padded
                               lattice nodes are unknowns (e.g. configs[2] after peeling: 0.33).  Applies to schemes
                               3 / 0 on lattices without periodic faces whose table fits the workspace; pressures of
                               all nodes are unchanged                                                        */
    PN_OPT_CONTRACT = 13,   /* 1 (default): when the unknowns are compacted (PN_OPT_COMPACT), solved nodes with exactly two
                               open bonds, both to solved nodes, are eliminated exactly beforehand -- a chain of them is
                               one series resistor between its two end nodes (the Schur complement of the balance
                               P:53) -- and take the resistance-weighted interpolation of the end pressures afterwards.
                               Near the threshold these "links" are 69 % of the unknowns left after peeling and the
                               reason for the slow convergence there.  0: never.  Pressures of all
                               nodes stay those of the full system.  Safety net: if the iteration on the reduced
                               system breaks down or stagnates before its budget is spent, pn_solve repeats the
                               solve once on the lattice kernels, without elimination and compaction (pn_info then
                               reports n_chain = 0, that kernel_scheme and the iterations of both attempts)    */
    PN_OPT_TILE = 14,       /* tile of the fused TMA kernel (scheme 3) on 3D lattices: 1 = 256 x 8 nodes, 2 = 128 x 16,
                               3 = 64 x 32, 0 (default) = automatic: a narrower tile where it fills its lanes at least 8 %
                               better than the next wider one (widths such as 192, 320 or 384 that leave a 256-wide tile
                               mostly empty); with any of them a width that does not fill its last tile is cut into equal
                               tiles                                                                           */
    PN_OPT_XDEFER = 10      /* 1 (default): the single-kernel scheme applies the fp32 solution update every OTHER
                               iteration, two search directions at once (the earlier one recovered from p and r):
                               40 instead of 44 bytes per node-iteration on average; 0: every iteration    */
};

/* Device bytes pn_create needs for an nx x ny x nz lattice (0 on a bad shape). */
size_t pn_workspace_bytes(int nx, int ny, int nz);

/* Create a handle.  nx, ny, nz >= 1 (nz == 1: 2D).  `device`: CUDA ordinal.  `cuda_stream`: a
 * cudaStream_t (NULL = the legacy default stream).  `workspace`: DEVICE memory, 256-byte aligned, at
 * least pn_workspace_bytes(nx, ny, nz) bytes, owned by the caller and left untouched by it until
 * pn_destroy.  Errors: PN_ERR_ARG, PN_ERR_WORKSPACE, PN_ERR_CUDA. */
int pn_create(pn_ctx** out, int nx, int ny, int nz, int device, void* cuda_stream, void* workspace,
              size_t workspace_bytes);

/* S0: hand the network to the library (it copies; the caller may free its arrays on return).
 * gx, gy, gz: nx*ny*nz floats each, forward-bond convention; gz must be NULL iff nz == 1.
 * `pointers_are_device` != 0: DEVICE pointers (device-to-device copy on the handle's stream);
 * 0: HOST pointers (pageable or pinned).  Every in-lattice bond must be finite and >= 0, else
 * PN_ERR_VALUE and the handle keeps no network.  Invalidates earlier pressures. */
int pn_set_conductances(pn_ctx* ctx, const float* gx, const float* gy, const float* gz,
                        int pointers_are_device);

/* S8(f) item 4 -- conductances that change between solves ("simulating a flow or transport process that may
 * take thousands of time steps").  Both calls change the network the handle holds WITHOUT the full S0 + S1 of a new
 * network: the next pn_solve in the same direction skips the labelling and peeling when no bond went from closed
 * (g == 0) to open or back (pn_info.labels_reused), rebuilds the solve copy, scaling and weights on the device, and
 * starts from the pressures of the previous solve (warm start) unless PN_OPT_X0 is 0.  Pressures and fluxes of the
 * previous solve become unavailable.  Values must be finite and >= 0: PN_ERR_VALUE; a bad axis / node index:
 * PN_ERR_ARG; on either error the handle keeps no network (as after a failed pn_set_conductances).  Needs a network:
 * PN_ERR_STATE before pn_set_conductances.
 *
 * pn_update_conductances: sparse.  Bond i of the list is the forward bond along `axis[i]` (0 = x, 1 = y, 2 = z; 2D:
 * 0 or 1) of node `node[i]` (n = i + nx*(j + ny*k)) and takes `value[i]`; `count` entries, all DISTINCT bonds.
 * Entries whose forward neighbour is off-lattice are stored and ignored as in pn_set_conductances.  HOST or DEVICE
 * pointers (all three alike).
 * pn_replace_conductances: all bonds; arguments as pn_set_conductances. */
int pn_update_conductances(pn_ctx* ctx, long long count, const int* axis, const long long* node, const float* value,
                           int pointers_are_device);
int pn_replace_conductances(pn_ctx* ctx, const float* gx, const float* gy, const float* gz, int pointers_are_device);

/* S1..S7: classify and prune clusters for `direction` (0 = x, 1 = y, 2 = z; the axis needs >= 3
 * node planes), then iterate until the true fp64 residual ||b - A x||_2 <= tol * ||b||_2
 * (0 < tol < 1).  Returns when the stream work of this solve has finished.  `info` may be NULL.
 * Returns PN_OK, PN_NO_SPANNING_CLUSTER, PN_MAX_ITERS, or an error. */
int pn_solve(pn_ctx* ctx, int direction, double tol, pn_info* info);

/* Pressures of the last solve on ALL nx*ny*nz nodes (fp64, node order n = i + nx*(j + ny*k)):
 * Dirichlet planes and pinned clusters hold their pin values.  `out`: nx*ny*nz doubles, DEVICE if
 * `pointer_is_device` else HOST.  Valid until the next pn_solve / pn_set_conductances. */
int pn_get_pressures(pn_ctx* ctx, double* out, int pointer_is_device);

/* Node class (PN_CLASS_*) of every node for the last solve's direction; nx*ny*nz bytes. */
int pn_get_classes(pn_ctx* ctx, signed char* out, int pointer_is_device);

/* S8, eq.(4) P:61 with mu = l = 1, dP = 1, L = n_a - 1, S = number of nodes in a plane normal to a:
 *   q_in  = sum over bonds leaving the inlet plane   g (1 - P_nbr)
 *   q_out = sum over bonds entering the outlet plane g (P_nbr - 0)
 *   g_eff = (q_in + q_out) / 2,   k_eff = g_eff (n_a - 1) / S.
 * HOST pointers; any may be NULL.  Needs a finished pn_solve (PN_ERR_STATE otherwise). */
int pn_flux(pn_ctx* ctx, double* q_in, double* q_out, double* g_eff, double* k_eff);

/* Dissipation estimate of the effective conductance: g_e = sum over ALL bonds of g (P_i - P_j)^2 (dP = 1; the energy
 * identity Q dP = sum g dP_bond^2 of the balance P:53 with eq.(4)).  Equal to g_eff at the exact solution, and
 * its error is quadratic in the error of the pressures where g_eff's (boundary fluxes) is linear: a cross-check that
 * holds to ~1e-12 already at a 1e-10 residual (S8(c) consequence (iv)).  HOST pointer.  Needs a finished pn_solve. */
int pn_dissipation(pn_ctx* ctx, double* g_e);

/* The same dissipation sum WITHOUT a handle, a workspace or any allocation -- for callers that may not allocate
 * device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 *   g_e = sum over all bonds g (P_i - P_j)^2        (energy identity of P:53 with eq.(4), dP = 1)
 * over the network AS THE CALLER HOLDS IT: gx, gy, gz in the layout of pn_set_conductances (forward-bond convention,
 * gz NULL iff nz == 1), `pressures` in the layout of pn_get_pressures (nx*ny*nz doubles).  Bit b of `periodic_mask`
 * (b = 0, 1, 2 for x, y, z): that axis wraps around, the forward entry of its last node being the bond back to the
 * first (PN_OPT_LATERAL = 1 with solve axis a: every bit but a); other forward entries that leave the lattice are
 * ignored.  With the pressures of a finished pn_solve the result equals pn_dissipation's up to the order of the sum
 * (pinned clusters are at one pressure: their bonds add exact zeros).
 * ALL pointers are DEVICE pointers on `device`, owned by the caller; `g_e` receives ONE double, written on
 * `cuda_stream` (NULL = the legacy default stream): the call only enqueues (one 4-byte memset + one kernel) and does
 * not synchronise.  The sum is taken over fixed chunks of 8192 nodes whose partial sums are added in chunk order: the
 * value does not depend on the GPU or on block scheduling.
 * Scratch: the chunk sums and an arrival counter live in a file-scope `static __device__` array of
 * PN_NOALLOC_MAX_NODES / 8192 + 32 doubles (about 256 KB), which every GPU that loads the library holds until exit.
 * Limit: nx*ny*nz <= PN_NOALLOC_MAX_NODES (2^28 = 268 435 456 nodes; 512^3 is 2^27), else PN_ERR_TOO_LARGE and nothing
 * is enqueued.  The array is shared by every call in the process: calls that may OVERLAP on one GPU (different
 * streams, different host threads) race on it and must be ordered by the caller; calls on one stream are safe.  The
 * counter is cleared at the start of every call; the chunk sums need no clearing (every chunk in use is rewritten).
 * Calls no cudaMalloc / cudaFree and no allocating library routine (first use on a device: cudaGetSymbolAddress and
 * cudaDeviceGetAttribute).  Errors: PN_ERR_ARG (null pointer, bad shape or mask, gz given for nz == 1 or missing for
 * nz > 1), PN_ERR_TOO_LARGE, PN_ERR_CUDA. */
#define PN_NOALLOC_MAX_NODES 268435456LL
int pn_dissipation_noalloc(int nx, int ny, int nz, const float* gx, const float* gy, const float* gz,
                           const double* pressures, int periodic_mask, double* g_e, int device, void* cuda_stream);

/* Tuning knobs (PN_OPT_*).  PN_ERR_ARG on an unknown key or out-of-range value. */
int pn_set_option(pn_ctx* ctx, int key, double value);

/* Kernel launches enqueued by this handle since pn_create (bench.py's `gpu_launches`). */
long long pn_launch_count(const pn_ctx* ctx);

/* Convergence record of the last pn_solve: the true fp64 relative residual ||b - A x||_2 / ||b||_2 at every
 * evaluation (S8(a) S3), the first entry being that of the initial guess; info->outer_cycles of them (at most
 * 256 are kept).  Copies min(count, capacity) values to the HOST array `out` and returns the count (>= 0), or
 * PN_ERR_ARG.  `out` may be NULL when capacity == 0 (query). */
int pn_residual_history(const pn_ctx* ctx, double* out, int capacity);

/* Release the handle (not the workspace).  NULL is allowed. */
int pn_destroy(pn_ctx* ctx);

/* Static text for a return code. */
const char* pn_strerror(int code);

/* Text of the last CUDA error seen by this handle ("" if none). */
const char* pn_last_error(const pn_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* PN_H */
