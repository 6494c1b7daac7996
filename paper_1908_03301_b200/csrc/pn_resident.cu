// pn_resident.cu -- the fp32 inner CG loop (SURVEY.md 8(a) S4 + S5 + S6) for 2D lattices whose vectors AND bond weights
// fit the shared memory of all SMs together: ONE persistent, cooperative launch per fp64 residual replacement, every
// CTA keeping its slab of rows on chip for the whole launch.
//
// SURVEY.md section 7 ("Small problems ... persistent cooperative kernel") and the paper's opposite extreme (two kernels
// and two host round trips per iteration).  A 1024^2 lattice is 25 MB of r, q, p, x_hat, wx, wz: launched one
// kernel per iteration (k_cg_fused_tma) it costs 22 us per iteration, almost all of it launch gap, TMA pipeline ramp
// and reduction tail.  Here, per iteration, a CTA touches global memory only for
//   * the first and last row of its slab (r, q, p), written to a small exchange array for its two neighbours, and the
//     two neighbour rows it reads from there (double-buffered by iteration parity);
//   * 4 partial sums, and one arrival at a device-side grid barrier.
// Arithmetic per node is that of k_cg_fused_tma (pn_fused_tma.cu): the residual update of iteration t-1 is deferred
// into iteration t and recomputed on the halo rows from the neighbours' r, q, p; beta_{t+1} is predicted from
// r.r, r.q, q.q; x_hat is updated every other iteration (PN_OPT_XDEFER).  After the barrier EVERY CTA adds the slots
// in the same fixed order and runs the same epilogue (pn_finish_F) on its own copy of the state: alpha, beta and the
// flags are bit-identical in all CTAs and from run to run.  CTA 0 stores the state at exit; all CTAs store their rows.
//
// A first version of this file streamed the slab through a TMA ring from L2, updating r, q, p in place (no second
// buffers: 100 MB instead of 151 MB at 2048^2).  Measured and dropped (profiles/r02_resident.md): at 2048^2 the 100 MB
// still do not stay in the 126 MB L2 (hit rate 60 %, DRAM traffic ~ the algorithmic bytes), and at 1024^2 the exposed
// TMA latency of a 9-step march per iteration costs what the launches did.  Larger 2D lattices, 3D lattices and
// periodic faces use k_cg_fused_tma.
#include "pn_internal.cuh"

namespace {

constexpr int RT = 1024;                          // threads per CTA
constexpr size_t RES_SMEM_MAX = 225 * 1024;       // dynamic shared memory the kernel may ask for
constexpr int RED_DOUBLES = 4 * 32 + 8;

__device__ __forceinline__ void red_release_add(unsigned int* p, unsigned int v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned int ld_relaxed(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// Grid barrier, called by ONE thread per CTA between two CTA barriers (the pattern of a cooperative grid sync): the
// CTA's writes are ordered before the release by the barrier before it, and the other CTAs' writes are visible to the
// whole CTA through the barrier after the acquire.  `target` = arrivals expected so far (a multiple of gridDim.x).
// The release is cumulative over what the CTA barrier ordered before it; the spin uses relaxed loads (an acquire load
// invalidates L1 on every poll) and ONE acquire fence once the count is reached.
__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int target) {
    red_release_add(bar, 1u);
    while (ld_relaxed(bar) < target) { }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
}

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4& v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 fma4(float a, const float4& x, const float4& y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ float dot4(const float4& a, const float4& b) { return a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w; }

// floats of shared memory for slabs of at most `rows` rows of px nodes: p with two halo rows, r, q, x_hat, wx,
// wz with the backward row, and two 4-float gaps so that the flat-index stencil (i - 1, i + 4) never leaves the arrays
__host__ __device__ inline size_t slab_floats(int px, int rows) { return (size_t)px * (6 * (size_t)rows + 3) + 8; }

__global__ void __launch_bounds__(RT, 1)
k_cg_resident2d(pn_geom g, pn_ptrs P, int rows_max, int max_launch_iters) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;   // same value in every CTA: nobody enters the barriers alone
    extern __shared__ __align__(16) float sh[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;
    const int px = g.px, px4 = px >> 2;
    const int k0 = (int)(((long long)c * g.nz) / G), k1 = (int)(((long long)(c + 1) * g.nz) / G);   // own rows
    const int rows = k1 - k0;
    const int own = rows * px;                       // floats of the own rows
    // flat layout as in HBM: row pitch px, a neighbour that does not exist meets a zero weight
    float* Pp = sh + 4;                               // rows + 2: halo row k0-1, own rows, halo row k1
    float* Wx = Pp + (size_t)(rows_max + 2) * px + 4; // own rows
    float* Wz = Wx + (size_t)rows_max * px;           // rows k0-1 .. k1-1 (row j of Wz = bond between rows k0-1+j and k0+j)
    float* Rr = Wz + (size_t)(rows_max + 1) * px;
    float* Qq = Rr + (size_t)rows_max * px;
    float* Xh = Qq + (size_t)rows_max * px;
    double* red = reinterpret_cast<double*>(sh + ((slab_floats(px, rows_max) + 1) & ~(size_t)1));
    pn_state* ls = reinterpret_cast<pn_state*>(red + RED_DOUBLES);     // this CTA's copy of the iteration state
    const int XR = 2 * G;                             // exchange rows per (parity, vector)
    float* __restrict__ xch = P.xchg;
    unsigned int* bar = P.gbar;
    unsigned int bar_target = 0;

    // ---- load the slab (once per launch) ----
    for (size_t i = tid; i < slab_floats(px, rows_max); i += RT) sh[i] = 0.f;
    if (tid == 0) *ls = *st;
    __syncthreads();
    {
        const long long base = (long long)k0 * px;
        for (int j = tid * 4; j < own; j += RT * 4) {
            st4(Pp + px + j, ld4(P.p + base + j));
            st4(Rr + j, ld4(P.r + base + j));
            st4(Qq + j, ld4(P.q + base + j));
            st4(Xh + j, ld4(P.xh + base + j));
            st4(Wx + j, ld4(P.w[0] + base + j));
        }
        for (int j = tid * 4; j < own + px; j += RT * 4) st4(Wz + j, ld4(P.w[2] + base - px + j));   // row -1 = the zero halo plane
        // the slab's first and last row of r, q, p as the neighbours want them in the first iteration (parity 0)
        const float* src[3] = {P.r, P.q, P.p};
#pragma unroll
        for (int v = 0; v < 3; ++v)
            for (int i = tid * 4; i < px; i += RT * 4) {
                st4(xch + ((long long)(v * XR + 2 * c)) * px + i, ld4(src[v] + base + i));
                st4(xch + ((long long)(v * XR + 2 * c + 1)) * px + i, ld4(src[v] + base + (own - px) + i));
            }
    }
    __syncthreads();
    if (tid == 0) { bar_target += G; grid_barrier(bar, bar_target); }
    __syncthreads();

    const bool has_lo = c > 0, has_hi = c < G - 1;   // a neighbouring slab below / above (else the halo row stays zero)
    for (int li = 0; li < max_launch_iters; ++li) {
        const int pin = li & 1, pout = pin ^ 1;                      // exchange parity read / written by this iteration
        const float beta = (float)ls->beta;
        const float al = (float)ls->alpha;                          // alpha_{t-1} (0 right after a residual replacement)
        const float nal = -al;
        // x_hat every other iteration, exactly as in k_cg_fused_tma
        const int xmode = ls->xpend ? 2 : ((ls->xskip_min > 0.0 && ls->beta >= ls->xskip_min) ? 0 : 1);
        const float c2 = xmode == 2 ? (float)(ls->alpha2 / ls->beta_prev) : 0.f;
        double a_rr = 0.0, a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;

        // ---- halo rows: the neighbours' r_{t-1}, q_{t-1}, p_{t-1} (read at L2: another SM wrote them) go in flight now ----
        float4 hr = make_float4(0.f, 0.f, 0.f, 0.f), hq = hr, hp = hr;
        const int hside = tid / px4, hi4 = tid - hside * px4;        // thread -> (halo row, float4); px <= 2048, so 2 * px4 <= RT
        const bool hdo = tid < 2 * px4 && (hside == 0 ? has_lo : has_hi);
        if (hdo) {
            const int slot = hside == 0 ? 2 * c - 1 : 2 * c + 2;
            hr = __ldcg(reinterpret_cast<const float4*>(xch + ((long long)((pin * 3 + 0) * XR + slot)) * px + 4 * hi4));
            hq = __ldcg(reinterpret_cast<const float4*>(xch + ((long long)((pin * 3 + 1) * XR + slot)) * px + 4 * hi4));
            hp = __ldcg(reinterpret_cast<const float4*>(xch + ((long long)((pin * 3 + 2) * XR + slot)) * px + 4 * hi4));
        }
        // ---- phase A: r_t = r - alpha q ; p_t = r_t + beta p ; x_hat (own rows, in shared memory) ----
        for (int j = tid * 4; j < own; j += RT * 4) {
            const float4 ro = ld4(Rr + j);                           // r_{t-1}
            const float4 po = ld4(Pp + px + j);
            const float4 rn = fma4(nal, ld4(Qq + j), ro);
            const float4 pn = fma4(beta, po, rn);
            st4(Rr + j, rn);
            st4(Pp + px + j, pn);
            if (xmode) {
                float4 xn = fma4(al, po, ld4(Xh + j));
                if (xmode == 2)
                    xn = make_float4(fmaf(c2, po.x - ro.x, xn.x), fmaf(c2, po.y - ro.y, xn.y),
                                     fmaf(c2, po.z - ro.z, xn.z), fmaf(c2, po.w - ro.w, xn.w));
                st4(Xh + j, xn);
            }
            if (j < px) {                                            // first own row -> the slab below reads it next iteration
                st4(xch + ((long long)((pout * 3 + 0) * XR + 2 * c)) * px + j, rn);
                st4(xch + ((long long)((pout * 3 + 2) * XR + 2 * c)) * px + j, pn);
            }
            if (j >= own - px) {
                st4(xch + ((long long)((pout * 3 + 0) * XR + 2 * c + 1)) * px + (j - (own - px)), rn);
                st4(xch + ((long long)((pout * 3 + 2) * XR + 2 * c + 1)) * px + (j - (own - px)), pn);
            }
            a_rr += (double)dot4(rn, rn);
        }
        if (hdo) st4(Pp + (hside == 0 ? 0 : px + own) + 4 * hi4, fma4(beta, hp, fma4(nal, hq, hr)));
        __syncthreads();
        // ---- phase C: q_t = p_t - W p_t ; the three sums with q ----
        for (int j = tid * 4; j < own; j += RT * 4) {
            const float* pc_ = Pp + px + j;
            const float4 pc = ld4(pc_), pzm = ld4(pc_ - px), pzp = ld4(pc_ + px);
            const float pl = pc_[-1], pr = pc_[4];
            const float4 gx = ld4(Wx + j);
            const float gxl = Wx[j - 1];
            const float4 gzm = ld4(Wz + j), gz = ld4(Wz + px + j);
            float4 q;
            q.x = gxl * pl + gx.x * pc.y + gzm.x * pzm.x + gz.x * pzp.x;
            q.y = gx.x * pc.x + gx.y * pc.z + gzm.y * pzm.y + gz.y * pzp.y;
            q.z = gx.y * pc.y + gx.z * pc.w + gzm.z * pzm.z + gz.z * pzp.z;
            q.w = gx.z * pc.z + gx.w * pr + gzm.w * pzm.w + gz.w * pzp.w;
            q.x = pc.x - q.x; q.y = pc.y - q.y; q.z = pc.z - q.z; q.w = pc.w - q.w;
            st4(Qq + j, q);
            if (j < px) st4(xch + ((long long)((pout * 3 + 1) * XR + 2 * c)) * px + j, q);
            if (j >= own - px) st4(xch + ((long long)((pout * 3 + 1) * XR + 2 * c + 1)) * px + (j - (own - px)), q);
            a_pq += (double)dot4(pc, q);
            a_rq += (double)dot4(ld4(Rr + j), q);
            a_qq += (double)dot4(q, q);
        }
        // ---- the four sums: warp -> CTA -> slots -> grid barrier -> every CTA adds the slots in the same order ----
        a_rr = pn_warp_sum(a_rr); a_pq = pn_warp_sum(a_pq); a_rq = pn_warp_sum(a_rq); a_qq = pn_warp_sum(a_qq);
        if (lane == 0) { red[wid] = a_rr; red[32 + wid] = a_pq; red[64 + wid] = a_rq; red[96 + wid] = a_qq; }
        __syncthreads();
        if (wid == 0) {
            // slot layout [parity][CTA][4]: one 32-byte sector per CTA
            double* my = P.slots + ((size_t)pin * PN_MAX_BLOCKS + c) * 4;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double v = pn_warp_sum(red[32 * k + lane]);
                if (lane == 0) my[k] = v;
            }
            if (lane == 0) { bar_target += G; grid_barrier(bar, bar_target); }
            __syncwarp();
            // all loads first (one round trip to L2), then the fixed-order sums: CTA b -> lane b % 32, ascending b per lane
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
            if (lane == 0) { red[128] = t0; red[129] = t1; red[130] = t2; red[131] = t3; }
            if (lane == 0) pn_finish_F(ls, red[128], red[129], red[130], red[131]);
        }
        __syncthreads();
        if (ls->flag != PN_FLAG_RUN) break;
    }
    // ---- back to HBM for S7 / S3 (and for a later launch that continues the same sequence) ----
    {
        const long long base = (long long)k0 * px;
        for (int j = tid * 4; j < own; j += RT * 4) {
            st4(P.p + base + j, ld4(Pp + px + j));
            st4(P.r + base + j, ld4(Rr + j));
            st4(P.q + base + j, ld4(Qq + j));
            st4(P.xh + base + j, ld4(Xh + j));
        }
    }
    if (c == 0 && tid == 0) *st = *ls;
}

int grid_size(const pn_geom& g) {
    int G = g.sms < PN_RESIDENT_MAX_CTAS ? g.sms : PN_RESIDENT_MAX_CTAS;
    if (g.nz < G) G = g.nz;
    return G;
}
size_t smem_bytes(const pn_geom& g) {
    const int G = grid_size(g);
    const int rows_max = (g.nz + G - 1) / G;
    return ((slab_floats(g.px, rows_max) + 1) & ~(size_t)1) * 4 + RED_DOUBLES * 8 + sizeof(pn_state) + 16;
}

}  // namespace

// 2D lattices (held as nx x 1 x rows) whose slabs -- rows / SMs rows of r, q, p, x_hat, wx, wz -- fit one SM's shared
// memory each (about 1.2 M nodes on 148 SMs), no periodic faces, the exchange array present in the workspace, and a
// device that launches cooperatively
bool pn_resident_supported(const pn_geom& g, const pn_ptrs& P) {
    return g.ny == 1 && g.nz >= 1 && g.px <= 2048 && !(g.wrap[0] | g.wrap[1] | g.wrap[2]) && P.xchg != nullptr && g.coop && g.sms > 0 &&
           smem_bytes(g) <= RES_SMEM_MAX;
}

cudaError_t pn_resident_init_device() {
    return cudaFuncSetAttribute(k_cg_resident2d, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES_SMEM_MAX);
}

// Runs inner iterations until a trigger (proxy convergence, reliable update due, budget, breakdown) or
// `max_launch_iters`; ONE launch.
cudaError_t pn_launch_cg_resident(const pn_geom& g, const pn_ptrs& P, int max_launch_iters, cudaStream_t st) {
    const int G = grid_size(g);
    int rows_max = (g.nz + G - 1) / G;
    cudaError_t e = cudaMemsetAsync(P.gbar, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    pn_geom gg = g;
    pn_ptrs PP = P;
    void* args[] = {(void*)&gg, (void*)&PP, (void*)&rows_max, (void*)&max_launch_iters};
    return cudaLaunchCooperativeKernel((const void*)k_cg_resident2d, dim3(G), dim3(RT), args, smem_bytes(g), st);
}
