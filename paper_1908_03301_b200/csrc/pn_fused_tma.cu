// pn_fused_tma.cu -- the whole fp32 inner CG iteration (SURVEY.md 8(a) S4 + S5 + S6) as ONE 2.5D, TMA-fed,
// warp-specialised persistent kernel for sm_100a: 44 B per node-iteration instead of the 48 B of the
// two-kernel form (SURVEY.md 8(d) "irreducible: g once + each of x, r, p, q read once and written once").
//
// Paper: K2 (SpMV + dot) and K3 (vector updates + dots) are two kernels because the update of
// the residual needs alpha = r.r / p.Ap, a grid-wide sum over the SpMV's output.  Here the
// residual update of iteration t-1 is deferred into the kernel of iteration t, where it is recomputed on
// the tile halo as well, so that one kernel per iteration remains:
//
//   kernel F(t):   r_t = r_{t-1} - alpha_{t-1} q_{t-1}          (tile + one-node halo, from r, q staged by TMA)
//                  p_t = r_t + beta_t p_{t-1}                   (tile + halo)  -> shared-memory plane ring
//                  x_hat += alpha_{t-1} p_{t-1}
//                  q_t = p_t - W p_t                            (7-point operator from the plane ring)
//                  sums:  rr = r_t.r_t   pq = p_t.q_t   rq = r_t.q_t   qq = q_t.q_t
//   last block:    alpha_t = rr / pq
//                  beta_{t+1} = ||r_t - alpha_t q_t||^2 / rr = (rr - 2 alpha_t rq + alpha_t^2 qq) / rr
//
// beta_{t+1} must be known before r_{t+1} exists; it is obtained from the three sums by expanding the
// square (exact in exact arithmetic; in fp32 the fp64-accumulated sums reproduce ||r_{t+1}||^2 to ~1e-7
// relative unless r shrinks by orders of magnitude in one step, and the NEXT kernel measures the true
// r_{t+1}.r_{t+1} anyway: alpha_{t+1} and the denominator of beta_{t+2} use the measured value).  A
// non-positive prediction raises the reliable-update flag, i.e. an fp64 residual replacement.
// r, p and q are double-buffered (index = iteration parity): a tile reads its neighbours' old values as halo.
//
// HBM bytes per node: reads r, q, p, x_hat, wx, wy, wz (28 B) + writes r, q, p, x_hat (16 B) = 44 B; 40 B with x_hat touched every
// other iteration; 36 B in the persistent form (PERSIST, 3D tiles), which does not store r at all: r_{t-1} = p_{t-1} -
// beta_{t-1} p_{t-2} is recovered from the last two search directions, kept in three rotating slots (512^3: 0.8627 -> 0.7473 ms
// per iteration, same iteration count).
#include <new>

#include "pn_tma.cuh"

namespace {

using namespace pn_tma;

template <int NBX_, int TY_, bool HAS_Y_, int S_, int BOXW_ = 256>
struct FCfg {
    static constexpr int NBX = NBX_, TY = TY_, S = S_;
    static constexpr bool HAS_Y = HAS_Y_;
    // where the CTA barrier of a plane step sits: at its END (phases A and C become independent instruction streams) or
    // between the phases.  Measured on one box (profiles/r01_barrier_placement.md): the end is 3.6 % faster on the 3D tile
    // (512^3); on the 2D tile it was 3.1 % slower with generic shared-memory accesses and is 0.7 % faster now that the 2D
    // tile uses LDS / STS (see the kernel's first lines)
    static constexpr bool BAR_END = true;
    static constexpr int BOXW = BOXW_;                     // nodes per box row (256 = the TMA box limit per dimension)
    static constexpr int LPR = BOXW / 4;                   // consumer lanes per box row (64, 32 or 16: whole warps, or two rows per warp)
    static_assert(BOXW % 64 == 0 && BOXW <= 256, "box rows of whole or half warps");
    static constexpr int TXW = BOXW * NBX;                 // tile width in nodes
    static constexpr int RH = TY + (HAS_Y ? 2 : 0);        // rows of r, q, p and p_new including the y halo
    static constexpr int RWY = TY + (HAS_Y ? 1 : 0);       // rows of the wy box (backward row included)
    static constexpr int W = TXW + 8;                      // p_new ring row: 4 pad + tile + 4 pad floats
    static constexpr int NCONS = LPR * NBX * TY;           // consumer threads: one float4 of nodes each
    static constexpr int NTHREADS = NCONS + 32;            // + one producer warp
    static constexpr int NHALO4 = HAS_Y ? 2 * LPR * NBX : 0;  // float4s in the two halo rows
    // stage layout (floats): three haloed vectors, then the weights
    static constexpr int VEC = NBX * RH * BOXW + 2 * a32(RH * 4);   // main boxes, left sliver, right sliver
    static constexpr int V_SL = NBX * RH * BOXW;
    static constexpr int V_SR = V_SL + a32(RH * 4);
    static constexpr int R_ = 0, Q_ = VEC, P_ = 2 * VEC;
    static constexpr int WX = 3 * VEC;
    static constexpr int WX_SL = WX + NBX * TY * BOXW;
    static constexpr int WY = WX_SL + a32(TY * 4);
    static constexpr int WZ = WY + (HAS_Y ? NBX * RWY * BOXW : 0);
    static constexpr int STAGE_FLOATS = WZ + NBX * TY * BOXW;
    static constexpr int RING_FLOATS = 4 * RH * W;
    static constexpr size_t SMEM_BYTES = (size_t)(S * STAGE_FLOATS + RING_FLOATS) * 4 + 2 * S * 8 + 64 * 8 + 1024;
    // transaction bytes per group of boxes
    static constexpr unsigned B_RQP = 3u * (NBX * RH * BOXW + 2 * RH * 4) * 4u;
    static constexpr unsigned B_W = (NBX * TY * BOXW + TY * 4 + (HAS_Y ? NBX * RWY * BOXW : 0)) * 4u;
    static constexpr unsigned B_WZ = NBX * TY * BOXW * 4u;
};

struct alignas(64) pn_fmaps {
    CUtensorMap v_main[3][2], v_slv[3][2];   // [r, q, p][buffer]
    CUtensorMap wx_main, wx_slv, wy, wz;
};

// PERSIST: the same kernel as ONE cooperative launch per fp64 residual replacement -- the iteration loop runs inside, the
// last-block epilogue becomes a grid barrier after which every CTA adds the per-CTA sums in the same fixed order and runs
// pn_finish_F on its own copy of the state (as k_cg_resident2d / k_cg_persist / k_cpersist do).  Saves the launch gap, the
// state reads and the reduction tail of every iteration (~17 us of 868 at 512^3); not with periodic faces (k_wrap_fix), and
// not on the 2D tile (measured slower there).
__device__ __forceinline__ void ft_grid_barrier(unsigned int* bar, unsigned int target) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(bar), "r"(1u) : "memory");
    unsigned int v;
    do { asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory"); } while (v < target);
    __threadfence();
}

// NARROW (single-box tiles only): the lattice's width is cut into ntx EQUAL tiles of tw <= 256 nodes (tw a multiple of 4) instead
// of 256-wide ones with a narrow remainder; the TMA boxes are tw wide (rows land in shared memory with pitch tw), lanes beyond
// tw idle.  A tile step costs ~1.4 us whatever its width against 1.9 us of memory time for a full 256 x 8 tile, so a narrow
// remainder tile is nearly as expensive as a full one: equal tiles (320^3: 259 -> 252 us) and, more so, the 128 x 16 tile for
// widths that fill 256-wide tiles badly (252 -> 230 us; FCfg3DN below) keep more of every step's lanes busy.
// r = ca * p1 + cb * p2 (ca in {0, 1}: exact)
__device__ __forceinline__ float4 rec4(float ca, const float4& p1, float cb, const float4& p2) {
    return make_float4(fmaf(cb, p2.x, ca * p1.x), fmaf(cb, p2.y, ca * p1.y), fmaf(cb, p2.z, ca * p1.z), fmaf(cb, p2.w, ca * p1.w));
}

template <class C, bool PERSIST, bool NARROW>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_cg_fused_tma(const __grid_constant__ pn_fmaps maps, pn_geom g, pn_ptrs P, int ntx, int nty, int nchunks, int lz,
               int max_launch_iters, int tw) {
    static_assert(!NARROW || C::NBX == 1, "equal narrow tiles: one box per tile");
    const int bw = NARROW ? tw : C::BOXW;        // pitch of a box row in shared memory = tile width
    const int txw = NARROW ? tw : C::TXW;
    pn_state* gst = P.st;
    if (gst->flag != PN_FLAG_RUN) return;
    __shared__ pn_state ls_;                 // PERSIST: this CTA's copy of the iteration state
    __shared__ double red2[4 * 32 + 8];      // PERSIST: warp partials of the four sums
    pn_state* st = PERSIST ? &ls_ : gst;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // The integer round trip on the base pointer makes every tile access a GENERIC load / store (the compiler can no longer
    // prove the shared address space); without it the compiler emits LDS / STS.  Measured, same box (profiles/
    // r01_barrier_placement.md): the 3D tile is 5 % FASTER with the generic form (0.8663 vs 0.9127 ms per iteration at 512^3),
    // the 2D tile 1.2 % faster with LDS (0.03402 vs 0.03447 ms at 2048^2) -- each gets what it measured best with.
    float* stages = C::HAS_Y ? reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023))
                             : reinterpret_cast<float*>(smem_raw);
    if (!C::HAS_Y && (smem_u32(smem_raw) & 127u) != 0u) __trap();   // TMA destinations need 128-byte alignment
    float* ring = stages + C::S * C::STAGE_FLOATS;
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + C::RING_FLOATS);
    uint64_t* empty = full + C::S;
    double* red = reinterpret_cast<double*>(empty + C::S);   // 32 doubles + 4 totals

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < C::S; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, C::NCONS / 32);
        }
        mbar_fence_init();
        if (PERSIST) ls_ = *gst;
    }
    __syncthreads();
    const int tiles = ntx * nty;
    const int total = tiles * nchunks;
    unsigned it = 0;                            // stage counter of this thread's role; runs on across iterations
    unsigned int bar_target = 0;
  for (int li = 0; li < max_launch_iters; ++li) {
    const float beta = (float)st->beta;
    const float al = (float)st->alpha;          // alpha_{t-1} (0 right after a residual replacement)
    const float nal = -al;
    const int par = st->iters & 1;              // buffers holding r_{t-1}, q_{t-1}, p_{t-1}
    // The residual is NOT stored (36 instead of 40 bytes per node and iteration).  Three direction slots {P.p, P.p2, P.r}
    // rotate with the iteration count: p_{t-1} in slot s1, p_{t-2} in s2, p_t goes to s0, and the kernel recovers
    //     r_{t-1} = p_{t-1} - beta_{t-1} p_{t-2}        (p_{t-1} = r_{t-1} + beta_{t-1} p_{t-2} read backwards; ca = 1, cb = -beta_{t-1})
    // Right after a residual replacement slot s2 holds the explicit residual k_residual64 wrote: ca = 0, cb = 1.  The recovered
    // residual differs from a stored one by a rounding of the size of ulp(p); iteration counts are unchanged.
    const int s1 = st->iters % 3, s2 = (st->iters + 2) % 3, s0 = (st->iters + 1) % 3;
    const float ca = st->rexp ? 0.f : 1.f;
    const float cb = st->rexp ? 1.f : -(float)st->beta_last;
    const float a2 = (float)st->alpha2;
    // x_hat is touched every OTHER iteration: xmode 0 = skip (alpha_{t-1} p_{t-1} stays owed), 2 = apply this
    // iteration's update and the owed one alpha_{t-2} p_{t-2}, whose direction this kernel loads anyway; 1 = plain update
    // (skipping disabled; a small beta also ends a skip, as in the kernels that recover p_{t-2} by a division).
    const int xmode = st->xpend ? 2 : ((st->xskip_min > 0.0 && st->beta >= st->xskip_min) ? 0 : 1);
    float* __restrict__ q_out = par ? P.q : P.q2;
    float* __restrict__ p_out = s0 == 0 ? P.p : (s0 == 1 ? P.p2 : P.r);
    double a_rr = 0.0, a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;

    if (tid >= C::NCONS) {
        // ================= producer warp: one elected lane issues every TMA load =================
        if (tid == C::NCONS) {
            if (PERSIST) asm volatile("fence.proxy.async;" ::: "memory");   // other CTAs' stores of the last iteration -> this one's TMA loads
            for (int item = blockIdx.x; item < total; item += gridDim.x) {
                const int chunk = item / tiles, t = item - chunk * tiles;
                const int tyi = t / ntx, txi = t - tyi * ntx;
                const int x0 = txi * txw, y0 = tyi * C::TY;
                // z-chunks: nchunks equal parts (3D tiles; 32-bit: chunk < 1200, nz < 2^21); fixed length lz, ragged last chunk (2D tile).  A compile-time choice:
                // the 2D instantiation is sensitive to its code generation (a run-time choice here cost it 27 %, 98 -> 125 us
                // per iteration at 4096^2, with 85 instead of 76 registers and the same chunks)
                const int k0 = C::HAS_Y ? (int)((unsigned)chunk * (unsigned)g.nz / (unsigned)nchunks) : chunk * lz;
                const int k1 = C::HAS_Y ? (int)((unsigned)(chunk + 1) * (unsigned)g.nz / (unsigned)nchunks) : min(k0 + lz, g.nz);
                const int yh = y0 - (C::HAS_Y ? 1 : 0);
                const unsigned b_rqp = NARROW ? 3u * (unsigned)(C::RH * bw + 2 * C::RH * 4) * 4u : C::B_RQP;
                const unsigned b_w = NARROW ? (unsigned)(C::TY * bw + C::TY * 4 + (C::HAS_Y ? C::RWY * bw : 0)) * 4u : C::B_W;
                const unsigned b_wz = NARROW ? (unsigned)(C::TY * bw) * 4u : C::B_WZ;
                for (int kk = k0 - 2; kk < k1; ++kk, ++it) {
                    const int s = it % C::S;
                    const unsigned ph = (it / C::S) & 1u;
                    mbar_wait(empty + s, ph ^ 1u);
                    float* sg = stages + s * C::STAGE_FLOATS;
                    const bool has_w = kk >= k0;
                    const bool has_wz = kk >= k0 - 1;
                    mbar_expect_tx(full + s, b_rqp + (has_w ? b_w : 0u) + (has_wz ? b_wz : 0u));
                    const int zp = kk + 2;   // plane kk+1 (+1: the tensor maps start at the leading halo plane)
                    const int zw = kk + 1;   // plane kk
#pragma unroll
                    for (int v = 0; v < 3; ++v) {
                        float* sv = sg + v * C::VEC;
                        // stage regions R_, Q_, P_: p_{t-2} (or the explicit residual), q_{t-1}, p_{t-1}; directions by slot, q by parity
                        const int sl = v == 0 ? s2 : s1;
                        const CUtensorMap* mm = v != 1 ? (sl == 2 ? &maps.v_main[0][0] : &maps.v_main[2][sl]) : &maps.v_main[1][par];
                        const CUtensorMap* ms = v != 1 ? (sl == 2 ? &maps.v_slv[0][0] : &maps.v_slv[2][sl]) : &maps.v_slv[1][par];
#pragma unroll
                        for (int b = 0; b < C::NBX; ++b)
                            tma_load_3d(sv + b * C::RH * C::BOXW, mm, x0 + b * C::BOXW, yh, zp, full + s);
                        tma_load_3d(sv + C::V_SL, ms, x0 - 4, yh, zp, full + s);
                        tma_load_3d(sv + C::V_SR, ms, x0 + txw, yh, zp, full + s);
                    }
                    if (has_w) {
#pragma unroll
                        for (int b = 0; b < C::NBX; ++b) {
                            tma_load_3d(sg + C::WX + b * C::TY * C::BOXW, &maps.wx_main, x0 + b * C::BOXW, y0, zw, full + s);
                            if (C::HAS_Y)
                                tma_load_3d(sg + C::WY + b * C::RWY * C::BOXW, &maps.wy, x0 + b * C::BOXW, yh, zw, full + s);
                        }
                        tma_load_3d(sg + C::WX_SL, &maps.wx_slv, x0 - 4, y0, zw, full + s);
                    }
                    if (has_wz) {
#pragma unroll
                        for (int b = 0; b < C::NBX; ++b)
                            tma_load_3d(sg + C::WZ + b * C::TY * C::BOXW, &maps.wz, x0 + b * C::BOXW, y0, zw, full + s);
                    }
                }
            }
        }
    } else {
        // ================= consumer warps ==========================================================
        const int lane = tid & 31;
        const int tx = tid % (C::LPR * C::NBX), ty = tid / (C::LPR * C::NBX);
        const int b = tx / C::LPR, c4 = tx % C::LPR;
        const int rrow = ty + (C::HAS_Y ? 1 : 0);               // own row in the haloed arrays
        const int rcol = 4 + b * C::BOXW + c4 * 4;              // own column in a ring row
        const int own_main = (b * C::RH + rrow) * bw + c4 * 4;   // own float4 inside the r / q / p main boxes
        const int own_ty = (b * C::TY + ty) * bw + c4 * 4;       // own float4 inside the wx / wz boxes
        const bool act = !NARROW || c4 * 4 < tw;                 // lanes beyond a narrow tile's width idle
        // the float4 of the two halo rows this thread also owns in phase A (the LAST warps take them)
        const int hidx = tid - (C::NCONS - C::NHALO4);
        const bool has_halo = C::HAS_Y && hidx >= 0;
        const int hb = has_halo ? hidx / (2 * C::LPR) : 0;
        const int hrow = has_halo ? (((hidx / C::LPR) & 1) ? C::RH - 1 : 0) : 0;
        const int hc4 = hidx % C::LPR;
        for (int item = blockIdx.x; item < total; item += gridDim.x) {
            const int chunk = item / tiles, t = item - chunk * tiles;
            const int tyi = t / ntx, txi = t - tyi * ntx;
            const int x0 = txi * txw, y0 = tyi * C::TY;
            const int k0 = C::HAS_Y ? (int)((unsigned)chunk * (unsigned)g.nz / (unsigned)nchunks) : chunk * lz;
            const int k1 = C::HAS_Y ? (int)((unsigned)(chunk + 1) * (unsigned)g.nz / (unsigned)nchunks) : min(k0 + lz, g.nz);
            const int x = x0 + b * C::BOXW + c4 * 4, y = y0 + ty;
            const bool inb = act && (x < g.px) && (y < g.ny);
            const long long nrow = (long long)y * g.px + x;
            float4 wzm = make_float4(0.f, 0.f, 0.f, 0.f);
            float4 r_cur = make_float4(0.f, 0.f, 0.f, 0.f);     // r_t on the own float4 of plane kk
            float4 xh_nxt = make_float4(0.f, 0.f, 0.f, 0.f);    // x_hat of plane kk+1, fetched one step ahead
            if (inb && xmode) xh_nxt = __ldcs(reinterpret_cast<const float4*>(P.xh + (long long)k0 * g.plane + nrow));
            bar_consumers(C::NCONS);   // the ring is rebuilt per item: nobody may still read the previous item's planes
            for (int kk = k0 - 2; kk < k1; ++kk, ++it) {
                const int s = it % C::S;
                const unsigned ph = (it / C::S) & 1u;
                // x_hat of plane kk+2 goes in flight now and is used one step later
                const float4 xh_use = xh_nxt;
                if (inb && xmode && kk + 2 >= k0 + 1 && kk + 2 < k1)
                    xh_nxt = __ldcs(reinterpret_cast<const float4*>(P.xh + (long long)(kk + 2) * g.plane + nrow));
                mbar_wait(full + s, ph);
                const float* sg = stages + s * C::STAGE_FLOATS;
                // ---- phase A: r_t, p_t on plane kk+1 (tile and halo) -> ring; own part -> HBM ----
                float* rw = ring + ((kk + 5) & 3) * (C::RH * C::W);
                float4 r_nxt;
                {
                    const float4 po = lds4(sg + C::P_ + own_main);
                    const float4 pR = lds4(sg + C::R_ + own_main);      // p_{t-2} (or the explicit residual)
                    const float4 ro = rec4(ca, po, cb, pR);              // r_{t-1}
                    r_nxt = fma4(nal, lds4(sg + C::Q_ + own_main), ro);
                    const float4 pn = fma4(beta, po, r_nxt);
                    if (act) *reinterpret_cast<float4*>(rw + rrow * C::W + rcol) = pn;
                    if (kk + 1 >= k0 && kk + 1 < k1 && inb) {
                        const long long n = (long long)(kk + 1) * g.plane + nrow;
                        __stcs(reinterpret_cast<float4*>(p_out + n), pn);
                        if (xmode) {
                            float4 xn = fma4(al, po, xh_use);
                            if (xmode == 2) xn = fma4(a2, pR, xn);      // the owed direction p_{t-2} is in the stage as it is
                            __stcs(reinterpret_cast<float4*>(P.xh + n), xn);
                        }
                        a_rr += (double)dot4(r_nxt, r_nxt);
                    }
                }
                if (has_halo && (!NARROW || hc4 * 4 < tw)) {
                    const int o = (hb * C::RH + hrow) * bw + hc4 * 4;
                    const float4 ph = lds4(sg + C::P_ + o), pRh = lds4(sg + C::R_ + o);
                    const float4 rn = fma4(nal, lds4(sg + C::Q_ + o), rec4(ca, ph, cb, pRh));
                    *reinterpret_cast<float4*>(rw + hrow * C::W + 4 + hb * C::BOXW + hc4 * 4) = fma4(beta, ph, rn);
                }
                if (tid < 2 * C::RH) {
                    const int side = tid / C::RH, row = tid - side * C::RH;
                    const int o = (side ? C::V_SR : C::V_SL) + row * 4;
                    const float4 ps = lds4(sg + C::P_ + o), pRs = lds4(sg + C::R_ + o);
                    const float4 rn = fma4(nal, lds4(sg + C::Q_ + o), rec4(ca, ps, cb, pRs));
                    *reinterpret_cast<float4*>(rw + row * C::W + (side ? 4 + txw : 0)) = fma4(beta, ps, rn);
                }
                if (!C::BAR_END) bar_consumers(C::NCONS);
                // ---- phase C: q_t(kk) = p_t - W p_t from the ring, weights from the stage.  Of plane kk+1, written just above,
                // it reads only this thread's own float4; everything it reads from other threads belongs to planes kk and kk-1,
                // complete since the barrier that ended the previous step: no barrier is NEEDED between the phases ----
                if (kk >= k0) {
                    const float* r0 = ring + ((kk + 4) & 3) * (C::RH * C::W) + rrow * C::W + rcol;
                    const float4 pc = lds4(r0);
                    const float4 pzm = lds4(ring + ((kk + 3) & 3) * (C::RH * C::W) + rrow * C::W + rcol);
                    const float4 pzp = lds4(rw + rrow * C::W + rcol);
                    float pl = __shfl_up_sync(0xffffffffu, pc.w, 1);
                    float pr = __shfl_down_sync(0xffffffffu, pc.x, 1);
                    if (lane == 0 || (C::LPR < 32 && c4 == 0)) pl = r0[-1];          // (c4 tests: a warp holds two rows when LPR == 16)
                    if (lane == 31 || (C::LPR < 32 && c4 == C::LPR - 1)) pr = r0[4];
                    const float4 gx = lds4(sg + C::WX + own_ty);
                    float gxl = __shfl_up_sync(0xffffffffu, gx.w, 1);
                    if (lane == 0 || (C::LPR < 32 && c4 == 0)) {
                        if (c4 != 0) gxl = sg[C::WX + own_ty - 1];
                        else if (b != 0) gxl = sg[C::WX + ((b - 1) * C::TY + ty) * C::BOXW + C::BOXW - 1];   // (b != 0: never NARROW)
                        else gxl = sg[C::WX_SL + ty * 4 + 3];
                    }
                    const float4 gz = lds4(sg + C::WZ + own_ty);
                    float4 q;
                    q.x = gxl * pl + gx.x * pc.y + wzm.x * pzm.x + gz.x * pzp.x;
                    q.y = gx.x * pc.x + gx.y * pc.z + wzm.y * pzm.y + gz.y * pzp.y;
                    q.z = gx.y * pc.y + gx.z * pc.w + wzm.z * pzm.z + gz.z * pzp.z;
                    q.w = gx.z * pc.z + gx.w * pr + wzm.w * pzm.w + gz.w * pzp.w;
                    if (C::HAS_Y) {
                        const float4 pym = lds4(r0 - C::W), pyp = lds4(r0 + C::W);
                        const int oy = (b * C::RWY + ty) * bw + c4 * 4;   // row ty of the wy box = lattice row y-1
                        const float4 gym = lds4(sg + C::WY + oy), gy = lds4(sg + C::WY + oy + bw);
                        q.x += gym.x * pym.x + gy.x * pyp.x;
                        q.y += gym.y * pym.y + gy.y * pyp.y;
                        q.z += gym.z * pym.z + gy.z * pyp.z;
                        q.w += gym.w * pym.w + gy.w * pyp.w;
                    }
                    q.x = pc.x - q.x; q.y = pc.y - q.y; q.z = pc.z - q.z; q.w = pc.w - q.w;
                    if (inb) {
                        __stcs(reinterpret_cast<float4*>(q_out + (long long)kk * g.plane + nrow), q);
                        a_pq += (double)dot4(pc, q);
                        a_rq += (double)dot4(r_cur, q);
                        a_qq += (double)dot4(q, q);
                    }
                    wzm = gz;
                } else if (kk == k0 - 1) {
                    wzm = lds4(sg + C::WZ + own_ty);   // wz(k0-1): the backward z bond of the first plane
                }
                r_cur = r_nxt;
                if (C::BAR_END) bar_consumers(C::NCONS);   // plane kk+1 of the ring complete before the next step's phase C reads its rows
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + s);
            }
        }
    }
    if (!PERSIST) {
        // ---- the four sums: warp -> block -> grid; the last block computes alpha_t and beta_{t+1} ----
        a_rr = pn_block_sum(a_rr, red);
        a_pq = pn_block_sum(a_pq, red);
        a_rq = pn_block_sum(a_rq, red);
        a_qq = pn_block_sum(a_qq, red);
        const double v4[4] = {a_rr, a_pq, a_rq, a_qq};
        if (pn_grid_sum<4>(v4, P.slots, &st->ticket, red, red + 32)) {
            if (threadIdx.x == 0) {
                if (g.wrap[0] | g.wrap[1] | g.wrap[2]) {   // periodic faces: k_wrap_fix adds the wrap bonds' part and finishes
                    st->part[0] = red[32]; st->part[1] = red[33]; st->part[2] = red[34]; st->part[3] = red[35];
                } else pn_finish_F(st, red[32], red[33], red[34], red[35]);
            }
        }
        return;
    }
    // ---- PERSIST: warp -> CTA -> slots [parity][CTA][4] -> grid barrier -> every CTA adds the slots in the same order ----
    {
        const int lane = tid & 31, wid = tid >> 5, pin = li & 1, G = (int)gridDim.x, c = (int)blockIdx.x;
        a_rr = pn_warp_sum(a_rr); a_pq = pn_warp_sum(a_pq); a_rq = pn_warp_sum(a_rq); a_qq = pn_warp_sum(a_qq);
        if (lane == 0) { red2[wid] = a_rr; red2[32 + wid] = a_pq; red2[64 + wid] = a_rq; red2[96 + wid] = a_qq; }
        __syncthreads();
        if (wid == 0) {
            constexpr int NW = C::NTHREADS / 32;
            double* my = P.slots + ((size_t)pin * PN_MAX_BLOCKS + c) * 4;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double v = pn_warp_sum(lane < NW ? red2[32 * k + lane] : 0.0);
                if (lane == 0) my[k] = v;
            }
            if (lane == 0) { bar_target += G; ft_grid_barrier(P.gbar, bar_target); }
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
            if (lane == 0) pn_finish_F(&ls_, t0, t1, t2, t3);
        }
        __syncthreads();
        if (ls_.flag != PN_FLAG_RUN) break;
    }
  }
    if (PERSIST && blockIdx.x == 0 && tid == 0) *gst = ls_;
}

// ---- host side ----------------------------------------------------------------------------------------
// width of the (equal) x tiles: 256-wide boxes per tile unless one box covers a tile and the width does not fill the last one
template <class C>
int tile_width(const pn_geom& g) {
    if (C::NBX != 1 || g.px % C::BOXW == 0) return C::TXW;
    const int ntx = (g.px + C::BOXW - 1) / C::BOXW;
    return ((g.px + ntx - 1) / ntx + 3) / 4 * 4;
}

template <class C>
bool build_maps(pn_fmaps* M, const pn_geom& g, const pn_ptrs& P) {
    const long long h = g.plane;
    const int bw = C::NBX == 1 ? tile_width<C>(g) : C::BOXW;
    const float* vec[3][2] = {{P.r, P.r2}, {P.q, P.q2}, {P.p, P.p2}};
    bool ok = true;
    for (int v = 0; v < 3; ++v)
        for (int bsel = 0; bsel < 2; ++bsel) {
            ok &= make_map(&M->v_main[v][bsel], g, vec[v][bsel] - h, bw, C::RH);
            ok &= make_map(&M->v_slv[v][bsel], g, vec[v][bsel] - h, 4, C::RH);
        }
    ok &= make_map(&M->wx_main, g, P.w[0] - h, bw, C::TY);
    ok &= make_map(&M->wx_slv, g, P.w[0] - h, 4, C::TY);
    ok &= make_map(&M->wy, g, P.w[1] - h, bw, C::RWY);
    ok &= make_map(&M->wz, g, P.w[2] - h, bw, C::TY);
    return ok;
}

template <class C>
cudaError_t launch_cfg(const pn_geom& g, const pn_ptrs& P, const pn_fmaps& M, int max_launch_iters, cudaStream_t st) {
    const int tw = tile_width<C>(g);
    const bool narrow = tw != C::TXW;
    const int ntx = (g.px + tw - 1) / tw, nty = (g.ny + C::TY - 1) / C::TY;
    const int sms = g.sms;
    // 3D tiles: equal z-chunks (choose_chunks); the 2D tile keeps round 1's fixed chunk length with a ragged last chunk (see
    // the kernel: its instantiation must not change)
    const int lz = C::HAS_Y ? 0 : choose_lz(g.nz, ntx * nty, sms, 44.0, 24.0);
    const int nchunks = C::HAS_Y ? choose_chunks(g.nz, ntx * nty, sms) : (g.nz + lz - 1) / lz;
    const long long total = (long long)ntx * nty * nchunks;
    const int nb = (int)(total < sms ? total : sms);
    if (max_launch_iters <= 0) {   // one iteration per launch
        if (narrow) k_cg_fused_tma<C, false, C::NBX == 1><<<nb, C::NTHREADS, C::SMEM_BYTES, st>>>(M, g, P, ntx, nty, nchunks, lz, 1, tw);
        else k_cg_fused_tma<C, false, false><<<nb, C::NTHREADS, C::SMEM_BYTES, st>>>(M, g, P, ntx, nty, nchunks, lz, 1, tw);
        return cudaGetLastError();
    }
    cudaError_t e = cudaMemsetAsync(P.gbar, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    pn_fmaps MM = M;
    pn_geom gg = g;
    pn_ptrs PP = P;
    int a_ntx = ntx, a_nty = nty, a_nch = nchunks, a_lz = lz, a_mi = max_launch_iters, a_tw = tw;
    void* args[] = {(void*)&MM, (void*)&gg, (void*)&PP, (void*)&a_ntx, (void*)&a_nty, (void*)&a_nch, (void*)&a_lz, (void*)&a_mi, (void*)&a_tw};
    const void* fn = narrow ? (const void*)k_cg_fused_tma<C, true, C::NBX == 1> : (const void*)k_cg_fused_tma<C, true, false>;
    return cudaLaunchCooperativeKernel(fn, dim3(nb), dim3(C::NTHREADS), args, C::SMEM_BYTES, st);
}

typedef FCfg<1, 8, true, 3> FCfg3D;    // 256 x 8 tile, y halo, 3 stages
typedef FCfg<1, 16, true, 3, 128> FCfg3DN;   // 128 x 16 tile for widths that fill 256-wide tiles badly (e.g. 320, 384)
typedef FCfg<1, 32, true, 3, 64> FCfg3DS;    // 64 x 32 tile for widths that fill 128-wide tiles badly too (e.g. 192, 320)
typedef FCfg<8, 1, false, 4> FCfg2D;   // 2048 x 1 tile (lattices held as nx x 1 x ny), 4 stages

// fraction of the consumer lanes of a tiling that hold lattice nodes
template <class C>
double lane_efficiency(const pn_geom& g) {
    const int ntx = (g.px + C::TXW - 1) / C::TXW, nty = (g.ny + C::TY - 1) / C::TY;
    return ((double)g.px / ((double)ntx * C::TXW)) * ((double)g.ny / ((double)nty * C::TY));
}

}  // namespace

bool pn_tma_supported() { return get_encoder() != nullptr; }

// cudaFuncSetAttribute is per device: pn_create calls this with the handle's device current
cudaError_t pn_fused_init_device() {
    cudaError_t e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3D, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3D::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3D, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3D::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3D, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3D::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3D, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3D::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DN, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DN::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DN, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DN::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DN, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DN::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DN, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DN::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DS, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DS::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DS, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DS::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DS, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DS::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg3DS, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg3DS::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg2D, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg2D::SMEM_BYTES);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cg_fused_tma<FCfg2D, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg2D::SMEM_BYTES);
    return e;
}

struct pn_fused_plan {
    pn_fmaps maps;
    int kind;      // 0: 2D tile, 1: 256 x 8, 2: 128 x 16, 3: 64 x 32
};

bool pn_fused_plan_build(pn_fused_plan** out, const pn_geom& g, const pn_ptrs& P) {
    if (!get_encoder()) return false;
    pn_fused_plan* pl = new (std::nothrow) pn_fused_plan;
    if (!pl) return false;
    // 3D: a narrower, taller tile where it fills its lanes at least 8 % better than the next wider one; of two that fill
    // equally the wider is the faster (512^3: 0.861 against 0.884 ms per iteration for 256 x 8 / 128 x 16; 256^3: 113.8 against
    // 115.2 us).  Measured with the tile forced (profiles/r02_small_lattices.md): 320^3 252 -> 230 us, 384^3 392 -> 371 us,
    // 260^3 161 -> 143 us with 128 x 16
    if (g.ny == 1) pl->kind = 0;
    else if (g.tile) pl->kind = g.tile;
    else {
        const double e1 = lane_efficiency<FCfg3D>(g), e2 = lane_efficiency<FCfg3DN>(g), e3 = lane_efficiency<FCfg3DS>(g);
        pl->kind = 1;
        double best = e1;
        if (e2 > 1.08 * best) { pl->kind = 2; best = e2; }
        if (e3 > 1.08 * best) { pl->kind = 3; best = e3; }
    }
    const bool ok = pl->kind == 0 ? build_maps<FCfg2D>(&pl->maps, g, P)
                    : (pl->kind == 1 ? build_maps<FCfg3D>(&pl->maps, g, P)
                                     : (pl->kind == 2 ? build_maps<FCfg3DN>(&pl->maps, g, P) : build_maps<FCfg3DS>(&pl->maps, g, P)));
    if (!ok) { delete pl; return false; }
    *out = pl;
    return true;
}

void pn_fused_plan_free(pn_fused_plan* pl) { delete pl; }

// max_launch_iters <= 0: ONE iteration (the launch a CUDA graph replays); > 0: a cooperative launch that iterates up to the
// next trigger (no periodic faces)
cudaError_t pn_launch_cg_fused(const pn_fused_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st, int max_launch_iters) {
    if (pl->kind == 0) return launch_cfg<FCfg2D>(g, P, pl->maps, max_launch_iters, st);
    if (pl->kind == 1) return launch_cfg<FCfg3D>(g, P, pl->maps, max_launch_iters, st);
    return pl->kind == 2 ? launch_cfg<FCfg3DN>(g, P, pl->maps, max_launch_iters, st) : launch_cfg<FCfg3DS>(g, P, pl->maps, max_launch_iters, st);
}
