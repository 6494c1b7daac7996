// pn_fused2_tma.cu -- the fp32 inner CG iteration (SURVEY.md 8(a) S4 + S5 + S6) as ONE kernel that never
// stores q = A p: 32 B per node-iteration on average instead of the 40 B of pn_fused_tma.cu.
//
// pn_fused_tma.cu writes q_t in iteration t only to read it back in iteration t+1 for the deferred residual
// update r_{t+1} = r_t - alpha_t q_t.  Here iteration t+1 RECOMPUTES q_t = p_t - W p_t from p_t, which it loads
// anyway (it needs it for p_{t+1} = r_{t+1} + beta p_t), on its tile plus a one-node halo; the operator is
// applied twice per node and iteration (once to the old direction for the residual, once to the new one for the
// dot products), the SMs have the room (the 40 B kernel issues on 27 % of the cycles), HBM does not:
//
//   kernel G(t):   q_{t-1} = p_{t-1} - W p_{t-1}                 tile + 1-node halo, from p_{t-1} on tile + 2-node halo
//                  r_t = r_{t-1} - alpha_{t-1} q_{t-1}           tile + halo
//                  p_t = r_t + beta_t p_{t-1}                    tile + halo -> shared-memory plane ring
//                  x_hat: every other iteration, as in pn_fused_tma.cu (PN_OPT_XDEFER)
//                  q_t = p_t - W p_t                             tile, registers only
//                  sums:  rr = r_t.r_t   pq = p_t.q_t   rq = r_t.q_t   qq = q_t.q_t   -> alpha_t, predicted beta_{t+1}
//
// HBM bytes per node: reads r, p, wx, wy, wz (20 B) + writes r, p (8 B) + x_hat (8 B every other iteration) = 32 B.
// The recomputed q on a halo node is bit-identical to the one its owner tile computes: both run stencil1() below.
//
// 2.5D: a CTA owns an (x, y) tile of 256 x 8 nodes and marches along z.  Two TMA rings with their own mbarriers:
//   P ring (4 slots): one plane of p_old, 12 rows (2-node y halo) + two 4-float x slivers
//   G ring (3 slots): one plane of r_old, wx, wz (10 rows each) and wy (11 rows) + slivers
// and a 4-plane shared-memory ring of p_new (10 rows).  Step a of the march: A = {q_old, r_new, p_new} on plane a
// (needs p_old(a-1..a+1), G(a), wz(a-1)), then C = {q_new, dot products} on plane a-1 (needs p_new(a-2..a), the
// weights of plane a-1 and wz(a-2), carried in registers).
// Not for periodic lateral faces (k_wrap_fix corrects a stored q) nor for 2D lattices: those stay on pn_fused_tma.cu.
#include <new>

#include "pn_tma.cuh"

namespace {

using namespace pn_tma;

template <int TY_, int SG_>
struct GCfg {
    static constexpr int BOXW = 256, TY = TY_;
    static constexpr int PR = TY + 4;                      // p_old rows  y0-2 .. y0+TY+1
    static constexpr int RR = TY + 2;                      // r, wx, wz, p_new rows  y0-1 .. y0+TY
    static constexpr int WYR = TY + 3;                     // wy rows  y0-2 .. y0+TY
    static constexpr int W = BOXW + 8;                     // p_new ring row: 4 pad + tile + 4 pad floats
    static constexpr int NCONS = 64 * TY;                  // consumer threads: one float4 of an own row each, plus ONE node of the
                                                           // two halo rows (2 x 256 nodes = NCONS) for step A
    static constexpr int NTHREADS = NCONS + 32;            // + one producer warp
    static constexpr int SP = 4, SG = SG_;                 // ring depths
    // P slot (floats)
    static constexpr int P_SL = PR * BOXW, P_SR = P_SL + a32(PR * 4), P_FLOATS = P_SR + a32(PR * 4);
    // G slot (floats): r | wx | wz | wy, each main box then left and right sliver
    static constexpr int V10 = RR * BOXW + 2 * a32(RR * 4);
    static constexpr int V10_SL = RR * BOXW, V10_SR = V10_SL + a32(RR * 4);
    static constexpr int R_ = 0, WX = V10, WZ = 2 * V10, WY = 3 * V10;
    static constexpr int WY_SL = WYR * BOXW, WY_SR = WY_SL + a32(WYR * 4);
    static constexpr int G_FLOATS = WY + WY_SR + a32(WYR * 4);
    static constexpr int RING_FLOATS = 4 * RR * W;   // 4 planes: step A of the next plane may start while a slower warp still reads a-2
    static constexpr size_t SMEM_BYTES = (size_t)(SP * P_FLOATS + SG * G_FLOATS + RING_FLOATS) * 4 + 2 * (SP + SG) * 8 + 64 * 8 + 1024;
    static constexpr unsigned B_P = (PR * BOXW + 2 * PR * 4) * 4u;
    static constexpr unsigned B_G = (3 * (RR * BOXW + 2 * RR * 4) + WYR * BOXW + 2 * WYR * 4) * 4u;
};

struct alignas(64) pn_gmaps {
    CUtensorMap p_main[2], p_slv[2], r_main[2], r_slv[2];   // [buffer]
    CUtensorMap wx_main, wx_slv, wz_main, wz_slv, wy_main, wy_slv;
};

// q at one node: the 7-point operator of the scaled system.  ONE definition, used for own nodes, halo rows and
// halo columns, so that a node's q has the same bits whichever tile computes it.
__device__ __forceinline__ float stencil1(float pc, float pl, float pr, float pym, float pyp, float pzm, float pzp, float gxl,
                                          float gx, float gym, float gy, float gzm, float gz) {
    float s = __fmul_rn(gxl, pl);
    s = fmaf(gx, pr, s);
    s = fmaf(gzm, pzm, s);
    s = fmaf(gz, pzp, s);
    s = fmaf(gym, pym, s);
    s = fmaf(gy, pyp, s);
    return __fsub_rn(pc, s);
}

// the operator on a float4 of consecutive nodes; pl / pr = the nodes left of .x / right of .w, gxl = the bond left of .x
__device__ __forceinline__ float4 stencil4(const float4& pc, float pl, float pr, const float4& pym, const float4& pyp,
                                           const float4& pzm, const float4& pzp, float gxl, const float4& gx, const float4& gym,
                                           const float4& gy, const float4& gzm, const float4& gz) {
    float4 q;
    q.x = stencil1(pc.x, pl, pc.y, pym.x, pyp.x, pzm.x, pzp.x, gxl, gx.x, gym.x, gy.x, gzm.x, gz.x);
    q.y = stencil1(pc.y, pc.x, pc.z, pym.y, pyp.y, pzm.y, pzp.y, gx.x, gx.y, gym.y, gy.y, gzm.y, gz.y);
    q.z = stencil1(pc.z, pc.y, pc.w, pym.z, pyp.z, pzm.z, pzp.z, gx.y, gx.z, gym.z, gy.z, gzm.z, gz.z);
    q.w = stencil1(pc.w, pc.z, pr, pym.w, pyp.w, pzm.w, pzp.w, gx.z, gx.w, gym.w, gy.w, gzm.w, gz.w);
    return q;
}

template <class C>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_cg_fused2_tma(const __grid_constant__ pn_gmaps maps, pn_geom g, pn_ptrs P, int ntx, int nty, int nchunks, int lz) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // no integer round trip on the base pointer: the compiler then proves the shared address space itself (LDS / STS, free
    // to schedule); TMA destinations need 128-byte alignment, checked rather than assumed
    float* pslots = reinterpret_cast<float*>(smem_raw);
    if ((smem_u32(smem_raw) & 127u) != 0u) __trap();
    float* gslots = pslots + C::SP * C::P_FLOATS;
    float* ring = gslots + C::SG * C::G_FLOATS;
    uint64_t* fullP = reinterpret_cast<uint64_t*>(ring + C::RING_FLOATS);
    uint64_t* emptyP = fullP + C::SP;
    uint64_t* fullG = emptyP + C::SP;
    uint64_t* emptyG = fullG + C::SG;
    double* red = reinterpret_cast<double*>(emptyG + C::SG);   // 32 doubles + 4 totals

    const int tid = threadIdx.x;
    const float beta = (float)st->beta;
    const float al = (float)st->alpha;          // alpha_{t-1} (0 right after a residual replacement)
    const float nal = -al;
    const int par = st->iters & 1;              // buffers holding r_{t-1}, p_{t-1}
    // x_hat every other iteration: same rule and same state as pn_fused_tma.cu (see there)
    const int xmode = st->xpend ? 2 : ((st->xskip_min > 0.0 && st->beta >= st->xskip_min) ? 0 : 1);
    const float c2 = xmode == 2 ? (float)(st->alpha2 / st->beta_prev) : 0.f;
    float* __restrict__ r_out = par ? P.r : P.r2;
    float* __restrict__ p_out = par ? P.p : P.p2;

    if (tid == 0) {
        for (int s = 0; s < C::SP; ++s) { mbar_init(fullP + s, 1); mbar_init(emptyP + s, C::NCONS / 32); }
        for (int s = 0; s < C::SG; ++s) { mbar_init(fullG + s, 1); mbar_init(emptyG + s, C::NCONS / 32); }
        mbar_fence_init();
    }
    __syncthreads();

    const int tiles = ntx * nty;
    const int total = tiles * nchunks;
    double a_rr = 0.0, a_pq = 0.0, a_rq = 0.0, a_qq = 0.0;

    if (tid >= C::NCONS) {
        // ================= producer warp: one elected lane issues every TMA load =================
        if (tid == C::NCONS) {
            unsigned itP = 0, itG = 0;
            for (int item = blockIdx.x; item < total; item += gridDim.x) {
                const int chunk = item / tiles, t = item - chunk * tiles;
                const int tyi = t / ntx, txi = t - tyi * ntx;
                const int x0 = txi * C::BOXW, y0 = tyi * C::TY, k0 = chunk * lz;
                const int k1 = min(k0 + lz, g.nz);
                for (int z = k0 - 2; z <= k1 + 1; ++z) {
                    const int zc = z + 1;   // the tensor maps start at the leading halo plane
                    {
                        const int s = itP % C::SP;
                        mbar_wait(emptyP + s, ((itP / C::SP) & 1u) ^ 1u);
                        mbar_expect_tx(fullP + s, C::B_P);
                        float* d = pslots + s * C::P_FLOATS;
                        tma_load_3d(d, &maps.p_main[par], x0, y0 - 2, zc, fullP + s);
                        tma_load_3d(d + C::P_SL, &maps.p_slv[par], x0 - 4, y0 - 2, zc, fullP + s);
                        tma_load_3d(d + C::P_SR, &maps.p_slv[par], x0 + C::BOXW, y0 - 2, zc, fullP + s);
                        ++itP;
                    }
                    if (z <= k1) {
                        const int s = itG % C::SG;
                        mbar_wait(emptyG + s, ((itG / C::SG) & 1u) ^ 1u);
                        mbar_expect_tx(fullG + s, C::B_G);
                        float* d = gslots + s * C::G_FLOATS;
                        tma_load_3d(d + C::R_, &maps.r_main[par], x0, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::R_ + C::V10_SL, &maps.r_slv[par], x0 - 4, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::R_ + C::V10_SR, &maps.r_slv[par], x0 + C::BOXW, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WX, &maps.wx_main, x0, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WX + C::V10_SL, &maps.wx_slv, x0 - 4, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WX + C::V10_SR, &maps.wx_slv, x0 + C::BOXW, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WZ, &maps.wz_main, x0, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WZ + C::V10_SL, &maps.wz_slv, x0 - 4, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WZ + C::V10_SR, &maps.wz_slv, x0 + C::BOXW, y0 - 1, zc, fullG + s);
                        tma_load_3d(d + C::WY, &maps.wy_main, x0, y0 - 2, zc, fullG + s);
                        tma_load_3d(d + C::WY + C::WY_SL, &maps.wy_slv, x0 - 4, y0 - 2, zc, fullG + s);
                        tma_load_3d(d + C::WY + C::WY_SR, &maps.wy_slv, x0 + C::BOXW, y0 - 2, zc, fullG + s);
                        ++itG;
                    }
                }
            }
        }
    } else {
        // ================= consumer warps: thread = (own row ra = 1..TY of the 10 p_new rows, float4 c4 of the row) =====
        const int lane = tid & 31;
        const int ra = (tid >> 6) + 1, c4 = tid & 63;
        const int o10 = ra * C::BOXW + c4 * 4;                 // own float4 in a 10-row box (r, wx, wz)
        const int oP = (ra + 1) * C::BOXW + c4 * 4;            // own float4 in the 12-row p_old box
        const int oY = (ra + 1) * C::BOXW + c4 * 4;            // own forward-y bonds in the 11-row wy box (row above: - BOXW)
        const int oR = ra * C::W + 4 + c4 * 4;                 // own float4 in a p_new ring plane
        unsigned itP = 0, itG = 0;                             // ring index of P(k0-2) / G(k0-2) of the current item
        for (int item = blockIdx.x; item < total; item += gridDim.x) {
            const int chunk = item / tiles, t = item - chunk * tiles;
            const int tyi = t / ntx, txi = t - tyi * ntx;
            const int x0 = txi * C::BOXW, y0 = tyi * C::TY, k0 = chunk * lz;
            const int k1 = min(k0 + lz, g.nz);
            const int x = x0 + c4 * 4, y = y0 - 1 + ra;
            const bool inb = (x < g.px) && (y < g.ny);
            const long long nrow = (long long)y * g.px + x;
            float4 wzC = make_float4(0.f, 0.f, 0.f, 0.f);       // wz(c-1) for step C
            float4 r_cur = make_float4(0.f, 0.f, 0.f, 0.f);     // r_t on the own float4 of plane a-1
            float4 xh_nxt = make_float4(0.f, 0.f, 0.f, 0.f);    // x_hat of the next own plane, fetched one step ahead
            if (inb && xmode) xh_nxt = *reinterpret_cast<const float4*>(P.xh + (long long)k0 * g.plane + nrow);
            bar_consumers(C::NCONS);   // the p_new ring is rebuilt per item: nobody may still read the previous item's planes
            mbar_wait(fullP + itP % C::SP, (itP / C::SP) & 1u);                    // P(k0-2)
            mbar_wait(fullP + (itP + 1) % C::SP, ((itP + 1) / C::SP) & 1u);        // P(k0-1)
            mbar_wait(fullG + itG % C::SG, (itG / C::SG) & 1u);                    // G(k0-2): its wz only
            // own float4 of p_old(a-1), p_old(a) and of wz(a-1) rotate through registers from plane to plane
            float4 pA_m = lds4(pslots + (itP % C::SP) * C::P_FLOATS + oP);
            float4 pA_c = lds4(pslots + ((itP + 1) % C::SP) * C::P_FLOATS + oP);
            float4 gA_zm = lds4(gslots + (itG % C::SG) * C::G_FLOATS + C::WZ + o10);
            float4 pn_m1 = make_float4(0.f, 0.f, 0.f, 0.f), pn_m2 = pn_m1;   // own p_new(a-1), p_new(a-2)
            for (int a = k0 - 1; a <= k1; ++a) {
                const unsigned iP = itP + (unsigned)(a - (k0 - 2)), iG = itG + (unsigned)(a - (k0 - 2));
                mbar_wait(fullP + (iP + 1) % C::SP, ((iP + 1) / C::SP) & 1u);      // P(a+1)
                mbar_wait(fullG + iG % C::SG, (iG / C::SG) & 1u);                  // G(a)
                const float* Pm = pslots + ((iP - 1) % C::SP) * C::P_FLOATS;
                const float* Pc = pslots + (iP % C::SP) * C::P_FLOATS;
                const float* Pp = pslots + ((iP + 1) % C::SP) * C::P_FLOATS;
                const float* Gc = gslots + (iG % C::SG) * C::G_FLOATS;
                const float* Gm = gslots + ((iG - 1) % C::SG) * C::G_FLOATS;
                float* ringA = ring + ((a + 4) & 3) * (C::RR * C::W);
                const bool own_plane = a >= k0 && a < k1;
                // x_hat of the next own plane goes in flight now and is used one step later
                const float4 xh_use = xh_nxt;
                if (inb && xmode && a + 1 >= k0 + 1 && a + 1 < k1)
                    xh_nxt = *reinterpret_cast<const float4*>(P.xh + (long long)(a + 1) * g.plane + nrow);
                // ---- step A: q_old, r_t, p_t on plane a (10 rows; the two halo columns below) ----
                float4 r_nxt, pn;
                {
                    const float4 pc = pA_c;
                    const float4 pzp = lds4(Pp + oP);
                    float pl = __shfl_up_sync(0xffffffffu, pc.w, 1);
                    float pr = __shfl_down_sync(0xffffffffu, pc.x, 1);
                    if (lane == 0) pl = c4 == 0 ? slds1(Pc + (C::P_SL + (ra + 1) * 4 + 3)) : (*(Pc + (oP - 1)));
                    if (lane == 31) pr = c4 == 63 ? slds1(Pc + (C::P_SR + (ra + 1) * 4)) : (*(Pc + (oP + 4)));
                    const float4 gx = lds4(Gc + C::WX + o10);
                    float gxl = __shfl_up_sync(0xffffffffu, gx.w, 1);
                    if (lane == 0) gxl = c4 == 0 ? (*(Gc + (C::WX + C::V10_SL + ra * 4 + 3))) : (*(Gc + (C::WX + o10 - 1)));
                    const float4 gz = lds4(Gc + C::WZ + o10);
                    const float4 q = stencil4(pc, pl, pr, lds4(Pc + oP - C::BOXW), lds4(Pc + oP + C::BOXW), pA_m, pzp,
                                              gxl, gx, lds4(Gc + C::WY + oY - C::BOXW), lds4(Gc + C::WY + oY), gA_zm, gz);
                    pA_m = pc; pA_c = pzp; gA_zm = gz;
                    const float4 ro = lds4(Gc + C::R_ + o10);       // r_{t-1}
                    r_nxt = fma4(nal, q, ro);
                    pn = fma4(beta, pc, r_nxt);
                    *reinterpret_cast<float4*>(ringA + oR) = (pn);
                    if (inb && own_plane) {
                        const long long n = (long long)a * g.plane + nrow;
                        *reinterpret_cast<float4*>(r_out + n) = r_nxt;
                        *reinterpret_cast<float4*>(p_out + n) = pn;
                        if (xmode) {
                            float4 xn = fma4(al, pc, xh_use);
                            if (xmode == 2)
                                xn = make_float4(fmaf(c2, pc.x - ro.x, xn.x), fmaf(c2, pc.y - ro.y, xn.y),
                                                 fmaf(c2, pc.z - ro.z, xn.z), fmaf(c2, pc.w - ro.w, xn.w));
                            *reinterpret_cast<float4*>(P.xh + n) = xn;
                        }
                        a_rr += (double)dot4(r_nxt, r_nxt);
                    }
                }
                for (int hn = tid; hn < 2 * C::BOXW; hn += C::NCONS) {
                    // nodes of the two halo rows (scalar; same stencil1 as their owner tile runs on them)
                    const int hr = hn < C::BOXW ? 0 : C::RR - 1, hx = hn & (C::BOXW - 1);
                    const int iP = (hr + 1) * C::BOXW + hx, i10 = hr * C::BOXW + hx;
                    const float pc = (*(Pc + (iP)));
                    const float pl = hx == 0 ? slds1(Pc + (C::P_SL + (hr + 1) * 4 + 3)) : (*(Pc + (iP - 1)));
                    const float pr = hx == C::BOXW - 1 ? slds1(Pc + (C::P_SR + (hr + 1) * 4)) : (*(Pc + (iP + 1)));
                    const float gxl = hx == 0 ? (*(Gc + (C::WX + C::V10_SL + hr * 4 + 3))) : (*(Gc + (C::WX + i10 - 1)));
                    const float q = stencil1(pc, pl, pr, (*(Pc + (iP - C::BOXW))), (*(Pc + (iP + C::BOXW))), (*(Pm + (iP))), (*(Pp + (iP))), gxl, (*(Gc + (C::WX + i10))),
                                             (*(Gc + (C::WY + i10))), (*(Gc + (C::WY + i10 + C::BOXW))), (*(Gm + (C::WZ + i10))), (*(Gc + (C::WZ + i10))));
                    const float rn = fmaf(nal, q, (*(Gc + (C::R_ + i10))));
                    ringA[hr * C::W + 4 + hx] = fmaf(beta, pc, rn);
                }
                if (tid < 2 * C::RR) {
                    // the nodes just left (side 0: column x0-1) and right (side 1: column x0+256) of the tile, 10 rows each
                    const int side = tid / C::RR, hr = tid - side * C::RR, hp = hr + 1;
                    const int ps = side ? C::P_SR + hp * 4 : C::P_SL + hp * 4 + 3;        // the node in a p_old sliver
                    const int gs = side ? C::V10_SR + hr * 4 : C::V10_SL + hr * 4 + 3;    // ... in a 10-row sliver
                    const int ys = side ? C::WY_SR + hp * 4 : C::WY_SL + hp * 4 + 3;      // ... in the wy sliver (own row)
                    const float pc = (*(Pc + (ps)));
                    const float pl = side ? (*(Pc + (hp * C::BOXW + C::BOXW - 1))) : (*(Pc + (ps - 1)));
                    const float pr = side ? (*(Pc + (ps + 1))) : (*(Pc + (hp * C::BOXW)));
                    const float gxl = side ? (*(Gc + (C::WX + hr * C::BOXW + C::BOXW - 1))) : (*(Gc + (C::WX + gs - 1)));
                    const float q = stencil1(pc, pl, pr, (*(Pc + (ps - 4))), (*(Pc + (ps + 4))), (*(Pm + (ps))), (*(Pp + (ps))), gxl, (*(Gc + (C::WX + gs))),
                                             (*(Gc + (C::WY + ys - 4))), (*(Gc + (C::WY + ys))), (*(Gm + (C::WZ + gs))), (*(Gc + (C::WZ + gs))));
                    const float rn = fmaf(nal, q, (*(Gc + (C::R_ + gs))));
                    ringA[hr * C::W + (side ? 4 + C::BOXW : 3)] = fmaf(beta, pc, rn);
                }
                // ---- step C: q_t on plane c = a-1; weights of plane c from G(a-1).  It reads, besides this thread's own
                // registers, only rows of ring plane a-1, complete since the barrier that ended the previous step: no
                // barrier between A and C, the two operator applications of a step are independent instruction streams ----
                {
                    const int c = a - 1;
                    const float4 gz = lds4(Gm + C::WZ + o10);
                    if (c >= k0) {
                        const float* r0 = ring + ((c + 4) & 3) * (C::RR * C::W) + oR;
                        const float4 pc = pn_m1;
                        float pl = __shfl_up_sync(0xffffffffu, pc.w, 1);
                        float pr = __shfl_down_sync(0xffffffffu, pc.x, 1);
                        if (lane == 0) pl = (*(r0 + (-1)));
                        if (lane == 31) pr = (*(r0 + (4)));
                        const float4 gx = lds4(Gm + C::WX + o10);
                        float gxl = __shfl_up_sync(0xffffffffu, gx.w, 1);
                        if (lane == 0) gxl = c4 == 0 ? (*(Gm + (C::WX + C::V10_SL + ra * 4 + 3))) : (*(Gm + (C::WX + o10 - 1)));
                        const float4 q = stencil4(pc, pl, pr, lds4(r0 - C::W), lds4(r0 + C::W),
                                                  pn_m2, pn, gxl, gx,
                                                  lds4(Gm + C::WY + oY - C::BOXW), lds4(Gm + C::WY + oY), wzC, gz);
                        if (inb) {
                            a_pq += (double)dot4(pc, q);
                            a_rq += (double)dot4(r_cur, q);
                            a_qq += (double)dot4(q, q);
                        }
                    }
                    wzC = gz;
                }
                r_cur = r_nxt;
                pn_m2 = pn_m1; pn_m1 = pn;
                bar_consumers(C::NCONS);   // ring plane a complete (rows written by other warps) before the next step's C reads it
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(emptyP + (iP - 1) % C::SP);     // P(a-1)
                    mbar_arrive(emptyG + (iG - 1) % C::SG);     // G(a-1)
                }
            }
            // the planes still held at the end of the chunk: P(k1), P(k1+1), G(k1)
            const unsigned nP = (unsigned)(k1 - k0 + 4), nG = (unsigned)(k1 - k0 + 3);
            if (lane == 0) {
                mbar_arrive(emptyP + (itP + nP - 2) % C::SP);
                mbar_arrive(emptyP + (itP + nP - 1) % C::SP);
                mbar_arrive(emptyG + (itG + nG - 1) % C::SG);
            }
            itP += nP;
            itG += nG;
        }
    }
    // ---- the four sums: warp -> block -> grid; the last block computes alpha_t and beta_{t+1} ----
    a_rr = pn_block_sum(a_rr, red);
    a_pq = pn_block_sum(a_pq, red);
    a_rq = pn_block_sum(a_rq, red);
    a_qq = pn_block_sum(a_qq, red);
    const double v4[4] = {a_rr, a_pq, a_rq, a_qq};
    if (pn_grid_sum<4>(v4, P.slots, &st->ticket, red, red + 32)) {
        if (threadIdx.x == 0) pn_finish_F(st, red[32], red[33], red[34], red[35]);
    }
}

template <class C>
bool build_gmaps(pn_gmaps* M, const pn_geom& g, const pn_ptrs& P) {
    const long long h = g.plane;
    const float* pv[2] = {P.p, P.p2};
    const float* rv[2] = {P.r, P.r2};
    bool ok = true;
    for (int b = 0; b < 2; ++b) {
        ok &= make_map(&M->p_main[b], g, pv[b] - h, C::BOXW, C::PR);
        ok &= make_map(&M->p_slv[b], g, pv[b] - h, 4, C::PR);
        ok &= make_map(&M->r_main[b], g, rv[b] - h, C::BOXW, C::RR);
        ok &= make_map(&M->r_slv[b], g, rv[b] - h, 4, C::RR);
    }
    ok &= make_map(&M->wx_main, g, P.w[0] - h, C::BOXW, C::RR);
    ok &= make_map(&M->wx_slv, g, P.w[0] - h, 4, C::RR);
    ok &= make_map(&M->wz_main, g, P.w[2] - h, C::BOXW, C::RR);
    ok &= make_map(&M->wz_slv, g, P.w[2] - h, 4, C::RR);
    ok &= make_map(&M->wy_main, g, P.w[1] - h, C::BOXW, C::WYR);
    ok &= make_map(&M->wy_slv, g, P.w[1] - h, 4, C::WYR);
    return ok;
}

}  // namespace

// 256 x 8 tile, G ring of 3: the loads lead the march by one plane.  GCfg<6, 4> (256 x 6 tile, G ring of 4, a lead of two
// planes, 127 registers) was measured too: 0.9651 vs 0.9665 ms per iteration at 512^3 -- no difference, the kernel is not
// waiting for a longer lead (profiles/r01_q_recompute_experiment.md).
typedef GCfg<8, 3> GC8;

struct pn_fused2_plan {
    pn_gmaps maps;
};

// 3D lattices with no-flux lateral faces only (see the header of this file)
bool pn_fused2_supported(const pn_geom& g) { return g.ny > 1 && !(g.wrap[0] | g.wrap[1] | g.wrap[2]); }

bool pn_fused2_plan_build(pn_fused2_plan** out, const pn_geom& g, const pn_ptrs& P) {
    if (!get_encoder() || !pn_fused2_supported(g)) return false;
    pn_fused2_plan* pl = new (std::nothrow) pn_fused2_plan;
    if (!pl) return false;
    if (!build_gmaps<GC8>(&pl->maps, g, P)) { delete pl; return false; }
    *out = pl;
    return true;
}

void pn_fused2_plan_free(pn_fused2_plan* pl) { delete pl; }

template <class C>
static cudaError_t launch_fused2(const pn_fused2_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_cg_fused2_tma<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const int ntx = (g.px + C::BOXW - 1) / C::BOXW, nty = (g.ny + C::TY - 1) / C::TY;
    const int sms = pn_sm_count();
    // per chunk and node column: 4 extra planes of p, 2 of r and the weights, 1 more of the weights' slot (wz of plane k0-2)
    const int lz = choose_lz(g.nz, ntx * nty, sms, 32.0, 4 * 4.0 + 3 * 16.0, 128);
    const int nchunks = (g.nz + lz - 1) / lz;
    const long long total = (long long)ntx * nty * nchunks;
    const int nb = (int)(total < sms ? total : sms);
    k_cg_fused2_tma<C><<<nb, C::NTHREADS, C::SMEM_BYTES, st>>>(pl->maps, g, P, ntx, nty, nchunks, lz);
    return cudaGetLastError();
}

cudaError_t pn_launch_cg_fused2(const pn_fused2_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st) {
    return launch_fused2<GC8>(pl, g, P, st);
}
