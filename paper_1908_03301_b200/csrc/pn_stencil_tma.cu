// pn_stencil_tma.cu -- S4: the matrix-free stencil kernel of the fp32 inner CG as a
// 2.5D, TMA-fed, warp-specialised persistent kernel for sm_100a.
//
//   p_new = r + beta p_old ;  x_hat += alpha_x p_old ;  q = p_new - W p_new ;  pq = p_new . q
//
// north_star (a): "stages 2.5D tiles in shared memory or via TMA for neighbour reuse, and uses
// coalesced, vectorised HBM loads".  The paper's K2 caches the search vector in shared memory
// because consecutive rows share entries; this kernel does the same for all three axes:
//   * a CTA owns an (x, y) tile of TXW x TY nodes and marches along z over a chunk of planes;
//   * one producer warp streams, per plane, the tiles of r, p_old (with a one-node halo in x and y),
//     x_hat and the three bond-weight arrays into a ring of shared-memory stages with
//     cp.async.bulk.tensor (TMA) + mbarrier transaction counts.  Out-of-lattice parts of a box are
//     zero-filled by the TMA unit, which together with zero bond weights IS the no-flux face;
//   * 16 consumer warps turn each stage into a plane of p_new (halo included) kept in a 4-deep
//     shared-memory ring, so that the seven-point operator at plane k reads p_new(k-1), p_new(k),
//     p_new(k+1) from shared memory: every r, p, w value is fetched from HBM once per tile;
//   * p.Ap is reduced warp -> block -> grid (last block done), alpha stays on the device.
// HBM bytes per node: reads r, p, x_hat, wx, wy, wz (24 B) + writes p, q, x_hat (12 B) = 36 B, plus
// the tile halo (2 rows in TY, 2 planes in the z chunk) which mostly hits L2.
#include <new>

#include "pn_tma.cuh"

namespace {

using namespace pn_tma;

template <int NBX_, int TY_, bool HAS_Y_, int S_>
struct Cfg {
    static constexpr int NBX = NBX_, TY = TY_, S = S_;
    static constexpr bool HAS_Y = HAS_Y_;
    static constexpr int BOXW = 256;                       // TMA box limit per dimension
    static constexpr int TXW = BOXW * NBX;                 // tile width in nodes
    static constexpr int RH = TY + (HAS_Y ? 2 : 0);        // rows of r, p and p_new including the y halo
    static constexpr int RWY = TY + (HAS_Y ? 1 : 0);       // rows of the wy box (backward row included)
    static constexpr int W = TXW + 8;                      // p_new ring row: 4 pad + tile + 4 pad floats
    static constexpr int NCONS = 64 * NBX * TY;            // consumer threads: one float4 of nodes each
    static constexpr int NTHREADS = NCONS + 32;            // + one producer warp
    // stage layout (floats)
    static constexpr int R_MAIN = 0;
    static constexpr int R_SL = R_MAIN + NBX * RH * BOXW;
    static constexpr int R_SR = R_SL + a32(RH * 4);
    static constexpr int P_MAIN = R_SR + a32(RH * 4);
    static constexpr int P_SL = P_MAIN + NBX * RH * BOXW;
    static constexpr int P_SR = P_SL + a32(RH * 4);
    static constexpr int XH = P_SR + a32(RH * 4);
    static constexpr int WX = XH + NBX * TY * BOXW;
    static constexpr int WX_SL = WX + NBX * TY * BOXW;
    static constexpr int WY = WX_SL + a32(TY * 4);
    static constexpr int WZ = WY + (HAS_Y ? NBX * RWY * BOXW : 0);
    static constexpr int STAGE_FLOATS = WZ + NBX * TY * BOXW;
    static constexpr int RING_FLOATS = 4 * RH * W;
    static constexpr size_t SMEM_BYTES = (size_t)(S * STAGE_FLOATS + RING_FLOATS) * 4 + 2 * S * 8 + 64 * 8 + 1024;
    // transaction bytes per group of boxes
    static constexpr unsigned B_RP = 2u * (NBX * RH * BOXW + 2 * RH * 4) * 4u;
    static constexpr unsigned B_XH = NBX * TY * BOXW * 4u;
    static constexpr unsigned B_W = (NBX * TY * BOXW + TY * 4 + (HAS_Y ? NBX * RWY * BOXW : 0)) * 4u;
    static constexpr unsigned B_WZ = NBX * TY * BOXW * 4u;
};

struct alignas(64) pn_tmaps {
    CUtensorMap r_main, r_slv, p_main[2], p_slv[2], xh, wx_main, wx_slv, wy, wz;
};


template <class C>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_stencil_tma(const __grid_constant__ pn_tmaps maps, pn_geom g, pn_ptrs P, int ntx, int nty, int nchunks, int lz) {
    pn_state* st = P.st;
    if (st->flag != PN_FLAG_RUN) return;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    float* stages = reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    float* ring = stages + C::S * C::STAGE_FLOATS;
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + C::RING_FLOATS);
    uint64_t* empty = full + C::S;
    double* red = reinterpret_cast<double*>(empty + C::S);   // 32 doubles + 1 total

    const int tid = threadIdx.x;
    const float beta = (float)st->beta;
    const float ax = (float)st->alpha_x;
    const int par = st->iters & 1;
    float* __restrict__ pout = par ? P.p : P.p2;

    if (tid == 0) {
        for (int s = 0; s < C::S; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, C::NCONS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int tiles = ntx * nty;
    const int total = tiles * nchunks;
    double acc = 0.0;

    if (tid >= C::NCONS) {
        // ================= producer warp: one elected lane issues every TMA load =================
        if (tid == C::NCONS) {
            const CUtensorMap* mp_main = &maps.p_main[par];
            const CUtensorMap* mp_slv = &maps.p_slv[par];
            unsigned it = 0;
            for (int item = blockIdx.x; item < total; item += gridDim.x) {
                const int chunk = item / tiles, t = item - chunk * tiles;
                const int tyi = t / ntx, txi = t - tyi * ntx;
                const int x0 = txi * C::TXW, y0 = tyi * C::TY, k0 = chunk * lz;
                const int k1 = min(k0 + lz, g.nz);
                const int yh = y0 - (C::HAS_Y ? 1 : 0);
                for (int kk = k0 - 2; kk < k1; ++kk, ++it) {
                    const int s = it % C::S;
                    const unsigned ph = (it / C::S) & 1u;
                    mbar_wait(empty + s, ph ^ 1u);
                    float* sg = stages + s * C::STAGE_FLOATS;
                    const bool has_xh = (kk + 1 >= k0) && (kk + 1 < k1);
                    const bool has_w = kk >= k0;
                    const bool has_wz = kk >= k0 - 1;
                    mbar_expect_tx(full + s, C::B_RP + (has_xh ? C::B_XH : 0u) + (has_w ? C::B_W : 0u) + (has_wz ? C::B_WZ : 0u));
                    const int zp = kk + 2;   // plane kk+1 (+1: the tensor maps start at the leading halo plane)
                    const int zw = kk + 1;   // plane kk
#pragma unroll
                    for (int b = 0; b < C::NBX; ++b) {
                        tma_load_3d(sg + C::R_MAIN + b * C::RH * C::BOXW, &maps.r_main, x0 + b * C::BOXW, yh, zp, full + s);
                        tma_load_3d(sg + C::P_MAIN + b * C::RH * C::BOXW, mp_main, x0 + b * C::BOXW, yh, zp, full + s);
                    }
                    tma_load_3d(sg + C::R_SL, &maps.r_slv, x0 - 4, yh, zp, full + s);
                    tma_load_3d(sg + C::R_SR, &maps.r_slv, x0 + C::TXW, yh, zp, full + s);
                    tma_load_3d(sg + C::P_SL, mp_slv, x0 - 4, yh, zp, full + s);
                    tma_load_3d(sg + C::P_SR, mp_slv, x0 + C::TXW, yh, zp, full + s);
                    if (has_xh) {
#pragma unroll
                        for (int b = 0; b < C::NBX; ++b)
                            tma_load_3d(sg + C::XH + b * C::TY * C::BOXW, &maps.xh, x0 + b * C::BOXW, y0, zp, full + s);
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
        const int tx = tid % (64 * C::NBX), ty = tid / (64 * C::NBX);
        const int b = tx >> 6, c4 = tx & 63;
        const int rrow = ty + (C::HAS_Y ? 1 : 0);               // own row in the haloed arrays
        const int rcol = 4 + b * C::BOXW + c4 * 4;              // own column in a ring row
        const int own_main = (b * C::RH + rrow) * C::BOXW + c4 * 4;   // own float4 inside r / p main boxes
        const int own_ty = (b * C::TY + ty) * C::BOXW + c4 * 4;       // own float4 inside x_hat / wx / wz boxes
        unsigned it = 0;
        for (int item = blockIdx.x; item < total; item += gridDim.x) {
            const int chunk = item / tiles, t = item - chunk * tiles;
            const int tyi = t / ntx, txi = t - tyi * ntx;
            const int x0 = txi * C::TXW, y0 = tyi * C::TY, k0 = chunk * lz;
            const int k1 = min(k0 + lz, g.nz);
            const int x = x0 + b * C::BOXW + c4 * 4, y = y0 + ty;
            const bool inb = (x < g.px) && (y < g.ny);
            const long long nrow = (long long)y * g.px + x;
            float4 wzm = make_float4(0.f, 0.f, 0.f, 0.f);
            bar_consumers(C::NCONS);   // the ring is rebuilt per item: nobody may still read the previous item's planes
            for (int kk = k0 - 2; kk < k1; ++kk, ++it) {
                const int s = it % C::S;
                const unsigned ph = (it / C::S) & 1u;
                mbar_wait(full + s, ph);
                const float* sg = stages + s * C::STAGE_FLOATS;
                // ---- phase A: p_new(kk+1) = r + beta p_old on the tile and its halo -> ring ----
                float* rw = ring + ((kk + 5) & 3) * (C::RH * C::W);
                for (int i = tid; i < C::NBX * C::RH * 64; i += C::NCONS) {
                    const int bb = i / (C::RH * 64), rem = i - bb * (C::RH * 64);
                    const int row = rem >> 6, cc = rem & 63;
                    const int o = (bb * C::RH + row) * C::BOXW + cc * 4;
                    const float4 v = fma4(beta, lds4(sg + C::P_MAIN + o), lds4(sg + C::R_MAIN + o));
                    *reinterpret_cast<float4*>(rw + row * C::W + 4 + bb * C::BOXW + cc * 4) = v;
                }
                if (tid < 2 * C::RH) {
                    const int side = tid / C::RH, row = tid - side * C::RH;
                    const float4 v = fma4(beta, lds4(sg + (side ? C::P_SR : C::P_SL) + row * 4),
                                          lds4(sg + (side ? C::R_SR : C::R_SL) + row * 4));
                    *reinterpret_cast<float4*>(rw + row * C::W + (side ? 4 + C::TXW : 0)) = v;
                }
                // ---- deferred solution update on plane kk+1 ----
                if (kk + 1 >= k0 && kk + 1 < k1 && inb) {
                    const float4 v = fma4(ax, lds4(sg + C::P_MAIN + own_main), lds4(sg + C::XH + own_ty));
                    *reinterpret_cast<float4*>(P.xh + (long long)(kk + 1) * g.plane + nrow) = v;
                }
                bar_consumers(C::NCONS);
                // ---- phase C: q(kk) = p_new - W p_new from the ring, weights from the stage ----
                if (kk >= k0) {
                    const float* r0 = ring + ((kk + 4) & 3) * (C::RH * C::W) + rrow * C::W + rcol;
                    const float4 pc = lds4(r0);
                    const float4 pzm = lds4(ring + ((kk + 3) & 3) * (C::RH * C::W) + rrow * C::W + rcol);
                    const float4 pzp = lds4(rw + rrow * C::W + rcol);
                    float pl = __shfl_up_sync(0xffffffffu, pc.w, 1);
                    float pr = __shfl_down_sync(0xffffffffu, pc.x, 1);
                    if (lane == 0) pl = r0[-1];
                    if (lane == 31) pr = r0[4];
                    const float4 gx = lds4(sg + C::WX + own_ty);
                    float gxl = __shfl_up_sync(0xffffffffu, gx.w, 1);
                    if (lane == 0) {
                        if (c4 != 0) gxl = sg[C::WX + own_ty - 1];
                        else if (b != 0) gxl = sg[C::WX + ((b - 1) * C::TY + ty) * C::BOXW + C::BOXW - 1];
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
                        const int oy = (b * C::RWY + ty) * C::BOXW + c4 * 4;   // row ty of the wy box = lattice row y-1
                        const float4 gym = lds4(sg + C::WY + oy), gy = lds4(sg + C::WY + oy + C::BOXW);
                        q.x += gym.x * pym.x + gy.x * pyp.x;
                        q.y += gym.y * pym.y + gy.y * pyp.y;
                        q.z += gym.z * pym.z + gy.z * pyp.z;
                        q.w += gym.w * pym.w + gy.w * pyp.w;
                    }
                    q.x = pc.x - q.x; q.y = pc.y - q.y; q.z = pc.z - q.z; q.w = pc.w - q.w;
                    if (inb) {
                        const long long n = (long long)kk * g.plane + nrow;
                        *reinterpret_cast<float4*>(pout + n) = pc;
                        *reinterpret_cast<float4*>(P.q + n) = q;
                        acc += (double)(pc.x * q.x + pc.y * q.y + pc.z * q.z + pc.w * q.w);
                    }
                    wzm = gz;
                } else if (kk == k0 - 1) {
                    wzm = lds4(sg + C::WZ + own_ty);   // wz(k0-1): the backward z bond of the first plane
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + s);
            }
        }
    }
    // ---- p.Ap: warp -> block -> grid; the last block computes alpha ----
    acc = pn_block_sum(acc, red);
    const double v1[1] = {acc};
    if (pn_grid_sum<1>(v1, P.slots, &st->ticket, red, red + 32)) {
        if (threadIdx.x == 0) {
            if (g.wrap[0] | g.wrap[1] | g.wrap[2]) st->part[0] = red[32];   // periodic faces: k_wrap_fix finishes
            else pn_finish_A(st, red[32]);
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------
template <class C>
bool build_maps(pn_tmaps* M, const pn_geom& g, const pn_ptrs& P) {
    const long long h = g.plane;
    bool ok = true;
    ok &= make_map(&M->r_main, g, P.r - h, C::BOXW, C::RH);
    ok &= make_map(&M->r_slv, g, P.r - h, 4, C::RH);
    ok &= make_map(&M->p_main[0], g, P.p - h, C::BOXW, C::RH);
    ok &= make_map(&M->p_main[1], g, P.p2 - h, C::BOXW, C::RH);
    ok &= make_map(&M->p_slv[0], g, P.p - h, 4, C::RH);
    ok &= make_map(&M->p_slv[1], g, P.p2 - h, 4, C::RH);
    ok &= make_map(&M->xh, g, P.xh - h, C::BOXW, C::TY);
    ok &= make_map(&M->wx_main, g, P.w[0] - h, C::BOXW, C::TY);
    ok &= make_map(&M->wx_slv, g, P.w[0] - h, 4, C::TY);
    ok &= make_map(&M->wy, g, P.w[1] - h, C::BOXW, C::RWY);
    ok &= make_map(&M->wz, g, P.w[2] - h, C::BOXW, C::TY);
    return ok;
}

template <class C>
cudaError_t launch_cfg(const pn_geom& g, const pn_ptrs& P, const pn_tmaps& M, cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_stencil_tma<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const int ntx = (g.px + C::TXW - 1) / C::TXW, nty = (g.ny + C::TY - 1) / C::TY;
    const int sms = pn_sm_count();
    const int lz = choose_lz(g.nz, ntx * nty, sms, 36.0, 16.0);
    const int nchunks = (g.nz + lz - 1) / lz;
    const long long total = (long long)ntx * nty * nchunks;
    const int nb = (int)(total < sms ? total : sms);
    k_stencil_tma<C><<<nb, C::NTHREADS, C::SMEM_BYTES, st>>>(M, g, P, ntx, nty, nchunks, lz);
    return cudaGetLastError();
}

typedef Cfg<1, 8, true, 3> Cfg3D;    // 256 x 8 tile, y halo, 3 stages
typedef Cfg<8, 1, false, 4> Cfg2D;   // 2048 x 1 tile (lattices held as nx x 1 x ny), 4 stages

}  // namespace

// Opaque per-launch-batch handle: the tensor maps of one (geometry, pointers) pair.
struct pn_tma_plan {
    pn_tmaps maps;
    bool is2d;
};

bool pn_tma_supported() { return get_encoder() != nullptr; }

bool pn_tma_plan_build(pn_tma_plan** out, const pn_geom& g, const pn_ptrs& P) {
    pn_tma_plan* pl = new (std::nothrow) pn_tma_plan;
    if (!pl) return false;
    pl->is2d = (g.ny == 1);
    const bool ok = pl->is2d ? build_maps<Cfg2D>(&pl->maps, g, P) : build_maps<Cfg3D>(&pl->maps, g, P);
    if (!ok) { delete pl; return false; }
    *out = pl;
    return true;
}

void pn_tma_plan_free(pn_tma_plan* pl) { delete pl; }

cudaError_t pn_launch_stencil_tma(const pn_tma_plan* pl, const pn_geom& g, const pn_ptrs& P, cudaStream_t st) {
    return pl->is2d ? launch_cfg<Cfg2D>(g, P, pl->maps, st) : launch_cfg<Cfg3D>(g, P, pl->maps, st);
}
