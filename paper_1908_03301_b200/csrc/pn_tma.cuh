// pn_tma.cuh -- sm_100a TMA / mbarrier PTX wrappers and the tensor-map encoder shared by the TMA-fed
// kernels of libpn (pn_fused_tma.cu).  Not part of the C ABI.
#pragma once
#include <cuda.h>  // CUtensorMap and enums only: the encoder is fetched with cudaGetDriverEntryPoint
#include <cuda_runtime.h>
#include <stdint.h>

#include "pn_internal.cuh"

namespace pn_tma {

constexpr int a32(int x) { return (x + 31) / 32 * 32; }  // TMA destinations: 128-byte (32-float) aligned

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    const uint32_t a = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tma_load_3d(float* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}
// named barrier 1 over the first n threads of the CTA (the consumer warps)
__device__ __forceinline__ void bar_consumers(int n) { asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory"); }

__device__ __forceinline__ float4 lds4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 fma4(float a, const float4& x, const float4& y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ float dot4(const float4& a, const float4& b) { return a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w; }

// ---- host side: tensor maps ------------------------------------------------------------------------
typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline encode_fn get_encoder() {
    static encode_fn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (encode_fn)p;
    }
    return fn;
}

// 3D map over a padded lattice array INCLUDING its two halo planes: dims (px, ny, nz + 2); box bx x by x 1.
// Parts of a box outside the array are zero-filled by the TMA unit.
inline bool make_map(CUtensorMap* m, const pn_geom& g, const float* base_with_halo, int bx, int by) {
    encode_fn enc = get_encoder();
    if (!enc) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.px, (cuuint64_t)g.ny, (cuuint64_t)g.nz + 2};
    const cuuint64_t strides[2] = {(cuuint64_t)g.px * 4, (cuuint64_t)g.plane * 4};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
    const cuuint32_t es[3] = {1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base_with_halo, dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// z-chunk length of the 2.5D march (2D tile): balance the persistent grid against the `extra_bytes_per_chunk_node` every
// chunk pays for its two extra leading planes (per node of a plane, against `bytes_per_node` of useful traffic)
inline int choose_lz(int nz, int tiles, int nblocks, double bytes_per_node, double extra_bytes_per_chunk_node, int max_lz = 64) {
    int best = 1;
    double best_eff = 0.0;
    for (int lz = 4; lz <= max_lz; ++lz) {
        const int chunks = (nz + lz - 1) / lz;
        const long long items = (long long)chunks * tiles;
        const long long rounds = (items + nblocks - 1) / nblocks;
        const double balance = (double)items / (double)(rounds * nblocks);
        const double halo = bytes_per_node / (bytes_per_node + extra_bytes_per_chunk_node / lz);
        const double eff = balance * halo;
        if (eff > best_eff + 1e-9) { best_eff = eff; best = lz; }
    }
    return best;
}

// z-chunks of the 2.5D march (3D tiles).  The nz planes of every tile are cut into `nchunks` EQUAL parts (chunk j = planes
// [j nz / nchunks, (j+1) nz / nchunks)); item = (chunk, tile), CTA c of the persistent grid takes items c, c + G, ...
// Every item pays two extra leading planes (its prologue).  Chosen: the count that minimises the plane steps of the
// busiest CTA, computed exactly; ties go to fewer chunks (less prologue traffic).  (Round 1 fixed a chunk LENGTH and
// left a ragged last chunk: 494 steps per CTA instead of 462 at 512^3, 40 instead of 34 at 192^3.)
inline int choose_chunks(int nz, int tiles, int nblocks) {
    thread_local int last_key[3] = {0, 0, 0}, last_val = 0;   // launchers ask again for every launch
    if (last_key[0] == nz && last_key[1] == tiles && last_key[2] == nblocks) return last_val;
    int best = 1;
    long long best_cost = -1;
    int max_chunks = nz / 4 > 1 ? nz / 4 : 1;
    long long cap = (8ll * nblocks + tiles - 1) / tiles;   // up to ~8 items per CTA, or 8 chunks per tile: beyond, only more prologues
    if (cap < 8) cap = 8;
    if (max_chunks > cap) max_chunks = (int)cap;
    for (int nch = 1; nch <= max_chunks; ++nch) {
        const long long items = (long long)nch * tiles;
        long long cost = 0;
        const long long ncta = items < nblocks ? items : nblocks;
        for (long long c = 0; c < ncta; ++c) {
            long long tot = 0;
            for (long long it = c; it < items; it += nblocks) {
                const long long j = it / tiles;
                tot += ((j + 1) * nz / nch - j * nz / nch) + 2;
            }
            if (tot > cost) cost = tot;
        }
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = nch; }
    }
    last_key[0] = nz; last_key[1] = tiles; last_key[2] = nblocks; last_val = best;
    return best;
}

}  // namespace pn_tma
