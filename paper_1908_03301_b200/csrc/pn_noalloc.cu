// pn_noalloc.cu -- pn_dissipation_noalloc (include/pn.h): the dissipation sum  G_E = sum over bonds g (P_i - P_j)^2
// (energy identity of P:53 with eq.(4); pn_outer.cu's k_dissipation is the handle-based form) for callers that
// may not allocate device memory.  The grid reduction's scratch -- one partial sum per chunk of 8192 nodes and the
// arrival counter of the "last block adds them up" step -- lives in a file-scope __device__ array instead of a
// caller-given workspace.  Every call in the process shares that array: overlapping calls on one GPU race on it.
//
// In HOST code the array's name is a host-side stand-in for the symbol, not a device address; the address is asked for
// once per device with cudaGetSymbolAddress (that device being current) and handed to the kernel as an argument.
#include "pn_internal.cuh"

#include <mutex>

namespace {

constexpr int NA_T = 256;                      // threads per block
constexpr int NA_CHUNK = 8192;                 // nodes per partial sum (fixed: the summation order is part of the result)
constexpr long long NA_MAX_CHUNKS = PN_NOALLOC_MAX_NODES / NA_CHUNK;   // 32768
constexpr int NA_TAIL = 32;                    // doubles after the chunk sums; the first holds the arrival counter
constexpr int NA_MAX_DEVICES = 64;

static_assert(PN_NOALLOC_MAX_NODES % NA_CHUNK == 0, "whole chunks");
static_assert((NA_MAX_CHUNKS * sizeof(double)) % 256 == 0, "the counter keeps the array's alignment");

// the scratch: NA_MAX_CHUNKS chunk sums, then the counter (256 KB + 256 B per GPU that loads the library)
static __device__ __align__(256) double pn_na_scratch[NA_MAX_CHUNKS + NA_TAIL];

struct na_device {
    std::once_flag once;
    cudaError_t err = cudaSuccess;
    double* scratch = nullptr;                 // DEVICE address of pn_na_scratch on this device
    int sms = 0;
};
na_device g_dev[NA_MAX_DEVICES];

// neighbour reached by the forward bond along one axis from coordinate c of n_b (stride sb), or -1 if there is none
__device__ __forceinline__ long long forward_node(long long n, int c, int n_b, long long sb, bool wraps) {
    if (c + 1 < n_b) return n + sb;
    return (wraps && n_b > 1) ? n - (long long)(n_b - 1) * sb : -1;
}

__global__ void __launch_bounds__(NA_T)
k_dissipation_noalloc(int nx, int ny, int nz, int pmask, const float* __restrict__ gx, const float* __restrict__ gy,
                      const float* __restrict__ gz, const double* __restrict__ P, double* scratch, long long nchunks,
                      double* __restrict__ out) {
    __shared__ double sm[32];
    __shared__ int s_last;
    const long long plane = (long long)nx * ny, n_all = plane * nz;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + NA_MAX_CHUNKS);
    for (long long c = blockIdx.x; c < nchunks; c += gridDim.x) {
        const long long lo = c * NA_CHUNK, hi = min(lo + NA_CHUNK, n_all);
        double e = 0.0;
        for (long long n = lo + threadIdx.x; n < hi; n += NA_T) {
            const long long row = n / nx;
            const int i = (int)(n - row * nx), j = (int)(row % ny), k = (int)(row / ny);
            const double xc = P[n];
            const float g0 = gx[n], g1 = gy[n], g2 = gz ? gz[n] : 0.f;
            if (g0 != 0.f) {
                const long long m = forward_node(n, i, nx, 1, pmask & 1);
                if (m >= 0) { const double d = P[m] - xc; e += (double)g0 * d * d; }
            }
            if (g1 != 0.f) {
                const long long m = forward_node(n, j, ny, nx, pmask & 2);
                if (m >= 0) { const double d = P[m] - xc; e += (double)g1 * d * d; }
            }
            if (g2 != 0.f) {
                const long long m = forward_node(n, k, nz, plane, pmask & 4);
                if (m >= 0) { const double d = P[m] - xc; e += (double)g2 * d * d; }
            }
        }
        e = pn_block_sum(e, sm);
        if (threadIdx.x == 0) scratch[c] = e;
    }
    // the block that arrives last adds the chunk sums in chunk order (a fixed tree: independent of the grid)
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1 ? 1 : 0;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double v = 0.0;
    for (long long c = threadIdx.x; c < nchunks; c += NA_T) v += __ldcg(scratch + c);
    v = pn_block_sum(v, sm);
    if (threadIdx.x == 0) { *out = v; *ticket = 0u; }
}

// once per device, with that device current: the symbol's address there and the SM count
void na_init_device(na_device* d, int device) {
    void* p = nullptr;
    d->err = cudaGetSymbolAddress(&p, pn_na_scratch);
    if (d->err != cudaSuccess) return;
    d->scratch = static_cast<double*>(p);
    d->err = cudaDeviceGetAttribute(&d->sms, cudaDevAttrMultiProcessorCount, device);
}

}  // namespace

extern "C" int pn_dissipation_noalloc(int nx, int ny, int nz, const float* gx, const float* gy, const float* gz,
                                      const double* pressures, int periodic_mask, double* g_e, int device,
                                      void* cuda_stream) {
    if (nx < 1 || ny < 1 || nz < 1 || !gx || !gy || !pressures || !g_e) return PN_ERR_ARG;
    if ((nz == 1) != (gz == nullptr)) return PN_ERR_ARG;
    if (periodic_mask < 0 || periodic_mask > 7) return PN_ERR_ARG;
    if (device < 0 || device >= NA_MAX_DEVICES) return PN_ERR_ARG;
    const long long plane = (long long)nx * ny;          // < 2^62; checked before it is multiplied again
    if (plane > PN_NOALLOC_MAX_NODES || plane * nz > PN_NOALLOC_MAX_NODES) return PN_ERR_TOO_LARGE;
    const long long n_all = plane * nz;

    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return PN_ERR_CUDA;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return PN_ERR_CUDA; }
    na_device* d = &g_dev[device];
    std::call_once(d->once, na_init_device, d, device);
    int rc = PN_OK;
    if (d->err != cudaSuccess || !d->scratch) {
        rc = PN_ERR_CUDA;
    } else {
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        const long long nchunks = (n_all + NA_CHUNK - 1) / NA_CHUNK;
        long long grid = (long long)d->sms * 8;
        if (grid > nchunks) grid = nchunks;
        // the counter must start at zero whatever an earlier (possibly failed) call left behind
        if (cudaMemsetAsync(d->scratch + NA_MAX_CHUNKS, 0, sizeof(unsigned int), st) != cudaSuccess) rc = PN_ERR_CUDA;
        if (rc == PN_OK) {
            k_dissipation_noalloc<<<(unsigned int)grid, NA_T, 0, st>>>(nx, ny, nz, periodic_mask, gx, gy, gz, pressures,
                                                                        d->scratch, nchunks, g_e);
            if (cudaGetLastError() != cudaSuccess) rc = PN_ERR_CUDA;
        }
    }
    if (prev != device) cudaSetDevice(prev);
    return rc;
}
