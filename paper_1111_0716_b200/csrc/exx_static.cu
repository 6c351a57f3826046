// exx_static.cu — exx_subspace_static (include/exx.h): the subspace matrix M = A^H B of exx_subspace for callers that must not
// allocate device memory.  Who that is: a host program whose GPU memory is entirely in the hands of another allocator (a framework's
// caching pool that has already reserved the card, or a batch job held to a fixed memory budget), so that a cudaMalloc from inside
// this library would either fail or take memory the owner believes it has; and a time-critical loop that cannot afford the
// device-wide synchronisation a cudaMalloc / cudaFree implies.  exx_subspace serves everyone else and grows its split-K scratch
// with cudaMalloc on demand; this file keeps the same scratch in a fixed array that is part of the loaded library image instead.
//
// What it costs: every GPU on which libexx is loaded carries EXX_STATIC_SCRATCH_BYTES (8 MiB) from the moment the module is loaded
// until the process exits, whether or not this entry point is ever called, and the size of the problem is capped
// (EXX_STATIC_MAX_NVEC vectors, EXX_STATIC_MAX_NPW plane waves).
//
// The kernels are a variant of the two in exx_subspace.cu (same DMMA m8n8k4 fragments, same fixed-order slice sum; tcgen05 has no
// fp64 kind) kept in this file so that the existing path is not touched.  Product code: shares nothing with oracle/.
#include <mutex>

#include "exx_internal.h"

namespace exx {
namespace {

constexpr size_t kScratchElems = (size_t)EXX_STATIC_SCRATCH_BYTES / sizeof(double2);
constexpr int kMaxDevices = 64;

// The split-K partial matrices partial[s][i][j].  In HOST code this name is only a handle for the runtime's symbol table: it is not a
// device address and must never be handed to a kernel.  The address on a given GPU comes from cudaGetSymbolAddress (scratch_for_device
// below); each device that loads the library has its own copy of the array.
static __device__ __align__(256) double2 g_static_scratch[kScratchElems];

std::mutex g_scratch_mutex;
double2* g_scratch_addr[kMaxDevices];  // per device ordinal, filled on the first call made with that device current

// Device address of g_static_scratch on the CURRENT device.  The first call per device asks the runtime (which also loads the module
// onto that device if nothing has yet); later calls read the cached pointer.  Allocates nothing.
int scratch_for_device(double2** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return EXX_ERR_BAD_ARG;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!p) return EXX_ERR_CUDA;
        g_scratch_addr[dev] = (double2*)p;
    }
    *out = g_scratch_addr[dev];
    return EXX_OK;
}

__device__ __forceinline__ void dmma884_s(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// One warp: a 32 x 32 tile of M over plane waves [s*chunk, min(npw, (s+1)*chunk)), chunk a multiple of 4; the 4 warps of a CTA take 4
// consecutive slices of the same tile.  Every element (s, i < nv, j < nv) of `partial` with s < nslices is WRITTEN here (an empty
// slice writes zeros), so nothing left in the array by an earlier call is ever read: the scratch needs no clearing.
constexpr int MI = 4, NJ = 4;
__global__ void __launch_bounds__(128) subspace_partial_static_kernel(const double2* __restrict__ A, const double2* __restrict__ Bm, int nv, int npw,
                                                                       int chunk, int nslices, double2* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tj_n = (nv + 8 * NJ - 1) / (8 * NJ);
    const int ti = blockIdx.x / tj_n, tj = blockIdx.x % tj_n, s = blockIdx.y * 4 + warp;
    if (s >= nslices) return;
    const int row = lane >> 2, kk = lane & 3;  // fragment coordinates: A (row, kk), B (kk, col = row)
    const int g0 = s * chunk, g1 = min(npw, g0 + chunk);
    const double2* a[MI];
    const double2* b[NJ];
    bool ia[MI], jb[NJ];
#pragma unroll
    for (int m = 0; m < MI; m++) {
        const int i = (ti * MI + m) * 8 + row;
        ia[m] = i < nv;
        a[m] = A + (size_t)min(i, nv - 1) * npw;
    }
#pragma unroll
    for (int n = 0; n < NJ; n++) {
        const int j = (tj * NJ + n) * 8 + row;
        jb[n] = j < nv;
        b[n] = Bm + (size_t)min(j, nv - 1) * npw;
    }
    double cr[MI][NJ][2], ci[MI][NJ][2];
#pragma unroll
    for (int m = 0; m < MI; m++)
#pragma unroll
        for (int n = 0; n < NJ; n++) cr[m][n][0] = cr[m][n][1] = ci[m][n][0] = ci[m][n][1] = 0.0;
    for (int g = g0 + kk; g < g1 + kk; g += 4) {  // the same trip count in every lane (mma.sync is warp-wide)
        double2 x[MI], y[NJ];
        const bool in = g < g1;
#pragma unroll
        for (int m = 0; m < MI; m++) x[m] = (in && ia[m]) ? a[m][g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int n = 0; n < NJ; n++) y[n] = (in && jb[n]) ? b[n][g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int m = 0; m < MI; m++)
#pragma unroll
            for (int n = 0; n < NJ; n++) {  // Re += ar br + ai bi, Im += ar bi - ai br
                dmma884_s(cr[m][n][0], cr[m][n][1], x[m].x, y[n].x);
                dmma884_s(cr[m][n][0], cr[m][n][1], x[m].y, y[n].y);
                dmma884_s(ci[m][n][0], ci[m][n][1], x[m].x, y[n].y);
                dmma884_s(ci[m][n][0], ci[m][n][1], -x[m].y, y[n].x);
            }
    }
    double2* p = partial + (size_t)s * nv * nv;
#pragma unroll
    for (int m = 0; m < MI; m++)
#pragma unroll
        for (int n = 0; n < NJ; n++) {
            const int oi = (ti * MI + m) * 8 + row, oj = (tj * NJ + n) * 8 + 2 * kk;
            if (oi < nv) {
                if (oj < nv) p[(size_t)oi * nv + oj] = make_double2(cr[m][n][0], ci[m][n][0]);
                if (oj + 1 < nv) p[(size_t)oi * nv + oj + 1] = make_double2(cr[m][n][1], ci[m][n][1]);
            }
        }
}

__global__ void subspace_reduce_static_kernel(const double2* __restrict__ partial, int n2, int nslices, double2* __restrict__ M) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n2) return;
    double2 s = make_double2(0.0, 0.0);
    for (int k = 0; k < nslices; k++) {  // fixed order: deterministic
        const double2 v = partial[(size_t)k * n2 + e];
        s.x += v.x;
        s.y += v.y;
    }
    M[e] = s;
}

}  // namespace
}  // namespace exx

using namespace exx;

extern "C" int exx_subspace_static(const double* a_dev, const double* b_dev, int nvec, int64_t npw, double* m_dev, void* cuda_stream) {
    if (!a_dev || !b_dev || !m_dev) return EXX_ERR_NULL;
    if (nvec < 1 || npw < 1) return EXX_ERR_BAD_ARG;
    if (nvec > EXX_STATIC_MAX_NVEC || npw > EXX_STATIC_MAX_NPW) {
        char msg[192];
        snprintf(msg, sizeof msg, "exx_subspace_static: nvec = %d, npw = %lld exceed the fixed limits (nvec <= %d, npw <= %d); use exx_subspace_block",
                 nvec, (long long)npw, EXX_STATIC_MAX_NVEC, EXX_STATIC_MAX_NPW);
        set_thread_error(msg);
        return EXX_ERR_LIMIT;
    }
    double2* scratch = nullptr;
    int rc = scratch_for_device(&scratch);  // first call on this device: cudaGetSymbolAddress; afterwards a table look-up
    if (rc) return rc;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int nv = nvec, np = (int)npw;
    const int tiles = ((nv + 8 * MI - 1) / (8 * MI)) * ((nv + 8 * NJ - 1) / (8 * NJ));
    // slices: about 8 warps per SM over the whole machine, but never more than the fixed array holds (>= 8 at the largest nvec)
    const int fit = (int)std::min<size_t>(256, kScratchElems / ((size_t)nv * nv));
    int nslices = std::max(1, std::min(fit, (sms * 8 + tiles - 1) / tiles));
    const int chunk = ((np + nslices - 1) / nslices + 3) / 4 * 4;
    nslices = (np + chunk - 1) / chunk;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    subspace_partial_static_kernel<<<dim3(tiles, (nslices + 3) / 4), 128, 0, st>>>((const double2*)a_dev, (const double2*)b_dev, nv, np, chunk, nslices,
                                                                                  scratch);
    subspace_reduce_static_kernel<<<(nv * nv + 255) / 256, 256, 0, st>>>(scratch, nv * nv, nslices, (double2*)m_dev);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "exx_subspace_static launch");
    return EXX_OK;
}
