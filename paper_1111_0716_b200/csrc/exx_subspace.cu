// exx_subspace.cu — the dense subspace matrix of the exchange operator, M_ij = <c_i | (V_x c)_j> within one k-point, as a
// complex fp64 GEMM on the fp64 tensor-core path (mma.sync m8n8k4 DMMA; tcgen05 has no fp64 kind).  BASELINE north_star:
// "tensor cores are used only if the optional dense subspace matrix <psi_i|V_x|psi_j> is built as a ZGEMM"; the paper's NSIM
// "matrix-matrix operations".  Product code: shares nothing with oracle/.
//
// M = A^H B with A = psi (nb x npw, row-major, npw contiguous) and B = V_x psi (same layout):
//   Re M_ij = sum_g (ar_ig br_jg + ai_ig bi_jg),   Im M_ij = sum_g (ar_ig bi_jg - ai_ig br_jg)
// i.e. four real m8n8k4 products per 4 plane waves.  A warp owns one 8 x 8 tile of M over one slice of the plane waves
// (split-K); the slices are added in a fixed order by a second kernel, so the result is deterministic.
#include "exx_internal.h"

namespace exx {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// partial[s][i][j] (complex) for slice s: plane waves [s*chunk, min(npw, (s+1)*chunk)); chunk is a multiple of 4
__global__ void __launch_bounds__(128) subspace_partial_kernel(const double2* __restrict__ A, const double2* __restrict__ Bm, int nb, int npw, int chunk,
                                                                double2* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tiles = (nb + 7) / 8;
    const int tile = blockIdx.x * 4 + warp;
    if (tile >= tiles * tiles) return;
    const int ti = tile / tiles, tj = tile % tiles, s = blockIdx.y;
    const int row = lane >> 2, kk = lane & 3;        // fragment coordinates: A (row, kk), B (kk, col = row)
    const int i = ti * 8 + row, j = tj * 8 + row;
    const int g0 = s * chunk, g1 = min(npw, g0 + chunk);
    const double2* a = A + (size_t)min(i, nb - 1) * npw;
    const double2* b = Bm + (size_t)min(j, nb - 1) * npw;
    const bool ia = i < nb, jb = j < nb;
    double cr0 = 0.0, cr1 = 0.0, ci0 = 0.0, ci1 = 0.0;
    for (int g = g0 + kk; g < g1 + kk; g += 4) {     // every lane makes the same number of trips (mma.sync is warp-wide)
        double2 x = make_double2(0.0, 0.0), y = make_double2(0.0, 0.0);
        if (g < g1) {
            if (ia) x = a[g];
            if (jb) y = b[g];
        }
        dmma884(cr0, cr1, x.x, y.x);
        dmma884(cr0, cr1, x.y, y.y);
        dmma884(ci0, ci1, x.x, y.y);
        dmma884(ci0, ci1, -x.y, y.x);
    }
    // accumulator fragment: row = lane / 4, columns 2 (lane % 4) and 2 (lane % 4) + 1
    const int oi = ti * 8 + row, oj = tj * 8 + 2 * kk;
    double2* p = partial + (size_t)s * nb * nb;
    if (oi < nb) {
        if (oj < nb) p[(size_t)oi * nb + oj] = make_double2(cr0, ci0);
        if (oj + 1 < nb) p[(size_t)oi * nb + oj + 1] = make_double2(cr1, ci1);
    }
}

__global__ void subspace_reduce_kernel(const double2* __restrict__ partial, int n2, int nslices, double2* __restrict__ M) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n2) return;
    double2 s = make_double2(0.0, 0.0);
    for (int k = 0; k < nslices; k++) {  // fixed order
        double2 v = partial[(size_t)k * n2 + e];
        s.x += v.x;
        s.y += v.y;
    }
    M[e] = s;
}

// nvec vectors per k-point in psi / vx (default: the context's nbands), M is nvec x nvec
int launch_subspace(exx_ctx* c, int ik, const double2* psi, const double2* vx, double2* M, int nvec) {
    const int nb = nvec > 0 ? nvec : c->nb, npw = c->npw[ik];
    const int64_t offk = c->off[ik] / c->nb * nb;
    const int tiles = (nb + 7) / 8;
    // slices: enough warps to fill the machine, chunks a multiple of 4 plane waves
    int nslices = std::max(1, std::min(64, (148 * 16 * 4) / std::max(1, tiles * tiles)));
    int chunk = ((npw + nslices - 1) / nslices + 3) / 4 * 4;
    nslices = (npw + chunk - 1) / chunk;
    const size_t need = sizeof(double2) * (size_t)nslices * nb * nb;
    if (need > c->subspace_bytes) {
        cudaFree(c->subspace_dev);
        c->subspace_dev = nullptr;
        c->subspace_bytes = 0;
        if (cudaMalloc((void**)&c->subspace_dev, need) != cudaSuccess) {
            cudaGetLastError();
            return EXX_ERR_ALLOC;
        }
        c->subspace_bytes = need;
        c->dev_bytes += need;
    }
    {
        LaunchScope ls(c, KC_SUBSPACE, 1);
        dim3 grid((tiles * tiles + 3) / 4, nslices);
        subspace_partial_kernel<<<grid, 128, 0, c->stream>>>(psi + offk, vx + offk, nb, npw, chunk, (double2*)c->subspace_dev);
    }
    {
        LaunchScope ls(c, KC_SUBSPACE, 0);
        subspace_reduce_kernel<<<(nb * nb + 255) / 256, 256, 0, c->stream>>>((const double2*)c->subspace_dev, nb * nb, nslices, M);
    }
    EXX_CUDA(c, cudaGetLastError());
    return EXX_OK;
}

}  // namespace exx
