// exx_subspace.cu — the dense subspace matrix of the exchange operator, M_ij = <c_i | (V_x c)_j> within one k-point, as a
// complex fp64 GEMM on the fp64 tensor-core path (mma.sync m8n8k4 DMMA; tcgen05 has no fp64 kind).  BASELINE north_star:
// "tensor cores are used only if the optional dense subspace matrix <psi_i|V_x|psi_j> is built as a ZGEMM"; the paper's NSIM
// "matrix-matrix operations".  Product code: shares nothing with oracle/.
//
// M = A^H B with A = psi (nb x npw, row-major, npw contiguous) and B = V_x psi (same layout):
//   Re M_ij = sum_g (ar_ig br_jg + ai_ig bi_jg),   Im M_ij = sum_g (ar_ig bi_jg - ai_ig br_jg)
// i.e. four real m8n8k4 products per 4 plane waves.  A warp owns one 32 x 32 tile of M (4 x 4 DMMA tiles of 8 x 8) over one slice of
// the plane waves (split-K); the slices are added in a fixed order by a second kernel, so the result is deterministic.
#include "exx_internal.h"

namespace exx {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// partial[s][i][j] (complex) for slice s: plane waves [s*chunk, min(npw, (s+1)*chunk)); chunk is a multiple of 4.
// A warp owns a (8 MI) x (8 NJ) tile of M for one slice: per 4 plane waves it loads MI + NJ complex fragments (one element per
// lane each) and issues 4 MI NJ DMMAs, so every fragment is reused NJ (MI) times from registers; the 4 warps of a CTA take 4
// consecutive slices of the same tile (their rows are shared in L1/L2).
template <int MI, int NJ>
__global__ void __launch_bounds__(128) subspace_partial_kernel(const double2* __restrict__ A, const double2* __restrict__ Bm, int nb, int npw, int chunk,
                                                                int nslices, double2* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tj_n = (nb + 8 * NJ - 1) / (8 * NJ);
    const int ti = blockIdx.x / tj_n, tj = blockIdx.x % tj_n, s = blockIdx.y * 4 + warp;
    if (s >= nslices) return;
    const int row = lane >> 2, kk = lane & 3;        // fragment coordinates: A (row, kk), B (kk, col = row)
    const int g0 = s * chunk, g1 = min(npw, g0 + chunk);
    const double2* a[MI];
    const double2* b[NJ];
    bool ia[MI], jb[NJ];
#pragma unroll
    for (int m = 0; m < MI; m++) {
        const int i = (ti * MI + m) * 8 + row;
        ia[m] = i < nb;
        a[m] = A + (size_t)min(i, nb - 1) * npw;
    }
#pragma unroll
    for (int n = 0; n < NJ; n++) {
        const int j = (tj * NJ + n) * 8 + row;
        jb[n] = j < nb;
        b[n] = Bm + (size_t)min(j, nb - 1) * npw;
    }
    double cr[MI][NJ][2], ci[MI][NJ][2];
#pragma unroll
    for (int m = 0; m < MI; m++)
#pragma unroll
        for (int n = 0; n < NJ; n++) cr[m][n][0] = cr[m][n][1] = ci[m][n][0] = ci[m][n][1] = 0.0;
    for (int g = g0 + kk; g < g1 + kk; g += 4) {     // every lane makes the same number of trips (mma.sync is warp-wide)
        double2 x[MI], y[NJ];
        const bool in = g < g1;
#pragma unroll
        for (int m = 0; m < MI; m++) x[m] = (in && ia[m]) ? a[m][g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int n = 0; n < NJ; n++) y[n] = (in && jb[n]) ? b[n][g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int m = 0; m < MI; m++)
#pragma unroll
            for (int n = 0; n < NJ; n++) {
                dmma884(cr[m][n][0], cr[m][n][1], x[m].x, y[n].x);
                dmma884(cr[m][n][0], cr[m][n][1], x[m].y, y[n].y);
                dmma884(ci[m][n][0], ci[m][n][1], x[m].x, y[n].y);
                dmma884(ci[m][n][0], ci[m][n][1], -x[m].y, y[n].x);
            }
    }
    // accumulator fragment: row = lane / 4, columns 2 (lane % 4) and 2 (lane % 4) + 1
    double2* p = partial + (size_t)s * nb * nb;
#pragma unroll
    for (int m = 0; m < MI; m++)
#pragma unroll
        for (int n = 0; n < NJ; n++) {
            const int oi = (ti * MI + m) * 8 + row, oj = (tj * NJ + n) * 8 + 2 * kk;
            if (oi < nb) {
                if (oj < nb) p[(size_t)oi * nb + oj] = make_double2(cr[m][n][0], ci[m][n][0]);
                if (oj + 1 < nb) p[(size_t)oi * nb + oj + 1] = make_double2(cr[m][n][1], ci[m][n][1]);
            }
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
    constexpr int MI = 4, NJ = 4;  // 32 x 32 tile of M per warp
    const int tiles = ((nb + 8 * MI - 1) / (8 * MI)) * ((nb + 8 * NJ - 1) / (8 * NJ));
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // slices: about 8 warps per SM over the whole machine, chunks a multiple of 4 plane waves
    int nslices = std::max(1, std::min(256, (sms * 8 + tiles - 1) / tiles));
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
        dim3 grid(tiles, (nslices + 3) / 4);
        subspace_partial_kernel<MI, NJ><<<grid, 128, 0, c->stream>>>(psi + offk, vx + offk, nb, npw, chunk, nslices, (double2*)c->subspace_dev);
    }
    {
        LaunchScope ls(c, KC_SUBSPACE, 0);
        subspace_reduce_kernel<<<(nb * nb + 255) / 256, 256, 0, c->stream>>>((const double2*)c->subspace_dev, nb * nb, nslices, M);
    }
    EXX_CUDA(c, cudaGetLastError());
    return EXX_OK;
}

}  // namespace exx
