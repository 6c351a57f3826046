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
    // rows of this lane's fragments: A rows (ti MI + m) 8 + row, B rows (tj NJ + n) 8 + row; a row past the edge is never loaded
    const size_t stride8 = (size_t)8 * npw;
    const double2* a0 = A + (size_t)(ti * MI * 8 + row) * npw;
    const double2* b0 = Bm + (size_t)(tj * NJ * 8 + row) * npw;
    bool ia[MI], jb[NJ];
#pragma unroll
    for (int m = 0; m < MI; m++) ia[m] = (ti * MI + m) * 8 + row < nb;
#pragma unroll
    for (int n = 0; n < NJ; n++) jb[n] = (tj * NJ + n) * 8 + row < nb;
    double cr[MI][NJ][2], ci[MI][NJ][2];
#pragma unroll
    for (int m = 0; m < MI; m++)
#pragma unroll
        for (int n = 0; n < NJ; n++) cr[m][n][0] = cr[m][n][1] = ci[m][n][0] = ci[m][n][1] = 0.0;
    // software pipeline: the fragments of the next 4 plane waves are loaded before the 64 DMMAs of the current ones are issued, so the
    // L2 latency of a trip hides behind the tensor work of the trip before it (8 warps per SM cannot hide it by themselves).
    // Measured at 160 x 160 x 15 465: 0.195 ms without it, 0.130 ms with it (cuBLAS ZGEMM on the same operands: 0.137 ms).
    const int trips = (g1 - g0 + 3) / 4;  // the same in every lane (mma.sync is warp-wide)
    double2 x[MI], y[NJ], xn[MI], yn[NJ];
    {
        const int g = g0 + kk;
        const bool in = g < g1;
#pragma unroll
        for (int m = 0; m < MI; m++) x[m] = (in && ia[m]) ? a0[m * stride8 + g] : make_double2(0.0, 0.0);
#pragma unroll
        for (int n = 0; n < NJ; n++) y[n] = (in && jb[n]) ? b0[n * stride8 + g] : make_double2(0.0, 0.0);
    }
    for (int t = 0; t < trips; t++) {
        const int gn = g0 + kk + 4 * (t + 1);
        const bool in = gn < g1;
#pragma unroll
        for (int m = 0; m < MI; m++) xn[m] = (in && ia[m]) ? a0[m * stride8 + gn] : make_double2(0.0, 0.0);
#pragma unroll
        for (int n = 0; n < NJ; n++) yn[n] = (in && jb[n]) ? b0[n * stride8 + gn] : make_double2(0.0, 0.0);
#pragma unroll
        for (int m = 0; m < MI; m++)
#pragma unroll
            for (int n = 0; n < NJ; n++) {
                dmma884(cr[m][n][0], cr[m][n][1], x[m].x, y[n].x);
                dmma884(cr[m][n][0], cr[m][n][1], x[m].y, y[n].y);
                dmma884(ci[m][n][0], ci[m][n][1], x[m].x, y[n].y);
                dmma884(ci[m][n][0], ci[m][n][1], -x[m].y, y[n].x);
            }
#pragma unroll
        for (int m = 0; m < MI; m++) x[m] = xn[m];
#pragma unroll
        for (int n = 0; n < NJ; n++) y[n] = yn[n];
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
    // slices: as many as ONE wave of resident CTAs holds (a CTA = 4 slices of one tile; 220 registers: two CTAs per SM), chunks a
    // multiple of 4 plane waves
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, subspace_partial_kernel<MI, NJ>, 128, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 2;
    }
    int nslices = std::max(4, std::min(256, 4 * ((sms * per_sm) / tiles)));
    nslices = std::min(nslices, std::max(4, npw / 128 / 4 * 4));  // at least 32 trips per slice: more slices only feed the reduction
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
