// exx_fused.cu — the fused three-pass pair pipeline (S2..S6) for cubic grids N = 8 R1, R1 in {6, 8, 9, 12, 16}
// (N = 48, 64, 72, 96, 128).  The per-thread phases live in exx_fused_phases.h; this file holds the kernels that
// run them between barriers, the permuted kernel tables, and the loop nest over k, n-tiles, q, m-tiles
// (k,q loops on the host, band loops on the device, innermost loop blocked).
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <vector>

#include "exx_internal.h"

#include "exx_dft.h"
namespace exx {
__constant__ cplx c_tw[48 + 64 + 72 + 96 + 128];
}
#include "exx_fused_phases.h"

namespace exx {

cplx h_tw[TW_TOTAL];  // host copy (source of the constant-memory upload)

struct FusedState {
    int R1 = 0;
    double* kperm_dev = nullptr;  // ntab tables, permuted order of pass B
    int tn = 0, tm = 0;
};

// ---------------------------------------------------------------------------------------------------------------
// pass A: rho = conj(u_m) u_n, z transform, first y step.  One CTA per (tile, m, n), n fastest so that the CTAs that
// share a u_m / u_n tile run back to back and the tile is fetched from HBM once.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT1, FusedCfg<R1>::MINB1) pass_a_kernel(const cplx* __restrict__ un_base, const cplx* __restrict__ uq_base,
                                                                    MTile mt, int tn, cplx* __restrict__ work) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U1, NT = FusedCfg<R1>::NT1;
    constexpr bool TWREG = FusedCfg<R1>::TWREG;
    static_assert(!TWREG || NT % R1 == 0, "TWREG needs a thread-invariant k1z");
    constexpr size_t Ng = (size_t)N * N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = S + U * R1 * N;
    const int tid = threadIdx.x;
    unsigned bid = blockIdx.x;
    const int n = bid % tn;
    bid /= tn;
    const int m = bid % mt.tm;
    const int tile = bid / mt.tm;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    cplx twr[8];
    if (TWREG)
        load_twr<R1>(tid, twr);
    else
        for (int i = tid; i < R1 * 8; i += NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    const cplx* un = un_base + (size_t)n * Ng;
    const cplx* um = uq_base + (size_t)mt.m_idx[m] * Ng;
    cplx* W = work + ((size_t)n * mt.tm + m) * Ng;
    p1_z1<R1, U, NT>(tid, un, um, x, yb, S);
    __syncthreads();
    p13_z8<R1, U, NT, -1, TWREG>(tid, S, T, twr);
    __syncthreads();
    p1_y1<R1, U, NT>(tid, S, W, x, yb);
}

// ---- bulk-copy (TMA, 1-D) and mbarrier helpers for pass B --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)), "l"(gsrc),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_all() {
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// pass B: second y step, x transform, K', inverse x, first inverse y step; in place on the pair's work box.  The tile
// (k1y, zb) is one contiguous run of the work box (layout widx): N rows of 512 bytes are bulk-copied (TMA) into the padded
// shared-memory tile, all five steps run in shared memory, and the rows are bulk-copied back.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) pass_b_kernel(cplx* __restrict__ work, const double* __restrict__ kperm, int npairs) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z, NT = FusedCfg<R1>::NT2, PX = P2Geo<Z>::PX;
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr uint32_t ROWB = 8 * Z * sizeof(cplx);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    __shared__ __align__(8) uint64_t bar;
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int pair = bid % npairs;
    const int tile = bid / npairs;
    const int k1y = tile / (N / Z);
    cplx* Wt = work + (size_t)pair * Ng + (size_t)tile * ((size_t)N * 8 * Z);
    const double* Kt = kperm + (size_t)tile * ((size_t)N * 8 * Z);
    if (tid == 0) mbar_init(&bar, 1);
    __syncthreads();
    if (tid == 0) mbar_arrive_expect_tx(&bar, ROWB * N);
    for (int x = tid; x < N; x += NT) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar);
    mbar_wait(&bar, 0);
    p2_y8<R1, Z, NT, -1>(tid, S, k1y);
    __syncthreads();
    p2_xR<R1, Z, NT, -1>(tid, S);
    __syncthreads();
    p2_x8<R1, Z, NT>(tid, S, Kt);
    __syncthreads();
    p2_xR<R1, Z, NT, +1>(tid, S);
    __syncthreads();
    p2_y8<R1, Z, NT, +1>(tid, S, k1y);
    fence_proxy_async_smem();
    __syncthreads();
    for (int x = tid; x < N; x += NT) bulk_s2g(Wt + x * 8 * Z, S + x * PX, ROWB);
    bulk_commit_wait_all();
}

// pass C: second inverse y step, inverse z, acc_n -= w f u_m v.  One CTA per (tile, n) loops over the m-tile with its
// accumulator tile in shared memory, then adds it to acc_n in global memory once (fixed summation order).
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT3, FusedCfg<R1>::MINB3) pass_c_kernel(const cplx* __restrict__ work, const cplx* __restrict__ uq_base, MTile mt,
                                                                    int tn, cplx* __restrict__ acc) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U3, NT = FusedCfg<R1>::NT3;
    constexpr bool TWREG = FusedCfg<R1>::TWREG, ACCREG = FusedCfg<R1>::ACCREG;
    static_assert(!TWREG || NT % R1 == 0, "TWREG needs a thread-invariant k1z");
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr int IT = (U * R1 * 8 + NT - 1) / NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    cplx* A = S + U * R1 * N;                       // unused when ACCREG
    cplx* T = A + (ACCREG ? 0 : U * R1 * N);
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int n = bid % tn;
    const int tile = bid / tn;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    cplx twr[8];
    if (TWREG)
        load_twr<R1>(tid, twr);
    else
        for (int i = tid; i < R1 * 8; i += NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    cplx accr[ACCREG ? IT * R1 : 1];
    if (ACCREG) {
#pragma unroll
        for (int i = 0; i < (ACCREG ? IT * R1 : 1); i++) accr[i] = mk(0.0, 0.0);
    }
    for (int m = 0; m < mt.tm; m++) {
        const cplx* W = work + ((size_t)n * mt.tm + m) * Ng;
        const cplx* um = uq_base + (size_t)mt.m_idx[m] * Ng;
        p3_y2inv<R1, U, NT>(tid, W, x, yb, S);
        __syncthreads();
        p13_z8<R1, U, NT, +1, TWREG>(tid, S, T, twr);
        __syncthreads();
        if (ACCREG)
            p3_zinv2_reg<R1, U, NT>(tid, S, um, mt.wf[m], x, yb, accr);
        else
            p3_zinv2<R1, U, NT>(tid, S, um, mt.wf[m], x, yb, A, m == 0);
        __syncthreads();
    }
    if (ACCREG)
        p3_flush_reg<R1, U, NT>(tid, accr, acc + (size_t)n * Ng, x, yb);
    else
        p3_flush<R1, U, NT>(tid, A, acc + (size_t)n * Ng, x, yb);
}

// ---------------------------------------------------------------------------------------------------------------
template <int R1>
struct Launch {
    static constexpr int N = 8 * R1, U1 = FusedCfg<R1>::U1, U3 = FusedCfg<R1>::U3, Z = FusedCfg<R1>::Z;
    static constexpr bool TWREG = FusedCfg<R1>::TWREG, ACCREG = FusedCfg<R1>::ACCREG;
    static constexpr size_t smem_a = sizeof(cplx) * ((size_t)U1 * R1 * N + (TWREG ? 0 : R1 * 8));
    static constexpr size_t smem_c = sizeof(cplx) * ((size_t)(ACCREG ? 1 : 2) * U3 * R1 * N + (TWREG ? 0 : R1 * 8));
    static constexpr size_t smem_b = sizeof(cplx) * ((size_t)N * P2Geo<Z>::PX);

    static int init(exx_ctx* c) {
        EXX_CUDA(c, cudaFuncSetAttribute(pass_a_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_b_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_c_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c));
        return EXX_OK;
    }
    // all pairs (n0..n0+tn) x mt of one (k, q): the three passes
    static int pairs(exx_ctx* c, const cplx* un_base, const cplx* uq_base, const MTile& mt, int tn, const double* kperm, cplx* work, cplx* acc) {
        const int npairs = tn * mt.tm;
        const unsigned tiles1 = N * (8 / U1), tiles3 = N * (8 / U3), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_PASS_A, npairs);
            pass_a_kernel<R1><<<tiles1 * npairs, FusedCfg<R1>::NT1, smem_a, c->stream>>>(un_base, uq_base, mt, tn, work);
        }
        {
            LaunchScope ls(c, KC_PASS_B, npairs);
            pass_b_kernel<R1><<<tiles2 * npairs, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, kperm, npairs);
        }
        {
            LaunchScope ls(c, KC_PASS_C, npairs);
            pass_c_kernel<R1><<<tiles3 * tn, FusedCfg<R1>::NT3, smem_c, c->stream>>>(work, uq_base, mt, tn, acc);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
};

#define EXX_DISPATCH_R1(R1v, EXPR)                  \
    switch (R1v) {                                  \
    case 6: { typedef Launch<6> L; EXPR; } break;   \
    case 8: { typedef Launch<8> L; EXPR; } break;   \
    case 9: { typedef Launch<9> L; EXPR; } break;   \
    case 12: { typedef Launch<12> L; EXPR; } break; \
    case 16: { typedef Launch<16> L; EXPR; } break; \
    default: return EXX_ERR_BAD_ARG;                \
    }

bool fused_supported(const exx_ctx* c) {
    int n = c->N[0];
    if (c->N[1] != n || c->N[2] != n) return false;
    return n == 48 || n == 64 || n == 72 || n == 96 || n == 128;
}

void fused_tiles(const exx_ctx* c, int* tn, int* tm) {
    // defaults: 16 x 16 pairs per batch (fewer, longer launches: measured 5 % faster than 4 x 16), shrunk so that the pair
    // workspace stays below ~4 GiB
#ifdef EXX_TUNE_TN
    int n = EXX_TUNE_TN, m = EXX_TUNE_TM;
#else
    int n = 16, m = 16;
#endif
    size_t box = sizeof(cplx) * (size_t)c->Ng;
    while ((size_t)n * m * box > ((size_t)4 << 30) && m > 4) m /= 2;
    while ((size_t)n * m * box > ((size_t)4 << 30) && n > 4) n /= 2;
    *tn = std::min(n, c->nb);
    *tm = std::min(m, c->nb);
}

int fused_create(exx_ctx* c) {
    FusedState* st = new (std::nothrow) FusedState();
    if (!st) return EXX_ERR_ALLOC;
    c->fused = st;
    st->R1 = c->N[0] / 8;
    // twiddles W_N^j for every supported N (long double angles), to constant memory
    {
        const int Ns[5] = {48, 64, 72, 96, 128};
        const int off[5] = {TwOff<6>::v, TwOff<8>::v, TwOff<9>::v, TwOff<12>::v, TwOff<16>::v};
        const long double tp = 6.283185307179586476925286766559005768L;
        for (int s = 0; s < 5; s++)
            for (int j = 0; j < Ns[s]; j++) {
                long double a = tp * j / Ns[s];
                h_tw[off[s] + j] = mk((double)cosl(a), (double)(-sinl(a)));
            }
        EXX_CUDA(c, cudaMemcpyToSymbol(c_tw, h_tw, sizeof(h_tw)));
    }
    // permuted kernel tables
    size_t Ng = (size_t)c->Ng;
    cudaError_t e = cudaMalloc((void**)&st->kperm_dev, sizeof(double) * Ng * c->ntab);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return EXX_ERR_ALLOC;
    }
    c->dev_bytes += sizeof(double) * Ng * c->ntab;
    std::vector<double> nat(Ng), perm(Ng);
    int Z = 4;
    EXX_DISPATCH_R1(st->R1, Z = L::Z);
    for (int t = 0; t < c->ntab; t++) {
        EXX_CUDA(c, cudaMemcpy(nat.data(), c->ktab_dev + (size_t)t * Ng, sizeof(double) * Ng, cudaMemcpyDeviceToHost));
        permute_ktable(st->R1, Z, nat.data(), perm.data());
        EXX_CUDA(c, cudaMemcpy(st->kperm_dev + (size_t)t * Ng, perm.data(), sizeof(double) * Ng, cudaMemcpyHostToDevice));
    }
    int rc = EXX_OK;
    EXX_DISPATCH_R1(st->R1, rc = L::init(c));
    return rc;
}

void fused_destroy(exx_ctx* c) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return;
    cudaFree(st->kperm_dev);
    delete st;
    c->fused = nullptr;
}

int fused_apply(exx_ctx* c, const double* occ, const double2* psi, double2* out) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return EXX_ERR_BAD_ARG;
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    c->path_used = 2;
    c->pruned_used = 0;
    if ((rc = compute_u_cache(c, psi))) return rc;
    int tn_max = (int)c->acc_boxes, tm_max = (int)std::min<size_t>(32, c->work_boxes / c->acc_boxes);
    if (c->opt_tile_n > 0) tn_max = (int)std::min<int64_t>(tn_max, c->opt_tile_n);
    if (c->opt_tile_m > 0) tm_max = (int)std::min<int64_t>(tm_max, c->opt_tile_m);
    c->tile_n_used = tn_max;
    c->tile_m_used = tm_max;
    cplx* work = (cplx*)c->work_dev;
    cplx* acc = (cplx*)c->acc_dev;
    for (int k = 0; k < nk; k++)
        for (int n0 = 0; n0 < nb; n0 += tn_max) {
            const int tn = std::min(tn_max, nb - n0);
            EXX_CUDA(c, cudaMemsetAsync(acc, 0, sizeof(cplx) * Ng * tn, c->stream));
            const cplx* un_base = (const cplx*)c->u_dev + ((size_t)k * nb + n0) * Ng;
            for (int q = 0; q < nk; q++) {
                const double* kperm = st->kperm_dev + (size_t)c->ktab_of[(size_t)k * nk + q] * Ng;
                const cplx* uq = (const cplx*)c->u_dev + (size_t)q * nb * Ng;
                MTile mt;
                mt.tm = 0;
                for (int m = 0; m <= nb; m++) {
                    if (m < nb && occ[q * nb + m] != 0.0) {
                        mt.m_idx[mt.tm] = m;
                        mt.wf[mt.tm] = c->kw[q] * occ[q * nb + m];
                        mt.tm++;
                    }
                    if (mt.tm == tm_max || (m == nb && mt.tm > 0)) {
                        EXX_DISPATCH_R1(st->R1, rc = L::pairs(c, un_base, uq, mt, tn, kperm, work, acc));
                        if (rc) return rc;
                        c->pairs_executed += (int64_t)tn * mt.tm;
                        c->pairs_ordered += (int64_t)tn * mt.tm;
                        mt.tm = 0;
                    }
                }
            }
            // S7: forward transform of the accumulators, gather onto sphere(k)
            if ((rc = launch_fft3d_generic(c, (double2*)acc, tn, -1))) return rc;
            if ((rc = launch_gather(c, k, (const double2*)acc, tn, out + c->off[k] + (int64_t)n0 * c->npw[k]))) return rc;
        }
    return EXX_OK;
}

}  // namespace exx
