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
    int32_t* fmap_dev = nullptr;  // per k: F-layout index of every sphere vector (offsets = exx_ctx::map_off)
    int tn = 0, tm = 0;
};

// ---------------------------------------------------------------------------------------------------------------
// pass A: rho = conj(u_b) u_a, z transform, first y step.  One CTA per (tile, pair), pair fastest so that the CTAs that
// share a u tile run back to back and the tile is fetched from HBM once.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT1, FusedCfg<R1>::MINB1) pass_a_kernel(const cplx* __restrict__ ua_base, const cplx* __restrict__ ub_base,
                                                                    AJob job, cplx* __restrict__ work) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U1, NT = FusedCfg<R1>::NT1;
    constexpr bool TWREG = FusedCfg<R1>::TWREG;
    static_assert(!TWREG || NT % R1 == 0, "TWREG needs a thread-invariant k1z");
    constexpr size_t Ng = (size_t)N * N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = S + U * R1 * N;
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int p = bid % job.npairs;
    const int tile = bid / job.npairs;
    const int pi = job.pi[p], pj = job.pj[p];
    const int x = tile / (8 / U), yb = tile % (8 / U);
    cplx twr[8];
    if (TWREG)
        load_twr<R1>(tid, twr);
    else
        for (int i = tid; i < R1 * 8; i += NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    const cplx* un = ua_base + (size_t)job.a_idx[pi] * Ng;
    const cplx* um = ub_base + (size_t)job.b_idx[pj] * Ng;
    cplx* W = work + (size_t)(pi * job.tb + pj) * Ng;
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
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) pass_b_kernel(cplx* __restrict__ work, const double* __restrict__ kperm, AJob job) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z, NT = FusedCfg<R1>::NT2, PX = P2Geo<Z>::PX;
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr uint32_t ROWB = 8 * Z * sizeof(cplx);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    __shared__ __align__(8) uint64_t bar;
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int p = bid % job.npairs;
    const int tile = bid / job.npairs;
    const int k1y = tile / (N / Z);
    cplx* Wt = work + (size_t)(job.pi[p] * job.tb + job.pj[p]) * Ng + (size_t)tile * ((size_t)N * 8 * Z);
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

// pass C: second inverse y step, inverse z, acc -= coef u v.  One CTA per (tile, row) loops over the row's columns with
// its accumulator tile on chip, then adds it to the row's accumulator box in global memory once (fixed summation order).
// Rows/columns are the a/b bands of the batch (CJob); the transposed sweep (cj) uses conj(v) and the a-band as multiplier.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT3, FusedCfg<R1>::MINB3) pass_c_kernel(const cplx* __restrict__ work, const cplx* __restrict__ usrc_base, CJob job,
                                                                    cplx* __restrict__ acc_base) {
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
    const int r = bid % job.nr;
    const int tile = bid / job.nr;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    const int cnt = job.cnt[r];
    const bool cj = job.cj != 0;
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
    for (int ci = 0; ci < cnt; ci++) {
        const int col = job.col[r][ci];
        const cplx* W = work + (size_t)(r * job.box_r + col * job.box_c) * Ng;
        const cplx* um = usrc_base + (size_t)job.src[col] * Ng;
        const double wf = job.coef[col];
        p3_y2inv<R1, U, NT>(tid, W, x, yb, S);
        __syncthreads();
        p13_z8<R1, U, NT, +1, TWREG>(tid, S, T, twr);
        __syncthreads();
        if (ACCREG)
            p3_zinv2_reg<R1, U, NT>(tid, S, um, wf, x, yb, accr, cj);
        else
            p3_zinv2<R1, U, NT>(tid, S, um, wf, x, yb, A, ci == 0, cj);
        __syncthreads();
    }
    if (cnt > 0) {
        if (ACCREG)
            p3_flush_reg<R1, U, NT>(tid, accr, acc_base + (size_t)job.tgt[r] * Ng, x, yb);
        else
            p3_flush<R1, U, NT>(tid, A, acc_base + (size_t)job.tgt[r] * Ng, x, yb);
    }
}

// ---- plain 3-D transforms through the same passes (S1, S7; F layout, see exx_fused_phases.h) ------------------------
// forward first half: natural box p of in_base -> work box p (z transform, first y step)
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT1, FusedCfg<R1>::MINB1) fft_a_kernel(const cplx* __restrict__ in_base, int nbox, cplx* __restrict__ work) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U1, NT = FusedCfg<R1>::NT1;
    constexpr bool TWREG = FusedCfg<R1>::TWREG;
    constexpr size_t Ng = (size_t)N * N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = S + U * R1 * N;
    const int tid = threadIdx.x;
    const int p = blockIdx.x % nbox, tile = blockIdx.x / nbox;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    cplx twr[8];
    if (TWREG)
        load_twr<R1>(tid, twr);
    else
        for (int i = tid; i < R1 * 8; i += NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    p1_z1_single<R1, U, NT>(tid, in_base + (size_t)p * Ng, x, yb, S);
    __syncthreads();
    p13_z8<R1, U, NT, -1, TWREG>(tid, S, T, twr);
    __syncthreads();
    p1_y1<R1, U, NT>(tid, S, work + (size_t)p * Ng, x, yb);
}

// the pass-B half, in place on work box p.  SIGN < 0: second y step, forward x (-> F layout); SIGN > 0: inverse x, first
// inverse y step (F layout ->)
template <int R1, int SIGN>
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) fft_b_kernel(cplx* __restrict__ work, int nbox) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z, NT = FusedCfg<R1>::NT2, PX = P2Geo<Z>::PX;
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr uint32_t ROWB = 8 * Z * sizeof(cplx);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    __shared__ __align__(8) uint64_t bar;
    const int tid = threadIdx.x;
    const int p = blockIdx.x % nbox, tile = blockIdx.x / nbox;
    const int k1y = tile / (N / Z);
    cplx* Wt = work + (size_t)p * Ng + (size_t)tile * ((size_t)N * 8 * Z);
    if (tid == 0) mbar_init(&bar, 1);
    __syncthreads();
    if (tid == 0) mbar_arrive_expect_tx(&bar, ROWB * N);
    for (int x = tid; x < N; x += NT) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar);
    mbar_wait(&bar, 0);
    if (SIGN < 0) {
        p2_y8<R1, Z, NT, -1>(tid, S, k1y);
        __syncthreads();
        p2_xR<R1, Z, NT, -1>(tid, S);
        __syncthreads();
        p2_x8_half<R1, Z, NT, -1>(tid, S);
    } else {
        p2_x8_half<R1, Z, NT, +1>(tid, S);
        __syncthreads();
        p2_xR<R1, Z, NT, +1>(tid, S);
        __syncthreads();
        p2_y8<R1, Z, NT, +1>(tid, S, k1y);
    }
    fence_proxy_async_smem();
    __syncthreads();
    for (int x = tid; x < N; x += NT) bulk_s2g(Wt + x * 8 * Z, S + x * PX, ROWB);
    bulk_commit_wait_all();
}

// inverse second half: work box p -> natural box p of out_base (second inverse y step, inverse z)
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT3, FusedCfg<R1>::MINB3) fft_c_kernel(const cplx* __restrict__ work, int nbox, cplx* __restrict__ out_base) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U3, NT = FusedCfg<R1>::NT3;
    constexpr bool TWREG = FusedCfg<R1>::TWREG;
    constexpr size_t Ng = (size_t)N * N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = S + U * R1 * N;
    const int tid = threadIdx.x;
    const int p = blockIdx.x % nbox, tile = blockIdx.x / nbox;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    cplx twr[8];
    if (TWREG)
        load_twr<R1>(tid, twr);
    else
        for (int i = tid; i < R1 * 8; i += NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    p3_y2inv<R1, U, NT>(tid, work + (size_t)p * Ng, x, yb, S);
    __syncthreads();
    p13_z8<R1, U, NT, +1, TWREG>(tid, S, T, twr);
    __syncthreads();
    p3_zinv2_store<R1, U, NT>(tid, S, out_base + (size_t)p * Ng, x, yb);
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
        EXX_CUDA(c, cudaFuncSetAttribute(fft_a_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a));
        EXX_CUDA(c, cudaFuncSetAttribute((fft_b_kernel<R1, -1>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute((fft_b_kernel<R1, +1>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute(fft_c_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c));
        return EXX_OK;
    }
    // passes A and B over the pairs of one batch
    static int pass_ab(exx_ctx* c, const cplx* ua_base, const cplx* ub_base, const AJob& job, const double* kperm, cplx* work) {
        const unsigned tiles1 = N * (8 / U1), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_PASS_A, job.npairs);
            pass_a_kernel<R1><<<tiles1 * job.npairs, FusedCfg<R1>::NT1, smem_a, c->stream>>>(ua_base, ub_base, job, work);
        }
        {
            LaunchScope ls(c, KC_PASS_B, job.npairs);
            pass_b_kernel<R1><<<tiles2 * job.npairs, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, kperm, job);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    // plain transforms of nbox boxes: forward natural in -> F layout in work; inverse F layout in work -> natural out
    static int fft_forward(exx_ctx* c, const cplx* in_base, int nbox, cplx* work) {
        const unsigned tiles1 = N * (8 / U1), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_a_kernel<R1><<<tiles1 * nbox, FusedCfg<R1>::NT1, smem_a, c->stream>>>(in_base, nbox, work);
        }
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_b_kernel<R1, -1><<<tiles2 * nbox, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, nbox);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    static int fft_inverse(exx_ctx* c, cplx* work, int nbox, cplx* out_base) {
        const unsigned tiles3 = N * (8 / U3), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_b_kernel<R1, +1><<<tiles2 * nbox, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, nbox);
        }
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_c_kernel<R1><<<tiles3 * nbox, FusedCfg<R1>::NT3, smem_c, c->stream>>>(work, nbox, out_base);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    static void fill_fmap(const int32_t* nat, int n, int32_t* out) {
        for (int i = 0; i < n; i++) {
            int j = nat[i];
            out[i] = (int32_t)findex<R1>(j / (N * N), (j / N) % N, j % N);
        }
    }
    // one accumulation sweep (pass C)
    static int pass_c(exx_ctx* c, const cplx* usrc_base, const CJob& job, int64_t units, const cplx* work, cplx* acc_base) {
        const unsigned tiles3 = N * (8 / U3);
        LaunchScope ls(c, KC_PASS_C, units);
        pass_c_kernel<R1><<<tiles3 * job.nr, FusedCfg<R1>::NT3, smem_c, c->stream>>>(work, usrc_base, job, acc_base);
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
    // sphere -> F layout maps for S1 / S7
    if (cudaMalloc((void**)&st->fmap_dev, sizeof(int32_t) * (size_t)std::max<int64_t>(1, c->map_off[c->nk])) != cudaSuccess) {
        cudaGetLastError();
        return EXX_ERR_ALLOC;
    }
    for (int k = 0; k < c->nk; k++) {
        std::vector<int32_t> fm(c->npw[k]);
        EXX_DISPATCH_R1(st->R1, L::fill_fmap(c->map_h[k].data(), c->npw[k], fm.data()));
        EXX_CUDA(c, cudaMemcpy(st->fmap_dev + c->map_off[k], fm.data(), sizeof(int32_t) * c->npw[k], cudaMemcpyHostToDevice));
    }
    int rc = EXX_OK;
    EXX_DISPATCH_R1(st->R1, rc = L::init(c));
    return rc;
}

void fused_destroy(exx_ctx* c) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return;
    cudaFree(st->kperm_dev);
    cudaFree(st->fmap_dev);
    delete st;
    c->fused = nullptr;
}

// The loop nest (k and q on the host, band loops on the device, innermost loop blocked).  Bands are cut into
// a-tiles (k-point k) and b-tiles (k-point q) of at most 16; every batch evaluates v for the pairs of one (a-tile, b-tile)
// block (passes A, B) and sweeps pass C once per side that receives a contribution.
//   plain mode:    all ordered (k, q); pair (a, b) evaluated iff f_b != 0;   acc_a -= w_q f_b u_b v
//   symmetry mode: k <= q, and a <= b when k == q; pair evaluated iff f_a != 0 or f_b != 0;
//                  acc_a -= w_q f_b u_b v   and (unless a == b)   acc_b -= w_k f_a u_a conj(v)
// using v_{bq,ak} = conj(v_{ak,bq}) (K real and K_{q-k}(g) = K_{k-q}(-g); exact on an alias-free grid).
int fused_apply(exx_ctx* c, const double* occ, const double2* psi, double2* out) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return EXX_ERR_BAD_ARG;
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    c->path_used = 2;
    c->pruned_used = 0;
    // S1: sphere coefficients -> F-layout work boxes (scatter) -> inverse transform through passes B/C -> u cache
    for (int k = 0; k < nk; k++) {
        const int bmax = (int)std::min<size_t>(c->work_boxes, (size_t)nb);
        for (int n0 = 0; n0 < nb; n0 += bmax) {
            const int bn = std::min(bmax, nb - n0);
            if ((rc = launch_scatter(c, k, psi + c->off[k] + (int64_t)n0 * c->npw[k], bn, (double2*)c->work_dev, st->fmap_dev + c->map_off[k]))) return rc;
            EXX_DISPATCH_R1(st->R1, rc = L::fft_inverse(c, (cplx*)c->work_dev, bn, (cplx*)c->u_dev + ((size_t)k * nb + n0) * Ng));
            if (rc) return rc;
        }
    }
    int ta_max = 16, tb_max = 16;
    while ((size_t)ta_max * tb_max > c->work_boxes && tb_max > 1) tb_max /= 2;
    while ((size_t)ta_max * tb_max > c->work_boxes && ta_max > 1) ta_max /= 2;
    if (c->opt_tile_n > 0) ta_max = (int)std::min<int64_t>(ta_max, c->opt_tile_n);
    if (c->opt_tile_m > 0) tb_max = (int)std::min<int64_t>(tb_max, c->opt_tile_m);
    const bool sym = c->opt_symmetry && c->alias_free;
    if (sym) ta_max = tb_max = std::min(ta_max, tb_max);  // diagonal blocks need matching tiles
    c->tile_n_used = ta_max;
    c->tile_m_used = tb_max;
    c->symmetry_used = sym ? 1 : 0;
    cplx* work = (cplx*)c->work_dev;
    cplx* acc = (cplx*)c->acc_dev;  // one accumulator box per (k, band)
    EXX_CUDA(c, cudaMemsetAsync(acc, 0, sizeof(cplx) * Ng * (size_t)nk * nb, c->stream));
    for (int k = 0; k < nk; k++)
        for (int q = sym ? k : 0; q < nk; q++) {
            const double* kperm = st->kperm_dev + (size_t)c->ktab_of[(size_t)k * nk + q] * Ng;
            const cplx* ua = (const cplx*)c->u_dev + (size_t)k * nb * Ng;
            const cplx* ub = (const cplx*)c->u_dev + (size_t)q * nb * Ng;
            // b-bands: in plain mode only bands with f != 0 take part as m
            std::vector<int> blist;
            for (int m = 0; m < nb; m++)
                if (sym || occ[q * nb + m] != 0.0) blist.push_back(m);
            for (int a0 = 0; a0 < nb; a0 += ta_max)
                for (size_t b0 = (sym && k == q) ? (size_t)a0 : 0; b0 < blist.size(); b0 += tb_max) {
                    const int ta = std::min(ta_max, nb - a0), tb = (int)std::min<size_t>(tb_max, blist.size() - b0);
                    AJob aj;
                    aj.npairs = 0;
                    aj.tb = tb;
                    bool ev[16][16];
                    for (int i = 0; i < ta; i++) aj.a_idx[i] = a0 + i;
                    for (int j = 0; j < tb; j++) aj.b_idx[j] = blist[b0 + j];
                    for (int i = 0; i < ta; i++)
                        for (int j = 0; j < tb; j++) {
                            const double fa = occ[k * nb + aj.a_idx[i]], fb = occ[q * nb + aj.b_idx[j]];
                            bool e = sym ? ((fa != 0.0 || fb != 0.0) && (k < q || aj.a_idx[i] <= aj.b_idx[j])) : (fb != 0.0);
                            ev[i][j] = e;
                            if (e) {
                                aj.pi[aj.npairs] = (unsigned char)i;
                                aj.pj[aj.npairs] = (unsigned char)j;
                                aj.npairs++;
                            }
                        }
                    if (aj.npairs == 0) continue;
                    EXX_DISPATCH_R1(st->R1, rc = L::pass_ab(c, ua, ub, aj, kperm, work));
                    if (rc) return rc;
                    c->pairs_executed += aj.npairs;
                    // side a: rows = a-bands, columns = b-bands with f_b != 0
                    {
                        CJob cj;
                        cj.nr = 0;
                        cj.box_r = tb;
                        cj.box_c = 1;
                        cj.cj = 0;
                        int64_t units = 0;
                        int rowbox[16];
                        for (int j = 0; j < tb; j++) {
                            cj.src[j] = aj.b_idx[j];
                            cj.coef[j] = c->kw[q] * occ[q * nb + aj.b_idx[j]];
                        }
                        for (int i = 0; i < ta; i++) {
                            int n = 0;
                            for (int j = 0; j < tb; j++)
                                if (ev[i][j] && occ[q * nb + aj.b_idx[j]] != 0.0) cj.col[cj.nr][n++] = (unsigned char)j;
                            if (n) {
                                cj.cnt[cj.nr] = n;
                                cj.tgt[cj.nr] = k * nb + aj.a_idx[i];
                                rowbox[cj.nr] = i;
                                cj.nr++;
                                units += n;
                            }
                        }
                        if (cj.nr) {
                            // rows were compacted: the work box of (row r, column c) is rowbox[r]*tb + c, so shift the work
                            // base per launch only when rows are contiguous; otherwise launch row by row groups
                            bool contiguous = true;
                            for (int r = 0; r < cj.nr; r++) contiguous = contiguous && rowbox[r] == rowbox[0] + r;
                            if (contiguous) {
                                EXX_DISPATCH_R1(st->R1, rc = L::pass_c(c, ub, cj, units, work + (size_t)rowbox[0] * tb * Ng, acc));
                                if (rc) return rc;
                            } else {
                                for (int r = 0; r < cj.nr; r++) {
                                    CJob one = cj;
                                    one.nr = 1;
                                    one.cnt[0] = cj.cnt[r];
                                    one.tgt[0] = cj.tgt[r];
                                    for (int n = 0; n < cj.cnt[r]; n++) one.col[0][n] = cj.col[r][n];
                                    EXX_DISPATCH_R1(st->R1, rc = L::pass_c(c, ub, one, cj.cnt[r], work + (size_t)rowbox[r] * tb * Ng, acc));
                                    if (rc) return rc;
                                }
                            }
                            c->pairs_ordered += units;
                        }
                    }
                    // side b (symmetry): rows = b-bands, columns = a-bands with f_a != 0, conj(v); the pair a == b is not repeated
                    if (sym) {
                        CJob cj;
                        cj.nr = 0;
                        cj.box_r = 1;
                        cj.box_c = tb;
                        cj.cj = 1;
                        int64_t units = 0;
                        int rowbox[16];
                        for (int i = 0; i < ta; i++) {
                            cj.src[i] = aj.a_idx[i];
                            cj.coef[i] = c->kw[k] * occ[k * nb + aj.a_idx[i]];
                        }
                        for (int j = 0; j < tb; j++) {
                            int n = 0;
                            for (int i = 0; i < ta; i++)
                                if (ev[i][j] && occ[k * nb + aj.a_idx[i]] != 0.0 && !(k == q && aj.a_idx[i] == aj.b_idx[j]))
                                    cj.col[cj.nr][n++] = (unsigned char)i;
                            if (n) {
                                cj.cnt[cj.nr] = n;
                                cj.tgt[cj.nr] = q * nb + aj.b_idx[j];
                                rowbox[cj.nr] = j;
                                cj.nr++;
                                units += n;
                            }
                        }
                        if (cj.nr) {
                            bool contiguous = true;
                            for (int r = 0; r < cj.nr; r++) contiguous = contiguous && rowbox[r] == rowbox[0] + r;
                            if (contiguous) {
                                EXX_DISPATCH_R1(st->R1, rc = L::pass_c(c, ua, cj, units, work + (size_t)rowbox[0] * Ng, acc));
                                if (rc) return rc;
                            } else {
                                for (int r = 0; r < cj.nr; r++) {
                                    CJob one = cj;
                                    one.nr = 1;
                                    one.cnt[0] = cj.cnt[r];
                                    one.tgt[0] = cj.tgt[r];
                                    for (int n = 0; n < cj.cnt[r]; n++) one.col[0][n] = cj.col[r][n];
                                    EXX_DISPATCH_R1(st->R1, rc = L::pass_c(c, ua, one, cj.cnt[r], work + (size_t)rowbox[r] * Ng, acc));
                                    if (rc) return rc;
                                }
                            }
                            c->pairs_ordered += units;
                        }
                    }
                }
        }
    // S7: forward transform of every accumulator through passes A/B (-> F layout), gather onto sphere(k)
    for (int k = 0; k < nk; k++) {
        const int bmax = (int)std::min<size_t>(c->work_boxes, (size_t)nb);
        for (int n0 = 0; n0 < nb; n0 += bmax) {
            const int bn = std::min(bmax, nb - n0);
            EXX_DISPATCH_R1(st->R1, rc = L::fft_forward(c, acc + ((size_t)k * nb + n0) * Ng, bn, work));
            if (rc) return rc;
            if ((rc = launch_gather(c, k, (const double2*)work, bn, out + c->off[k] + (int64_t)n0 * c->npw[k], st->fmap_dev + c->map_off[k]))) return rc;
        }
    }
    return EXX_OK;
}

}  // namespace exx
