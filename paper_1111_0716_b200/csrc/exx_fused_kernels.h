// exx_fused_kernels.h — the kernels of the fused passes and their launchers (Launch<R1>), mode-generic like
// exx_fused_phases.h: exx_fused.cu includes it once per (EXX_NS, EXX_REAL) — exx / double for the fp64 product path, exx32 /
// float for the mixed-precision pair pipeline.  Product code: shares nothing with oracle/.
#include "exx_fused_phases.h"

namespace EXX_NS {
#ifdef EXX_SECOND_MODE  // names of exx_internal.h that the first mode (namespace exx) sees directly
using ::exx::AJob;
using ::exx::CJob;
using ::exx::DJob;
using ::exx::RJob;
using ::exx::RowMask;
using ::exx::KC_PASS_R;
using ::exx::KC_SCATTER;
using ::exx::LaunchScope;
using ::exx::KC_PASS_A;
using ::exx::KC_PASS_B;
using ::exx::KC_PASS_C;
using ::exx::KC_FFT_FUSED;
using ::exx::KC_ENERGY;
using ::exx::EJob;
using ::exx::TMAX;
using ::exx::pair_sum_kernel;
using ::exx::band_energy_kernel;
#endif

cplx h_tw[TW_TOTAL];  // host copy of the twiddle tables (source of the constant-memory upload)

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
    // .read: wait only until the shared-memory source has been read (the CTA may then retire and free its tile); the global
    // writes are complete at the kernel boundary, which is where the next pass starts
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// pass B: second y step, x transform, K', inverse x, first inverse y step; in place on the pair's work box.  The tile
// (k1y, zb) is one contiguous run of the work box (layout widx): N rows of 512 bytes are bulk-copied (TMA) into the padded
// shared-memory tile, all five steps run in shared memory, and the rows are bulk-copied back.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) pass_b_kernel(cplx* __restrict__ work, const real* __restrict__ kperm, AJob job) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z, NT = FusedCfg<R1>::NT2, PX = P2Geo<Z>::PX;
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr uint32_t ROWB = 8 * Z * sizeof(cplx);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    // the tile arrives in chunks of NT / Z rows, one mbarrier each: iteration i of the first step touches chunk i only, so it can
    // start as soon as that chunk has landed
    constexpr int CR = NT / Z, NCH = (N + CR - 1) / CR;
    static_assert(NT % Z == 0, "chunks are whole rows");
    __shared__ __align__(8) uint64_t bar[NCH];
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int p = bid % job.npairs;
    const int tile = bid / job.npairs;
    const int k1y = tile / (N / Z);
    cplx* Wt = work + (size_t)(job.pi[p] * job.tb + job.pj[p]) * Ng + (size_t)tile * ((size_t)N * 8 * Z);
    const real* Kt = kperm + (size_t)tile * ((size_t)N * 8 * Z);
    if (tid < NCH) mbar_init(&bar[tid], 1);
    __syncthreads();
    if (tid < NCH) mbar_arrive_expect_tx(&bar[tid], ROWB * (uint32_t)((tid + 1) * CR <= N ? CR : N - tid * CR));
    for (int x = tid; x < N; x += NT) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar[x / CR]);
    p2_y8<R1, Z, NT, -1>(tid, S, k1y, [&](int i) { mbar_wait(&bar[i], 0); });
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

// Energy route (E2): pass B cut after the forward x transform.  Instead of multiplying by K' and
// transforming back, the CTA sums K'(g) |rho^(g)|^2 over its tile in a fixed order (thread-serial, xor-shuffle tree, warps in
// order) and writes ONE double: epart[pair * tiles + tile].  The work box is only read.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) pass_b_energy_kernel(const cplx* __restrict__ work, const real* __restrict__ kperm, AJob job,
                                                                                         double* __restrict__ epart) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z, NT = FusedCfg<R1>::NT2, PX = P2Geo<Z>::PX;
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr uint32_t ROWB = 8 * Z * sizeof(cplx);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    constexpr int CR = NT / Z, NCH = (N + CR - 1) / CR;
    static_assert(NT % Z == 0, "chunks are whole rows");
    __shared__ __align__(8) uint64_t bar[NCH];
    __shared__ double wsum[(NT + 31) / 32];
    const int tid = threadIdx.x;
    const unsigned bid = blockIdx.x;
    const int p = bid % job.npairs;
    const int tile = bid / job.npairs;
    const int k1y = tile / (N / Z);
    const cplx* Wt = work + (size_t)(job.pi[p] * job.tb + job.pj[p]) * Ng + (size_t)tile * ((size_t)N * 8 * Z);
    const real* Kt = kperm + (size_t)tile * ((size_t)N * 8 * Z);
    if (tid < NCH) mbar_init(&bar[tid], 1);
    __syncthreads();
    if (tid < NCH) mbar_arrive_expect_tx(&bar[tid], ROWB * (uint32_t)((tid + 1) * CR <= N ? CR : N - tid * CR));
    for (int x = tid; x < N; x += NT) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar[x / CR]);
    p2_y8<R1, Z, NT, -1>(tid, S, k1y, [&](int i) { mbar_wait(&bar[i], 0); });
    __syncthreads();
    p2_xR<R1, Z, NT, -1>(tid, S);
    __syncthreads();
    double e = p2_x8_energy<R1, Z, NT>(tid, S, Kt);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((tid & 31) == 0) wsum[tid >> 5] = e;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < (NT + 31) / 32; w++) t += wsum[w];
        epart[(size_t)p * (R1 * (N / Z)) + tile] = t;
    }
}

#ifndef EXX_SECOND_MODE
// pairsum[p] = sum over the tiles of pair p, fixed order: lane-strided serial sums, then an xor-shuffle tree.  One warp per pair.
__global__ void pair_sum_kernel(const double* __restrict__ epart, int ntiles, double* __restrict__ pairsum) {
    const double* e = epart + (size_t)blockIdx.x * ntiles;
    double s = 0.0;
    for (int t = threadIdx.x; t < ntiles; t += 32) s += e[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) pairsum[blockIdx.x] = s;
}
// band_e2[band] += (w f)_band * sum over the band's pairs of (w f)_partner * pairsum: one thread per band and side, pairs in list
// order, side a before side b (a diagonal block has the same bands on both sides), launches serial on the stream: deterministic.
__global__ void band_energy_kernel(AJob job, EJob ej, const double* __restrict__ pairsum_g, double* __restrict__ band_e2) {
    const int t = threadIdx.x;
    __shared__ double pairsum[TMAX * TMAX];  // staged once: the serial loops below then run at shared-memory latency
    for (int p = t; p < job.npairs; p += blockDim.x) pairsum[p] = pairsum_g[p];
    __syncthreads();
    if (t < TMAX) {
        double s = 0.0;
        bool any = false;
        for (int p = 0; p < job.npairs; p++)
            if (job.pi[p] == t) s += ej.wb[job.pj[p]] * pairsum[p], any = true;
        if (any) band_e2[ej.tgt_a + job.a_idx[t]] += ej.wa[t] * s;
    }
    __syncthreads();
    if (t >= TMAX && ej.sym) {
        const int j = t - TMAX;
        double s = 0.0;
        bool any = false;
        for (int p = 0; p < job.npairs; p++)
            if (job.pj[p] == j && !(ej.same_k && job.a_idx[job.pi[p]] == job.b_idx[j])) s += ej.wa[job.pi[p]] * pairsum[p], any = true;
        if (any) band_e2[ej.tgt_b + job.b_idx[j]] += ej.wb[j] * s;
    }
}
#endif

// pass C: second inverse y step, inverse z, acc -= coef u v.  One CTA per (tile, row) loops over the row's columns with
// its accumulator tile on chip, then adds it to the row's accumulator box in global memory once (fixed summation order).
// Rows/columns are the a/b bands of the batch (CJob); the transposed sweep (cj) uses conj(v) and the a-band as multiplier.
template <int R1>
__global__ void __launch_bounds__(FusedCfg<R1>::NT3, FusedCfg<R1>::MINB3) pass_c_kernel(const cplx* __restrict__ work, const cplx* __restrict__ usrc_base, CJob job,
                                                                    acc_c* __restrict__ acc_base) {
    constexpr int N = 8 * R1, U = FusedCfg<R1>::U3, NT = FusedCfg<R1>::NT3;
    constexpr bool TWREG = FusedCfg<R1>::TWREG, ACCREG = FusedCfg<R1>::ACCREG, STAGE3 = FusedCfg<R1>::STAGE3 >= 1, STAGEU = FusedCfg<R1>::STAGE3 >= 2;
    static_assert(!TWREG || NT % R1 == 0, "TWREG needs a thread-invariant k1z");
    constexpr size_t Ng = (size_t)N * N * N;
    constexpr int IT = (U * R1 * 8 + NT - 1) / NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S = reinterpret_cast<cplx*>(smem_raw);
    acc_c* A = reinterpret_cast<acc_c*>(S + U * R1 * N);  // fp64 accumulator tile; unused when ACCREG
    cplx* T = reinterpret_cast<cplx*>(A + (ACCREG ? 0 : U * R1 * N));
    cplx* G = T + (TWREG ? 0 : R1 * 8);  // STAGE3: per-thread slots for the next column's work-box elements
    cplx* G2 = G + Slots<R1, U, NT>::COUNT;  // ... and for this column's u elements
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
    acc_c accr[ACCREG ? IT * R1 : 1];
    if (ACCREG) {
#pragma unroll
        for (int i = 0; i < (ACCREG ? IT * R1 : 1); i++) accr[i] = mka(0.0, 0.0);
    }
    if (STAGE3 && cnt > 0) {
        p3_stage<R1, U, NT>(tid, work + (size_t)(r * job.box_r + job.col[r][0] * job.box_c) * Ng, x, yb, G);
        stage_commit();
    }
    for (int ci = 0; ci < cnt; ci++) {
        const int col = job.col[r][ci];
        const cplx* W = work + (size_t)(r * job.box_r + col * job.box_c) * Ng;
        const cplx* um = usrc_base + (size_t)job.src[col] * Ng;
        const double wf = job.coef[col];
        if (STAGE3) {
            // this column's elements were requested one column ago; the next column's are requested as soon as the slots
            // have been read (the transform consumes them first, so the copies cannot overtake the reads)
            stage_wait<0>();
            p3_y2inv_staged<R1, U, NT>(tid, G, S);
            if (STAGEU) p3_stage_u<R1, U, NT>(tid, um, x, yb, G2);  // group 1: this column's u elements, consumed two barriers from here
            stage_commit();
            if (ci + 1 < cnt) p3_stage<R1, U, NT>(tid, work + (size_t)(r * job.box_r + job.col[r][ci + 1] * job.box_c) * Ng, x, yb, G);
            stage_commit();                             // group 2 (possibly empty): the next column's work-box elements
        } else {
            p3_y2inv<R1, U, NT>(tid, W, x, yb, S);
        }
        __syncthreads();
        p13_z8<R1, U, NT, +1, TWREG>(tid, S, T, twr);
        __syncthreads();
        if (STAGEU) stage_wait<1>();  // the u elements have landed; the next column's work-box elements may still be in flight
        if (ACCREG)
            p3_zinv2_reg<R1, U, NT, STAGEU>(tid, S, um, wf, x, yb, accr, cj, G2);
        else
            p3_zinv2<R1, U, NT, STAGEU>(tid, S, um, wf, x, yb, A, ci == 0, cj, G2);
        __syncthreads();
    }
    if (cnt > 0) {
        if (ACCREG)
            p3_flush_reg<R1, U, NT>(tid, accr, acc_base + (size_t)job.tgt[r] * Ng, x, yb);
        else
            p3_flush<R1, U, NT>(tid, A, acc_base + (size_t)job.tgt[r] * Ng, x, yb);
    }
}


// ---- dual sweep (pair symmetry): one inverse transform per pair, both accumulations ----------------------------------------
// CTA = (tile, row group): RG warp groups of NT3 threads, group wg owns row g*RG + wg of the batch: its two tiles S (columns
// alternate between them), its staging slots G (next column's work-box elements), its slots UA ((-w_k f_a) u_a of the row, loaded
// once) and its register accumulators.  The column's u_b elements are staged once per CTA, one column ahead, into G2[column parity].
// Per column: [y step] group barrier [8-point z step] group barrier [last z step; side a into registers; side b = P written over
// the thread's own elements of S] CTA barrier [P tiles of the groups added in group order -> partial box (row group, column)].
// The one CTA barrier also hands over the next column's u_b slots; the reduction reads the tiles the next column does not write.
// Every sum has a fixed order: deterministic.
__device__ __forceinline__ void group_barrier(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

template <int R1>
struct DualGeo {
    static constexpr int N = 8 * R1, U = FusedCfg<R1>::U3, NT = FusedCfg<R1>::NT3, RG = FusedCfg<R1>::RG > 0 ? FusedCfg<R1>::RG : 1;
    static constexpr int TILE = U * R1 * N;
    static constexpr int SL = Slots<R1, U, NT>::COUNT;  // slots of one step of one group
    static constexpr size_t smem = sizeof(cplx) * ((size_t)RG * (2 * TILE + 2 * SL) + 2 * SL + R1 * 8);
};

template <int R1>
__global__ void __launch_bounds__(DualGeo<R1>::RG * DualGeo<R1>::NT, 1) pass_c_dual_kernel(const cplx* __restrict__ work, const cplx* __restrict__ ua_base,
                                                                                        const cplx* __restrict__ ub_base, DJob job,
                                                                                        acc_c* __restrict__ acc_base, cplx* __restrict__ part_base) {
    typedef DualGeo<R1> D;
    constexpr int N = D::N, U = D::U, NT = D::NT, RG = D::RG, TILE = D::TILE, SL = D::SL;
    constexpr int ITU = (U * R1 * 8 + NT - 1) / NT;
    constexpr size_t Ng = (size_t)N * N * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* S0 = reinterpret_cast<cplx*>(smem_raw);  // [parity][group][TILE]
    cplx* G0 = S0 + 2 * RG * TILE;
    cplx* UA0 = G0 + RG * SL;
    cplx* G2 = UA0 + RG * SL;  // [parity][SL]
    cplx* T = G2 + 2 * SL;
    const int tid_cta = threadIdx.x;
    const int wg = tid_cta / NT, tid = tid_cta - wg * NT;
    cplx* G = G0 + wg * SL;
    cplx* UA = UA0 + wg * SL;
    const unsigned bid = blockIdx.x;
    const int g = bid % job.nrg;
    const int tile = bid / job.nrg;
    const int x = tile / (8 / U), yb = tile % (8 / U);
    const int row = g * RG + wg;
    const bool rowok = row < job.ta;
    const unsigned ev = rowok ? job.ev[row] : 0u, bs = rowok ? job.bside[row] : 0u;
    unsigned cta_ev = 0u;
#pragma unroll
    for (int w = 0; w < RG; w++)
        if (g * RG + w < job.ta) cta_ev |= job.ev[g * RG + w];
    for (int i = tid_cta; i < R1 * 8; i += RG * NT) T[tidx(i >> 3, i & 7)] = c_tw[TwOff<R1>::v + (i >> 3) * (i & 7)];
    cplx twr[8];  // (TWREG is not used by the dual sweep)
    acc_c accr[ITU * R1];
#pragma unroll
    for (int i = 0; i < ITU * R1; i++) accr[i] = mka(0.0, 0.0);
    const size_t rowbox = (size_t)row * job.tb;
    unsigned rem = cta_ev;
    if (bs) p3_stage_u<R1, U, NT>(tid, ua_base + (size_t)job.a_src[rowok ? row : 0] * Ng, x, yb, UA);
    if (rem) {
        const int c0 = __ffs(rem) - 1;
        if (ev >> c0 & 1u) p3_stage<R1, U, NT>(tid, work + (rowbox + c0) * Ng, x, yb, G);
        if (job.amask >> c0 & 1u) p3_stage_u_share<R1, U, NT, RG>(wg, tid, ub_base + (size_t)job.b_src[c0] * Ng, x, yb, G2);
    }
    stage_commit();
    stage_wait<0>();
    if (bs) p3_scale_slots<R1, U, NT>(tid, UA, (real)(-job.coef_a[row]));
    __syncthreads();  // twiddle table; the first column's u_b slots
    int par = 0;
    while (rem) {
        const int c = __ffs(rem) - 1;
        rem &= rem - 1;
        const bool act = ev >> c & 1u;
        cplx* S = S0 + (par * RG + wg) * TILE;
        if (act) p3_y2inv_staged<R1, U, NT>(tid, G, S);
        if (rem) {  // the next column's work-box elements (this group's row) and this thread's share of its u_b elements
            const int cn = __ffs(rem) - 1;
            if (ev >> cn & 1u) p3_stage<R1, U, NT>(tid, work + (rowbox + cn) * Ng, x, yb, G);
            if (job.amask >> cn & 1u) p3_stage_u_share<R1, U, NT, RG>(wg, tid, ub_base + (size_t)job.b_src[cn] * Ng, x, yb, G2 + (par ^ 1) * SL);
        }
        stage_commit();
        group_barrier(1 + wg, NT);
        if (act) p13_z8<R1, U, NT, +1, false>(tid, S, T, twr);
        group_barrier(1 + wg, NT);
        if (act) p3_zinv2_dual<R1, U, NT>(tid, S, G2 + par * SL, UA, job.coef_b[c], job.amask >> c & 1u, bs >> c & 1u, accr);
        unsigned gm = 0u;
#pragma unroll
        for (int w = 0; w < RG; w++)
            if (g * RG + w < job.ta && (job.bside[g * RG + w] >> c & 1u)) gm |= 1u << w;
        stage_wait<0>();
        __syncthreads();  // P tiles complete; the next column's u_b slots complete; this column's u_b slots free
        if (gm) p3_reduce_b<R1, U, NT, RG>(wg, tid, S0 + par * RG * TILE, TILE, gm, part_base + ((size_t)g * job.tb + c) * Ng, x, yb);
        par ^= 1;
    }
    if (ev & job.amask) p3_flush_reg<R1, U, NT>(tid, accr, acc_base + (size_t)job.a_tgt[row] * Ng, x, yb);
}

// pass R: acc[tgt[col]] += sum_g partial[g*tb + col] over the row groups that wrote one, in group order (fixed: deterministic)
template <int DUMMY>
__global__ void __launch_bounds__(256) pass_r_kernel(const cplx* __restrict__ part, RJob job, acc_c* __restrict__ acc_base, size_t Ng) {
    const int col = blockIdx.y;
    const unsigned gm = job.gmask[col];
    if (!gm) return;
    acc_c* acc = acc_base + (size_t)job.tgt[col] * Ng;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < Ng; p += (size_t)gridDim.x * blockDim.x) {
        double sx = 0.0, sy = 0.0;
        for (int g = 0; g < job.nrg; g++)
            if (gm >> g & 1u) {
                cplx v = part[((size_t)g * job.tb + col) * Ng + p];
                sx += (double)v.x;
                sy += (double)v.y;
            }
        acc_c a = acc[p];
        acc[p] = mka(a.x + sx, a.y + sy);
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
// inverse y step (F layout ->).  Sphere pruning (S1/S7): bit x of `rows` says whether F-layout x row x can hold a
// sphere coefficient (|kx| <= gmax).  The inverse (S1) bulk-copies only those rows in and zero-fills the others on chip (they are
// never read from the box, so the scatter need not clear them); the forward (S7) writes only those rows back (the gather reads
// no other).  All ones = plain transform.
template <int R1, int SIGN>
__global__ void __launch_bounds__(FusedCfg<R1>::NT2, FusedCfg<R1>::MINB2) fft_b_kernel(cplx* __restrict__ work, int nbox, RowMask rows) {
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
    if (SIGN > 0) {
        int nrows = 0;
#pragma unroll
        for (int i = 0; i < 4; i++) nrows += __popc(rows.w[i]);
        if (tid == 0) mbar_arrive_expect_tx(&bar, ROWB * (uint32_t)nrows);
        for (int x = tid; x < N; x += NT)
            if (rows.w[x >> 5] >> (x & 31) & 1u) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar);
        if (nrows < N) {
            for (int e = tid; e < N * 8 * Z; e += NT) {
                const int x = e / (8 * Z);
                if (!(rows.w[x >> 5] >> (x & 31) & 1u)) S[x * PX + (e - x * 8 * Z)] = mk(EXX_RC(0.0), EXX_RC(0.0));
            }
        }
        mbar_wait(&bar, 0);
        if (nrows < N) __syncthreads();  // the zero rows were written by other threads
    } else {
        if (tid == 0) mbar_arrive_expect_tx(&bar, ROWB * N);
        for (int x = tid; x < N; x += NT) bulk_g2s(S + x * PX, Wt + x * 8 * Z, ROWB, &bar);
        mbar_wait(&bar, 0);
    }
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
    for (int x = tid; x < N; x += NT)
        if (SIGN > 0 || (rows.w[x >> 5] >> (x & 31) & 1u)) bulk_s2g(Wt + x * 8 * Z, S + x * PX, ROWB);
    bulk_commit_wait_all();
}

// clears the F-layout x rows of `rows` in nbox work boxes (the only rows the pruned inverse transform reads): S1's scatter target
template <int R1>
__global__ void __launch_bounds__(256) zero_rows_kernel(cplx* __restrict__ work, RowMask rows) {
    constexpr int N = 8 * R1, Z = FusedCfg<R1>::Z;
    constexpr size_t Ng = (size_t)N * N * N;
    // one CTA per (box, pass-B tile): N rows of 8 Z elements
    cplx* Wt = work + (size_t)blockIdx.y * Ng + (size_t)blockIdx.x * ((size_t)N * 8 * Z);
    for (int e = threadIdx.x; e < N * 8 * Z; e += blockDim.x) {
        const int x = e / (8 * Z);
        if (rows.w[x >> 5] >> (x & 31) & 1u) Wt[e] = mk(EXX_RC(0.0), EXX_RC(0.0));
    }
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
    static constexpr bool TWREG = FusedCfg<R1>::TWREG, ACCREG = FusedCfg<R1>::ACCREG, STAGE3 = FusedCfg<R1>::STAGE3 >= 1, STAGEU = FusedCfg<R1>::STAGE3 >= 2;
    static constexpr int IT3S = (U3 * N + FusedCfg<R1>::NT3 - 1) / FusedCfg<R1>::NT3;  // items per thread in pass C's first step
    static constexpr size_t smem_a = sizeof(cplx) * ((size_t)U1 * R1 * N + (TWREG ? 0 : R1 * 8));
    static constexpr size_t smem_c = sizeof(cplx) * ((size_t)U3 * R1 * N + (TWREG ? 0 : R1 * 8)) + sizeof(acc_c) * (ACCREG ? 0 : (size_t)U3 * R1 * N);
    static constexpr int IT3U = (U3 * R1 * 8 + FusedCfg<R1>::NT3 - 1) / FusedCfg<R1>::NT3;  // ... and in its last step
    static constexpr size_t smem_c3 = smem_c + sizeof(cplx) * (size_t)((STAGE3 ? 1 : 0) + (STAGEU ? 1 : 0)) * Slots<R1, FusedCfg<R1>::U3, FusedCfg<R1>::NT3>::COUNT;  // pass_c_kernel
    static constexpr size_t smem_b = sizeof(cplx) * ((size_t)N * P2Geo<Z>::PX);

    static constexpr int RG = FusedCfg<R1>::RG;  // dual sweep: rows per CTA (0: not built for this grid)
    static constexpr size_t smem_d = DualGeo<R1>::smem;

    static int init(exx_ctx* c) {
        if (RG > 0) EXX_CUDA(c, cudaFuncSetAttribute(pass_c_dual_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_d));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_a_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_b_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_c_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c3));
        EXX_CUDA(c, cudaFuncSetAttribute(pass_b_energy_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute(fft_a_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a));
        EXX_CUDA(c, cudaFuncSetAttribute((fft_b_kernel<R1, -1>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute((fft_b_kernel<R1, +1>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));
        EXX_CUDA(c, cudaFuncSetAttribute(fft_c_kernel<R1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c));
        return EXX_OK;
    }
    // passes A and B over the pairs of one batch
    static int pass_ab(exx_ctx* c, const cplx* ua_base, const cplx* ub_base, const AJob& job, const real* kperm, cplx* work) {
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
    // energy route: pass A, the forward half of pass B with the K' |rho^|^2 sum, and the two small fixed-order reductions
    static int pass_a_energy(exx_ctx* c, const cplx* ua_base, const cplx* ub_base, const AJob& job, const EJob& ej, const real* kperm, cplx* work,
                             double* epart, double* pairsum, double* band_e2) {
        const unsigned tiles1 = N * (8 / U1), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_PASS_A, job.npairs);
            pass_a_kernel<R1><<<tiles1 * job.npairs, FusedCfg<R1>::NT1, smem_a, c->stream>>>(ua_base, ub_base, job, work);
        }
        {
            LaunchScope ls(c, KC_PASS_B, job.npairs);
            pass_b_energy_kernel<R1><<<tiles2 * job.npairs, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, kperm, job, epart);
        }
        {
            LaunchScope ls(c, KC_ENERGY, job.npairs);
            pair_sum_kernel<<<job.npairs, 32, 0, c->stream>>>(epart, (int)tiles2, pairsum);
        }
        {
            LaunchScope ls(c, KC_ENERGY, job.npairs);
            band_energy_kernel<<<1, 2 * TMAX, 0, c->stream>>>(job, ej, pairsum, band_e2);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    // plain transforms of nbox boxes: forward natural in -> F layout in work; inverse F layout in work -> natural out
    static RowMask all_rows() {
        RowMask m;
        for (int i = 0; i < 4; i++) m.w[i] = 0u;
        for (int x = 0; x < N; x++) m.w[x >> 5] |= 1u << (x & 31);  // exactly N bits: the kernel counts them for its transfer size
        return m;
    }
    // F-layout x rows that hold frequencies |kx| <= gmax
    static RowMask sphere_rows(int gmax) {
        RowMask m;
        for (int i = 0; i < 4; i++) m.w[i] = 0u;
        for (int kx = 0; kx < N; kx++) {
            const int g = 2 * kx < N ? kx : kx - N;
            if (g >= -gmax && g <= gmax) {
                const int xpos = 8 * (kx % R1) + kx / R1;
                m.w[xpos >> 5] |= 1u << (xpos & 31);
            }
        }
        return m;
    }
    static int zero_rows(exx_ctx* c, cplx* work, int nbox, const RowMask& rows) {
        LaunchScope ls(c, KC_SCATTER, 0);
        zero_rows_kernel<R1><<<dim3(R1 * (N / Z), nbox), 256, 0, c->stream>>>(work, rows);
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    static int fft_forward(exx_ctx* c, const cplx* in_base, int nbox, cplx* work, const RowMask& rows = all_rows()) {
        const unsigned tiles1 = N * (8 / U1), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_a_kernel<R1><<<tiles1 * nbox, FusedCfg<R1>::NT1, smem_a, c->stream>>>(in_base, nbox, work);
        }
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_b_kernel<R1, -1><<<tiles2 * nbox, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, nbox, rows);
        }
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    static int fft_inverse(exx_ctx* c, cplx* work, int nbox, cplx* out_base, const RowMask& rows = all_rows()) {
        const unsigned tiles3 = N * (8 / U3), tiles2 = R1 * (N / Z);
        {
            LaunchScope ls(c, KC_FFT_FUSED, nbox);
            fft_b_kernel<R1, +1><<<tiles2 * nbox, FusedCfg<R1>::NT2, smem_b, c->stream>>>(work, nbox, rows);
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
    // the dual sweep (pair symmetry) and the reduction of its partial boxes
    static int pass_c_dual(exx_ctx* c, const cplx* ua_base, const cplx* ub_base, const DJob& job, int64_t units, const cplx* work, acc_c* acc_base,
                           cplx* part) {
        const unsigned tiles3 = N * (8 / U3);
        LaunchScope ls(c, KC_PASS_C, units);
        pass_c_dual_kernel<R1><<<tiles3 * job.nrg, DualGeo<R1>::RG * FusedCfg<R1>::NT3, smem_d, c->stream>>>(work, ua_base, ub_base, job, acc_base, part);
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    static int pass_r(exx_ctx* c, const RJob& job, int64_t units, const cplx* part, acc_c* acc_base) {
        LaunchScope ls(c, KC_PASS_R, units);
        const size_t Ng = (size_t)N * N * N;
        pass_r_kernel<0><<<dim3((unsigned)((Ng + 511) / 512), job.ncol), 256, 0, c->stream>>>(part, job, acc_base, Ng);
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
    // one accumulation sweep (pass C)
    static int pass_c(exx_ctx* c, const cplx* usrc_base, const CJob& job, int64_t units, const cplx* work, acc_c* acc_base) {
        const unsigned tiles3 = N * (8 / U3);
        LaunchScope ls(c, KC_PASS_C, units);
        pass_c_kernel<R1><<<tiles3 * job.nr, FusedCfg<R1>::NT3, smem_c3, c->stream>>>(work, usrc_base, job, acc_base);
        EXX_CUDA(c, cudaGetLastError());
        return EXX_OK;
    }
};

// twiddles W_N^j for every supported N (long double angles), to this mode's constant memory
inline int upload_twiddles(exx_ctx* c) {
    const long double tp = 6.283185307179586476925286766559005768L;
    for (int r1 = 1; r1 <= 16; r1++)
        for (int j = 0; j < 8 * r1; j++) {
            long double a = tp * j / (8 * r1);
            h_tw[4 * r1 * (r1 - 1) + j] = mk((real)cosl(a), (real)(-sinl(a)));
        }
    EXX_CUDA(c, cudaMemcpyToSymbol(c_tw, h_tw, sizeof(h_tw)));
    return EXX_OK;
}

}  // namespace EXX_NS
