// exx_fused.cu — host side of the fused three-pass pair pipeline (S1..S7) for cubic grids N = 8 R1, R1 in {2, 4, 5, 6, 8, 9, 10, 12, 16}
// (N = 16, 32, 40, 48, 64, 72, 80, 96, 128).  The per-thread phases live in exx_fused_phases.h, the kernels and launchers in
// exx_fused_kernels.h (compiled twice: fp64 and fp32); this file holds the permuted kernel tables, the F-layout sphere maps and
// the loop nest over k, q and band-pair batches
// (k,q loops on the host, band loops on the device, innermost loop blocked).
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <vector>

#include "exx_internal.h"
#include "exx_shard.h"

#include "exx_fused_kernels.h"  // fp64 mode: namespace exx, real = double

// mixed-precision mode (EXX_OPT_PRECISION = 1): the same phases, kernels and launchers in fp32
#undef EXX_NS
#undef EXX_REAL
#define EXX_NS exx32
#define EXX_REAL float
#define EXX_SECOND_MODE
#include "exx_fused_kernels.h"
#undef EXX_SECOND_MODE

namespace exx {

struct FusedState {
    int R1 = 0;
    double* kperm_dev = nullptr;  // ntab tables, permuted order of pass B
    int32_t* fmap_dev = nullptr;  // per k: F-layout index of every sphere vector (offsets = exx_ctx::map_off)
    // mixed precision (allocated on first use): fp32 copies of the u cache and of the permuted kernel tables
    exx32::cplx* u32_dev = nullptr;
    float* kperm32_dev = nullptr;
    // energy route (fused_energy): per-CTA partial sums of one batch, per-pair sums, per-band sums
    double* epart_dev = nullptr;
    double* pairsum_dev = nullptr;
    double* band_e2_dev = nullptr;
    // exx_apply_to: real-space boxes of the trial vectors phi (allocated on first use, nk*nb boxes like the u cache)
    cplx* uphi_dev = nullptr;
    size_t uphi_boxes = 0;
    // dual sweep of pass C (pair symmetry): partial boxes of the second side, one per (row group, column) of a batch
    // (allocated by fused_ensure_part before the first dual sweep; an allocation that failed is remembered and not retried at that size)
    cplx* part_dev = nullptr;
    size_t part_boxes = 0;
    size_t part_refused = 0;
};

#define EXX_DISPATCH_R1(R1v, EXPR)                  \
    switch (R1v) {                                  \
    case 2: { typedef Launch<2> L; EXPR; } break;   \
    case 4: { typedef Launch<4> L; EXPR; } break;   \
    case 5: { typedef Launch<5> L; EXPR; } break;   \
    case 10: { typedef Launch<10> L; EXPR; } break; \
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
    return n == 16 || n == 32 || n == 40 || n == 48 || n == 64 || n == 72 || n == 80 || n == 96 || n == 128;
}

void fused_tiles(const exx_ctx* c, int* tn, int* tm) {
    // defaults: EXX_DEFAULT_TILE^2 pairs per batch (fewer, longer launches and fewer accumulator round trips: 16 x 16 measured
    // 5 % faster than 4 x 16, 32 x 32 another 3 % at C4a), shrunk so that the pair workspace stays below EXX_WORK_CAP_GIB
#ifdef EXX_TUNE_TN
    int n = EXX_TUNE_TN, m = EXX_TUNE_TM;
#else
    int n = EXX_DEFAULT_TILE, m = EXX_DEFAULT_TILE;
#endif
    size_t box = sizeof(cplx) * (size_t)c->Ng;
    const size_t cap = (size_t)EXX_WORK_CAP_GIB << 30;
    while ((size_t)n * m * box > cap && m > 4) m /= 2;
    while ((size_t)n * m * box > cap && n > 4) n /= 2;
    *tn = std::min(n, c->nb);
    *tm = std::min(m, c->nb);
}

int fused_create(exx_ctx* c) {
    FusedState* st = new (std::nothrow) FusedState();
    if (!st) return EXX_ERR_ALLOC;
    c->fused = st;
    st->R1 = c->N[0] / 8;
    if (int rct = upload_twiddles(c)) return rct;
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
        permute_ktable(st->R1, Z, exx::KVW, nat.data(), perm.data());
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
    {
        const size_t tiles2 = (size_t)st->R1 * (c->N[0] / Z);
        if (cudaMalloc((void**)&st->epart_dev, sizeof(double) * TMAX * TMAX * tiles2) != cudaSuccess ||
            cudaMalloc((void**)&st->pairsum_dev, sizeof(double) * TMAX * TMAX) != cudaSuccess ||
            cudaMalloc((void**)&st->band_e2_dev, sizeof(double) * (size_t)c->nk * c->nb) != cudaSuccess) {
            cudaGetLastError();
            return EXX_ERR_ALLOC;
        }
        c->dev_bytes += sizeof(double) * (TMAX * TMAX * (tiles2 + 1) + (size_t)c->nk * c->nb);
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
    cudaFree(st->u32_dev);
    cudaFree(st->kperm32_dev);
    cudaFree(st->epart_dev);
    cudaFree(st->pairsum_dev);
    cudaFree(st->band_e2_dev);
    cudaFree(st->uphi_dev);
    cudaFree(st->part_dev);
    delete st;
    c->fused = nullptr;
}

// Stand-alone batched 3-D transform through the fused passes (S8(f)-3; the paper's third intercept, offloads
// FFT3D calls above a size threshold).  Forward: natural-order boxes `in` -> F-layout boxes `out`.  Inverse: F-layout boxes
// `in` (used as scratch, destroyed) -> natural-order boxes `out`.  Needs only the twiddles and kernel attributes, none of the
// per-band buffers.
int fused_fft3d(exx_ctx* c, double2* in, int nbatch, int sign, double2* out) {
    if (!fused_supported(c)) return EXX_ERR_BAD_GRID;
    const int R1 = c->N[0] / 8;
    int rc = EXX_OK;
    if (!c->fft_ready) {
        if ((rc = upload_twiddles(c))) return rc;
        EXX_DISPATCH_R1(R1, rc = L::init(c));
        if (rc) return rc;
        c->fft_ready = true;
    }
    const size_t Ng = (size_t)c->Ng;
    const int bmax = 1 << 12;  // keeps every grid well below 2^31 CTAs
    for (int b0 = 0; b0 < nbatch; b0 += bmax) {
        const int bn = std::min(bmax, nbatch - b0);
        if (sign < 0) {
            EXX_DISPATCH_R1(R1, rc = L::fft_forward(c, (const cplx*)in + (size_t)b0 * Ng, bn, (cplx*)out + (size_t)b0 * Ng));
        } else {
            EXX_DISPATCH_R1(R1, rc = L::fft_inverse(c, (cplx*)in + (size_t)b0 * Ng, bn, (cplx*)out + (size_t)b0 * Ng));
        }
        if (rc) return rc;
    }
    return EXX_OK;
}
int fused_findex(const exx_ctx* c, int32_t* host_out) {
    if (!fused_supported(c)) return EXX_ERR_BAD_GRID;
    const int R1 = c->N[0] / 8, N = c->N[0];
    std::vector<int32_t> nat((size_t)N);
    for (int kx = 0; kx < N; kx++)
        for (int ky = 0; ky < N; ky++) {
            for (int kz = 0; kz < N; kz++) nat[kz] = (int32_t)(((int64_t)kx * N + ky) * N + kz);
            EXX_DISPATCH_R1(R1, L::fill_fmap(nat.data(), N, host_out + ((size_t)kx * N + ky) * N));
        }
    return EXX_OK;
}

__global__ void to_float_kernel(const double* __restrict__ in, float* __restrict__ out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = (float)in[i];
}
static int init_mode32(exx_ctx* c, int R1) {
    switch (R1) {
    case 2: return exx32::Launch<2>::init(c);
    case 4: return exx32::Launch<4>::init(c);
    case 5: return exx32::Launch<5>::init(c);
    case 10: return exx32::Launch<10>::init(c);
    case 6: return exx32::Launch<6>::init(c);
    case 8: return exx32::Launch<8>::init(c);
    case 9: return exx32::Launch<9>::init(c);
    case 12: return exx32::Launch<12>::init(c);
    case 16: return exx32::Launch<16>::init(c);
    default: return EXX_ERR_BAD_ARG;
    }
}

// the mode of the pair pipeline: fp64 (product default) or fp32 transforms with fp64 accumulation
struct ModeD {
    typedef exx::cplx cplx;
    typedef double real;
    template <int R1>
    using L = exx::Launch<R1>;
};
struct ModeF {
    typedef exx32::cplx cplx;
    typedef float real;
    template <int R1>
    using L = exx32::Launch<R1>;
};
#define EXX_DISPATCH_M(R1v, EXPR)                                      \
    switch (R1v) {                                                     \
    case 2: { typedef typename M::template L<2> L; EXPR; } break;      \
    case 4: { typedef typename M::template L<4> L; EXPR; } break;      \
    case 5: { typedef typename M::template L<5> L; EXPR; } break;      \
    case 10: { typedef typename M::template L<10> L; EXPR; } break;    \
    case 6: { typedef typename M::template L<6> L; EXPR; } break;      \
    case 8: { typedef typename M::template L<8> L; EXPR; } break;      \
    case 9: { typedef typename M::template L<9> L; EXPR; } break;      \
    case 12: { typedef typename M::template L<12> L; EXPR; } break;    \
    case 16: { typedef typename M::template L<16> L; EXPR; } break;    \
    default: return EXX_ERR_BAD_ARG;                                   \
    }

template <class M>
static int pair_loop(exx_ctx* c, FusedState* st, const double* occ, const typename M::cplx* u_base, typename M::cplx* work,
                     const typename M::real* kperm_base, acc_c* acc, bool sym, int ta_max, int tb_max,
                     const typename M::cplx* ua_base = nullptr /* a-bands from another set of boxes (exx_apply_to; needs !sym) */,
                     int na = -1 /* ... na of them per k-point, boxes (k * na + a) */) {
    if (!ua_base) ua_base = u_base;
    if (na < 0) na = c->nb;
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    // the batch list and its owners (exx_shard.h); one shard = the whole list
    std::vector<PairBlock> blocks;
    plan_blocks(nk, nb, occ, sym, ta_max, tb_max, (int)c->opt_shard_count, blocks, na);
    std::vector<int> blist;
    int bl_q = -1;
    for (const PairBlock& blk : blocks) {
        if (blk.shard != (int)c->opt_shard_rank) continue;
        const int k = blk.k, q = blk.q;
        const typename M::real* kperm = kperm_base + (size_t)c->ktab_of[(size_t)k * nk + q] * Ng;
        const typename M::cplx* ua = ua_base + (size_t)k * na * Ng;
        const typename M::cplx* ub = u_base + (size_t)q * nb * Ng;
        if (bl_q != q) b_list(nb, occ, q, sym, blist), bl_q = q;
        const int a0 = blk.a0, ta = blk.ta, tb = blk.tb;
        const size_t b0 = (size_t)blk.b0;
        AJob aj;
        aj.npairs = 0;
        aj.tb = tb;
        bool ev[TMAX][TMAX];
        for (int i = 0; i < ta; i++) aj.a_idx[i] = a0 + i;
        for (int j = 0; j < tb; j++) aj.b_idx[j] = blist[b0 + j];
        for (int i = 0; i < ta; i++)
            for (int j = 0; j < tb; j++) {
                const double fa = aj.a_idx[i] < nb ? occ[k * nb + aj.a_idx[i]] : 0.0, fb = occ[q * nb + aj.b_idx[j]];
                bool e = pair_evaluated(sym, k, q, aj.a_idx[i], aj.b_idx[j], fa, fb);
                ev[i][j] = e;
                if (e) {
                    aj.pi[aj.npairs] = (unsigned char)i;
                    aj.pj[aj.npairs] = (unsigned char)j;
                    aj.npairs++;
                }
            }
        if (aj.npairs == 0) continue;
        EXX_DISPATCH_M(st->R1, rc = L::pass_ab(c, ua, ub, aj, kperm, work));
        if (rc) return rc;
        c->pairs_executed += aj.npairs;
        int dual_rg = 0;
        EXX_DISPATCH_M(st->R1, dual_rg = L::RG);
        if (sym && dual_rg > 0 && c->opt_dual && st->part_dev && (size_t)((ta + dual_rg - 1) / dual_rg) * tb <= st->part_boxes) {
            // dual sweep: every pair box is transformed back ONCE; side a accumulates on chip per row, side b goes
            // through one partial box per (row group, column), added to the b-bands' accumulators by pass R in row-group order
            DJob dj;
            RJob rj;
            dj.ta = ta, dj.tb = tb, dj.nrg = (ta + dual_rg - 1) / dual_rg, dj.amask = 0u;
            rj.ncol = tb, rj.tb = tb, rj.nrg = dj.nrg;
            int64_t units_a = 0, units_b = 0, boxes = 0, parts = 0;
            for (int j = 0; j < tb; j++) {
                dj.b_src[j] = aj.b_idx[j];
                dj.coef_b[j] = c->kw[q] * occ[q * nb + aj.b_idx[j]];
                if (occ[q * nb + aj.b_idx[j]] != 0.0) dj.amask |= 1u << j;
                rj.tgt[j] = q * nb + aj.b_idx[j];
                rj.gmask[j] = 0u;
            }
            for (int i = 0; i < ta; i++) {
                const double fa = occ[k * nb + aj.a_idx[i]];
                dj.a_tgt[i] = k * na + aj.a_idx[i];
                dj.a_src[i] = aj.a_idx[i];
                dj.coef_a[i] = c->kw[k] * fa;
                dj.ev[i] = dj.bside[i] = 0u;
                for (int j = 0; j < tb; j++) {
                    if (!ev[i][j]) continue;
                    const bool sa = (dj.amask >> j & 1u) != 0, sb = fa != 0.0 && !(k == q && aj.a_idx[i] == aj.b_idx[j]);
                    if (!sa && !sb) continue;
                    dj.ev[i] |= 1u << j;
                    boxes++;
                    if (sa) units_a++;
                    if (sb) {
                        dj.bside[i] |= 1u << j, units_b++;
                        if (!(rj.gmask[j] >> (i / dual_rg) & 1u)) rj.gmask[j] |= 1u << (i / dual_rg), parts++;
                    }
                }
            }
            for (int i = ta; i < TMAX; i++) dj.ev[i] = dj.bside[i] = 0u, dj.a_tgt[i] = dj.a_src[i] = 0, dj.coef_a[i] = 0.0;
            for (int j = tb; j < TMAX; j++) dj.b_src[j] = 0, dj.coef_b[j] = 0.0, rj.tgt[j] = 0, rj.gmask[j] = 0u;
            if (boxes) {
                EXX_DISPATCH_M(st->R1, rc = L::pass_c_dual(c, ua, ub, dj, boxes, work, acc, (typename M::cplx*)st->part_dev));
                if (rc) return rc;
            }
            if (parts) {
                EXX_DISPATCH_M(st->R1, rc = L::pass_r(c, rj, parts, (const typename M::cplx*)st->part_dev, acc));
                if (rc) return rc;
            }
            c->pairs_ordered += units_a + units_b;
            continue;
        }
        // side a: rows = a-bands, columns = b-bands with f_b != 0
        {
            CJob cj;
            cj.nr = 0;
            cj.box_r = tb;
            cj.box_c = 1;
            cj.cj = 0;
            int64_t units = 0;
            int rowbox[TMAX];
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
                    cj.tgt[cj.nr] = k * na + aj.a_idx[i];
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
                    EXX_DISPATCH_M(st->R1, rc = L::pass_c(c, ub, cj, units, work + (size_t)rowbox[0] * tb * Ng, acc));
                    if (rc) return rc;
                } else {
                    for (int r = 0; r < cj.nr; r++) {
                        CJob one = cj;
                        one.nr = 1;
                        one.cnt[0] = cj.cnt[r];
                        one.tgt[0] = cj.tgt[r];
                        for (int n = 0; n < cj.cnt[r]; n++) one.col[0][n] = cj.col[r][n];
                        EXX_DISPATCH_M(st->R1, rc = L::pass_c(c, ub, one, cj.cnt[r], work + (size_t)rowbox[r] * tb * Ng, acc));
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
            int rowbox[TMAX];
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
                    EXX_DISPATCH_M(st->R1, rc = L::pass_c(c, ua, cj, units, work + (size_t)rowbox[0] * Ng, acc));
                    if (rc) return rc;
                } else {
                    for (int r = 0; r < cj.nr; r++) {
                        CJob one = cj;
                        one.nr = 1;
                        one.cnt[0] = cj.cnt[r];
                        one.tgt[0] = cj.tgt[r];
                        for (int n = 0; n < cj.cnt[r]; n++) one.col[0][n] = cj.col[r][n];
                        EXX_DISPATCH_M(st->R1, rc = L::pass_c(c, ua, one, cj.cnt[r], work + (size_t)rowbox[r] * Ng, acc));
                        if (rc) return rc;
                    }
                }
                c->pairs_ordered += units;
            }
        }
    }
    return EXX_OK;
}

// S1: sphere coefficients -> F-layout work boxes (scatter) -> inverse transform through passes B/C -> u cache
// nvec vectors per k-point (default nb), packed like psi; box (k, n) goes to u_out[(k * stride + n) * Ng] (stride default nb)
static int fused_u_cache(exx_ctx* c, FusedState* st, const double2* psi, cplx* u_out = nullptr, int nvec = -1, int stride = -1) {
    if (!u_out) u_out = (cplx*)c->u_dev;
    if (nvec < 0) nvec = c->nb;
    if (stride < 0) stride = c->nb;
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    for (int k = 0; k < nk; k++) {
        const int bmax = (int)std::min<size_t>(c->work_boxes, (size_t)nvec);
        const int64_t offk = c->off[k] / nb * nvec;
        for (int n0 = 0; n0 < nvec; n0 += bmax) {
            const int bn = std::min(bmax, nvec - n0);
            if (c->opt_prune_rows) {
                // sphere pruning: only the x rows with |kx| <= gmax are cleared, scattered into and read by the inverse transform
                RowMask rows;
                EXX_DISPATCH_R1(st->R1, rows = L::sphere_rows(c->gmax[0]));
                EXX_DISPATCH_R1(st->R1, rc = L::zero_rows(c, (cplx*)c->work_dev, bn, rows));
                if (rc) return rc;
                if ((rc = launch_scatter(c, k, psi + offk + (int64_t)n0 * c->npw[k], bn, (double2*)c->work_dev, st->fmap_dev + c->map_off[k], false))) return rc;
                EXX_DISPATCH_R1(st->R1, rc = L::fft_inverse(c, (cplx*)c->work_dev, bn, u_out + ((size_t)k * stride + n0) * Ng, rows));
            } else {
                if ((rc = launch_scatter(c, k, psi + offk + (int64_t)n0 * c->npw[k], bn, (double2*)c->work_dev, st->fmap_dev + c->map_off[k]))) return rc;
                EXX_DISPATCH_R1(st->R1, rc = L::fft_inverse(c, (cplx*)c->work_dev, bn, u_out + ((size_t)k * stride + n0) * Ng));
            }
            if (rc) return rc;
        }
    }
    return EXX_OK;
}

// The partial boxes of the dual sweep, one per (row group, column) of a ta_max x tb_max batch, are made here, right before the first
// apply that can use them (pair symmetry on, EXX_OPT_DUAL_SWEEP on, a grid with a dual kernel) — never for contexts that run without
// the symmetry or with two sweeps.  They come on top of the pair workspace EXX_WORK_CAP_GIB bounds (at most 1/RG of it: 0.25x at
// 72^3, 0.5x at 96^3).  If the device cannot give them the apply is not refused: pair_loop sees no buffer and runs two sweeps.
static int fused_ensure_part(exx_ctx* c, FusedState* st, bool sym, int ta_max, int tb_max) {
    int rg = 0;
    EXX_DISPATCH_R1(st->R1, rg = L::RG);
    if (!sym || !c->opt_dual || rg <= 0) return EXX_OK;
    const size_t Ng = (size_t)c->Ng;
    const size_t need = (size_t)((ta_max + rg - 1) / rg) * tb_max;
    if (need <= st->part_boxes || (st->part_refused && need >= st->part_refused)) return EXX_OK;
    if (st->part_dev) {  // a larger batch than before (tile options changed)
        cudaFree(st->part_dev);
        c->dev_bytes -= sizeof(cplx) * Ng * st->part_boxes;
        st->part_dev = nullptr;
        st->part_boxes = 0;
    }
    if (test_fail_alloc("part") || cudaMalloc((void**)&st->part_dev, sizeof(cplx) * Ng * need) != cudaSuccess) {
        cudaGetLastError();  // out of memory is not an error of this call: two sweeps need no partial boxes
        st->part_dev = nullptr;
        st->part_refused = need;
        return EXX_OK;
    }
    st->part_boxes = need;
    c->dev_bytes += sizeof(cplx) * Ng * need;
    return EXX_OK;
}

// bands per side of a batch and whether the pair symmetry applies (options, workspace, shards); recorded in the counters
static void fused_batch_shape(exx_ctx* c, int* ta, int* tb, bool* symmetry) {
    int ta_max = TMAX, tb_max = TMAX;
    fused_tiles(c, &ta_max, &tb_max);
    if (c->opt_shard_count > 1) ta_max = std::min(ta_max, EXX_SHARD_TILE), tb_max = std::min(tb_max, EXX_SHARD_TILE);
    while ((size_t)ta_max * tb_max > c->work_boxes && tb_max > 1) tb_max /= 2;
    while ((size_t)ta_max * tb_max > c->work_boxes && ta_max > 1) ta_max /= 2;
    if (c->opt_tile_n > 0) ta_max = (int)std::min<int64_t>(ta_max, c->opt_tile_n);
    if (c->opt_tile_m > 0) tb_max = (int)std::min<int64_t>(tb_max, c->opt_tile_m);
    const bool sym = c->opt_symmetry && c->alias_free;
    if (sym) ta_max = tb_max = std::min(ta_max, tb_max);  // diagonal blocks need matching tiles
    c->tile_n_used = ta_max;
    c->tile_m_used = tb_max;
    c->symmetry_used = sym ? 1 : 0;
    *ta = ta_max, *tb = tb_max, *symmetry = sym;
}

// mixed precision: fp32 copies of the permuted kernel tables (built once) and of the u cache (refreshed for this psi)
static int fused_mode32_ready(exx_ctx* c, FusedState* st) {
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    const size_t nbox = (size_t)nk * nb;
    if (!st->u32_dev) {
        if (cudaMalloc((void**)&st->u32_dev, sizeof(exx32::cplx) * Ng * nbox) != cudaSuccess ||
            cudaMalloc((void**)&st->kperm32_dev, sizeof(float) * Ng * c->ntab) != cudaSuccess) {
            cudaGetLastError();
            return EXX_ERR_ALLOC;
        }
        c->dev_bytes += sizeof(exx32::cplx) * Ng * nbox + sizeof(float) * Ng * c->ntab;
        if ((rc = exx32::upload_twiddles(c))) return rc;
        if ((rc = init_mode32(c, st->R1))) return rc;
        // the fp32 mode reads K' four values per load: its own permutation of the natural tables
        std::vector<double> nat(Ng), perm(Ng);
        std::vector<float> permf(Ng);
        int Z = 4;
        EXX_DISPATCH_R1(st->R1, Z = L::Z);
        for (int t = 0; t < c->ntab; t++) {
            EXX_CUDA(c, cudaMemcpy(nat.data(), c->ktab_dev + (size_t)t * Ng, sizeof(double) * Ng, cudaMemcpyDeviceToHost));
            permute_ktable(st->R1, Z, exx32::KVW, nat.data(), perm.data());
            for (size_t i = 0; i < Ng; i++) permf[i] = (float)perm[i];
            EXX_CUDA(c, cudaMemcpy(st->kperm32_dev + (size_t)t * Ng, permf.data(), sizeof(float) * Ng, cudaMemcpyHostToDevice));
        }
        EXX_CUDA(c, cudaDeviceSynchronize());  // pageable copies may still be in flight; one-time set-up
    }
    to_float_kernel<<<2048, 256, 0, c->stream>>>((const double*)c->u_dev, (float*)st->u32_dev, 2 * Ng * nbox);
    EXX_CUDA(c, cudaGetLastError());
    return EXX_OK;
}

// The loop nest (k and q on the host, band loops on the device, innermost loop blocked).  Bands are cut into
// a-tiles (k-point k) and b-tiles (k-point q) of at most TMAX; every batch evaluates v for the pairs of one (a-tile, b-tile)
// block (passes A, B) and sweeps pass C once per side that receives a contribution.
//   plain mode:    all ordered (k, q); pair (a, b) evaluated iff f_b != 0;   acc_a -= w_q f_b u_b v
//   symmetry mode: k <= q, and a <= b when k == q; pair evaluated iff f_a != 0 or f_b != 0;
//                  acc_a -= w_q f_b u_b v   and (unless a == b)   acc_b -= w_k f_a u_a conj(v)
// using v_{bq,ak} = conj(v_{ak,bq}) (K real and K_{q-k}(g) = K_{k-q}(-g); exact on an alias-free grid).
int fused_apply(exx_ctx* c, const double* occ, const double2* psi, double2* out, const double2* phi, int nphi) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return EXX_ERR_BAD_ARG;
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    c->path_used = 2;
    c->pruned_used = 0;
    if (!(c->opt_keep_u && c->u_valid)) {  // EXX_OPT_KEEP_U: psi unchanged since the previous call, its real-space boxes still stand
        if ((rc = fused_u_cache(c, st, psi))) return rc;
        c->u_valid = true;
    }
    if (phi) {  // exx_apply_to: the a-bands of every pair are the trial vectors
        if (st->uphi_boxes < (size_t)nk * nphi) {  // grown on demand; accumulators of the trial vectors sit behind their boxes
            cudaFree(st->uphi_dev);
            st->uphi_dev = nullptr;
            c->dev_bytes -= 2 * sizeof(cplx) * Ng * st->uphi_boxes;
            st->uphi_boxes = 0;
            if (cudaMalloc((void**)&st->uphi_dev, 2 * sizeof(cplx) * Ng * (size_t)nk * nphi) != cudaSuccess) {
                cudaGetLastError();
                return EXX_ERR_ALLOC;
            }
            st->uphi_boxes = (size_t)nk * nphi;
            c->dev_bytes += 2 * sizeof(cplx) * Ng * st->uphi_boxes;
        }
        if ((rc = fused_u_cache(c, st, phi, st->uphi_dev, nphi, nphi))) return rc;
    }
    const int na = phi ? nphi : nb;  // a-bands per k-point
    int ta_max, tb_max;
    bool sym;
    fused_batch_shape(c, &ta_max, &tb_max, &sym);
    if (phi) sym = false, c->symmetry_used = 0;  // v_{b,a} = conj(v_{a,b}) pairs two bands of ONE set; here a and b come from different sets
    if ((rc = fused_ensure_part(c, st, sym, ta_max, tb_max))) return rc;
    cplx* work = (cplx*)c->work_dev;
    // one accumulator box per (k, band), always fp64; exx_apply_to: per (k, trial vector), behind the trial vectors' boxes
    acc_c* acc = phi ? (acc_c*)(st->uphi_dev + Ng * st->uphi_boxes) : (acc_c*)c->acc_dev;
    EXX_CUDA(c, cudaMemsetAsync(acc, 0, sizeof(acc_c) * Ng * (size_t)nk * na, c->stream));
    c->precision_used = 0;
    if (c->opt_precision == 1 && !phi) {
        // mixed precision (the paper's second mode): pair transforms, kernel multiply and the product with u in fp32;
        // S1, S7 and every accumulator stay fp64
        if ((rc = fused_mode32_ready(c, st))) return rc;
        if ((rc = pair_loop<ModeF>(c, st, occ, st->u32_dev, (exx32::cplx*)c->work_dev, st->kperm32_dev, acc, sym, ta_max, tb_max))) return rc;
        c->precision_used = 1;
    } else {
        if ((rc = pair_loop<ModeD>(c, st, occ, (const cplx*)c->u_dev, work, st->kperm_dev, acc, sym, ta_max, tb_max, phi ? st->uphi_dev : nullptr, na))) return rc;
    }
    // S7: forward transform of every accumulator through passes A/B (-> F layout), gather onto sphere(k)
    for (int k = 0; k < nk; k++) {
        const int bmax = (int)std::min<size_t>(c->work_boxes, (size_t)na);
        const int64_t offk = c->off[k] / nb * na;
        for (int n0 = 0; n0 < na; n0 += bmax) {
            const int bn = std::min(bmax, na - n0);
            if (c->opt_prune_rows) {  // the gather reads sphere points only: rows with |kx| > gmax are not written back
                RowMask rows;
                EXX_DISPATCH_R1(st->R1, rows = L::sphere_rows(c->gmax[0]));
                EXX_DISPATCH_R1(st->R1, rc = L::fft_forward(c, (const cplx*)(acc + ((size_t)k * na + n0) * Ng), bn, work, rows));
            } else {
                EXX_DISPATCH_R1(st->R1, rc = L::fft_forward(c, (const cplx*)(acc + ((size_t)k * na + n0) * Ng), bn, work));
            }
            if (rc) return rc;
            if ((rc = launch_gather(c, k, (const double2*)work, bn, out + offk + (int64_t)n0 * c->npw[k], st->fmap_dev + c->map_off[k]))) return rc;
        }
    }
    return EXX_OK;
}

// ---- energy route (E2) ------------------------------------------------------------------------------------------------------
// E_x = -1/2 sum_{k,q} w_k w_q sum_{a,b} f_a f_b sum_g K'_{k-q}(g) |rho^_{ak,bq}(g)|^2   ((E2); equal to (E1)
// on any grid because K' is real: Parseval).  Only pairs with f_a != 0 and f_b != 0 count, no inverse transform and no pass C:
// passes A and the forward half of B per pair, then fixed-order sums.  With the pair symmetry an unordered pair is transformed
// once and credited to both bands (|rho^_{bq,ak}(g)|^2 K'_{q-k}(g) summed over g is the same number).
template <class M>
static int pair_energy_loop(exx_ctx* c, FusedState* st, const double* occ, const typename M::cplx* u_base, typename M::cplx* work,
                            const typename M::real* kperm_base, bool sym, int ta_max, int tb_max) {
    int rc;
    const int nb = c->nb, nk = c->nk;
    const size_t Ng = (size_t)c->Ng;
    std::vector<PairBlock> blocks;
    plan_blocks(nk, nb, occ, sym, ta_max, tb_max, (int)c->opt_shard_count, blocks);
    std::vector<int> blist;
    int bl_q = -1;
    for (const PairBlock& blk : blocks) {
        if (blk.shard != (int)c->opt_shard_rank) continue;
        const int k = blk.k, q = blk.q;
        const typename M::real* kperm = kperm_base + (size_t)c->ktab_of[(size_t)k * nk + q] * Ng;
        const typename M::cplx* ua = u_base + (size_t)k * nb * Ng;
        const typename M::cplx* ub = u_base + (size_t)q * nb * Ng;
        if (bl_q != q) b_list(nb, occ, q, sym, blist), bl_q = q;
        const int a0 = blk.a0, ta = blk.ta, tb = blk.tb;
        const size_t b0 = (size_t)blk.b0;
        AJob aj;
        EJob ej;
        aj.npairs = 0;
        aj.tb = tb;
        ej.tgt_a = k * nb, ej.tgt_b = q * nb, ej.sym = sym ? 1 : 0, ej.same_k = k == q ? 1 : 0;
        for (int i = 0; i < TMAX; i++) ej.wa[i] = ej.wb[i] = 0.0;
        for (int i = 0; i < ta; i++) aj.a_idx[i] = a0 + i, ej.wa[i] = c->kw[k] * occ[k * nb + a0 + i];
        for (int j = 0; j < tb; j++) aj.b_idx[j] = blist[b0 + j], ej.wb[j] = c->kw[q] * occ[q * nb + blist[b0 + j]];
        int64_t ordered = 0;
        for (int i = 0; i < ta; i++)
            for (int j = 0; j < tb; j++) {
                const double fa = occ[k * nb + aj.a_idx[i]], fb = occ[q * nb + aj.b_idx[j]];
                if (fa == 0.0 || fb == 0.0 || !pair_evaluated(sym, k, q, aj.a_idx[i], aj.b_idx[j], fa, fb)) continue;
                aj.pi[aj.npairs] = (unsigned char)i;
                aj.pj[aj.npairs] = (unsigned char)j;
                aj.npairs++;
                ordered += (sym && !(k == q && aj.a_idx[i] == aj.b_idx[j])) ? 2 : 1;
            }
        if (aj.npairs == 0) continue;
        EXX_DISPATCH_M(st->R1, rc = L::pass_a_energy(c, ua, ub, aj, ej, kperm, work, st->epart_dev, st->pairsum_dev, st->band_e2_dev));
        if (rc) return rc;
        c->pairs_executed += aj.npairs;
        c->pairs_ordered += ordered;
    }
    return EXX_OK;
}

// band_e2_host[k nb + n] = w_k f_nk sum_{q,m} w_q f_mq sum_g K' |rho^|^2  (this shard's batches); the caller applies the -1/2.
// Synchronises the stream.
int fused_energy(exx_ctx* c, const double* occ, const double2* psi, double* band_e2_host) {
    FusedState* st = (FusedState*)c->fused;
    if (!st) return EXX_ERR_BAD_ARG;
    int rc;
    const int nb = c->nb, nk = c->nk;
    c->path_used = 2;
    c->pruned_used = 0;
    if (!(c->opt_keep_u && c->u_valid)) {  // EXX_OPT_KEEP_U: psi unchanged since the previous call, its real-space boxes still stand
        if ((rc = fused_u_cache(c, st, psi))) return rc;
        c->u_valid = true;
    }
    int ta_max, tb_max;
    bool sym;
    fused_batch_shape(c, &ta_max, &tb_max, &sym);
    EXX_CUDA(c, cudaMemsetAsync(st->band_e2_dev, 0, sizeof(double) * (size_t)nk * nb, c->stream));
    c->precision_used = 0;
    if (c->opt_precision == 1) {
        if ((rc = fused_mode32_ready(c, st))) return rc;
        if ((rc = pair_energy_loop<ModeF>(c, st, occ, st->u32_dev, (exx32::cplx*)c->work_dev, st->kperm32_dev, sym, ta_max, tb_max))) return rc;
        c->precision_used = 1;
    } else {
        if ((rc = pair_energy_loop<ModeD>(c, st, occ, (const cplx*)c->u_dev, (cplx*)c->work_dev, st->kperm_dev, sym, ta_max, tb_max))) return rc;
    }
    EXX_CUDA(c, cudaMemcpyAsync(band_e2_host, st->band_e2_dev, sizeof(double) * (size_t)nk * nb, cudaMemcpyDeviceToHost, c->stream));
    EXX_CUDA(c, cudaStreamSynchronize(c->stream));
    return EXX_OK;
}

}  // namespace exx
