// exx_internal.h — context layout and launch helpers shared by the translation units of libexx.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/exx.h"

namespace exx {

// kernel classes for launch counting / event timing (EXX_INFO_NUM_KERNEL_CLASSES entries)
enum KClass {
    KC_SCATTER = 0,
    KC_GATHER = 1,
    KC_FFT_AXIS = 2,     // generic per-axis FFT
    KC_CODENSITY = 3,    // generic rho = conj(u_m) u_n
    KC_KMUL = 4,         // generic v^ = K' rho^
    KC_ACCUM = 5,        // generic acc -= w f u_m v
    KC_ENERGY = 6,
    KC_PASS_A = 7,       // fused: co-density + forward (y,z)-plane transform
    KC_PASS_B = 8,       // fused: forward x, K', inverse x
    KC_PASS_C = 9,       // fused: inverse (y,z)-plane transform, times f_m u_m, accumulate
    KC_SUBSPACE = 10,    // subspace ZGEMM (DMMA) + its slice reduction
    KC_FFT_FUSED = 11,   // plain 3-D transforms (S1, S7) through the fused passes; unit = one box pass
    KC_PASS_R = 12,      // fused, pair symmetry: partial boxes of the dual sweep's second side added to the accumulators
    KC_COUNT = 13
};

struct Plan1D {
    int n = 0;
    int nst = 0;
    int radix[16] = {0};
    double2* tw_dev = nullptr;  // n entries exp(-2 pi i j / n)
};

struct EventRec {
    cudaEvent_t a, b;
    int kclass;
};

}  // namespace exx

struct exx_ctx {
    int N[3];
    int64_t Ng;
    double A[9], B[9], omega;
    int nk, nb;
    std::vector<double> kfrac, kw;
    double ecut;
    exx_kernel_params kp;
    int gmax[3];                      // max |g_i| over all spheres
    bool alias_free;                  // 4*gmax_i + 1 <= N_i for all i

    std::vector<int> npw;
    std::vector<int64_t> off;         // nk+1, complex elements
    std::vector<std::vector<int32_t>> map_h;
    std::vector<int64_t> map_off;     // nk+1 offsets into map_dev
    int32_t* map_dev = nullptr;

    std::vector<int> ktab_of;         // nk*nk -> table index
    int ntab = 0;
    std::vector<std::vector<double>> ktab_dk;  // per table the delta-kappa triple
    double* ktab_dev = nullptr;       // ntab * Ng, K'(g) = K/(Omega Ng^2), C order

    exx::Plan1D plan[3];

    cudaStream_t stream = nullptr;
    double2* u_dev = nullptr;         // nk*nb boxes, u_nk(r)
    double2* work_dev = nullptr;      // pair workspace
    double2* acc_dev = nullptr;       // accumulators of one n-tile
    size_t work_boxes = 0, acc_boxes = 0;
    double2* vx_dev = nullptr;        // internal V_x psi buffer (exx_energy with NULL, exx_apply_host)
    double2* psi_stage_dev = nullptr; // exx_apply_host staging
    double2* uphi1_dev = nullptr;     // exx_apply_to on the generic path: one box, the current trial vector in real space
    double* band_dot_dev = nullptr;   // nk*nb Re<c|Vc>
    double* band_e_dev = nullptr;     // nk*nb + 1: per-band energies, then total
    double* occw_dev = nullptr;       // nk*nb: 1/2 w_k f_nk
    int64_t* band_off_dev = nullptr;  // nk*nb: offset of band (k,n) in psi (complex elements)
    int* band_len_dev = nullptr;      // nk*nb: npw(k)
    double* host_pinned = nullptr;    // nk*nb + 1 doubles, pinned
    void* subspace_dev = nullptr;     // split-K partials of exx_subspace (grown on demand)
    size_t subspace_bytes = 0;
    size_t dev_bytes = 0;

    // fused path state (exx_fused.cu)
    void* fused = nullptr;

    // compact work grid (EXX_OPT_PRUNE): a second context of the same problem on the smallest supported cubic grid that still
    // holds every product the method forms without wrap-around (N >= 4 gmax + 1); owned by this context.  big_alloc: the
    // real-space cache, pair workspace, accumulators and fused tables of THIS grid exist (allocated in exx_create when there is
    // no inner context, else on the first apply with pruning switched off).
    bool fft_ready = false;           // twiddles/attributes of the fused kernels set up for exx_fft3d_fused
    exx_ctx* inner = nullptr;
    bool inner_larger = false;        // the inner grid has MORE points than this one (taken for its fused kernels only)
    bool big_alloc = false;
    int last_pruned = 0;

    // options
    int64_t opt_path = 0, opt_tile_n = 0, opt_tile_m = 0, opt_prune = 1, opt_profile = 0, opt_symmetry = 1, opt_precision = 0;
    int64_t opt_keep_u = 0;        // 1: the caller promises psi is unchanged since the previous call: S1 of psi is skipped (fused path)
    bool u_valid = false;          // the u cache holds S1 of the psi of the previous call (fused path)
    int64_t opt_energy_route = 0;  // 0 auto (pair-density route E2 where the fused path runs), 1 always E1 from V_x psi
    int64_t energy_route_used = 0;
    int64_t opt_prune_rows = 1;    // S1/S7 on the fused path: 1 = skip the F-layout x rows outside the spheres (see RowMask)
    int64_t opt_dual = 1;          // pair symmetry: 1 = one dual sweep of pass C per batch (default), 0 = two single sweeps
    int64_t opt_shard_count = 1, opt_shard_rank = 0;  // S8(f)-4: this context runs shard rank of count (exx_shard.h)

    // counters of the last apply
    int64_t symmetry_used = 0, precision_used = 0;
    int64_t launches = 0, pairs_ordered = 0, pairs_executed = 0, path_used = 0, tile_n_used = 0, tile_m_used = 0, pruned_used = 0;
    int64_t launches_by_class[exx::KC_COUNT] = {0};
    int64_t units_by_class[exx::KC_COUNT] = {0};   // box passes (generic) or pairs (fused) processed
    std::vector<exx::EventRec> events;
    std::vector<cudaEvent_t> event_pool;
    size_t event_pool_used = 0;

    std::string last_error;
};

namespace exx {

void set_thread_error(const std::string& s);
// Test hook for the out-of-memory branches, which a 180 GB device never takes by itself: while the environment variable
// EXX_TEST_FAIL_ALLOC names `tag`, the device allocation carrying that tag reports failure without calling cudaMalloc.
// Tags: "part" (partial boxes of the dual sweep), "acc" (accumulator boxes in ensure_big).  One getenv per tagged allocation.
bool test_fail_alloc(const char* tag);
int cuda_fail(exx_ctx* c, cudaError_t e, const char* what);

#define EXX_CUDA(c, call)                                         \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return exx::cuda_fail((c), e__, #call); \
    } while (0)

// launch bookkeeping: count, optionally bracket with events
struct LaunchScope {
    exx_ctx* c;
    int kclass;
    cudaEvent_t a = nullptr, b = nullptr;
    LaunchScope(exx_ctx* c_, int k, int64_t units = 0);
    ~LaunchScope();
};

// ---- generic kernels (exx_kernels.cu) ----
struct MTile {
    int tm;
    int m_idx[32];     // band indices within k-point q
    double wf[32];     // w_q * f_mq
};
// one batch of band pairs for the fused passes: a-bands (k-point ka) x b-bands (k-point kb), at most TMAX x TMAX.
// Pair p = (pi[p], pj[p]) evaluates v = IFFT K' FFT[conj(u_b) u_a]; its work box is pi*tb + pj.
constexpr int TMAX = 32;  // most bands per side of a batch
#ifndef EXX_DEFAULT_TILE
#define EXX_DEFAULT_TILE 32  // bands per side of a batch unless EXX_OPT_TILE_N/M say otherwise (32 vs 16: C4a -3 %, C2 -11 %)
#endif
#ifndef EXX_SHARD_TILE
#define EXX_SHARD_TILE 16    // ... when the batches are shared out over shards (more, smaller batches balance better)
#endif
#ifndef EXX_WORK_CAP_GIB
#define EXX_WORK_CAP_GIB 16  // the pair workspace (tile_n x tile_m boxes) is kept below this
#endif
struct AJob {
    int npairs, tb;
    int a_idx[TMAX], b_idx[TMAX];      // band indices within their k-points
    unsigned char pi[TMAX * TMAX], pj[TMAX * TMAX];
};
// one accumulation sweep of pass C: CTA row r owns accumulator box tgt[r] and loops over its cnt[r] columns:
//   acc[tgt[r]] -= coef[c] * u[src[c]] * (cj ? conj(v) : v),   v in work box r*box_r + c*box_c
struct CJob {
    int nr, box_r, box_c, cj;
    int tgt[TMAX], cnt[TMAX], src[TMAX];
    double coef[TMAX];
    unsigned char col[TMAX][TMAX];
};
// the dual sweep of pass C (pair symmetry): CTA (tile, row group) walks the columns; row i (a-band) x column j
// (b-band), work box i*tb + j.  ev[i] bit j: the pair was transformed; side a (acc_a -= coef_b[j] u_b v) runs where amask has bit
// j (f_b != 0); side b (acc_b -= coef_a[i] u_a conj v) where bside[i] has bit j (f_a != 0 and not the diagonal pair).
struct DJob {
    int ta, tb, nrg;
    int a_tgt[TMAX];            // accumulator box of row i
    int a_src[TMAX], b_src[TMAX];  // u boxes of row i / column j (within ua_base / ub_base)
    double coef_a[TMAX], coef_b[TMAX];
    unsigned ev[TMAX], bside[TMAX];
    unsigned amask;
};
// pass R: acc[tgt[j]] += sum over the row groups g with bit g of gmask[j] of partial box g*tb + j, in group order
struct RJob {
    int ncol, tb, nrg;
    int tgt[TMAX];
    unsigned gmask[TMAX];
};
// F-layout x rows (bit xpos) of a box that a pruned plain transform reads (inverse, S1) or writes (forward, S7)
struct RowMask {
    uint32_t w[4];
};
// weights of one batch on the energy route: band (a,k) gets  wa[i] * sum_j wb[j] S_ij,  band (b,q) (pair symmetry) the mirror image
struct EJob {
    double wa[TMAX], wb[TMAX];   // w_k f_a, w_q f_b
    int tgt_a, tgt_b;            // k*nb, q*nb: first entry of the k-point's bands in the per-band energy array
    int sym, same_k;             // pair symmetry on; k == q (then the pair a == b is counted once)
};
int fft_generic_init(exx_ctx* c);
int launch_scatter(exx_ctx* c, int ik, const double2* coef, int nbatch, double2* box, const int32_t* map = nullptr, bool clear = true);  // map: override (F layout); clear: zero the boxes first
int launch_gather(exx_ctx* c, int ik, const double2* box, int nbatch, double2* coef, const int32_t* map = nullptr);
int launch_fft3d_generic(exx_ctx* c, double2* box, int nbatch, int sign);
int launch_codensity_tile(exx_ctx* c, const double2* un_base, int n0, int tn, const double2* uq_base, const MTile& mt, double2* work);
int launch_kmul(exx_ctx* c, const double* ktab, double2* work, int nboxes);
int launch_accumulate_tile(exx_ctx* c, const double2* uq_base, const MTile& mt, int tn, const double2* work, double2* acc);
int launch_energy(exx_ctx* c, const double2* psi, const double2* vx);
int launch_subspace(exx_ctx* c, int ik, const double2* psi, const double2* vx, double2* M, int nvec = -1);  // exx_subspace.cu
int compute_u_cache(exx_ctx* c, const double2* psi);  // exx_api.cu: S1 for every band

// ---- fused path (exx_fused.cu) ----
bool fused_supported(const exx_ctx* c);
void fused_tiles(const exx_ctx* c, int* tn, int* tm);
int fused_create(exx_ctx* c);
void fused_destroy(exx_ctx* c);
int fused_apply(exx_ctx* c, const double* occ, const double2* psi, double2* out, const double2* phi = nullptr, int nphi = 0);  // phi, nphi: exx_apply_to
int fused_energy(exx_ctx* c, const double* occ, const double2* psi, double* band_e2_host);  // E2 route: per-band sums w f w f K'|rho^|^2
int fused_fft3d(exx_ctx* c, double2* in, int nbatch, int sign, double2* out);
int fused_findex(const exx_ctx* c, int32_t* host_out);

}  // namespace exx
