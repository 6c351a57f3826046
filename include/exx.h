/*
 * exx.h — C ABI of libexx: plane-wave Fock-exchange operator V_x|psi_nk> and exchange energy E_x on one B200.
 *
 * The operation (PAPER.md = arXiv 1111.0716; P:Lnn is line nn of it):
 *   - FOCK_ACC "applies the Fock exchange operator"; the exchange energy is Eq. 2;
 *   - four nested loops, two over k-points k,q and two over bands n,m; the band loops run on the GPU and every
 *     operation inside them stays on the device;
 *   - FFTs, scatter/gather "used to express cutoffs", data-manipulation kernels;
 *   - library contexts created/destroyed at the start/end of the program.
 * On the FFT grid this is definition (D) of DESIGN.md section 2 (Hartree atomic units, no spin factor):
 *   u_nk(r_j)       = sum_{g in sphere(k)} c_nk(g) e^{+i G.r_j}
 *   rho~_{nk,mq}(g) = (1/Ng) sum_j conj(u_mq(r_j)) u_nk(r_j) e^{-i G.r_j}
 *   v_{nk,mq}(r_j)  = (1/Omega) sum_g K(|k-q+G|) rho~_{nk,mq}(g) e^{+i G.r_j}
 *   (V_x u)_nk(r_j) = - sum_q w_q sum_m f_mq u_mq(r_j) v_{nk,mq}(r_j)
 *   (V_x c)_nk(g)   = (1/Ng) sum_j (V_x u)_nk(r_j) e^{-i G.r_j},  g in sphere(k) = { g : |k+G|^2/2 < E_cut }
 *   E_x             = 1/2 sum_k w_k sum_n f_nk Re <c_nk | (V_x c)_nk>
 *
 * Conventions
 *   - complex numbers: interleaved (re, im) fp64.  All arithmetic is fp64.
 *   - FFT box: C order, index (j1*N2 + j2)*N3 + j3; integer frequency g_i = j_i if 2 j_i < N_i else j_i - N_i.
 *   - sphere(k) is listed by ascending box index; exx_index_map returns that list (bit-exact contract).
 *   - psi / out layout: k-major, then band, then sphere index: element (k,n,ig) at
 *       exx_psi_offset(k) + n*npw(k) + ig   (complex elements),  exx_psi_offset(k) = nbands * sum_{k'<k} npw(k').
 *   - pointers named *_dev are device (HBM) pointers, *_host are host pointers; both are owned by the caller.
 *     The context owns its index maps, kernel tables, the real-space cache u_nk(r) and all workspaces; they are
 *     allocated in exx_create and freed in exx_destroy, and the calls allocate nothing — with these exceptions, each made on
 *     first use, kept until exx_destroy and counted in EXX_INFO_WORKSPACE_BYTES:
 *       - exx_apply / exx_energy: the first call that runs the dual sweep (pair symmetry, EXX_OPT_DUAL_SWEEP = 1, a grid with a
 *         dual kernel) makes its partial boxes (at most tile_n/RG x tile_m boxes; if the device refuses, two sweeps run instead);
 *         the first call after EXX_OPT_PRUNE was switched off on a context with a compact work grid makes the full-grid buffers;
 *         the first call with EXX_OPT_PRECISION = 1 makes the fp32 copies of u_nk(r) and of the kernel tables;
 *       - exx_apply_to: boxes and accumulators of the trial vectors (again when nphi grows);
 *       - exx_subspace / exx_subspace_block: the split-K partial matrices (again when they grow);
 *       - exx_apply_host: one device copy of psi.
 *     exx_subspace_static never allocates.
 *   - every call returns EXX_OK (0) or a negative error code; no exceptions, no abort, nothing printed.
 *     On error, output arguments are left untouched.  exx_last_error() gives detail for EXX_ERR_CUDA.
 *   - work is enqueued on the CUDA stream given to exx_create (a cudaStream_t cast to void*; NULL = default
 *     stream).  exx_apply returns without synchronising; exx_energy and the *_host calls synchronise that stream.
 */
#ifndef EXX_H
#define EXX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct exx_ctx exx_ctx; /* opaque */

typedef struct {
    int kind;     /* 0: bare Coulomb 4 pi/Q^2, term at k-q+G = 0 set to 0;
                     1: HSE short range (4 pi/Q^2)(1 - exp(-Q^2/(4 mu^2))), term at k-q+G = 0 is pi/mu^2 */
    double mu;    /* bohr^-1, used when kind == 1 (HSE06: 0.106) */
    double scale; /* multiplies K (1.0 in all BASELINE configs; HSE06's 1/4 mixing is NOT applied implicitly) */
} exx_kernel_params;

enum {
    EXX_OK = 0,
    EXX_ERR_NULL = -1,        /* a required pointer is NULL */
    EXX_ERR_BAD_GRID = -2,    /* N_i not of the form 2^a 3^b 5^c (>= 2), N_i > 1024, or the cutoff sphere does not fit the box */
    EXX_ERR_BAD_LATTICE = -3, /* zero or non-finite cell volume */
    EXX_ERR_BAD_CUTOFF = -4,  /* E_cut <= 0 or non-finite, or an empty sphere */
    EXX_ERR_BAD_KERNEL = -5,  /* unknown kind, mu <= 0 for HSE, non-finite scale */
    EXX_ERR_BAD_OCC = -6,     /* an occupation is negative or non-finite */
    EXX_ERR_ALLOC = -7,       /* host or device allocation failed */
    EXX_ERR_CUDA = -8,        /* a CUDA call or kernel launch failed; see exx_last_error */
    EXX_ERR_BAD_ARG = -9,     /* index out of range, nk/nbands < 1, weights not finite, unknown option */
    EXX_ERR_ALIAS = -10,      /* out aliases psi */
    EXX_ERR_LIMIT = -11       /* a size is beyond the fixed capacity of an entry point that allocates nothing (exx_subspace_static);
                                 exx_last_error(NULL) names the limit */
};

/* Options (exx_set_option / exx_get_option).  All but EXX_OPT_PRECISION are tuning knobs: results differ only by rounding
 * order (<= 1e-13 relative, tested).  EXX_OPT_PRECISION = 1 changes the arithmetic (see below). */
enum {
    EXX_OPT_PATH = 1,       /* 0 auto (fused kernels when the grid is supported, else generic), 1 generic per-axis kernels, 2 fused */
    EXX_OPT_TILE_N = 2,     /* bands per row tile of a pair batch (0 = auto: 32, or 16 when sharded; at most 32; shrunk to fit the workspace) */
    EXX_OPT_TILE_M = 3,     /* bands per column tile of a pair batch (0 = auto, as above; at most 32) */
    EXX_OPT_PRUNE = 4,      /* 1 (default): run the pair pipeline on the compact work grid when there is one (see EXX_INFO_COMPACT_GRID);
                               0: always transform the caller's full grid */
    EXX_OPT_PROFILE = 5,    /* 1: bracket every kernel launch with CUDA events so exx_get_kernel_time works (slower) */
    EXX_OPT_PRECISION = 8,  /* 0 (default): fp64 throughout.  1: mixed precision, the paper's second mode ("some or all of the
                               FFTs in single precision"): the pair transforms, the kernel multiply and the product with u_m run in fp32
                               (fused path only); S1, S7, every accumulator and E_x stay fp64.  Agrees with fp64 to ~1e-6 relative
                               (the paper reports 1e-5); NOT covered by the 1e-10 / 1e-11 parity bars */
    EXX_OPT_SYMMETRY = 6,   /* 1 (default): evaluate each unordered band pair once and use v_{mq,nk} = conj(v_{nk,mq}) for the second
                               accumulation (fused path on alias-free grids only; see EXX_INFO_SYMMETRY); 0: every ordered pair */
    EXX_OPT_SHARD_COUNT = 9,  /* P >= 1 (default 1): this context is shard EXX_OPT_SHARD_RANK of P (one process per GPU, SURVEY.md
                               S8(f)-4; the paper's multi-device runs are MPI over processes, Table V).  exx_apply then
                               runs only this shard's share of the pair work and `out` holds a PARTIAL V_x psi: the sum of `out` over
                               the P shards is the full result (the caller adds them, e.g. one all-reduce; the binding's
                               apply_sharded does).  Fused path: the pair batches of exx_shard_plan; generic path: output rows
                               (k,n) with (k nbands + n) mod P = rank, the other rows of `out` zero */
    EXX_OPT_SHARD_RANK = 10, /* 0 .. P-1 (default 0); exx_apply returns EXX_ERR_BAD_ARG while rank >= P */
    EXX_OPT_KEEP_U = 12,    /* 1: the caller promises that psi is the same as in the previous exx_apply / exx_apply_to / exx_energy call on this
                               context (same work grid): the real-space images u_nk(r) kept from that call are used and S1 of psi is
                               skipped (fused path; the generic kernels ignore it).  For an eigensolver that calls exx_apply_to on many
                               blocks of trial vectors between two updates of the orbitals.  0 (default): S1 of psi in every call.
                               Set it back to 0 for the first call after psi changes */
    EXX_OPT_DUAL_SWEEP = 13, /* pair symmetry only.  1 (default): the last pass transforms every pair box back ONCE and feeds both
                               accumulations (acc_a -= w_q f_b u_b v on chip, acc_b -= w_k f_a u_a conj(v) through one partial box per
                               (row group, column) that a small reduction kernel adds in a fixed order); 0: two sweeps of the last
                               pass, the second repeating the inverse y/z steps (grids without a dual kernel always do this).
                               Results differ by rounding order only (fp64 mode); both are deterministic.  With EXX_OPT_PRECISION = 1
                               the dual sweep adds the second side's products of one row group (at most 4 rows) in fp32 before they
                               reach the fp64 accumulators, where two sweeps add each product in fp64: there the two differ at fp32
                               rounding level, inside that mode's 1e-5 bar.  The partial boxes are allocated by the first apply
                               that uses them; if the device refuses them, two sweeps run */
    EXX_OPT_PRUNE_SPHERE = 14, /* fused path, S1 and S7 ("the sphere is ~2 % of the box").  1 (default): the inverse
                               transform of the bands reads, and the forward transform of the accumulators writes, only the
                               x rows of the frequency box with |g_x| <= max |g_x| of the spheres (46 % of the rows at C4a); the
                               scatter clears only those.  0: whole boxes.  Bit-identical results */
    EXX_OPT_ENERGY_ROUTE = 11 /* what exx_energy does when it is given no V_x psi.  0 (default): the pair-density route
                               E_x = -1/2 sum w_k w_q f_nk f_mq sum_g K'_{k-q}(g) |rho^_{nk,mq}(g)|^2 (form (E2) of DESIGN.md section 2:
                               Eq. 2 of PAPER.md, L127-130, written in reciprocal space) wherever the fused kernels run: the co-density
                               and the forward transform only, pairs of two occupied bands only, no inverse transform and no
                               accumulation (2.7x less work than V_x psi at C4a); otherwise, and with 1, V_x psi into an
                               internal buffer and then (E1).  Both give the same number up to rounding (K' is real: Parseval) */
};

/* Counters (exx_get_info), all for the most recent exx_apply on this context unless stated. */
enum {
    EXX_INFO_LAUNCHES = 1,        /* kernels launched */
    EXX_INFO_PAIRS_ORDERED = 2,   /* ordered band-pair exchange evaluations covered: sum over (k,q) of Nb * Nocc(q) */
    EXX_INFO_PAIRS_EXECUTED = 3,  /* pair FFT round trips actually executed (== ordered unless a symmetry is exploited) */
    EXX_INFO_PATH_USED = 4,       /* 1 generic, 2 fused */
    EXX_INFO_WORKSPACE_BYTES = 5, /* device bytes owned by the context */
    EXX_INFO_NCOEF = 6,           /* complex elements in psi / out */
    EXX_INFO_TILE_N = 7,
    EXX_INFO_TILE_M = 8,
    EXX_INFO_PRUNED = 9,          /* 1 if the last apply ran on the compact work grid */
    EXX_INFO_NUM_KERNEL_CLASSES = 10,  /* how many kernel classes exx_get_kernel_time knows (the value, not this enum) */
    EXX_INFO_WORK_GRID = 11,      /* N of the (cubic) grid the last apply transformed; first axis of the caller's grid if not compacted */
    EXX_INFO_SYMMETRY = 13,       /* 1 if the last apply used the pair symmetry (then PAIRS_EXECUTED < PAIRS_ORDERED) */
    EXX_INFO_PRECISION = 15,      /* 0 fp64, 1 mixed: what the last apply ran in */
    EXX_INFO_ENERGY_ROUTE = 16,   /* most recent exx_energy: 1 = (E1) from V_x psi, 2 = pair-density route (E2); 0 before any */
    EXX_INFO_COMPACT_GRID = 12    /* (no apply needed) N of the compact work grid, 0 if none: the smallest supported cubic grid with
                                     N >= 4 max|g_i| + 1, used when the caller's box is itself alias-free (N_i >= 4 max|g_i| + 1) and the
                                     cubic grid has fewer points — or, if the caller's grid has no fused kernels (non-cubic, or a cubic
                                     size outside the fused list), at most 4x as many.  No product the method forms wraps around on
                                     either grid, so V_x psi on the sphere is the same up to rounding */
};

/* Create a context.  grid: N1,N2,N3.  lattice: 9 doubles, row i = a_i in bohr.  kfrac: nk*3 fractional reciprocal
 * coordinates kappa (k = sum kappa_i b_i, a_i.b_j = 2 pi delta_ij).  kweight: nk weights w_k (the caller makes them
 * sum to 1).  All host pointers, read during the call only.  Builds index maps, the kernel tables
 * K'_{k-q}(g) = K(|k-q+G|)/(Omega Ng^2) for every distinct k-q, twiddle tables and workspaces (host work + H2D). */
int exx_create(exx_ctx** out, const int grid[3], const double lattice[9], int nk, const double* kfrac_host,
               const double* kweight_host, double ecut_hartree, const exx_kernel_params* kp, int nbands, void* cuda_stream);
int exx_destroy(exx_ctx* ctx);

/* Queries (host). */
int exx_npw(const exx_ctx* ctx, int ik, int* npw);
int exx_index_map(const exx_ctx* ctx, int ik, int32_t* host_out /* npw(ik) entries */);
int exx_psi_offset(const exx_ctx* ctx, int ik /* 0..nk; nk gives the total */, int64_t* complex_elems);
int exx_set_option(exx_ctx* ctx, int option, int64_t value);
int exx_get_option(const exx_ctx* ctx, int option, int64_t* value);
int exx_get_info(const exx_ctx* ctx, int what, int64_t* value);
/* Per kernel class `kclass` (0 .. EXX_INFO_NUM_KERNEL_CLASSES-1), for the most recent exx_apply: launch count, work
 * units (generic kernels and fused_fft_pass: box passes, i.e. one read + one write of an FFT box; fused passes A/B: band pairs;
 * fused pass C: accumulation sweeps, one per pair and side — or, for the dual sweep of EXX_OPT_DUAL_SWEEP, pair boxes, each serving
 * both sides; fused pass R: partial boxes added to the accumulators), and — with
 * EXX_OPT_PROFILE = 1 — the device time from CUDA events on the context's stream (0 otherwise).  Synchronises.
 * exx_kernel_class_name gives the class name (static string, NULL if out of range). */
int exx_get_kernel_time(exx_ctx* ctx, int kclass, double* ms_total, int64_t* launches, int64_t* units);
const char* exx_kernel_class_name(int kclass);

/* Host only, no context and no GPU needed: how the fused path's pair batches are shared out among `nshards` shards.  The
 * loop nest over (k, q, a-tile, b-tile) gives one batch per tile x tile block of band pairs
 * (tile = 0: the default, 32 for one shard and 16 for several; at most 32); batches are handed out longest first to the least loaded shard — deterministic, so every rank
 * computes the same plan.  occ_host: nk*nbands.  symmetry: as EXX_OPT_SYMMETRY (the caller says whether it applies).
 * Outputs (each nshards entries, either may be NULL): pairs_out = pair densities the shard transforms (passes A, B);
 * passes_out = fused pass executions (2 per pair + 1 per accumulation sweep), the load that is balanced.
 * The plan describes what a context runs only when `tile` is the tile that context uses: a context may shrink its tile below the
 * default (pair workspace cap on grids of 128^3 and more, EXX_OPT_TILE_N/M), so pass the value EXX_INFO_TILE_N reports after an
 * apply when the counts must match a particular context (totals over all shards do not depend on the tile). */
int exx_shard_plan(int nk, int nbands, const double* occ_host, int symmetry, int tile, int nshards, int64_t* pairs_out, int64_t* passes_out);

/* V_x applied to every band: out(k,n,:) = (V_x c)_nk.  psi_dev/out_dev: device, exx_psi_offset(nk) complex elements
 * each, 16-byte aligned, must not overlap.  occ_host: nk*nbands occupations f_nk in [0, inf), host, read during the
 * call.  Bands with f = 0 are skipped as m (they contribute exactly 0) and kept as n.  Asynchronous on the stream. */
int exx_apply(exx_ctx* ctx, const double* psi_dev, const double* occ_host, double* out_dev);

/* The same operator applied to OTHER vectors: out(k,i,:) = (V_x[psi, occ] phi_ki)(g), g in sphere(k), i.e. definition (D) above with
 * u_nk replaced, in the co-density only, by the real-space image of phi_ki.  This is FOCK_ACC inside an iterative eigensolver
 * (applied to blocks of NSIM bands, L143): the orbitals psi with occupations occ define the operator, a block of
 * trial vectors phi receives it.  phi_dev / out_dev: nphi >= 1 vectors per k-point (any count, not tied to nbands), packed like
 * psi: element (k,i,ig) at nphi * sum_{k'<k} npw(k') + i*npw(k) + ig; device, 16-byte aligned; out may overlap neither psi nor
 * phi.  phi == psi (nphi = nbands) gives exx_apply's result, without the pair symmetry, which couples two bands of one set:
 * EXX_INFO_SYMMETRY reads 0.  Always fp64 (EXX_OPT_PRECISION is ignored).  Shards, tiles, pruning and paths as for exx_apply.
 * The first call, and any call with a larger nphi than before, allocates the trial vectors' real-space boxes and accumulators
 * (2 nk nphi boxes).  Asynchronous on the stream. */
int exx_apply_to(exx_ctx* ctx, const double* psi_dev, const double* occ_host, const double* phi_dev, int nphi, double* out_dev);

/* E_x = 1/2 sum w_k f_nk Re<c_nk|(V_x c)_nk> (Eq. 2).  If vxpsi_dev_or_null is NULL the library evaluates E_x
 * from psi alone: by the pair-density route (EXX_OPT_ENERGY_ROUTE = 0, fused kernels; the counters of exx_get_info then describe
 * this call) or by applying V_x into an internal buffer first.  ex_host: 1 double.  per_band_host_or_null: nk*nbands terms
 * 1/2 w_k f_nk Re<c|V_x c> (or NULL); they add up to E_x.  With shards (EXX_OPT_SHARD_COUNT > 1) and no V_x psi given, the
 * result is this shard's partial sum.  Synchronises the stream. */
int exx_energy(exx_ctx* ctx, const double* psi_dev, const double* occ_host, const double* vxpsi_dev_or_null, double* ex_host,
               double* per_band_host_or_null);

/* Subspace matrix of the exchange operator within k-point ik (BASELINE north_star "optional dense subspace matrix
 * <psi_i|V_x|psi_j>"; the paper's NSIM matrix-matrix work):  m_dev[i*nbands + j] = sum_g conj(c_i(g)) (V_x c)_j(g),
 * nbands x nbands complex128, row-major, device.  psi_dev / vxpsi_dev: the packed arrays of exx_apply (all k-points).
 * A ZGEMM on the fp64 tensor-core path (DMMA), split over the plane waves and reduced in a fixed order (deterministic).
 * Asynchronous on the stream.  Hermitian when vxpsi = V_x psi and every band is occupied. */
int exx_subspace(exx_ctx* ctx, int ik, const double* psi_dev, const double* vxpsi_dev, double* m_dev);

/* The same matrix for a block of trial vectors (the layout of exx_apply_to: nphi vectors per k-point in phi_dev and vphi_dev):
 * m_dev[i*nphi + j] = sum_g conj(phi_i(g)) vphi_j(g) within k-point ik, nphi x nphi complex128, row-major, device — the projected
 * operator <phi_i|V_x|phi_j> an iterative eigensolver builds from exx_apply_to's output.  Asynchronous. */
int exx_subspace_block(exx_ctx* ctx, int ik, const double* phi_dev, const double* vphi_dev, int nphi, double* m_dev);

/* The subspace matrix once more, for callers that must not allocate device memory:  m_dev[i*nvec + j] = sum_g conj(a_i(g)) b_j(g),
 * nvec x nvec complex128, row-major.  Needs no context (exx_create allocates), and calls no cudaMalloc, cudaFree or any other
 * allocating routine, on any call, successful or not.
 *   Who needs this: a program whose GPU memory is wholly managed by someone else — a framework's caching pool that has reserved the
 *   card, a job held to a fixed memory budget — where an allocation made behind the owner's back fails or steals what was promised
 *   elsewhere; and a latency-critical loop that cannot take the device-wide synchronisation cudaMalloc and cudaFree bring.
 *   Everyone else should call exx_subspace / exx_subspace_block, which have no size limit.
 * a_dev, b_dev: nvec vectors of npw complex128 each, vector i at element i*npw (for one k-point of the packed psi / V_x psi arrays:
 * the pointers psi_dev + 2*exx_psi_offset(ik) doubles, with npw = exx_npw(ik)); m_dev: nvec*nvec complex128; all three are device
 * pointers on the CURRENT device, 16-byte aligned, owned by the caller; inputs are only read, m_dev may not overlap them.
 * cuda_stream: a cudaStream_t of the current device cast to void* (NULL = default stream).  Asynchronous on that stream.
 *   The split-K scratch of the ZGEMM lives in a fixed array inside the library image: EXX_STATIC_SCRATCH_BYTES of every GPU that
 *   loads libexx stay occupied until the process exits, whether this call is used or not.  Hence the limits: 1 <= nvec <=
 *   EXX_STATIC_MAX_NVEC and 1 <= npw <= EXX_STATIC_MAX_NPW; beyond them the call returns EXX_ERR_LIMIT, launches nothing and leaves
 *   m_dev untouched (exx_last_error(NULL) then says which limit).
 *   The first call a process makes with a given device current looks up that device's address of the array (and may make the CUDA
 *   runtime load the library's kernels onto it): make that first call during set-up, outside any stream capture.
 *   All calls on one device share the one array.  Nothing in it has to start at zero — each call overwrites every element it later
 *   reads — so calls that follow one another on a stream, or are otherwise ordered, are independent.  Two calls whose kernels may
 *   run at the same time on one GPU (different streams without an event between them, or two host threads) race on the array and
 *   both results are garbage: order them.
 * Deterministic (fixed slice order); agrees with exx_subspace to rounding order (the number of slices may differ). */
#define EXX_STATIC_SCRATCH_BYTES (8 << 20) /* 8 MiB: 8 slices at nvec = 256, 20 at nvec = 160 */
#define EXX_STATIC_MAX_NVEC 256
#define EXX_STATIC_MAX_NPW (1 << 24)
int exx_subspace_static(const double* a_dev, const double* b_dev, int nvec, int64_t npw, double* m_dev, void* cuda_stream);

/* Same as exx_apply (+ exx_energy when ex_host_or_null != NULL) on HOST buffers: copies psi to the device, applies,
 * copies out back; synchronises.  Pinned host memory makes the copies asynchronous, pageable memory works too. */
int exx_apply_host(exx_ctx* ctx, const double* psi_host, const double* occ_host, double* out_host, double* ex_host_or_null);

/* Building blocks exposed for parity tests and stand-alone use (all asynchronous on the stream, device pointers):
 * exx_scatter: box(b, map_k[ig]) = coef(b, ig), zero elsewhere; exx_gather: the reverse (pure data movement, bit exact);
 * exx_fft3d: in-place unnormalised 3-D transform of nbatch boxes, sign = -1 forward (e^{-i G.r}), +1 inverse;
 * exx_to_real: u = scatter + inverse transform (step S1). */
int exx_scatter(exx_ctx* ctx, int ik, const double* coef_dev, int nbatch, double* box_dev);
int exx_gather(exx_ctx* ctx, int ik, const double* box_dev, int nbatch, double* coef_dev);
int exx_fft3d(exx_ctx* ctx, double* box_dev, int nbatch, int sign);
int exx_to_real(exx_ctx* ctx, int ik, const double* coef_dev, int nbatch, double* box_dev);
/* Stand-alone batched 3-D transform through the fused passes (cubic N = 16, 32, 40, 48, 64, 72, 80, 96, 128; EXX_ERR_BAD_GRID otherwise): two
 * passes per transform instead of the three of exx_fft3d.  The frequency side lives in the library's "F layout":
 * exx_findex gives, for every natural C-order frequency index ((kx*N + ky)*N + kz), its position in an F-layout box.
 *   sign = -1: in_dev natural-order boxes (unchanged) -> out_dev F-layout boxes, unnormalised forward transform
 *   sign = +1: in_dev F-layout boxes (used as scratch: destroyed) -> out_dev natural-order boxes, unnormalised inverse
 * in_dev != out_dev, nbatch boxes of Ng complex128 each; asynchronous on the stream. */
int exx_fft3d_fused(exx_ctx* ctx, double* in_dev, int nbatch, int sign, double* out_dev);
int exx_findex(const exx_ctx* ctx, int32_t* host_out /* Ng entries */);
/* K'_{k-q}(g) as the library tabulated it (host_out: Ng doubles, C order). */
int exx_kernel_table(const exx_ctx* ctx, int ik, int iq, double* host_out);

/* Measurement aid ("report both fractions"): the fp64 vector-pipe peak of the current device, measured by a
 * chain-free DFMA loop (8 independent accumulators per thread, 2 flops per DFMA, every SM filled; CUDA events, best of 3).
 * *gflops_host receives GFLOP/s.  Not on the hot path; synchronises the stream.  The fused passes are plain fp64 FMA/ADD/MUL code
 * (tcgen05 has no fp64 kind), so this is the ALU roofline bench.py quotes beside the HBM one. */
int exx_measure_fp64_peak(void* cuda_stream, double* gflops_host);

const char* exx_strerror(int code);
const char* exx_last_error(const exx_ctx* ctx_or_null); /* detail of the last EXX_ERR_CUDA (thread-local if ctx NULL) */
int exx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EXX_H */
