// exx_api.cu — the C ABI of libexx (include/exx.h): host-side plan (index maps, kernel tables, twiddles,
// workspaces), the loop nest over k, q, n-tiles, m-tiles, and the generic pipeline S1..S8.
// Product code: shares nothing with oracle/.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <new>

#include "exx_internal.h"
#include "exx_shard.h"

namespace exx {

static thread_local std::string g_thread_error;
void set_thread_error(const std::string& s) { g_thread_error = s; }
bool test_fail_alloc(const char* tag) {
    const char* v = getenv("EXX_TEST_FAIL_ALLOC");
    return v && !strcmp(v, tag);
}

int cuda_fail(exx_ctx* c, cudaError_t e, const char* what) {
    std::string s = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
    if (c) c->last_error = s;
    g_thread_error = s;
    return EXX_ERR_CUDA;
}

LaunchScope::LaunchScope(exx_ctx* c_, int k, int64_t units) : c(c_), kclass(k) {
    c->launches++;
    c->launches_by_class[k]++;
    c->units_by_class[k] += units;
    if (c->opt_profile) {
        if (c->event_pool_used + 2 > c->event_pool.size()) {
            for (int i = 0; i < 256; i++) {
                cudaEvent_t e;
                if (cudaEventCreate(&e) != cudaSuccess) return;
                c->event_pool.push_back(e);
            }
        }
        a = c->event_pool[c->event_pool_used++];
        b = c->event_pool[c->event_pool_used++];
        cudaEventRecord(a, c->stream);
    }
}
LaunchScope::~LaunchScope() {
    if (a && b) {
        cudaEventRecord(b, c->stream);
        c->events.push_back({a, b, kclass});
    }
}

static const char* kclass_names[KC_COUNT] = {"scatter", "gather", "fft_axis_generic", "codensity", "kernel_multiply",
                                             "accumulate", "energy", "fused_pass_a", "fused_pass_b", "fused_pass_c", "subspace_zgemm", "fused_fft_pass",
                                             "fused_pass_r"};

// ---- host arithmetic of S0 (index maps, kernel tables).  Evaluation order of |t.B|^2 is fixed (A11). ----
static inline int fold(int j, int n) { return (2 * j < n) ? j : j - n; }
static double norm2_frac(const double B[9], const double t[3]) {
    double s = 0.0;
    for (int cc = 0; cc < 3; cc++) {
        double x = (t[0] * B[cc] + t[1] * B[3 + cc]) + t[2] * B[6 + cc];
        s = s + x * x;
    }
    return s;
}
static bool is_2a3b(int n) {  // 2^a 3^b 5^c
    if (n < 2) return false;
    while (n % 2 == 0) n /= 2;
    while (n % 3 == 0) n /= 3;
    while (n % 5 == 0) n /= 5;
    return n == 1;
}
static void make_plan(Plan1D& p, int n) {
    p.n = n;
    p.nst = 0;
    int m = n;
    while (m % 4 == 0) { p.radix[p.nst++] = 4; m /= 4; }
    while (m % 2 == 0) { p.radix[p.nst++] = 2; m /= 2; }
    while (m % 3 == 0) { p.radix[p.nst++] = 3; m /= 3; }
    while (m % 5 == 0) { p.radix[p.nst++] = 5; m /= 5; }
}

static double kernel_value(const exx_kernel_params& kp, const double B[9], const double t[3]) {
    const double pi = 3.14159265358979323846264338327950288;
    bool zero = (t[0] == 0.0 && t[1] == 0.0 && t[2] == 0.0);
    if (kp.kind == 0) {
        if (zero) return 0.0;
        return kp.scale * (4.0 * pi / norm2_frac(B, t));
    }
    if (zero) return kp.scale * (pi / (kp.mu * kp.mu));
    double q2 = norm2_frac(B, t);
    double x = q2 / (4.0 * kp.mu * kp.mu);
    return kp.scale * ((4.0 * pi / q2) * (-expm1(-x)));
}

static void free_ctx(exx_ctx* c) {
    if (!c) return;
    if (c->inner) free_ctx(c->inner);
    fused_destroy(c);
    cudaFree(c->map_dev);
    cudaFree(c->ktab_dev);
    for (int i = 0; i < 3; i++) cudaFree(c->plan[i].tw_dev);
    cudaFree(c->u_dev);
    cudaFree(c->work_dev);
    cudaFree(c->acc_dev);
    cudaFree(c->vx_dev);
    cudaFree(c->psi_stage_dev);
    cudaFree(c->uphi1_dev);
    cudaFree(c->band_dot_dev);
    cudaFree(c->band_e_dev);
    cudaFree(c->occw_dev);
    cudaFree(c->band_off_dev);
    cudaFree(c->band_len_dev);
    cudaFree(c->subspace_dev);
    if (c->host_pinned) cudaFreeHost(c->host_pinned);
    for (auto e : c->event_pool) cudaEventDestroy(e);
    delete c;
}

template <typename T>
static int dev_alloc(exx_ctx* c, T** p, size_t count, const char* test_tag = nullptr) {
    size_t bytes = sizeof(T) * (count ? count : 1);
    cudaError_t e = (test_tag && test_fail_alloc(test_tag)) ? cudaErrorMemoryAllocation : cudaMalloc((void**)p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        c->last_error = "cudaMalloc of " + std::to_string(bytes) + " bytes failed";
        set_thread_error(c->last_error);
        return EXX_ERR_ALLOC;
    }
    c->dev_bytes += bytes;
    return EXX_OK;
}

}  // namespace exx

namespace exx {
// S1: u_nk(r) for every band (batches bounded so a launch never exceeds ~2^28 elements)
int compute_u_cache(exx_ctx* c, const double2* psi) {
    int rc;
    const int nb = c->nb, nk = c->nk;
    const int64_t Ng = c->Ng;
    for (int k = 0; k < nk; k++) {
        int bmax = (int)std::max<int64_t>(1, std::min<int64_t>(nb, ((int64_t)1 << 28) / Ng));
        for (int n0 = 0; n0 < nb; n0 += bmax) {
            int bn = std::min(bmax, nb - n0);
            double2* box = c->u_dev + ((size_t)k * nb + n0) * Ng;
            if ((rc = launch_scatter(c, k, psi + c->off[k] + (int64_t)n0 * c->npw[k], bn, box))) return rc;
            if ((rc = launch_fft3d_generic(c, box, bn, +1))) return rc;
        }
    }
    return EXX_OK;
}
}  // namespace exx

using namespace exx;

extern "C" {

int exx_version(void) { return 100; }

const char* exx_strerror(int code) {
    switch (code) {
    case EXX_OK: return "ok";
    case EXX_ERR_NULL: return "null pointer";
    case EXX_ERR_BAD_GRID: return "bad grid (each N_i must be 2^a 3^b 5^c, 2 <= N_i <= 1024, and hold the cutoff sphere)";
    case EXX_ERR_BAD_LATTICE: return "bad lattice (zero or non-finite volume)";
    case EXX_ERR_BAD_CUTOFF: return "bad cutoff";
    case EXX_ERR_BAD_KERNEL: return "bad kernel parameters";
    case EXX_ERR_BAD_OCC: return "bad occupation (negative or non-finite)";
    case EXX_ERR_ALLOC: return "allocation failed";
    case EXX_ERR_CUDA: return "CUDA error";
    case EXX_ERR_BAD_ARG: return "bad argument";
    case EXX_ERR_ALIAS: return "out aliases psi";
    case EXX_ERR_LIMIT: return "size beyond the fixed capacity of a no-allocation entry point";
    default: return "unknown error";
    }
}
const char* exx_last_error(const exx_ctx* c) { return c ? c->last_error.c_str() : g_thread_error.c_str(); }
const char* exx_kernel_class_name(int k) { return (k >= 0 && k < KC_COUNT) ? kclass_names[k] : nullptr; }

static int ensure_big(exx_ctx* c);

static int create_impl(exx_ctx** out, const int grid[3], const double lattice[9], int nk, const double* kfrac, const double* kweight,
                       double ecut, const exx_kernel_params* kp, int nbands, void* cuda_stream, bool allow_inner) {
    if (!out || !grid || !lattice || !kfrac || !kweight || !kp) return EXX_ERR_NULL;
    if (nk < 1 || nbands < 1) return EXX_ERR_BAD_ARG;
    for (int i = 0; i < 3; i++)
        if (!is_2a3b(grid[i]) || grid[i] > 1024) return EXX_ERR_BAD_GRID;
    if (!(ecut > 0.0) || !std::isfinite(ecut)) return EXX_ERR_BAD_CUTOFF;
    if (kp->kind != 0 && kp->kind != 1) return EXX_ERR_BAD_KERNEL;
    if (kp->kind == 1 && !(kp->mu > 0.0 && std::isfinite(kp->mu))) return EXX_ERR_BAD_KERNEL;
    if (!std::isfinite(kp->scale)) return EXX_ERR_BAD_KERNEL;
    for (int i = 0; i < nk; i++) {
        if (!std::isfinite(kweight[i])) return EXX_ERR_BAD_ARG;
        for (int d = 0; d < 3; d++)
            if (!std::isfinite(kfrac[3 * i + d])) return EXX_ERR_BAD_ARG;
    }
    const double* a = lattice;
    double det = a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) + a[2] * (a[3] * a[7] - a[4] * a[6]);
    if (!std::isfinite(det) || det == 0.0) return EXX_ERR_BAD_LATTICE;

    exx_ctx* c = new (std::nothrow) exx_ctx();
    if (!c) return EXX_ERR_ALLOC;
    int rc = EXX_OK;
    auto fail = [&](int code) { std::string keep = c->last_error; free_ctx(c); set_thread_error(keep); return code; };
    try {
        memcpy(c->N, grid, sizeof(int) * 3);
        c->Ng = (int64_t)grid[0] * grid[1] * grid[2];
        if (c->Ng > (int64_t)INT32_MAX) return fail(EXX_ERR_BAD_GRID);
        memcpy(c->A, lattice, sizeof(double) * 9);
        c->omega = fabs(det);
        const double twopi = 6.283185307179586476925286766559;
        for (int i = 0; i < 3; i++) {
            const double *p = a + 3 * ((i + 1) % 3), *q = a + 3 * ((i + 2) % 3);
            c->B[3 * i + 0] = twopi * (p[1] * q[2] - p[2] * q[1]) / det;
            c->B[3 * i + 1] = twopi * (p[2] * q[0] - p[0] * q[2]) / det;
            c->B[3 * i + 2] = twopi * (p[0] * q[1] - p[1] * q[0]) / det;
        }
        c->nk = nk;
        c->nb = nbands;
        c->kfrac.assign(kfrac, kfrac + 3 * nk);
        c->kw.assign(kweight, kweight + nk);
        c->ecut = ecut;
        c->kp = *kp;
        c->stream = (cudaStream_t)cuda_stream;

        // ---- S0a: sphere(k) = { g : |k+G|^2/2 < ecut } by enumerating the bounding box of the sphere
        // (|g_i + kappa_i| = |(k+G).a_i|/2pi <= sqrt(2 ecut) |a_i| / 2pi), checking it fits, sorting by box index.
        c->npw.resize(nk);
        c->off.assign(nk + 1, 0);
        c->map_h.resize(nk);
        c->map_off.assign(nk + 1, 0);
        int gmin[3] = {0, 0, 0}, gmax[3] = {0, 0, 0};
        for (int k = 0; k < nk; k++) {
            int lo[3], hi[3];
            for (int i = 0; i < 3; i++) {
                double alen = sqrt(a[3 * i] * a[3 * i] + a[3 * i + 1] * a[3 * i + 1] + a[3 * i + 2] * a[3 * i + 2]);
                double r = sqrt(2.0 * ecut) * alen / twopi;
                lo[i] = (int)floor(-r - kfrac[3 * k + i]) - 1;
                hi[i] = (int)ceil(r - kfrac[3 * k + i]) + 1;
            }
            std::vector<int32_t>& m = c->map_h[k];
            for (int g1 = lo[0]; g1 <= hi[0]; g1++)
                for (int g2 = lo[1]; g2 <= hi[1]; g2++)
                    for (int g3 = lo[2]; g3 <= hi[2]; g3++) {
                        double t[3] = {(double)g1 + kfrac[3 * k], (double)g2 + kfrac[3 * k + 1], (double)g3 + kfrac[3 * k + 2]};
                        double e = 0.5 * norm2_frac(c->B, t);
                        if (!(e < ecut)) continue;
                        int g[3] = {g1, g2, g3};
                        int j[3];
                        for (int i = 0; i < 3; i++) {
                            // representable range of folded frequencies: [-(N/2), (N-1)/2] (integer division)
                            if (g[i] < -(grid[i] / 2) || g[i] > (grid[i] - 1) / 2) return fail(EXX_ERR_BAD_GRID);
                            j[i] = g[i] < 0 ? g[i] + grid[i] : g[i];
                            gmin[i] = std::min(gmin[i], g[i]);
                            gmax[i] = std::max(gmax[i], g[i]);
                        }
                        m.push_back((int32_t)(((int64_t)j[0] * grid[1] + j[1]) * grid[2] + j[2]));
                    }
            if (m.empty()) return fail(EXX_ERR_BAD_CUTOFF);
            std::sort(m.begin(), m.end());
            c->npw[k] = (int)m.size();
            c->off[k + 1] = c->off[k] + (int64_t)nbands * c->npw[k];
            c->map_off[k + 1] = c->map_off[k] + c->npw[k];
        }
        c->alias_free = true;
        for (int i = 0; i < 3; i++) {
            c->gmax[i] = std::max(gmax[i], -gmin[i]);
            if (4 * c->gmax[i] + 1 > grid[i]) c->alias_free = false;
        }
        if ((rc = dev_alloc(c, &c->map_dev, (size_t)c->map_off[nk]))) return fail(rc);
        for (int k = 0; k < nk; k++)
            if (cudaMemcpy(c->map_dev + c->map_off[k], c->map_h[k].data(), sizeof(int32_t) * c->npw[k], cudaMemcpyHostToDevice) != cudaSuccess)
                return fail(cuda_fail(c, cudaGetLastError(), "H2D index map"));

        // ---- S0b: K'_{dk}(g) = K(|dk + G|)/(Omega Ng^2), one table per distinct dk = kappa_k - kappa_q
        c->ktab_of.assign((size_t)nk * nk, -1);
        std::map<std::vector<double>, int> seen;
        for (int k = 0; k < nk; k++)
            for (int q = 0; q < nk; q++) {
                std::vector<double> dk = {kfrac[3 * k] - kfrac[3 * q], kfrac[3 * k + 1] - kfrac[3 * q + 1], kfrac[3 * k + 2] - kfrac[3 * q + 2]};
                auto it = seen.find(dk);
                if (it == seen.end()) {
                    it = seen.emplace(dk, c->ntab++).first;
                    c->ktab_dk.push_back(dk);
                }
                c->ktab_of[(size_t)k * nk + q] = it->second;
            }
        if ((rc = dev_alloc(c, &c->ktab_dev, (size_t)c->ntab * c->Ng))) return fail(rc);
        {
            std::vector<double> tab((size_t)c->Ng);
            const double norm = c->omega * (double)c->Ng * (double)c->Ng;
            for (int t = 0; t < c->ntab; t++) {
                const std::vector<double>& dk = c->ktab_dk[t];
                for (int j1 = 0; j1 < grid[0]; j1++)
                    for (int j2 = 0; j2 < grid[1]; j2++)
                        for (int j3 = 0; j3 < grid[2]; j3++) {
                            double tt[3] = {dk[0] + (double)fold(j1, grid[0]), dk[1] + (double)fold(j2, grid[1]), dk[2] + (double)fold(j3, grid[2])};
                            tab[((size_t)j1 * grid[1] + j2) * grid[2] + j3] = kernel_value(c->kp, c->B, tt) / norm;
                        }
                if (cudaMemcpy(c->ktab_dev + (size_t)t * c->Ng, tab.data(), sizeof(double) * c->Ng, cudaMemcpyHostToDevice) != cudaSuccess)
                    return fail(cuda_fail(c, cudaGetLastError(), "H2D kernel table"));
            }
        }

        // ---- S0c: twiddles exp(-2 pi i j / n), angles in long double
        for (int ax = 0; ax < 3; ax++) {
            make_plan(c->plan[ax], grid[ax]);
            int n = grid[ax];
            std::vector<double2> tw(n);
            const long double tp = 6.283185307179586476925286766559005768L;
            for (int j = 0; j < n; j++) {
                long double ang = tp * (long double)j / (long double)n;
                tw[j] = make_double2((double)cosl(ang), (double)(-sinl(ang)));
            }
            if ((rc = dev_alloc(c, &c->plan[ax].tw_dev, (size_t)n))) return fail(rc);
            if (cudaMemcpy(c->plan[ax].tw_dev, tw.data(), sizeof(double2) * n, cudaMemcpyHostToDevice) != cudaSuccess)
                return fail(cuda_fail(c, cudaGetLastError(), "H2D twiddles"));
        }

        // ---- workspaces
        int nbt = nk * nbands;
        if ((rc = dev_alloc(c, &c->vx_dev, (size_t)c->off[nk]))) return fail(rc);
        if ((rc = dev_alloc(c, &c->band_dot_dev, (size_t)nbt))) return fail(rc);
        if ((rc = dev_alloc(c, &c->band_e_dev, (size_t)nbt + 1))) return fail(rc);
        if ((rc = dev_alloc(c, &c->occw_dev, (size_t)nbt))) return fail(rc);
        if (cudaMallocHost((void**)&c->host_pinned, sizeof(double) * (2 * (size_t)nbt + 2)) != cudaSuccess) {
            cudaGetLastError();
            return fail(EXX_ERR_ALLOC);
        }
        if ((rc = dev_alloc(c, &c->band_off_dev, (size_t)nbt))) return fail(rc);
        if ((rc = dev_alloc(c, &c->band_len_dev, (size_t)nbt))) return fail(rc);
        {
            std::vector<int64_t> bo(nbt);
            std::vector<int> bl(nbt);
            for (int k = 0; k < nk; k++)
                for (int n = 0; n < nbands; n++) {
                    bo[k * nbands + n] = c->off[k] + (int64_t)n * c->npw[k];
                    bl[k * nbands + n] = c->npw[k];
                }
            cudaMemcpy(c->band_off_dev, bo.data(), sizeof(int64_t) * nbt, cudaMemcpyHostToDevice);
            cudaMemcpy(c->band_len_dev, bl.data(), sizeof(int) * nbt, cudaMemcpyHostToDevice);
        }
        if ((rc = fft_generic_init(c))) { exx_destroy(c); return rc; }
        // compact work grid: smallest fused-capable cubic grid with N >= 4 gmax + 1, if it has fewer points than the caller's box —
        // or, when the caller's grid has no fused kernels (non-cubic, or a cubic size outside the list), at most 4x its points:
        // the fused passes are ~7x faster per point than the generic per-axis kernels, and every alias-free grid gives the same
        // V_x psi on the sphere
        if (allow_inner && c->alias_free) {
            int need = 0;
            for (int i = 0; i < 3; i++) need = std::max(need, 4 * c->gmax[i] + 1);
            const int cand[9] = {16, 32, 40, 48, 64, 72, 80, 96, 128};
            for (int ci = 0; ci < 9; ci++)
                if (cand[ci] >= need) {
                    int64_t nw = cand[ci];
                    const bool smaller = nw * nw * nw < c->Ng;
                    if (smaller || (!fused_supported(c) && nw * nw * nw <= 4 * c->Ng)) {
                        int g3[3] = {cand[ci], cand[ci], cand[ci]};
                        exx_ctx* in = nullptr;
                        if (create_impl(&in, g3, lattice, nk, kfrac, kweight, ecut, kp, nbands, cuda_stream, false) == EXX_OK) {
                            bool same = true;  // same spheres in the same order (ordering is grid-independent, checked anyway)
                            for (int k = 0; k < nk; k++) same = same && in->npw[k] == c->npw[k];
                            if (same) {
                                c->inner = in;
                                c->inner_larger = !smaller;
                            } else
                                free_ctx(in);
                        }
                    }
                    break;
                }
        }
        if (!c->inner)
            if ((rc = ensure_big(c))) { exx_destroy(c); return rc; }
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { rc = cuda_fail(c, e, "exx_create sync"); exx_destroy(c); return rc; }
    } catch (const std::bad_alloc&) {
        return fail(EXX_ERR_ALLOC);
    }
    *out = c;
    return EXX_OK;
}

// the buffers that scale with nbands * Ng: real-space cache, pair workspace, accumulators, fused tables
static int ensure_big(exx_ctx* c) {
    if (c->big_alloc) return EXX_OK;
    // a failure part-way (out of memory) frees what this call allocated, so that a retry starts clean instead of leaking
    const size_t bytes_before = c->dev_bytes;
    auto undo = [&](int code) {
        if (c->fused) fused_destroy(c);
        cudaFree(c->u_dev), cudaFree(c->work_dev), cudaFree(c->acc_dev);
        c->u_dev = c->work_dev = c->acc_dev = nullptr;
        c->work_boxes = c->acc_boxes = 0;
        c->dev_bytes = bytes_before;  // EXX_INFO_WORKSPACE_BYTES counts what the context holds, not what it once tried to get
        return code;
    };
    int rc;
    int nbt = c->nk * c->nb;
    if ((rc = dev_alloc(c, &c->u_dev, (size_t)nbt * c->Ng))) return undo(rc);
    // generic pipeline: one n at a time, up to 16 m per tile, at most ~1 GiB of pair workspace;
    // fused pipeline: tn x tm pairs per batch (work) and tn accumulators
    size_t box_bytes = sizeof(double2) * (size_t)c->Ng;
    size_t wb = std::max<size_t>(1, std::min<size_t>(16, ((size_t)1 << 30) / box_bytes));
    c->work_boxes = wb;
    c->acc_boxes = 1;
    if (fused_supported(c)) {
        int tn, tm;
        fused_tiles(c, &tn, &tm);
        c->acc_boxes = (size_t)c->nk * c->nb;  // the fused loop nest keeps one accumulator per (k, band)
        c->work_boxes = std::max<size_t>(wb, (size_t)tn * tm);
    }
    if ((rc = dev_alloc(c, &c->work_dev, c->work_boxes * c->Ng))) return undo(rc);
    if ((rc = dev_alloc(c, &c->acc_dev, c->acc_boxes * c->Ng, "acc"))) return undo(rc);
    if (fused_supported(c))
        if ((rc = fused_create(c))) return undo(rc);
    c->big_alloc = true;
    return EXX_OK;
}

int exx_create(exx_ctx** out, const int grid[3], const double lattice[9], int nk, const double* kfrac, const double* kweight,
               double ecut, const exx_kernel_params* kp, int nbands, void* cuda_stream) {
    return create_impl(out, grid, lattice, nk, kfrac, kweight, ecut, kp, nbands, cuda_stream, true);
}

int exx_destroy(exx_ctx* c) {
    if (!c) return EXX_ERR_NULL;
    cudaStreamSynchronize(c->stream);
    free_ctx(c);
    return EXX_OK;
}

int exx_npw(const exx_ctx* c, int ik, int* npw) {
    if (!c || !npw) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_ERR_BAD_ARG;
    *npw = c->npw[ik];
    return EXX_OK;
}
int exx_index_map(const exx_ctx* c, int ik, int32_t* host_out) {
    if (!c || !host_out) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_ERR_BAD_ARG;
    memcpy(host_out, c->map_h[ik].data(), sizeof(int32_t) * c->npw[ik]);
    return EXX_OK;
}
int exx_psi_offset(const exx_ctx* c, int ik, int64_t* complex_elems) {
    if (!c || !complex_elems) return EXX_ERR_NULL;
    if (ik < 0 || ik > c->nk) return EXX_ERR_BAD_ARG;
    *complex_elems = c->off[ik];
    return EXX_OK;
}
int exx_kernel_table(const exx_ctx* c, int ik, int iq, double* host_out) {
    if (!c || !host_out) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk || iq < 0 || iq >= c->nk) return EXX_ERR_BAD_ARG;
    int t = c->ktab_of[(size_t)ik * c->nk + iq];
    cudaStreamSynchronize(c->stream);
    if (cudaMemcpy(host_out, c->ktab_dev + (size_t)t * c->Ng, sizeof(double) * c->Ng, cudaMemcpyDeviceToHost) != cudaSuccess)
        return cuda_fail(const_cast<exx_ctx*>(c), cudaGetLastError(), "D2H kernel table");
    return EXX_OK;
}

int exx_set_option(exx_ctx* c, int option, int64_t value) {
    if (!c) return EXX_ERR_NULL;
    switch (option) {
    case EXX_OPT_PATH:
        if (value < 0 || value > 2) return EXX_ERR_BAD_ARG;
        if (value == 2 && !fused_supported(c)) return EXX_ERR_BAD_ARG;
        c->opt_path = value;
        return EXX_OK;
    case EXX_OPT_TILE_N:
        if (value < 0 || value > TMAX) return EXX_ERR_BAD_ARG;
        c->opt_tile_n = value;
        return EXX_OK;
    case EXX_OPT_TILE_M:
        if (value < 0 || value > TMAX) return EXX_ERR_BAD_ARG;
        c->opt_tile_m = value;
        return EXX_OK;
    case EXX_OPT_PRUNE:
        c->opt_prune = value ? 1 : 0;
        return EXX_OK;
    case EXX_OPT_PROFILE:
        c->opt_profile = value ? 1 : 0;
        return EXX_OK;
    case EXX_OPT_SYMMETRY:
        c->opt_symmetry = value ? 1 : 0;
        return EXX_OK;
    case EXX_OPT_PRECISION:
        if (value != 0 && value != 1) return EXX_ERR_BAD_ARG;
        c->opt_precision = value;
        return EXX_OK;
    case EXX_OPT_SHARD_COUNT:
        if (value < 1 || value > 65536) return EXX_ERR_BAD_ARG;
        c->opt_shard_count = value;
        return EXX_OK;
    case EXX_OPT_SHARD_RANK:
        if (value < 0 || value > 65535) return EXX_ERR_BAD_ARG;
        c->opt_shard_rank = value;
        return EXX_OK;
    case EXX_OPT_ENERGY_ROUTE:
        if (value != 0 && value != 1) return EXX_ERR_BAD_ARG;
        c->opt_energy_route = value;
        return EXX_OK;
    case EXX_OPT_KEEP_U:
        c->opt_keep_u = value ? 1 : 0;
        return EXX_OK;
    case EXX_OPT_DUAL_SWEEP:
        c->opt_dual = value ? 1 : 0;
        return EXX_OK;
    case EXX_OPT_PRUNE_SPHERE:
        c->opt_prune_rows = value ? 1 : 0;
        return EXX_OK;
    default: return EXX_ERR_BAD_ARG;
    }
}
int exx_get_option(const exx_ctx* c, int option, int64_t* value) {
    if (!c || !value) return EXX_ERR_NULL;
    switch (option) {
    case EXX_OPT_PATH: *value = c->opt_path; return EXX_OK;
    case EXX_OPT_TILE_N: *value = c->opt_tile_n; return EXX_OK;
    case EXX_OPT_TILE_M: *value = c->opt_tile_m; return EXX_OK;
    case EXX_OPT_PRUNE: *value = c->opt_prune; return EXX_OK;
    case EXX_OPT_PROFILE: *value = c->opt_profile; return EXX_OK;
    case EXX_OPT_SYMMETRY: *value = c->opt_symmetry; return EXX_OK;
    case EXX_OPT_PRECISION: *value = c->opt_precision; return EXX_OK;
    case EXX_OPT_SHARD_COUNT: *value = c->opt_shard_count; return EXX_OK;
    case EXX_OPT_SHARD_RANK: *value = c->opt_shard_rank; return EXX_OK;
    case EXX_OPT_ENERGY_ROUTE: *value = c->opt_energy_route; return EXX_OK;
    case EXX_OPT_KEEP_U: *value = c->opt_keep_u; return EXX_OK;
    case EXX_OPT_DUAL_SWEEP: *value = c->opt_dual; return EXX_OK;
    case EXX_OPT_PRUNE_SPHERE: *value = c->opt_prune_rows; return EXX_OK;
    default: return EXX_ERR_BAD_ARG;
    }
}
int exx_get_info(const exx_ctx* c, int what, int64_t* value) {
    if (!c || !value) return EXX_ERR_NULL;
    switch (what) {
    case EXX_INFO_LAUNCHES: *value = c->launches; return EXX_OK;
    case EXX_INFO_PAIRS_ORDERED: *value = c->pairs_ordered; return EXX_OK;
    case EXX_INFO_PAIRS_EXECUTED: *value = c->pairs_executed; return EXX_OK;
    case EXX_INFO_PATH_USED: *value = c->path_used; return EXX_OK;
    case EXX_INFO_WORKSPACE_BYTES: *value = (int64_t)c->dev_bytes + (c->inner ? (int64_t)c->inner->dev_bytes : 0); return EXX_OK;
    case EXX_INFO_WORK_GRID: *value = (c->inner && c->last_pruned) ? c->inner->N[0] : c->N[0]; return EXX_OK;
    case EXX_INFO_COMPACT_GRID: *value = c->inner ? c->inner->N[0] : 0; return EXX_OK;
    case EXX_INFO_NCOEF: *value = c->off[c->nk]; return EXX_OK;
    case EXX_INFO_TILE_N: *value = c->tile_n_used; return EXX_OK;
    case EXX_INFO_TILE_M: *value = c->tile_m_used; return EXX_OK;
    case EXX_INFO_PRUNED: *value = c->pruned_used; return EXX_OK;
    case EXX_INFO_SYMMETRY: *value = c->symmetry_used; return EXX_OK;
    case EXX_INFO_PRECISION: *value = c->precision_used; return EXX_OK;
    case EXX_INFO_ENERGY_ROUTE: *value = c->energy_route_used; return EXX_OK;
    case EXX_INFO_NUM_KERNEL_CLASSES: *value = KC_COUNT; return EXX_OK;
    default: return EXX_ERR_BAD_ARG;
    }
}
int exx_get_kernel_time(exx_ctx* c, int kclass, double* ms_total, int64_t* launches, int64_t* units) {
    if (!c || !ms_total || !launches || !units) return EXX_ERR_NULL;
    if (kclass < 0 || kclass >= KC_COUNT) return EXX_ERR_BAD_ARG;
    if (c->inner && c->last_pruned) return exx_get_kernel_time(c->inner, kclass, ms_total, launches, units);
    EXX_CUDA(c, cudaStreamSynchronize(c->stream));
    double ms = 0.0;
    for (const EventRec& r : c->events)
        if (r.kclass == kclass) {
            float t = 0.f;
            EXX_CUDA(c, cudaEventElapsedTime(&t, r.a, r.b));
            ms += t;
        }
    *ms_total = ms;
    *launches = c->launches_by_class[kclass];
    *units = c->units_by_class[kclass];
    return EXX_OK;
}

// ---- building blocks ----
int exx_scatter(exx_ctx* c, int ik, const double* coef_dev, int nbatch, double* box_dev) {
    if (!c || !coef_dev || !box_dev) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk || nbatch < 0) return EXX_ERR_BAD_ARG;
    if (nbatch == 0) return EXX_OK;
    return launch_scatter(c, ik, (const double2*)coef_dev, nbatch, (double2*)box_dev);
}
int exx_gather(exx_ctx* c, int ik, const double* box_dev, int nbatch, double* coef_dev) {
    if (!c || !coef_dev || !box_dev) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk || nbatch < 0) return EXX_ERR_BAD_ARG;
    if (nbatch == 0) return EXX_OK;
    return launch_gather(c, ik, (const double2*)box_dev, nbatch, (double2*)coef_dev);
}
int exx_fft3d(exx_ctx* c, double* box_dev, int nbatch, int sign) {
    if (!c || !box_dev) return EXX_ERR_NULL;
    if (nbatch < 0 || (sign != 1 && sign != -1)) return EXX_ERR_BAD_ARG;
    if (nbatch == 0) return EXX_OK;
    return launch_fft3d_generic(c, (double2*)box_dev, nbatch, sign);
}
int exx_fft3d_fused(exx_ctx* c, double* in_dev, int nbatch, int sign, double* out_dev) {
    if (!c || !in_dev || !out_dev) return EXX_ERR_NULL;
    if (nbatch < 0 || (sign != 1 && sign != -1) || in_dev == out_dev) return EXX_ERR_BAD_ARG;
    if (nbatch == 0) return EXX_OK;
    return fused_fft3d(c, (double2*)in_dev, nbatch, sign, (double2*)out_dev);
}
int exx_findex(const exx_ctx* c, int32_t* host_out) {
    if (!c || !host_out) return EXX_ERR_NULL;
    return fused_findex(c, host_out);
}
int exx_to_real(exx_ctx* c, int ik, const double* coef_dev, int nbatch, double* box_dev) {
    int rc = exx_scatter(c, ik, coef_dev, nbatch, box_dev);
    if (rc) return rc;
    return exx_fft3d(c, box_dev, nbatch, +1);
}

static int check_occ(const exx_ctx* c, const double* occ) {
    for (int i = 0; i < c->nk * c->nb; i++)
        if (!(occ[i] >= 0.0) || !std::isfinite(occ[i])) return EXX_ERR_BAD_OCC;
    return EXX_OK;
}

static void reset_counters(exx_ctx* c) {
    c->launches = 0;
    for (int i = 0; i < KC_COUNT; i++) c->launches_by_class[i] = c->units_by_class[i] = 0;
    c->events.clear();
    c->event_pool_used = 0;
    c->pairs_ordered = c->pairs_executed = 0;
    c->symmetry_used = 0;
    c->precision_used = 0;
}

// Generic pipeline, steps S1..S7 as separate kernels.
static int apply_generic(exx_ctx* c, const double2* psi, const double* occ, double2* out, const double2* phi, int nphi) {
    int rc;
    const int nb = c->nb, nk = c->nk;
    const int64_t Ng = c->Ng;
    c->path_used = 1;
    c->pruned_used = 0;
    c->u_valid = false;  // EXX_OPT_KEEP_U is a promise about the fused path's cache only
    if ((rc = compute_u_cache(c, psi))) return rc;
    int tm_max = (int)std::min<size_t>(c->work_boxes, 32);
    if (c->opt_tile_m > 0) tm_max = (int)std::min<int64_t>(tm_max, c->opt_tile_m);
    c->tile_n_used = 1;
    c->tile_m_used = tm_max;
    const int na = phi ? nphi : nb;  // output rows per k-point
    for (int k = 0; k < nk; k++)
        for (int n = 0; n < na; n++) {
            double2* out_row = out + c->off[k] / nb * na + (int64_t)n * c->npw[k];
            if ((int64_t)(k * na + n) % c->opt_shard_count != c->opt_shard_rank) {
                // another shard's output row: zero here, so that the sum over shards is the full result
                EXX_CUDA(c, cudaMemsetAsync(out_row, 0, sizeof(double2) * (size_t)c->npw[k], c->stream));
                continue;
            }
            EXX_CUDA(c, cudaMemsetAsync(c->acc_dev, 0, sizeof(double2) * (size_t)Ng, c->stream));
            // the row's real-space box: u_nk from the cache, or (exx_apply_to) the trial vector phi_nk transformed now
            const double2* un_base = c->u_dev + (size_t)k * nb * Ng;
            int un_idx = n;
            if (phi) {
                if (!c->uphi1_dev)
                    if ((rc = dev_alloc(c, &c->uphi1_dev, (size_t)Ng))) return rc;
                if ((rc = launch_scatter(c, k, phi + c->off[k] / nb * na + (int64_t)n * c->npw[k], 1, c->uphi1_dev))) return rc;
                if ((rc = launch_fft3d_generic(c, c->uphi1_dev, 1, +1))) return rc;
                un_base = c->uphi1_dev;
                un_idx = 0;
            }
            for (int q = 0; q < nk; q++) {
                const double* ktab = c->ktab_dev + (size_t)c->ktab_of[(size_t)k * nk + q] * Ng;
                const double2* uq = c->u_dev + (size_t)q * nb * Ng;
                MTile mt;
                mt.tm = 0;
                for (int m = 0; m <= nb; m++) {
                    if (m < nb && occ[q * nb + m] != 0.0) {
                        mt.m_idx[mt.tm] = m;
                        mt.wf[mt.tm] = c->kw[q] * occ[q * nb + m];
                        mt.tm++;
                    }
                    if (mt.tm == tm_max || (m == nb && mt.tm > 0)) {
                        if ((rc = launch_codensity_tile(c, un_base, un_idx, 1, uq, mt, c->work_dev))) return rc;
                        if ((rc = launch_fft3d_generic(c, c->work_dev, mt.tm, -1))) return rc;
                        if ((rc = launch_kmul(c, ktab, c->work_dev, mt.tm))) return rc;
                        if ((rc = launch_fft3d_generic(c, c->work_dev, mt.tm, +1))) return rc;
                        if ((rc = launch_accumulate_tile(c, uq, mt, 1, c->work_dev, c->acc_dev))) return rc;
                        c->pairs_executed += mt.tm;
                        c->pairs_ordered += mt.tm;
                        mt.tm = 0;
                    }
                }
            }
            // S7: forward transform of the accumulator, gather onto sphere(k) (the 1/(Omega Ng^2) is inside K')
            if ((rc = launch_fft3d_generic(c, c->acc_dev, 1, -1))) return rc;
            if ((rc = launch_gather(c, k, c->acc_dev, 1, out_row))) return rc;
        }
    return EXX_OK;
}

static void options_to_inner(const exx_ctx* c, exx_ctx* in) {
    in->opt_path = c->opt_path == 1 ? 1 : 0;
    in->opt_tile_n = c->opt_tile_n;
    in->opt_tile_m = c->opt_tile_m;
    in->opt_profile = c->opt_profile;
    in->opt_symmetry = c->opt_symmetry;
    in->opt_precision = c->opt_precision;
    in->opt_keep_u = c->opt_keep_u;
    in->opt_dual = c->opt_dual;
    in->opt_prune_rows = c->opt_prune_rows;
    in->opt_shard_count = c->opt_shard_count;
    in->opt_shard_rank = c->opt_shard_rank;
}
static void counters_from_inner(exx_ctx* c, const exx_ctx* in, int rc) {
    c->launches = in->launches;
    c->pairs_ordered = in->pairs_ordered;
    c->pairs_executed = in->pairs_executed;
    c->path_used = in->path_used;
    c->tile_n_used = in->tile_n_used;
    c->tile_m_used = in->tile_m_used;
    c->symmetry_used = in->symmetry_used;
    c->precision_used = in->precision_used;
    c->pruned_used = 1;
    c->last_pruned = 1;
    if (rc) c->last_error = in->last_error;
}

static int apply_impl(exx_ctx* c, const double2* psi, const double* occ, double2* out, const double2* phi = nullptr, int nphi = 0) {
    reset_counters(c);
    if (c->opt_shard_rank >= c->opt_shard_count) return EXX_ERR_BAD_ARG;
    // (an inner grid that was taken only because it has fused kernels is pointless when the generic kernels are asked for)
    if (c->inner && c->opt_prune && !(c->inner_larger && c->opt_path == 1)) {
        // compact work grid: same spheres, same psi/out layout, every product alias-free on both grids
        exx_ctx* in = c->inner;
        options_to_inner(c, in);
        int rc = apply_impl(in, psi, occ, out, phi, nphi);
        counters_from_inner(c, in, rc);
        return rc;
    }
    c->last_pruned = 0;
    {
        int rc = ensure_big(c);
        if (rc) return rc;
    }
    bool use_fused = fused_supported(c) && c->opt_path != 1;
    if (use_fused) return fused_apply(c, occ, psi, out, phi, nphi);
    return apply_generic(c, psi, occ, out, phi, nphi);
}

int exx_apply(exx_ctx* c, const double* psi_dev, const double* occ_host, double* out_dev) {
    if (!c || !psi_dev || !occ_host || !out_dev) return EXX_ERR_NULL;
    int rc = check_occ(c, occ_host);
    if (rc) return rc;
    const char *p = (const char*)psi_dev, *o = (const char*)out_dev;
    size_t bytes = sizeof(double2) * (size_t)c->off[c->nk];
    if (p < o + bytes && o < p + bytes) return EXX_ERR_ALIAS;
    return apply_impl(c, (const double2*)psi_dev, occ_host, (double2*)out_dev);
}

int exx_apply_to(exx_ctx* c, const double* psi_dev, const double* occ_host, const double* phi_dev, int nphi, double* out_dev) {
    if (!c || !psi_dev || !occ_host || !phi_dev || !out_dev) return EXX_ERR_NULL;
    if (nphi < 1 || nphi > 65536) return EXX_ERR_BAD_ARG;
    int rc = check_occ(c, occ_host);
    if (rc) return rc;
    const char *p = (const char*)psi_dev, *f = (const char*)phi_dev, *o = (const char*)out_dev;
    const size_t bytes_psi = sizeof(double2) * (size_t)c->off[c->nk], bytes_phi = bytes_psi / c->nb * nphi;
    if ((p < o + bytes_phi && o < p + bytes_psi) || (f < o + bytes_phi && o < f + bytes_phi)) return EXX_ERR_ALIAS;
    return apply_impl(c, (const double2*)psi_dev, occ_host, (double2*)out_dev, (const double2*)phi_dev, nphi);
}

static int energy_impl(exx_ctx* c, const double2* psi, const double* occ, const double2* vx, double* ex, double* per_band) {
    int nbt = c->nk * c->nb;
    double* h = c->host_pinned;
    for (int k = 0; k < c->nk; k++)
        for (int n = 0; n < c->nb; n++) h[k * c->nb + n] = 0.5 * c->kw[k] * occ[k * c->nb + n];
    EXX_CUDA(c, cudaMemcpyAsync(c->occw_dev, h, sizeof(double) * nbt, cudaMemcpyHostToDevice, c->stream));
    int rc = launch_energy(c, psi, vx);
    if (rc) return rc;
    double* res = h + nbt;
    EXX_CUDA(c, cudaMemcpyAsync(res, c->band_e_dev, sizeof(double) * (nbt + 1), cudaMemcpyDeviceToHost, c->stream));
    EXX_CUDA(c, cudaStreamSynchronize(c->stream));
    *ex = res[nbt];
    if (per_band) memcpy(per_band, res, sizeof(double) * nbt);
    return EXX_OK;
}

// E_x without V_x psi: the pair-density route (E2), where the fused kernels run.  Same recursion onto the compact
// work grid as apply_impl.  EXX_E2_UNAVAILABLE: this context would run the generic kernels; the caller falls back to (E1).
static const int EXX_E2_UNAVAILABLE = 1;
static int energy_pairs_run(exx_ctx* c, const double2* psi, const double* occ, double* band_e2_host) {
    reset_counters(c);
    if (c->opt_shard_rank >= c->opt_shard_count) return EXX_ERR_BAD_ARG;
    if (c->inner && c->opt_prune && !(c->inner_larger && c->opt_path == 1)) {
        exx_ctx* in = c->inner;
        options_to_inner(c, in);
        int rc = energy_pairs_run(in, psi, occ, band_e2_host);
        if (rc != EXX_E2_UNAVAILABLE) counters_from_inner(c, in, rc);
        return rc;
    }
    if (!(fused_supported(c) && c->opt_path != 1)) return EXX_E2_UNAVAILABLE;
    c->last_pruned = 0;
    int rc = ensure_big(c);
    if (rc) return rc;
    return fused_energy(c, occ, psi, band_e2_host);
}
static int energy_pairs_impl(exx_ctx* c, const double2* psi, const double* occ, double* ex, double* per_band) {
    const int nbt = c->nk * c->nb;
    double* h = c->host_pinned;
    int rc = energy_pairs_run(c, psi, occ, h);
    if (rc) return rc;
    // fixed order: bands ascending within k-points ascending
    double e = 0.0;
    for (int i = 0; i < nbt; i++) {
        h[i] *= -0.5;
        e += h[i];
    }
    *ex = e;
    if (per_band) memcpy(per_band, h, sizeof(double) * nbt);
    return EXX_OK;
}

int exx_energy(exx_ctx* c, const double* psi_dev, const double* occ_host, const double* vxpsi_dev_or_null, double* ex_host,
               double* per_band_host_or_null) {
    if (!c || !psi_dev || !occ_host || !ex_host) return EXX_ERR_NULL;
    int rc = check_occ(c, occ_host);
    if (rc) return rc;
    const double2* vx = (const double2*)vxpsi_dev_or_null;
    c->energy_route_used = 1;
    if (!vx) {
        if (c->opt_energy_route == 0) {
            rc = energy_pairs_impl(c, (const double2*)psi_dev, occ_host, ex_host, per_band_host_or_null);
            if (rc != EXX_E2_UNAVAILABLE) {
                if (rc == EXX_OK) c->energy_route_used = 2;
                return rc;
            }
        }
        if ((rc = apply_impl(c, (const double2*)psi_dev, occ_host, c->vx_dev))) return rc;
        vx = c->vx_dev;
    }
    return energy_impl(c, (const double2*)psi_dev, occ_host, vx, ex_host, per_band_host_or_null);
}

int exx_shard_plan(int nk, int nbands, const double* occ_host, int symmetry, int tile, int nshards, int64_t* pairs_out, int64_t* passes_out) {
    if (!occ_host) return EXX_ERR_NULL;
    if (nk < 1 || nbands < 1 || nshards < 1 || tile < 0 || tile > TMAX) return EXX_ERR_BAD_ARG;
    for (int i = 0; i < nk * nbands; i++)
        if (!(occ_host[i] >= 0.0) || !std::isfinite(occ_host[i])) return EXX_ERR_BAD_OCC;
    const int t = std::min(tile ? tile : (nshards > 1 ? std::min(EXX_DEFAULT_TILE, EXX_SHARD_TILE) : EXX_DEFAULT_TILE), nbands);
    std::vector<PairBlock> blocks;
    plan_blocks(nk, nbands, occ_host, symmetry != 0, t, t, nshards, blocks);
    for (int s = 0; s < nshards; s++) {
        if (pairs_out) pairs_out[s] = 0;
        if (passes_out) passes_out[s] = 0;
    }
    for (const PairBlock& b : blocks) {
        if (pairs_out) pairs_out[b.shard] += b.npairs;
        if (passes_out) passes_out[b.shard] += b.cost();
    }
    return EXX_OK;
}

int exx_subspace(exx_ctx* c, int ik, const double* psi_dev, const double* vxpsi_dev, double* m_dev) {
    if (!c || !psi_dev || !vxpsi_dev || !m_dev) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_ERR_BAD_ARG;
    return launch_subspace(c, ik, (const double2*)psi_dev, (const double2*)vxpsi_dev, (double2*)m_dev);
}

int exx_subspace_block(exx_ctx* c, int ik, const double* phi_dev, const double* vphi_dev, int nphi, double* m_dev) {
    if (!c || !phi_dev || !vphi_dev || !m_dev) return EXX_ERR_NULL;
    if (ik < 0 || ik >= c->nk || nphi < 1 || nphi > 65536) return EXX_ERR_BAD_ARG;
    return launch_subspace(c, ik, (const double2*)phi_dev, (const double2*)vphi_dev, (double2*)m_dev, nphi);
}

int exx_apply_host(exx_ctx* c, const double* psi_host, const double* occ_host, double* out_host, double* ex_host_or_null) {
    if (!c || !psi_host || !occ_host || !out_host) return EXX_ERR_NULL;
    int rc = check_occ(c, occ_host);
    if (rc) return rc;
    size_t ncoef = (size_t)c->off[c->nk];
    if (!c->psi_stage_dev)
        if ((rc = dev_alloc(c, &c->psi_stage_dev, ncoef))) return rc;
    EXX_CUDA(c, cudaMemcpyAsync(c->psi_stage_dev, psi_host, sizeof(double2) * ncoef, cudaMemcpyHostToDevice, c->stream));
    if ((rc = apply_impl(c, c->psi_stage_dev, occ_host, c->vx_dev))) return rc;
    EXX_CUDA(c, cudaMemcpyAsync(out_host, c->vx_dev, sizeof(double2) * ncoef, cudaMemcpyDeviceToHost, c->stream));
    if (ex_host_or_null) return energy_impl(c, c->psi_stage_dev, occ_host, c->vx_dev, ex_host_or_null, nullptr);
    EXX_CUDA(c, cudaStreamSynchronize(c->stream));
    return EXX_OK;
}

}  // extern "C"
