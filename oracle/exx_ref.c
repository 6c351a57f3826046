/*
 * exx_ref.c — the ORACLE: a plain, slow, obviously-correct CPU implementation of the plane-wave
 * Fock-exchange operator V_x|psi_nk> and the exchange energy E_x.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call anything in oracle/.  It shares no code,
 * header, table generator or helper with the CUDA library (paper_1111_0716_b200/csrc); neither imports
 * the other.
 *
 * What it follows (P:Lnn = /root/reference/PAPER.md line nn; S8c = SURVEY.md section 8(c), definition (D)):
 *   - P:L127-130, Eq. 2: E_x = -(e^2/2) sum_{kn,qm} f_kn f_qm  iint phi*_kn(r) phi*_qm(r') phi_kn(r') phi_qm(r)/|r-r'|
 *     (the paper prints the "magnitude"; sign and Hartree units per DESIGN.md reading A2).
 *   - P:L107: "FOCK_ACC applies the Fock exchange operator" -> V_x psi_nk.
 *   - P:L127: four nested loops, k and q over k-points, n and m over bands.
 *   - P:L119: scatter/gather "used to express cutoffs" -> the sphere <-> box index map.
 * On the discrete FFT grid Eq. 2 becomes definition (D), written out here literally:
 *
 *   u_nk(r_j)       = sum_{g in sphere(k)} c_nk(g) exp(+2 pi i sum_i g_i j_i / N_i)
 *   rho~_{nk,mq}(g) = (1/Ng) sum_j conj(u_mq(r_j)) u_nk(r_j) exp(-2 pi i sum_i g_i j_i / N_i)
 *   v_{nk,mq}(r_j)  = (1/Omega) sum_g K(|k-q+G(g)|) rho~_{nk,mq}(g) exp(+2 pi i sum_i g_i j_i / N_i)
 *   (V_x u)_nk(r_j) = - sum_q w_q sum_m f_mq u_mq(r_j) v_{nk,mq}(r_j)
 *   (V_x c)_nk(g)   = (1/Ng) sum_j (V_x u)_nk(r_j) exp(-2 pi i sum_i g_i j_i / N_i),   g in sphere(k)
 *   E_x (E1)        = 1/2 sum_k w_k sum_n f_nk Re sum_g conj(c_nk(g)) (V_x c)_nk(g)
 *   E_x (E2)        = -1/2 (1/Omega) sum_{k,q} w_k w_q sum_{n,m} f_nk f_mq sum_g K(|k-q+G|) |rho~_{nk,mq}(g)|^2
 *   K bare: 4 pi/Q^2, 0 where Q = 0;   K HSE: (4 pi/Q^2)(1 - exp(-Q^2/(4 mu^2))), pi/mu^2 where Q = 0.
 *
 * The sums over j and g are evaluated with this file's own recursive mixed-radix FFT (exact same sums, fewer
 * operations); exx_ref_apply_direct evaluates (D) with no FFT at all (cyclic sums in reciprocal space), and
 * exx_ref_dft1d is the O(N^2) definition the FFT is pinned to.  No blocking, fusion or reordering beyond that.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed form for single-plane-wave bands, Hermiticity, global-phase
 * covariance, unitary-mix covariance, E1 == E2, E_x <= 0, FFT path == no-FFT path, supercell == k-point sampling,
 * HSE limits, brute-force index maps, FFT == naive DFT, Parseval.  Every function here has a pin; none is
 * "parity unpinned".
 *
 * Precision: IEEE fp64 throughout, compiled with -ffp-contract=off (no FMA contraction).
 * Layout: complex numbers are (re,im) interleaved doubles.  psi/out: k-major, then band, then sphere index:
 *   element (k,n,ig) at offset(k) + n*Npw(k) + ig, offset(k) = Nb * sum_{k'<k} Npw(k').
 * Boxes are C-order: index (j1*N2 + j2)*N3 + j3.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define EXX_REF_OK 0
#define EXX_REF_ERR_NULL -1
#define EXX_REF_ERR_BAD_GRID -2
#define EXX_REF_ERR_BAD_LATTICE -3
#define EXX_REF_ERR_BAD_CUTOFF -4
#define EXX_REF_ERR_BAD_KERNEL -5
#define EXX_REF_ERR_BAD_OCC -6
#define EXX_REF_ERR_ALLOC -7
#define EXX_REF_ERR_BAD_ARG -8

typedef struct exx_ref_ctx {
    int N[3];
    int64_t Ng;
    double A[9];     /* lattice rows a_i (bohr) */
    double B[9];     /* reciprocal rows b_i, a_i . b_j = 2 pi delta_ij */
    double omega;    /* |det A| */
    int nk, nb;
    double *kfrac;   /* nk*3 fractional reciprocal coordinates kappa */
    double *kw;      /* nk weights */
    double ecut;
    int kind;        /* 0 bare, 1 HSE short range */
    double mu, scale;
    int *npw;        /* nk */
    int64_t *off;    /* nk+1, complex elements */
    int32_t **map;   /* nk arrays of npw[k] box indices, ascending */
} exx_ref_ctx;

/* ------------------------------------------------------------------------------------------------ */
/* frequency folding (reading A9): g = j if 2j < N else j - N  (numpy fftfreq convention)   */
static int fold(int j, int n) { return (2 * j < n) ? j : j - n; }

/* |t . B|^2 for fractional vector t (row vector times rows b_i), evaluated in the fixed order of reading A11 */
static double norm2_frac(const double B[9], const double t[3]) {
    double s = 0.0;
    for (int c = 0; c < 3; c++) {
        double x = (t[0] * B[0 * 3 + c] + t[1] * B[1 * 3 + c]) + t[2] * B[2 * 3 + c];
        s = s + x * x;
    }
    return s;
}

/* Coulomb kernel K(Q) for Q = t.B with t = kappa_k - kappa_q + g (fractional). "Q = 0" is decided on t exactly. */
static double coulomb_kernel(const exx_ref_ctx *c, const double t[3]) {
    const double pi = 3.14159265358979323846264338327950288;
    int zero = (t[0] == 0.0 && t[1] == 0.0 && t[2] == 0.0);
    if (c->kind == 0) {
        if (zero) return 0.0;
        return c->scale * (4.0 * pi / norm2_frac(c->B, t));
    } else {
        if (zero) return c->scale * (pi / (c->mu * c->mu));
        double q2 = norm2_frac(c->B, t);
        double x = q2 / (4.0 * c->mu * c->mu);
        return c->scale * ((4.0 * pi / q2) * (-expm1(-x)));
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* 1-D transforms.  sign = -1: X[k] = sum_j x[j] exp(-2 pi i j k/n) (forward); sign = +1: inverse, unnormalised. */

/* exp(sign * 2 pi i * j / n), j reduced mod n, angle evaluated in long double */
static cplx root_of_unity(int64_t j, int n, int sign) {
    const long double twopi = 6.283185307179586476925286766559005768L;
    j %= n;
    if (j < 0) j += n;
    long double a = twopi * (long double)j / (long double)n;
    return (double)cosl(a) + I * (double)(sign * sinl(a));
}

/* the definition, O(n^2) */
void exx_ref_dft1d(int n, int sign, const double *in, double *out) {
    const cplx *x = (const cplx *)in;
    cplx *X = (cplx *)out;
    for (int k = 0; k < n; k++) {
        cplx s = 0.0;
        for (int j = 0; j < n; j++) s += x[j] * root_of_unity((int64_t)j * k, n, sign);
        X[k] = s;
    }
}

static int smallest_factor(int n) {
    for (int p = 2; (int64_t)p * p <= n; p++)
        if (n % p == 0) return p;
    return n;
}

/* recursive decimation in time, any n: split by the smallest prime factor p of n into p sub-transforms of
 * length m = n/p over the residue classes j = r (mod p), then X[k + q m] = sum_r W_n^{(k+qm) r} Y_r[k].
 * tw[j] = exp(sign 2 pi i j / n0) for the top-level n0; a level of length n uses stride n0/n into it. */
static void fft_rec(int n, const cplx *in, int istride, cplx *out, const cplx *tw, int n0, cplx *scratch) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_factor(n);
    int m = n / p;
    for (int r = 0; r < p; r++) fft_rec(m, in + (int64_t)r * istride, istride * p, out + (int64_t)r * m, tw, n0, scratch + n);
    int tws = n0 / n;
    for (int k = 0; k < m; k++) {
        for (int q = 0; q < p; q++) {
            int kk = k + q * m;
            cplx s = 0.0;
            for (int r = 0; r < p; r++) s += out[r * m + k] * tw[(((int64_t)kk * r) % n) * tws];
            scratch[kk] = s;
        }
    }
    memcpy(out, scratch, sizeof(cplx) * (size_t)n);
}

static int fft_depth_scratch(int n) { /* total scratch needed by fft_rec: n + n/p + ... */
    int s = 0;
    while (n > 1) { s += n; n /= smallest_factor(n); }
    return s + 1;
}

void exx_ref_fft1d(int n, int sign, const double *in, double *out) {
    cplx *tw = malloc(sizeof(cplx) * (size_t)n);
    cplx *scratch = malloc(sizeof(cplx) * (size_t)fft_depth_scratch(n));
    for (int j = 0; j < n; j++) tw[j] = root_of_unity(j, n, sign);
    fft_rec(n, (const cplx *)in, 1, (cplx *)out, tw, n, scratch);
    free(tw);
    free(scratch);
}

/* 3-D transform of a C-order box, in place: 1-D transforms along axis 2, then 1, then 0. */
static void fft3d(const int N[3], int sign, cplx *box) {
    int nmax = N[0] > N[1] ? N[0] : N[1];
    if (N[2] > nmax) nmax = N[2];
    cplx *pin = malloc(sizeof(cplx) * (size_t)nmax);
    cplx *pout = malloc(sizeof(cplx) * (size_t)nmax);
    cplx *scratch = malloc(sizeof(cplx) * (size_t)(2 * nmax + 64));
    for (int ax = 2; ax >= 0; ax--) {
        int n = N[ax];
        cplx *tw = malloc(sizeof(cplx) * (size_t)n);
        for (int j = 0; j < n; j++) tw[j] = root_of_unity(j, n, sign);
        int64_t stride = (ax == 2) ? 1 : (ax == 1 ? N[2] : (int64_t)N[1] * N[2]);
        int64_t Ng = (int64_t)N[0] * N[1] * N[2];
        for (int64_t base = 0; base < Ng; base++) {
            /* base runs over the box points whose coordinate along ax is 0 */
            int64_t j_ax = (base / stride) % n;
            if (j_ax != 0) continue;
            for (int j = 0; j < n; j++) pin[j] = box[base + j * stride];
            fft_rec(n, pin, 1, pout, tw, n, scratch);
            for (int j = 0; j < n; j++) box[base + j * stride] = pout[j];
        }
        free(tw);
    }
    free(pin);
    free(pout);
    free(scratch);
}

void exx_ref_fft3d(const int N[3], int sign, double *box) { fft3d(N, sign, (cplx *)box); }

/* ------------------------------------------------------------------------------------------------ */
static int valid_grid_len(int n) { return n >= 1; } /* the oracle's FFT handles any length */

int exx_ref_destroy(exx_ref_ctx *c) {
    if (!c) return EXX_REF_ERR_NULL;
    if (c->map)
        for (int k = 0; k < c->nk; k++) free(c->map[k]);
    free(c->map);
    free(c->npw);
    free(c->off);
    free(c->kfrac);
    free(c->kw);
    free(c);
    return EXX_REF_OK;
}

int exx_ref_create(exx_ref_ctx **out, const int grid[3], const double lattice[9], int nk, const double *kfrac,
                   const double *kweight, double ecut, int kind, double mu, double scale, int nbands) {
    if (!out || !grid || !lattice || !kfrac || !kweight) return EXX_REF_ERR_NULL;
    if (nk < 1 || nbands < 1) return EXX_REF_ERR_BAD_ARG;
    for (int i = 0; i < 3; i++)
        if (!valid_grid_len(grid[i])) return EXX_REF_ERR_BAD_GRID;
    if (!(ecut > 0.0) || !isfinite(ecut)) return EXX_REF_ERR_BAD_CUTOFF;
    if (kind != 0 && kind != 1) return EXX_REF_ERR_BAD_KERNEL;
    if (kind == 1 && !(mu > 0.0)) return EXX_REF_ERR_BAD_KERNEL;
    if (!isfinite(scale)) return EXX_REF_ERR_BAD_KERNEL;
    const double *a = lattice;
    double det = a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) + a[2] * (a[3] * a[7] - a[4] * a[6]);
    if (!isfinite(det) || det == 0.0) return EXX_REF_ERR_BAD_LATTICE;

    exx_ref_ctx *c = calloc(1, sizeof(*c));
    if (!c) return EXX_REF_ERR_ALLOC;
    memcpy(c->N, grid, sizeof(int) * 3);
    c->Ng = (int64_t)grid[0] * grid[1] * grid[2];
    memcpy(c->A, lattice, sizeof(double) * 9);
    c->omega = fabs(det);
    /* reciprocal rows: b_i = 2 pi (a_j x a_k)/det, cyclic */
    const double twopi = 6.283185307179586476925286766559;
    for (int i = 0; i < 3; i++) {
        const double *p = a + 3 * ((i + 1) % 3), *q = a + 3 * ((i + 2) % 3);
        c->B[3 * i + 0] = twopi * (p[1] * q[2] - p[2] * q[1]) / det;
        c->B[3 * i + 1] = twopi * (p[2] * q[0] - p[0] * q[2]) / det;
        c->B[3 * i + 2] = twopi * (p[0] * q[1] - p[1] * q[0]) / det;
    }
    c->nk = nk;
    c->nb = nbands;
    c->ecut = ecut;
    c->kind = kind;
    c->mu = mu;
    c->scale = scale;
    c->kfrac = malloc(sizeof(double) * 3 * (size_t)nk);
    c->kw = malloc(sizeof(double) * (size_t)nk);
    c->npw = calloc((size_t)nk, sizeof(int));
    c->off = calloc((size_t)nk + 1, sizeof(int64_t));
    c->map = calloc((size_t)nk, sizeof(int32_t *));
    if (!c->kfrac || !c->kw || !c->npw || !c->off || !c->map) { exx_ref_destroy(c); return EXX_REF_ERR_ALLOC; }
    memcpy(c->kfrac, kfrac, sizeof(double) * 3 * (size_t)nk);
    memcpy(c->kw, kweight, sizeof(double) * (size_t)nk);

    /* sphere(k) = { g : |k+G|^2/2 < ecut }, strict, listed by ascending C-order box index (reading A11) */
    for (int k = 0; k < nk; k++) {
        int32_t *m = malloc(sizeof(int32_t) * (size_t)c->Ng);
        if (!m) { exx_ref_destroy(c); return EXX_REF_ERR_ALLOC; }
        int cnt = 0;
        for (int j1 = 0; j1 < grid[0]; j1++)
            for (int j2 = 0; j2 < grid[1]; j2++)
                for (int j3 = 0; j3 < grid[2]; j3++) {
                    double t[3] = {(double)fold(j1, grid[0]) + kfrac[3 * k + 0], (double)fold(j2, grid[1]) + kfrac[3 * k + 1],
                                   (double)fold(j3, grid[2]) + kfrac[3 * k + 2]};
                    double e = 0.5 * norm2_frac(c->B, t);
                    if (e < ecut) m[cnt++] = (int32_t)(((int64_t)j1 * grid[1] + j2) * grid[2] + j3);
                }
        c->npw[k] = cnt;
        c->map[k] = realloc(m, sizeof(int32_t) * (size_t)(cnt > 0 ? cnt : 1));
        c->off[k + 1] = c->off[k] + (int64_t)nbands * cnt;
    }
    *out = c;
    return EXX_REF_OK;
}

int exx_ref_npw(const exx_ref_ctx *c, int ik, int *npw) {
    if (!c || !npw) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_REF_ERR_BAD_ARG;
    *npw = c->npw[ik];
    return EXX_REF_OK;
}
int exx_ref_index_map(const exx_ref_ctx *c, int ik, int32_t *host_out) {
    if (!c || !host_out) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_REF_ERR_BAD_ARG;
    memcpy(host_out, c->map[ik], sizeof(int32_t) * (size_t)c->npw[ik]);
    return EXX_REF_OK;
}
int exx_ref_psi_offset(const exx_ref_ctx *c, int ik, int64_t *complex_elems) {
    if (!c || !complex_elems) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik > c->nk) return EXX_REF_ERR_BAD_ARG;
    *complex_elems = c->off[ik];
    return EXX_REF_OK;
}
double exx_ref_omega(const exx_ref_ctx *c) { return c ? c->omega : 0.0; }
int exx_ref_recip(const exx_ref_ctx *c, double B[9]) {
    if (!c || !B) return EXX_REF_ERR_NULL;
    memcpy(B, c->B, sizeof(double) * 9);
    return EXX_REF_OK;
}

/* K(|k-q+G(g)|) for every g of the box (C-order, folded frequencies; reading A8: whole box) */
int exx_ref_kernel_table(const exx_ref_ctx *c, int ik, int iq, double *K) {
    if (!c || !K) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik >= c->nk || iq < 0 || iq >= c->nk) return EXX_REF_ERR_BAD_ARG;
    const int *N = c->N;
    double dk[3];
    for (int i = 0; i < 3; i++) dk[i] = c->kfrac[3 * ik + i] - c->kfrac[3 * iq + i];
    for (int j1 = 0; j1 < N[0]; j1++)
        for (int j2 = 0; j2 < N[1]; j2++)
            for (int j3 = 0; j3 < N[2]; j3++) {
                double t[3] = {dk[0] + (double)fold(j1, N[0]), dk[1] + (double)fold(j2, N[1]), dk[2] + (double)fold(j3, N[2])};
                K[((int64_t)j1 * N[1] + j2) * N[2] + j3] = coulomb_kernel(c, t);
            }
    return EXX_REF_OK;
}

/* u_nk(r_j) = sum_{g in sphere(k)} c_nk(g) exp(+i G.r_j): scatter, then unnormalised inverse transform */
static void to_real(const exx_ref_ctx *c, int ik, const cplx *coef, cplx *box) {
    memset(box, 0, sizeof(cplx) * (size_t)c->Ng);
    for (int ig = 0; ig < c->npw[ik]; ig++) box[c->map[ik][ig]] = coef[ig];
    fft3d(c->N, +1, box);
}
int exx_ref_to_real(const exx_ref_ctx *c, int ik, const double *coef, double *box) {
    if (!c || !coef || !box) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_REF_ERR_BAD_ARG;
    to_real(c, ik, (const cplx *)coef, (cplx *)box);
    return EXX_REF_OK;
}

static int check_occ(const exx_ref_ctx *c, const double *occ) {
    for (int i = 0; i < c->nk * c->nb; i++)
        if (!(occ[i] >= 0.0) || !isfinite(occ[i])) return EXX_REF_ERR_BAD_OCC;
    return EXX_REF_OK;
}

/* all u_mq(r) with f_mq != 0, plus optionally all (needed as n); returns array of nk*nb pointers (NULL if skipped) */
static cplx **all_real(const exx_ref_ctx *c, const cplx *psi, const double *occ, const unsigned char *need) {
    cplx **u = calloc((size_t)c->nk * c->nb, sizeof(cplx *));
    if (!u) return NULL;
    int fail = 0;
#pragma omp parallel for schedule(dynamic)
    for (int i = 0; i < c->nk * c->nb; i++) {
        int k = i / c->nb, n = i % c->nb;
        if (occ[i] == 0.0 && !(need && need[i])) continue;
        u[i] = malloc(sizeof(cplx) * (size_t)c->Ng);
        if (!u[i]) { fail = 1; continue; }
        to_real(c, k, psi + c->off[k] + (int64_t)n * c->npw[k], u[i]);
    }
    if (fail) {
        for (int i = 0; i < c->nk * c->nb; i++) free(u[i]);
        free(u);
        return NULL;
    }
    return u;
}
static void free_real(const exx_ref_ctx *c, cplx **u) {
    if (!u) return;
    for (int i = 0; i < c->nk * c->nb; i++) free(u[i]);
    free(u);
}

static int nthreads_max(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int exx_ref_num_threads(void) { return nthreads_max(); }

/* Rows (k,n) of V_x c by definition (D).  rows = nrows pairs (ik, n); out_rows: for row r, npw(ik_r) complex
 * numbers, concatenated in the order given.  OpenMP over the pairs (q,m) of a row; per-thread partial sums are
 * added in thread order, so the result is deterministic for a given thread count. */
int exx_ref_apply_rows(const exx_ref_ctx *c, const double *psi_, const double *occ, int nrows, const int *rows, double *out_rows_) {
    if (!c || !psi_ || !occ || !rows || !out_rows_) return EXX_REF_ERR_NULL;
    int rc = check_occ(c, occ);
    if (rc) return rc;
    const cplx *psi = (const cplx *)psi_;
    cplx *out_rows = (cplx *)out_rows_;
    const int64_t Ng = c->Ng;
    unsigned char *need = calloc((size_t)c->nk * c->nb, 1);
    if (!need) return EXX_REF_ERR_ALLOC;
    for (int r = 0; r < nrows; r++) {
        int k = rows[2 * r], n = rows[2 * r + 1];
        if (k < 0 || k >= c->nk || n < 0 || n >= c->nb) { free(need); return EXX_REF_ERR_BAD_ARG; }
        need[k * c->nb + n] = 1;
    }
    cplx **u = all_real(c, psi, occ, need);
    free(need);
    if (!u) return EXX_REF_ERR_ALLOC;

    int nt = nthreads_max();
    cplx *acc_t = malloc(sizeof(cplx) * (size_t)Ng * nt);
    cplx *work_t = malloc(sizeof(cplx) * (size_t)Ng * nt);
    double *K = malloc(sizeof(double) * (size_t)Ng * c->nk);
    if (!acc_t || !work_t || !K) { free(acc_t); free(work_t); free(K); free_real(c, u); return EXX_REF_ERR_ALLOC; }

    int64_t opos = 0;
    for (int r = 0; r < nrows; r++) {
        int k = rows[2 * r], n = rows[2 * r + 1];
        const cplx *un = u[k * c->nb + n];
        for (int q = 0; q < c->nk; q++) exx_ref_kernel_table(c, k, q, K + (int64_t)q * Ng);
        memset(acc_t, 0, sizeof(cplx) * (size_t)Ng * nt);
#pragma omp parallel num_threads(nt)
        {
#ifdef _OPENMP
            int t = omp_get_thread_num();
#else
            int t = 0;
#endif
            cplx *acc = acc_t + (int64_t)t * Ng, *w = work_t + (int64_t)t * Ng;
#pragma omp for schedule(static)
            for (int qm = 0; qm < c->nk * c->nb; qm++) {
                int q = qm / c->nb;
                double f = occ[qm];
                if (f == 0.0) continue; /* reading A16: f = 0 bands contribute exactly 0 */
                const cplx *um = u[qm];
                const double *Kq = K + (int64_t)q * Ng;
                for (int64_t j = 0; j < Ng; j++) w[j] = conj(um[j]) * un[j];          /* co-density on the grid     */
                fft3d(c->N, -1, w);                                                   /* sum_j ... exp(-i G.r_j)    */
                for (int64_t g = 0; g < Ng; g++) w[g] = (Kq[g] * (w[g] / (double)Ng)) / c->omega; /* K rho~ / Omega */
                fft3d(c->N, +1, w);                                                   /* v(r_j)                     */
                double wf = c->kw[q] * f;
                for (int64_t j = 0; j < Ng; j++) acc[j] -= wf * (um[j] * w[j]);
            }
        }
        for (int t = 1; t < nt; t++)
            for (int64_t j = 0; j < Ng; j++) acc_t[j] += acc_t[(int64_t)t * Ng + j];
        fft3d(c->N, -1, acc_t);
        for (int ig = 0; ig < c->npw[k]; ig++) out_rows[opos + ig] = acc_t[c->map[k][ig]] / (double)Ng;
        opos += c->npw[k];
    }
    free(acc_t);
    free(work_t);
    free(K);
    free_real(c, u);
    return EXX_REF_OK;
}

/* V_x c for every (k,n): out has the layout of psi. */
int exx_ref_apply(const exx_ref_ctx *c, const double *psi, const double *occ, double *out) {
    if (!c || !psi || !occ || !out) return EXX_REF_ERR_NULL;
    int nrows = c->nk * c->nb;
    int *rows = malloc(sizeof(int) * 2 * (size_t)nrows);
    if (!rows) return EXX_REF_ERR_ALLOC;
    for (int i = 0; i < nrows; i++) { rows[2 * i] = i / c->nb; rows[2 * i + 1] = i % c->nb; }
    int rc = exx_ref_apply_rows(c, psi, occ, nrows, rows, out); /* rows in (k,n) order == psi layout */
    free(rows);
    return rc;
}

/* The operator of (D), built from the orbitals psi and their occupations, applied to OTHER vectors phi (same layout as psi:
 * nb vectors per k-point on sphere(k)) -- what FOCK_ACC does inside an iterative eigensolver, where it acts on the trial
 * wavefunctions while the occupied orbitals define the operator (blocks of NSIM bands):
 *   t_ik(r_j)         = sum_{g in sphere(k)} phi_ik(g) exp(+2 pi i sum g_i j_i / N_i)
 *   rho~(g)           = (1/Ng) sum_j conj(u_mq(r_j)) t_ik(r_j) exp(-...)
 *   v(r_j)            = (1/Omega) sum_g K(|k-q+G|) rho~(g) exp(+...)
 *   (V_x t)_ik(r_j)   = - sum_q w_q sum_m f_mq u_mq(r_j) v(r_j),      out_ik(g) = (1/Ng) sum_j (V_x t)_ik(r_j) exp(-...), g in sphere(k)
 * i.e. (D) with u_nk replaced by t_ik in the co-density only.  phi and out hold nphi vectors per k-point (any nphi >= 1), packed like
 * psi: element (k,i,ig) at nphi * sum_{k'<k} npw(k') + i*npw(k) + ig.  Plain loops: rows in parallel, the (q,m) sum of a row serial in
 * loop order.  Pins (tests/test_oracle_exchange.py): closed-form eigenvalue for plane waves, phi = psi gives exx_ref_apply,
 * Hermiticity and negativity of <phi_i|V_x phi_j>, linearity in phi. */
int exx_ref_apply_to(const exx_ref_ctx *c, const double *psi_, const double *occ, const double *phi_, int nphi, double *out_) {
    if (!c || !psi_ || !occ || !phi_ || !out_) return EXX_REF_ERR_NULL;
    if (nphi < 1) return EXX_REF_ERR_BAD_ARG;
    int rc = check_occ(c, occ);
    if (rc) return rc;
    const cplx *psi = (const cplx *)psi_, *phi = (const cplx *)phi_;
    cplx *out = (cplx *)out_;
    const int64_t Ng = c->Ng;
    cplx **u = all_real(c, psi, occ, NULL); /* the occupied orbitals in real space */
    if (!u) return EXX_REF_ERR_ALLOC;
    int fail = 0;
#pragma omp parallel for schedule(dynamic)
    for (int i = 0; i < c->nk * nphi; i++) {
        int k = i / nphi, n = i % nphi;
        const int64_t offk = (c->off[k] / c->nb) * nphi; /* nphi * sum_{k'<k} npw(k') */
        cplx *t = malloc(sizeof(cplx) * (size_t)Ng), *w = malloc(sizeof(cplx) * (size_t)Ng), *acc = calloc((size_t)Ng, sizeof(cplx));
        double *K = malloc(sizeof(double) * (size_t)Ng);
        if (!t || !w || !acc || !K) {
            fail = 1;
        } else {
            to_real(c, k, phi + offk + (int64_t)n * c->npw[k], t);
            for (int q = 0; q < c->nk; q++) {
                exx_ref_kernel_table(c, k, q, K);
                for (int m = 0; m < c->nb; m++) {
                    double f = occ[q * c->nb + m];
                    if (f == 0.0) continue;
                    const cplx *um = u[q * c->nb + m];
                    for (int64_t j = 0; j < Ng; j++) w[j] = conj(um[j]) * t[j];
                    fft3d(c->N, -1, w);
                    for (int64_t g = 0; g < Ng; g++) w[g] = (K[g] * (w[g] / (double)Ng)) / c->omega;
                    fft3d(c->N, +1, w);
                    double wf = c->kw[q] * f;
                    for (int64_t j = 0; j < Ng; j++) acc[j] -= wf * (um[j] * w[j]);
                }
            }
            fft3d(c->N, -1, acc);
            cplx *o = out + offk + (int64_t)n * c->npw[k];
            for (int ig = 0; ig < c->npw[k]; ig++) o[ig] = acc[c->map[k][ig]] / (double)Ng;
        }
        free(t);
        free(w);
        free(acc);
        free(K);
    }
    free_real(c, u);
    return fail ? EXX_REF_ERR_ALLOC : EXX_REF_OK;
}

/* (E1): E_x = 1/2 sum_k w_k sum_n f_nk Re <c_nk | (V_x c)_nk>; per_band (optional) gets the nk*nb terms. */
int exx_ref_energy(const exx_ref_ctx *c, const double *psi_, const double *occ, const double *vxpsi_, double *ex, double *per_band) {
    if (!c || !psi_ || !occ || !vxpsi_ || !ex) return EXX_REF_ERR_NULL;
    int rc = check_occ(c, occ);
    if (rc) return rc;
    const cplx *psi = (const cplx *)psi_, *vx = (const cplx *)vxpsi_;
    double e = 0.0;
    for (int k = 0; k < c->nk; k++)
        for (int n = 0; n < c->nb; n++) {
            const cplx *a = psi + c->off[k] + (int64_t)n * c->npw[k], *b = vx + c->off[k] + (int64_t)n * c->npw[k];
            double s = 0.0;
            for (int ig = 0; ig < c->npw[k]; ig++) s += creal(conj(a[ig]) * b[ig]);
            double t = 0.5 * c->kw[k] * occ[k * c->nb + n] * s;
            if (per_band) per_band[k * c->nb + n] = t;
            e += t;
        }
    *ex = e;
    return EXX_REF_OK;
}

/* Subspace matrix of the exchange operator within k-point ik (BASELINE north_star: "the optional dense subspace matrix
 * <psi_i|V_x|psi_j>"; the paper's NSIM "matrix-matrix operations"):
 *   M[i*nb + j] = sum_{g in sphere(ik)} conj(c_i(g)) (V_x c)_j(g),   i, j = 0..nb-1, row-major complex, plain triple loop.
 * Pins (tests/test_oracle_exchange.py): numpy.einsum (independent library), Hermiticity when every band is occupied,
 * E_x = 1/2 sum w_k f_n Re M_nn. */
int exx_ref_subspace(const exx_ref_ctx *c, int ik, const double *psi_, const double *vxpsi_, double *m_) {
    if (!c || !psi_ || !vxpsi_ || !m_) return EXX_REF_ERR_NULL;
    if (ik < 0 || ik >= c->nk) return EXX_REF_ERR_BAD_ARG;
    const cplx *psi = (const cplx *)psi_ + c->off[ik], *vx = (const cplx *)vxpsi_ + c->off[ik];
    cplx *m = (cplx *)m_;
    const int64_t npw = c->npw[ik];
    for (int i = 0; i < c->nb; i++)
        for (int j = 0; j < c->nb; j++) {
            cplx s = 0.0;
            for (int64_t ig = 0; ig < npw; ig++) s += conj(psi[i * npw + ig]) * vx[j * npw + ig];
            m[(int64_t)i * c->nb + j] = s;
        }
    return EXX_REF_OK;
}

/* (E2): E_x = -1/2 (1/Omega) sum_{k,q} w_k w_q sum_{n,m} f f sum_g K |rho~|^2 — forward transforms only. */
int exx_ref_energy_e2(const exx_ref_ctx *c, const double *psi_, const double *occ, double *ex) {
    if (!c || !psi_ || !occ || !ex) return EXX_REF_ERR_NULL;
    int rc = check_occ(c, occ);
    if (rc) return rc;
    const cplx *psi = (const cplx *)psi_;
    const int64_t Ng = c->Ng;
    cplx **u = all_real(c, psi, occ, NULL);
    if (!u) return EXX_REF_ERR_ALLOC;
    int nt = nthreads_max();
    cplx *work_t = malloc(sizeof(cplx) * (size_t)Ng * nt);
    double *K = malloc(sizeof(double) * (size_t)Ng);
    double *part = calloc((size_t)nt, sizeof(double));
    if (!work_t || !K || !part) { free(work_t); free(K); free(part); free_real(c, u); return EXX_REF_ERR_ALLOC; }
    double e = 0.0;
    for (int k = 0; k < c->nk; k++)
        for (int q = 0; q < c->nk; q++) {
            exx_ref_kernel_table(c, k, q, K);
            int np = c->nb * c->nb;
            memset(part, 0, sizeof(double) * (size_t)nt);
#pragma omp parallel num_threads(nt)
            {
#ifdef _OPENMP
                int t = omp_get_thread_num();
#else
                int t = 0;
#endif
                cplx *w = work_t + (int64_t)t * Ng;
#pragma omp for schedule(static)
                for (int p = 0; p < np; p++) {
                    int n = p / c->nb, m = p % c->nb;
                    double fn = occ[k * c->nb + n], fm = occ[q * c->nb + m];
                    if (fn == 0.0 || fm == 0.0) continue;
                    const cplx *un = u[k * c->nb + n], *um = u[q * c->nb + m];
                    for (int64_t j = 0; j < Ng; j++) w[j] = conj(um[j]) * un[j];
                    fft3d(c->N, -1, w);
                    double s = 0.0;
                    for (int64_t g = 0; g < Ng; g++) {
                        cplx r = w[g] / (double)Ng;
                        s += K[g] * (creal(r) * creal(r) + cimag(r) * cimag(r));
                    }
                    part[t] += fn * fm * s;
                }
            }
            double s = 0.0;
            for (int t = 0; t < nt; t++) s += part[t];
            e += -0.5 * c->kw[k] * c->kw[q] * s / c->omega;
        }
    *ex = e;
    free(work_t);
    free(K);
    free(part);
    free_real(c, u);
    return EXX_REF_OK;
}

/* (D) with no FFT at all (oracle component O3; for small grids): both transforms written as explicit CYCLIC sums
 * in reciprocal space, all index arithmetic mod N_i (reading A10 — the method lives on the discrete grid):
 *   rho~(g')   = sum_{g'' in sphere(k)} conj(c_mq(g'' - g')) c_nk(g'')
 *   (V_x c)(g) = -(1/Omega) sum_q w_q sum_m f_mq sum_{g'} c_mq(g - g') K(|k-q+G(g')|) rho~(g')        g in sphere(k)
 */
int exx_ref_apply_direct(const exx_ref_ctx *c, const double *psi_, const double *occ, double *out_) {
    if (!c || !psi_ || !occ || !out_) return EXX_REF_ERR_NULL;
    int rc = check_occ(c, occ);
    if (rc) return rc;
    const cplx *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
    const int *N = c->N;
    const int64_t Ng = c->Ng;
    /* every band as a full box of coefficients, zero outside its sphere */
    cplx **cb = calloc((size_t)c->nk * c->nb, sizeof(cplx *));
    if (!cb) return EXX_REF_ERR_ALLOC;
    for (int i = 0; i < c->nk * c->nb; i++) {
        int k = i / c->nb, n = i % c->nb;
        cb[i] = calloc((size_t)Ng, sizeof(cplx));
        for (int ig = 0; ig < c->npw[k]; ig++) cb[i][c->map[k][ig]] = psi[c->off[k] + (int64_t)n * c->npw[k] + ig];
    }
#define IDX3(a, b, d) ((((int64_t)(a)) * N[1] + (b)) * N[2] + (d))
#define MODN(x, n) ((((x) % (n)) + (n)) % (n))
    for (int k = 0; k < c->nk; k++) {
#pragma omp parallel for schedule(dynamic)
        for (int n = 0; n < c->nb; n++) {
            cplx *rho = malloc(sizeof(cplx) * (size_t)Ng);
            cplx *res = calloc((size_t)c->npw[k], sizeof(cplx));
            double *Kl = malloc(sizeof(double) * (size_t)Ng);
            const cplx *cn = cb[k * c->nb + n];
            for (int q = 0; q < c->nk; q++) {
                exx_ref_kernel_table(c, k, q, Kl);
                for (int m = 0; m < c->nb; m++) {
                    double f = occ[q * c->nb + m];
                    if (f == 0.0) continue;
                    const cplx *cm = cb[q * c->nb + m];
                    /* rho~(g') for every g' of the box */
                    for (int p1 = 0; p1 < N[0]; p1++)
                        for (int p2 = 0; p2 < N[1]; p2++)
                            for (int p3 = 0; p3 < N[2]; p3++) {
                                cplx s = 0.0;
                                for (int ig = 0; ig < c->npw[k]; ig++) {
                                    int32_t b = c->map[k][ig];
                                    int s1 = b / (N[1] * N[2]), s2 = (b / N[2]) % N[1], s3 = b % N[2];
                                    s += conj(cm[IDX3(MODN(s1 - p1, N[0]), MODN(s2 - p2, N[1]), MODN(s3 - p3, N[2]))]) * cn[b];
                                }
                                rho[IDX3(p1, p2, p3)] = s;
                            }
                    /* (V_x c)(g) -= w_q f (1/Omega) sum_{g'} c_m(g - g') K(g') rho~(g') */
                    for (int ig = 0; ig < c->npw[k]; ig++) {
                        int32_t b = c->map[k][ig];
                        int g1 = b / (N[1] * N[2]), g2 = (b / N[2]) % N[1], g3 = b % N[2];
                        cplx s = 0.0;
                        for (int p1 = 0; p1 < N[0]; p1++)
                            for (int p2 = 0; p2 < N[1]; p2++)
                                for (int p3 = 0; p3 < N[2]; p3++) {
                                    int64_t gp = IDX3(p1, p2, p3);
                                    s += cm[IDX3(MODN(g1 - p1, N[0]), MODN(g2 - p2, N[1]), MODN(g3 - p3, N[2]))] * (Kl[gp] * rho[gp]);
                                }
                        res[ig] -= (c->kw[q] * f / c->omega) * s;
                    }
                }
            }
            memcpy(out + c->off[k] + (int64_t)n * c->npw[k], res, sizeof(cplx) * (size_t)c->npw[k]);
            free(rho);
            free(res);
            free(Kl);
        }
    }
#undef IDX3
#undef MODN
    for (int i = 0; i < c->nk * c->nb; i++) free(cb[i]);
    free(cb);
    return EXX_REF_OK;
}

const char *exx_ref_strerror(int code) {
    switch (code) {
    case EXX_REF_OK: return "ok";
    case EXX_REF_ERR_NULL: return "null pointer";
    case EXX_REF_ERR_BAD_GRID: return "bad grid";
    case EXX_REF_ERR_BAD_LATTICE: return "bad lattice (zero volume)";
    case EXX_REF_ERR_BAD_CUTOFF: return "bad cutoff";
    case EXX_REF_ERR_BAD_KERNEL: return "bad kernel parameters";
    case EXX_REF_ERR_BAD_OCC: return "bad occupation (negative or non-finite)";
    case EXX_REF_ERR_ALLOC: return "allocation failed";
    case EXX_REF_ERR_BAD_ARG: return "bad argument";
    default: return "unknown error";
    }
}
