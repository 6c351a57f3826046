// exx_fused_phases.h — the per-thread phases of the three fused passes, written as
// __host__ __device__ functions of (tid, tile) so that exx_fused.cu can run them between __syncthreads() and
// exx_host_emu.cpp can run the very same index logic thread by thread on the CPU (host logic test, no GPU).
// Product code: shares nothing with oracle/.
//
// Grid N = 8 R1 per axis (cubic), R1 in {2, 4, 5, 6, 8, 9, 10, 12, 16}.  Every 1-D transform of length N is two in-register steps
//   n = 8 n1 + n2, k = k1 + R1 k2:   R1-point DFT over n1 (stride 8)  ->  twiddle W_N^(n2 k1)  ->  8-point DFT over n2
// done in place, so a frequency k sits at position pos(k) = 8 (k mod R1) + k div R1; the inverse runs the two steps
// backwards and lands in natural order.  The pair pipeline (S2..S6) is cut at the two points where a full exchange
// through memory is unavoidable:
//   pass A (p1_*): rho = conj(u_m) u_n; z transform (both steps); first y step          tile: one x, U values of y mod 8
//   pass B (p2_*): second y step; x transform; times K'; inverse x; first inverse y step  tile: one k1y, Z positions of z
//   pass C (p3_*): second inverse y step; inverse z; acc -= w f u_m v                     tile: as pass A, loops over m
// With pair symmetry (v_{mq,nk} = conj v_{nk,mq}) pass C runs a second time with the roles of the bands swapped (cj).
//
// Like exx_dft.h this header is mode-generic: included once per (EXX_NS, EXX_REAL); accumulators are always fp64 (acc_c).
#include <stddef.h>

#include "exx_dft.h"

#ifndef EXX_ACC_C_DEFINED
#define EXX_ACC_C_DEFINED
namespace exx_acc {
struct alignas(16) acc_c {  // fp64 complex accumulator element, whatever the mode of the transforms
    double x, y;
};
}  // namespace EXX_NS_acc
#endif

namespace EXX_NS {
using exx_acc::acc_c;
EXX_HD acc_c mka(double x, double y) {
    acc_c r;
    r.x = x;
    r.y = y;
    return r;
}

// twiddle tables W_N^j, j < N = 8 R1, for every R1 <= 16, in one array (constant memory on the device): table R1 starts at
// sum_{r < R1} 8 r = 4 R1 (R1 - 1)
constexpr int TW_TOTAL = 4 * 17 * 16;
template <int R1>
struct TwOff {
    static constexpr int v = 4 * R1 * (R1 - 1);
};

#if defined(__CUDACC__)
__constant__ cplx c_tw[TW_TOTAL];  // one table per mode (this header is included in exactly one .cu)
#endif
extern cplx h_tw[TW_TOTAL];
#undef EXX_TW
#if defined(__CUDA_ARCH__)
#define EXX_TW(R1, j) c_tw[TwOff<R1>::v + (j)]
#else
#define EXX_TW(R1, j) h_tw[TwOff<R1>::v + (j)]
#endif

// per-grid launch geometry.  Passes A and C work on tiles of U*R1 rows (one x, U values of y mod 8) with NT1 / NT3 threads;
// pass B on tiles of Z z-positions with NT2 threads.  Thread counts are chosen so that every step's item count is a small
// multiple of the CTA size.  TWREG: the z twiddles W_N^(j k1z) live in 7 registers per thread (needs NT % R1 == 0 so that a
// thread's k1z never changes) instead of a shared-memory table; ACCREG: pass C keeps its accumulator tile in registers
// instead of shared memory; STAGE3 >= 1: pass C fetches the next column's work-box elements into per-thread shared-memory slots
// with cp.async while it transforms the current column (no registers held across the load latency); STAGE3 = 2: the u elements
// of the last step likewise, two barriers ahead.
constexpr int s3(int dflt) {
#ifdef EXX_STAGE3_ALL  // tuning builds: one level for every grid
    return EXX_STAGE3_ALL;
#else
    return dflt;
#endif
}
constexpr int rg(int dflt) {
#ifdef EXX_DUAL_RG_ALL  // tuning builds: one value for every grid (0 switches the dual sweep off)
    return EXX_DUAL_RG_ALL;
#else
    return dflt;
#endif
}
template <int R1>
struct FusedCfgBase;
template <>
struct FusedCfgBase<2> {
    static constexpr int U1 = 8, NT1 = 128, U3 = 8, NT3 = 128, Z = 4, NT2 = 64;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(0);
    static constexpr int MINB1 = 1, MINB2 = 1, MINB3 = 1;
    static constexpr int RG = rg(4);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<4> {
    static constexpr int U1 = 4, NT1 = 128, U3 = 4, NT3 = 128, Z = 4, NT2 = 128;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(2);
    static constexpr int MINB1 = 1, MINB2 = 6, MINB3 = 1;
    static constexpr int RG = rg(4);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<5> {
    static constexpr int U1 = 4, NT1 = 160, U3 = 4, NT3 = 160, Z = 4, NT2 = 160;
    static constexpr bool TWREG = false, ACCREG = true;
    static constexpr int STAGE3 = s3(2);
    static constexpr int MINB1 = 1, MINB2 = 6, MINB3 = 1;
    static constexpr int RG = rg(0);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<10> {
    static constexpr int U1 = 1, NT1 = 128, U3 = 1, NT3 = 128, Z = 4, NT2 = 160;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(1);
    static constexpr int MINB1 = 1, MINB2 = 4, MINB3 = 1;
    static constexpr int RG = rg(2);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<6> {
    static constexpr int U1 = 2, NT1 = 96, U3 = 2, NT3 = 96, Z = 4, NT2 = 64;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(2);
    static constexpr int MINB1 = 1, MINB2 = 6, MINB3 = 1;  // min CTAs per SM asked of the compiler (register cap)
    static constexpr int RG = rg(4);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<8> {
    static constexpr int U1 = 2, NT1 = 128, U3 = 2, NT3 = 128, Z = 4, NT2 = 96;
    static constexpr bool TWREG = false, ACCREG = true;
    static constexpr int STAGE3 = s3(2);
    static constexpr int MINB1 = 1, MINB2 = 6, MINB3 = 1;
    static constexpr int RG = rg(0);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<9> {
    static constexpr int U1 = 2, NT1 = 160, U3 = 1, NT3 = 96, Z = 4, NT2 = 96;
    static constexpr bool TWREG = false, ACCREG = true;
    static constexpr int STAGE3 = s3(2);
    static constexpr int MINB1 = 1, MINB2 = 5, MINB3 = 1;
    static constexpr int RG = rg(4);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<12> {
    static constexpr int U1 = 1, NT1 = 96, U3 = 1, NT3 = 96, Z = 4, NT2 = 128;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(1);
    static constexpr int MINB1 = 1, MINB2 = 4, MINB3 = 1;
    static constexpr int RG = rg(2);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <>
struct FusedCfgBase<16> {
    static constexpr int U1 = 1, NT1 = 128, U3 = 1, NT3 = 128, Z = 4, NT2 = 256;
    static constexpr bool TWREG = false, ACCREG = false;
    static constexpr int STAGE3 = s3(1);
    static constexpr int MINB1 = 1, MINB2 = 2, MINB3 = 1;
    static constexpr int RG = rg(0);  // rows per CTA of the dual sweep (5.4b); 0: two single sweeps (measured faster at 40^3 and 64^3)
};
template <int R1>
struct FusedCfg : FusedCfgBase<R1> {};

// tuning sweeps: -DEXX_TUNE_R1=<R1> plus any of EXX_TUNE_{U1,NT1,U3,NT3,NT2,MINB1,MINB2,MINB3,TWREG,ACCREG,STAGE3} overrides that grid
#ifdef EXX_TUNE_R1
#ifndef EXX_TUNE_U1
#define EXX_TUNE_U1 FusedCfgBase<EXX_TUNE_R1>::U1
#endif
#ifndef EXX_TUNE_NT1
#define EXX_TUNE_NT1 FusedCfgBase<EXX_TUNE_R1>::NT1
#endif
#ifndef EXX_TUNE_U3
#define EXX_TUNE_U3 FusedCfgBase<EXX_TUNE_R1>::U3
#endif
#ifndef EXX_TUNE_NT3
#define EXX_TUNE_NT3 FusedCfgBase<EXX_TUNE_R1>::NT3
#endif
#ifndef EXX_TUNE_NT2
#define EXX_TUNE_NT2 FusedCfgBase<EXX_TUNE_R1>::NT2
#endif
#ifndef EXX_TUNE_MINB1
#define EXX_TUNE_MINB1 FusedCfgBase<EXX_TUNE_R1>::MINB1
#endif
#ifndef EXX_TUNE_MINB2
#define EXX_TUNE_MINB2 FusedCfgBase<EXX_TUNE_R1>::MINB2
#endif
#ifndef EXX_TUNE_MINB3
#define EXX_TUNE_MINB3 FusedCfgBase<EXX_TUNE_R1>::MINB3
#endif
#ifndef EXX_TUNE_TWREG
#define EXX_TUNE_TWREG FusedCfgBase<EXX_TUNE_R1>::TWREG
#endif
#ifndef EXX_TUNE_ACCREG
#define EXX_TUNE_ACCREG FusedCfgBase<EXX_TUNE_R1>::ACCREG
#endif
#ifndef EXX_TUNE_STAGE3
#define EXX_TUNE_STAGE3 FusedCfgBase<EXX_TUNE_R1>::STAGE3
#endif
template <>
struct FusedCfg<EXX_TUNE_R1> {
    static constexpr int U1 = EXX_TUNE_U1, NT1 = EXX_TUNE_NT1, U3 = EXX_TUNE_U3, NT3 = EXX_TUNE_NT3, Z = 4, NT2 = EXX_TUNE_NT2;
    static constexpr bool TWREG = EXX_TUNE_TWREG, ACCREG = EXX_TUNE_ACCREG;
    static constexpr int STAGE3 = EXX_TUNE_STAGE3;
    static constexpr int MINB1 = EXX_TUNE_MINB1, MINB2 = EXX_TUNE_MINB2, MINB3 = EXX_TUNE_MINB3;
    static constexpr int RG = FusedCfgBase<EXX_TUNE_R1>::RG;
};
#endif

// ---- shared-memory layouts -------------------------------------------------------------------------------------
// passes A/C: S[row][k1z][j], XOR swizzle of j with (row R1 + k1z) & 7 and 4 (u & 1): conflict-free for the three access patterns
// (lanes along j; lanes along (row,k1z); lanes along the position 8 k1z + j), no padding.
template <int R1>
EXX_HD int sidx(int u, int r, int k1z, int j) {  // row = u R1 + r
    int row = u * R1 + r;
    if (sizeof(real) == 4) {
        // 8-byte elements: a half-warp (16 lanes) is served together and the bank is the low 4 bits of the element index.
        // Bit 3 of the index is the parity of it = row R1 + k1z, so swizzling j with the next three bits of it makes 16
        // consecutive (row, k1z) items, 16 consecutive positions of a row, and 2 rows x 8 j (R1 odd) all conflict-free.
        return row * (8 * R1) + k1z * 8 + (j ^ (((row * R1 + k1z) >> 1) & 7));
    }
    return row * (8 * R1) + k1z * 8 + (j ^ (((row * R1 + k1z) & 7) ^ ((u & 1) << 2)));
}
// the pair work box W between the passes: [k1y][kzpos / 4][x][n2y][kzpos % 4] — a pass-B tile (k1y, zb) is one
// contiguous run of N*32 elements (bulk-copied), and passes A/C touch it in runs of 4 U elements
template <int R1>
EXX_HD size_t widx(int k1y, int kzpos, int x, int n2y) {
    constexpr int N = 8 * R1;
    return ((((size_t)k1y * (N / 4) + (kzpos >> 2)) * N + x) * 8 + n2y) * 4 + (kzpos & 3);
}
// z twiddle table in shared memory: T[k1z][j] = W_N^(j k1z), same swizzle idea
EXX_HD int tidx(int k1z, int j) { return k1z * 8 + (j ^ (k1z & 7)); }

// pass B: S[xpos][k2y][kzl], x pitch padded so that lanes along (xpos, kzl) are conflict-free
template <int Z>
struct P2Geo {
    static constexpr int PX = 8 * Z + (Z == 8 ? 0 : Z);
};
template <int Z>
EXX_HD int s2idx(int xpos, int e) {  // e = k2y Z + kzl
    return xpos * P2Geo<Z>::PX + e;
}

// ================================================================================================================
// pass A
template <int R1, int U, int NT>
EXX_HD void p1_z1(int tid, const cplx* __restrict__ un, const cplx* __restrict__ um, int x, int yb, cplx* S) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
            cplx a[R1], b[R1], v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) {
                a[j] = un[base + j * 8];
                b[j] = um[base + j * 8];
            }
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = conj_mul(b[j], a[j]);  // rho = conj(u_m) u_n   (S2)
            dft<R1, -1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) S[sidx<R1>(u, n1y, j, n2z)] = v[j];
        }
    }
}

// per-thread z twiddles for TWREG: twr[j] = W_N^(j k1z) with k1z = tid mod R1
template <int R1>
EXX_HD void load_twr(int tid, cplx* twr) {
    int k1z = tid % R1;
#pragma unroll
    for (int j = 0; j < 8; j++) twr[j] = EXX_TW(R1, j * k1z);
}

template <int R1, int U, int NT, int SIGN, bool TWREG>
EXX_HD void p13_z8(int tid, cplx* S, const cplx* T, const cplx* twr) {
    // the 8-point z step on items (row, k1z).  SIGN < 0: twiddle then forward DFT; SIGN > 0: inverse DFT then conj twiddle
    constexpr int NI = U * R1 * R1, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it / R1, k1z = it - row * R1;
            int u = row / R1, r = row - u * R1;
            cplx v[8], w[8];
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = S[sidx<R1>(u, r, k1z, j)];
            if (TWREG) {
#pragma unroll
                for (int j = 1; j < 8; j++) w[j] = twr[j];
            } else {
                // three table reads (W^k, W^2k, W^4k) and four products instead of seven reads: the shared-memory
                // data pipe, not the fp64 pipe, is what these kernels run out of
                w[1] = T[tidx(k1z, 1)];
                w[2] = T[tidx(k1z, 2)];
                w[4] = T[tidx(k1z, 4)];
                w[3] = w[1] * w[2];
                w[5] = w[4] * w[1];
                w[6] = w[4] * w[2];
                w[7] = w[4] * w[3];
            }
            if (SIGN < 0) {
#pragma unroll
                for (int j = 1; j < 8; j++) v[j] = v[j] * w[j];
                dft<8, -1>(v);
            } else {
                dft<8, +1>(v);
#pragma unroll
                for (int j = 1; j < 8; j++) v[j] = mul_conj_b(v[j], w[j]);
            }
#pragma unroll
            for (int j = 0; j < 8; j++) S[sidx<R1>(u, r, k1z, j)] = v[j];
        }
    }
}

template <int R1, int U, int NT>
EXX_HD void p1_y1(int tid, const cplx* S, cplx* __restrict__ W, int x, int yb) {
    // items (kzblk, u, kzl), kzl fastest: 4 U consecutive lanes store one contiguous run of W
    constexpr int N = 8 * R1, NI = U * N, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int kzl = it & 3, u = (it >> 2) % U, kzpos = (it / (4 * U)) * 4 + kzl;
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[sidx<R1>(u, j, kzpos >> 3, kzpos & 7)];
            dft<R1, -1>(v);
            size_t base = widx<R1>(0, kzpos, x, yb * U + u);
#pragma unroll
            for (int j = 0; j < R1; j++) W[base + (size_t)j * (N / 4) * N * 32] = v[j];  // k1y = j
        }
    }
}

// ================================================================================================================
// pass B.  Tile: rows k1y*8 + n2y (n2y < 8), all x, z positions zb*Z .. zb*Z+Z-1.
// host stand-in for the bulk copies: tile rows W[tile][x][32] <-> S[x * PX ..]
template <int R1, int Z>
inline void p2_copy_rows(cplx* S, cplx* Wt, bool load) {
    constexpr int N = 8 * R1, PX = P2Geo<Z>::PX;
    for (int x = 0; x < N; x++)
        for (int e = 0; e < 8 * Z; e++) {
            if (load)
                S[x * PX + e] = Wt[x * 8 * Z + e];
            else
                Wt[x * 8 * Z + e] = S[x * PX + e];
        }
}

// called by p2_y8 before iteration i touches its rows (rows i NT/Z .. (i+1) NT/Z - 1): the kernel waits there for the bulk copy of
// that chunk of rows; the host emulation and the later steps pass nothing
struct NoWait {
    EXX_HD void operator()(int) const {}
};
template <int R1, int Z, int NT, int SIGN, class WAIT = NoWait>
EXX_HD void p2_y8(int tid, cplx* S, int k1y, WAIT wait = WAIT()) {
    // items (xpos, kzl), in place in shared memory.  SIGN < 0: y twiddle W_N^(n2y k1y) (uniform per CTA), forward 8-point
    // DFT over n2y;  SIGN > 0: inverse 8-point DFT over k2y, conjugate twiddle.
    constexpr int N = 8 * R1, NI = N * Z, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        wait(i);
        if (it < NI) {
            int xpos = it / Z, kzl = it - xpos * Z;
            cplx v[8];
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = S[s2idx<Z>(xpos, j * Z + kzl)];
            if (SIGN < 0) {
#pragma unroll
                for (int j = 1; j < 8; j++) v[j] = v[j] * EXX_TW(R1, j * k1y);
                dft<8, -1>(v);
            } else {
                dft<8, +1>(v);
#pragma unroll
                for (int j = 1; j < 8; j++) v[j] = mul_conj_b(v[j], EXX_TW(R1, j * k1y));
            }
#pragma unroll
            for (int j = 0; j < 8; j++) S[s2idx<Z>(xpos, j * Z + kzl)] = v[j];
        }
    }
}

template <int R1, int Z, int NT, int SIGN>
EXX_HD void p2_xR(int tid, cplx* S) {
    // the R1-point x step on items (n2x, rem = k2y*Z + kzl).  Forward: DFT then twiddle W_N^(n2x k1x); inverse: DFT only
    // (the conjugate twiddle was applied at the end of p2_x8).
    constexpr int NI = 8 * 8 * Z, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int n2x = it / (8 * Z), rem = it - n2x * (8 * Z);
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[s2idx<Z>(j * 8 + n2x, rem)];
            dft<R1, SIGN>(v);
            if (SIGN < 0) {
#pragma unroll
                for (int j = 1; j < R1; j++) v[j] = v[j] * EXX_TW(R1, n2x * j);
            }
#pragma unroll
            for (int j = 0; j < R1; j++) S[s2idx<Z>(j * 8 + n2x, rem)] = v[j];
        }
    }
}

// K' is read 16 bytes at a time (KVW consecutive k2x values); the tile's slice of the permuted table is [k2x / KVW][item][k2x % KVW],
// so the lanes of a warp (consecutive items) read one contiguous run per load
constexpr int KVW = 16 / sizeof(real);
struct alignas(16) kvec {
    real v[KVW];
};

template <int R1, int Z, int NT>
EXX_HD void p2_x8(int tid, cplx* S, const real* __restrict__ Kt) {
    // items (k1x, rem): second forward x step, times K' (S4), first inverse x step, conjugate twiddle.
    // Kt: this tile's slice of the permuted kernel table (layout above).
    constexpr int NI = R1 * 8 * Z, IT = (NI + NT - 1) / NT;
    const kvec* __restrict__ Kv = reinterpret_cast<const kvec*>(Kt);
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int k1x = it / (8 * Z), rem = it - k1x * (8 * Z);
            cplx v[8];
            real kk[8];
#pragma unroll
            for (int jv = 0; jv < 8 / KVW; jv++) {
                kvec q = Kv[(size_t)jv * NI + it];
#pragma unroll
                for (int e = 0; e < KVW; e++) kk[jv * KVW + e] = q.v[e];
            }
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = S[s2idx<Z>(k1x * 8 + j, rem)];
            dft<8, -1>(v);
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = scale(kk[j], v[j]);
            dft<8, +1>(v);
#pragma unroll
            for (int j = 1; j < 8; j++) v[j] = mul_conj_b(v[j], EXX_TW(R1, j * k1x));
#pragma unroll
            for (int j = 0; j < 8; j++) S[s2idx<Z>(k1x * 8 + j, rem)] = v[j];
        }
    }
}

// Energy route (E2 of DESIGN.md section 2): second forward x step only, then this thread's share of
//   sum_g K'(g) |rho^(g)|^2   (fp64 whatever the mode of the transforms).  Nothing is written back to the tile.
template <int R1, int Z, int NT>
EXX_HD double p2_x8_energy(int tid, const cplx* S, const real* __restrict__ Kt) {
    constexpr int NI = R1 * 8 * Z, IT = (NI + NT - 1) / NT;
    const kvec* __restrict__ Kv = reinterpret_cast<const kvec*>(Kt);
    double e = 0.0;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int k1x = it / (8 * Z), rem = it - k1x * (8 * Z);
            cplx v[8];
            real kk[8];
#pragma unroll
            for (int jv = 0; jv < 8 / KVW; jv++) {
                kvec q = Kv[(size_t)jv * NI + it];
#pragma unroll
                for (int e2 = 0; e2 < KVW; e2++) kk[jv * KVW + e2] = q.v[e2];
            }
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = S[s2idx<Z>(k1x * 8 + j, rem)];
            dft<8, -1>(v);
#pragma unroll
            for (int j = 0; j < 8; j++) e += (double)kk[j] * ((double)v[j].x * (double)v[j].x + (double)v[j].y * (double)v[j].y);
        }
    }
    return e;
}

// ================================================================================================================
// pass C
template <int R1, int U, int NT>
EXX_HD void p3_y2inv(int tid, const cplx* __restrict__ W, int x, int yb, cplx* S) {
    constexpr int N = 8 * R1, NI = U * N, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int kzl = it & 3, u = (it >> 2) % U, kzpos = (it / (4 * U)) * 4 + kzl;
            size_t base = widx<R1>(0, kzpos, x, yb * U + u);
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = W[base + (size_t)j * (N / 4) * N * 32];
            dft<R1, +1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) S[sidx<R1>(u, j, kzpos >> 3, kzpos & 7)] = v[j];
        }
    }
}

// STAGE3: the same step with the work-box elements fetched ahead of time.  Element j of item tid + i NT lives in the slot
// G[(i R1 + j) NT + tid], written and read by this thread only (no barrier needed): p3_stage copies them there (cp.async on the
// device, one element each, so the thread does not wait for them; a plain copy on the host), p3_y2inv_staged consumes them.
// slot of element j of item tid + i NT: (i R1 + j) slot_stride + tid; a step has U N = 8 U R1 items, and when they fit one round
// (NT >= items) the idle threads get no slots
template <int R1, int U, int NT>
struct Slots {
    static constexpr int IT = (8 * U * R1 + NT - 1) / NT, STRIDE = IT == 1 ? 8 * U * R1 : NT;
    static constexpr int COUNT = IT * R1 * STRIDE;  // slots of one step: work-box elements of the first step or u elements of the last one
};
EXX_HD void stage_elem(cplx* dst, const cplx* src) {
#if defined(__CUDA_ARCH__)
    if (sizeof(cplx) == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
#else
    *dst = *src;
#endif
}
// copies are grouped (stage_commit closes a group, possibly an empty one); stage_wait<P> returns when at most the P most
// recent groups of this thread are still in flight
EXX_HD void stage_commit() {
#if defined(__CUDA_ARCH__)
    asm volatile("cp.async.commit_group;" ::: "memory");
#endif
}
template <int P>
EXX_HD void stage_wait() {
#if defined(__CUDA_ARCH__)
    asm volatile("cp.async.wait_group %0;" ::"n"(P) : "memory");
#endif
}
template <int R1, int U, int NT>
EXX_HD void p3_stage(int tid, const cplx* __restrict__ W, int x, int yb, cplx* G) {
    static_assert(sizeof(cplx) == 16 || sizeof(cplx) == 8, "cplx size");
    constexpr int N = 8 * R1, NI = U * N, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int kzl = it & 3, u = (it >> 2) % U, kzpos = (it / (4 * U)) * 4 + kzl;
            size_t base = widx<R1>(0, kzpos, x, yb * U + u);
#pragma unroll
            for (int j = 0; j < R1; j++) stage_elem(G + (i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid, W + base + (size_t)j * (N / 4) * N * 32);
        }
    }
}
// the u_m elements of the last step, same scheme: element j of item tid + i NT in slot G2[(i R1 + j) NT + tid]
template <int R1, int U, int NT>
EXX_HD void p3_stage_u(int tid, const cplx* __restrict__ um, int x, int yb, cplx* G2) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
#pragma unroll
            for (int j = 0; j < R1; j++) stage_elem(G2 + (i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid, um + base + j * 8);
        }
    }
}
template <int R1, int U, int NT>
EXX_HD void p3_y2inv_staged(int tid, const cplx* G, cplx* S) {
    constexpr int N = 8 * R1, NI = U * N, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int kzl = it & 3, u = (it >> 2) % U, kzpos = (it / (4 * U)) * 4 + kzl;
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = G[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid];
            dft<R1, +1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) S[sidx<R1>(u, j, kzpos >> 3, kzpos & 7)] = v[j];
        }
    }
}

template <int R1, int U, int NT, bool USTG = false>
EXX_HD void p3_zinv2(int tid, const cplx* S, const cplx* __restrict__ um, double wf, int x, int yb, acc_c* A, bool first, bool cj = false,
                     const cplx* G2 = nullptr) {
    // items (row, n2z): last inverse z step, then acc -= (w_q f_m) u_m v   (S6); A is this CTA's private accumulator tile
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
            cplx b[R1], v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) b[j] = USTG ? G2[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid] : um[base + j * 8];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[sidx<R1>(u, n1y, j, n2z)];
            dft<R1, +1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) {
                cplx p = b[j] * (cj ? mk(v[j].x, -v[j].y) : v[j]);  // cj: the transposed pair uses conj(v)
                acc_c* a = A + row * N + j * 8 + n2z;
                if (first)
                    *a = mka(-wf * p.x, -wf * p.y);
                else
                    *a = mka(a->x - wf * p.x, a->y - wf * p.y);
            }
        }
    }
}

template <int R1, int U, int NT>
EXX_HD void p3_flush(int tid, const acc_c* A, acc_c* __restrict__ accg, int x, int yb) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
#pragma unroll
            for (int j = 0; j < R1; j++) {
                acc_c g = accg[base + j * 8], a = A[row * N + j * 8 + n2z];
                accg[base + j * 8] = mka(g.x + a.x, g.y + a.y);
            }
        }
    }
}

// register-accumulator variants (ACCREG): acc[i*R1 + j] belongs to item tid + i*NT, element n1z = j
template <int R1, int U, int NT, bool USTG = false>
EXX_HD void p3_zinv2_reg(int tid, const cplx* S, const cplx* __restrict__ um, double wf, int x, int yb, acc_c* acc, bool cj = false,
                         const cplx* G2 = nullptr) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
            cplx b[R1], v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) b[j] = USTG ? G2[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid] : um[base + j * 8];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[sidx<R1>(u, n1y, j, n2z)];
            dft<R1, +1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) {
                cplx p = b[j] * (cj ? mk(v[j].x, -v[j].y) : v[j]);  // cj: the transposed pair uses conj(v)
                acc[i * R1 + j] = mka(acc[i * R1 + j].x - wf * p.x, acc[i * R1 + j].y - wf * p.y);
            }
        }
    }
}

template <int R1, int U, int NT>
EXX_HD void p3_flush_reg(int tid, const acc_c* acc, acc_c* __restrict__ accg, int x, int yb) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
#pragma unroll
            for (int j = 0; j < R1; j++) accg[base + j * 8] = mka(accg[base + j * 8].x + acc[i * R1 + j].x, accg[base + j * 8].y + acc[i * R1 + j].y);
        }
    }
}

// ---- dual sweep (pair symmetry): ONE inverse transform of a pair's box feeds both accumulations --------------------------
// A CTA of RG warp groups (NT threads each) owns RG rows (a-bands) of the batch for one tile and walks the columns (b-bands) in
// lockstep.  Group wg transforms box (row, column) in its own tile S and, in the last step, adds
//     side a:  acc_a -= (w_q f_b) u_b v                 into its register accumulators (flushed once after the loop), and writes
//     side b:  P = (-w_k f_a) u_a conj(v)               over its own elements of S (each thread owns the elements it read),
// UA holding (-w_k f_a) u_a of the group's row and UB the column's u_b, both in per-thread slots (element j of item tid + i NT at
// slot (i R1 + j) NT + tid).  After a barrier p3_reduce_b adds the P tiles of the contributing groups in group order and stores
// the sum to the column's partial box; pass_r_kernel later adds the partial boxes of a column, in row-group order, to acc_b.
template <int R1, int U, int NT>
EXX_HD void p3_zinv2_dual(int tid, cplx* S, const cplx* UB, const cplx* UA, double wfb, bool do_a, bool do_b, acc_c* acc) {
    constexpr int NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[sidx<R1>(u, n1y, j, n2z)];
            dft<R1, +1>(v);
            if (do_a) {
#pragma unroll
                for (int j = 0; j < R1; j++) {
                    cplx p = UB[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid] * v[j];
                    acc[i * R1 + j] = mka(acc[i * R1 + j].x - wfb * p.x, acc[i * R1 + j].y - wfb * p.y);
                }
            }
            if (do_b) {
#pragma unroll
                for (int j = 0; j < R1; j++) S[sidx<R1>(u, n1y, j, n2z)] = mul_conj_b(UA[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid], v[j]);
            }
        }
    }
}

// UA slots <- coef * u (this thread's elements of the group's row; the slots are private to the thread)
template <int R1, int U, int NT>
EXX_HD void p3_scale_slots(int tid, cplx* UA, real coef) {
    constexpr int NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++)
        if (tid + i * NT < NI) {
#pragma unroll
            for (int j = 0; j < R1; j++) UA[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid] = scale(coef, UA[(i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid]);
        }
}

// the column's u_b elements, staged ONCE per CTA: group wg copies the elements j = wg, wg + RG, ... of every item into the shared
// slots, every group reads all of them after the next CTA barrier
template <int R1, int U, int NT, int RG>
EXX_HD void p3_stage_u_share(int wg, int tid, const cplx* __restrict__ um, int x, int yb, cplx* G2) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
#pragma unroll
            for (int j = 0; j < R1; j++)
                if (j % RG == wg) stage_elem(G2 + (i * R1 + j) * Slots<R1, U, NT>::STRIDE + tid, um + base + j * 8);
        }
    }
}

// partial box of (row group, column) <- sum over the contributing groups (bit g of gmask), in group order, of their P tiles;
// thread (wg, tid) handles the elements j = wg, wg + RG, ... of its item.  tile_stride = elements between the groups' S tiles.
template <int R1, int U, int NT, int RG>
EXX_HD void p3_reduce_b(int wg, int tid, const cplx* S0, int tile_stride, unsigned gmask, cplx* __restrict__ part, int x, int yb) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
#pragma unroll
            for (int j = 0; j < R1; j++)
                if (j % RG == wg) {
                    cplx s = mk(EXX_RC(0.0), EXX_RC(0.0));
#pragma unroll
                    for (int g = 0; g < RG; g++)
                        if (gmask >> g & 1u) s = s + S0[g * tile_stride + sidx<R1>(u, n1y, j, n2z)];
                    part[base + j * 8] = s;
                }
        }
    }
}

// ================================================================================================================
// Plain 3-D transforms with the same passes (S1: sphere coefficients -> u(r); S7: accumulator -> sphere coefficients).
// Frequency-domain boxes live in the "F layout": what pass B holds after its forward x steps, written back tile by tile:
//   findex(kx, ky, kz) = widx(k1y, kzpos, xpos, k2y) with xpos = 8 (kx mod R1) + kx div R1, kzpos = 8 (kz mod R1) + kz div R1,
//   k1y = ky mod R1, k2y = ky div R1.
// Forward  = pass A (one input, no product) + pass B forward half (y8, xR, x8)  -> F layout, then gather through findex.
// Inverse  = scatter through findex, pass B inverse half (x8, xR, y8) + pass C without multiply/accumulate -> natural box.
template <int R1>
EXX_HD size_t findex(int kx, int ky, int kz) {
    return widx<R1>(ky % R1, 8 * (kz % R1) + kz / R1, 8 * (kx % R1) + kx / R1, ky / R1);
}

template <int R1, int U, int NT>
EXX_HD void p1_z1_single(int tid, const cplx* __restrict__ un, int x, int yb, cplx* S) {
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = un[base + j * 8];
            dft<R1, -1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) S[sidx<R1>(u, n1y, j, n2z)] = v[j];
        }
    }
}

template <int R1, int Z, int NT, int SIGN>
EXX_HD void p2_x8_half(int tid, cplx* S) {
    // items (k1x, rem).  SIGN < 0: second forward x step only;  SIGN > 0: first inverse x step + conjugate twiddle
    constexpr int NI = R1 * 8 * Z, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int k1x = it / (8 * Z), rem = it - k1x * (8 * Z);
            cplx v[8];
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = S[s2idx<Z>(k1x * 8 + j, rem)];
            dft<8, SIGN>(v);
            if (SIGN > 0) {
#pragma unroll
                for (int j = 1; j < 8; j++) v[j] = mul_conj_b(v[j], EXX_TW(R1, j * k1x));
            }
#pragma unroll
            for (int j = 0; j < 8; j++) S[s2idx<Z>(k1x * 8 + j, rem)] = v[j];
        }
    }
}

template <int R1, int U, int NT>
EXX_HD void p3_zinv2_store(int tid, const cplx* S, cplx* __restrict__ out, int x, int yb) {
    // last inverse z step, stored to a natural-order box (no multiply, no accumulation)
    constexpr int N = 8 * R1, NI = U * R1 * 8, IT = (NI + NT - 1) / NT;
#pragma unroll
    for (int i = 0; i < IT; i++) {
        int it = tid + i * NT;
        if (it < NI) {
            int row = it >> 3, n2z = it & 7;
            int u = row / R1, n1y = row - u * R1;
            size_t base = ((size_t)x * N + (n1y * 8 + yb * U + u)) * N + n2z;
            cplx v[R1];
#pragma unroll
            for (int j = 0; j < R1; j++) v[j] = S[sidx<R1>(u, n1y, j, n2z)];
            dft<R1, +1>(v);
#pragma unroll
            for (int j = 0; j < R1; j++) out[base + j * 8] = v[j];
        }
    }
}

// ================================================================================================================
// Host side of the layout: K' in natural C order -> the order pass B reads it in,
//   [k1y][zb][k2x / vw][k1x][k2y][kzl][k2x % vw]  with kx = k1x + R1 k2x, ky = k1y + R1 k2y, zpos = zb Z + kzl = 8 k1z + k2z,
//   kz = k1z + R1 k2z; vw = values per 16-byte load in the mode that reads the table (2 in fp64, 4 in fp32).
inline void permute_ktable(int R1, int Z, int vw, const double* nat, double* perm) {
    const int N = 8 * R1;
    size_t o = 0;
    for (int k1y = 0; k1y < R1; k1y++)
        for (int zb = 0; zb < N / Z; zb++)
            for (int jv = 0; jv < 8 / vw; jv++)
                for (int k1x = 0; k1x < R1; k1x++)
                    for (int k2y = 0; k2y < 8; k2y++)
                        for (int kzl = 0; kzl < Z; kzl++)
                            for (int e = 0; e < vw; e++) {
                                int k2x = jv * vw + e, zpos = zb * Z + kzl, k1z = zpos >> 3, k2z = zpos & 7;
                                int kx = k1x + R1 * k2x, ky = k1y + R1 * k2y, kz = k1z + R1 * k2z;
                                perm[o++] = nat[((size_t)kx * N + ky) * N + kz];
                            }
}

}  // namespace EXX_NS
