// exx_host_emu.cpp — CPU execution of the fused passes' per-thread phases (exx_fused_phases.h), thread by thread and
// tile by tile, exactly as exx_fused.cu schedules them on the device.  Built only by tests/test_fused_host_emulation.py
// (g++, no CUDA); it lets the index/layout logic of the kernels be checked without a GPU.  Not part of libexx.so.
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "exx_fused_phases.h"

namespace exx {
cplx h_tw[TW_TOTAL];

static void fill_tw() {
    const long double tp = 6.283185307179586476925286766559005768L;
    for (int r1 = 1; r1 <= 16; r1++)
        for (int j = 0; j < 8 * r1; j++) {
            long double a = tp * j / (8 * r1);
            h_tw[4 * r1 * (r1 - 1) + j] = mk((double)cosl(a), (double)(-sinl(a)));
        }
}

template <int R1>
static void emu_pair(const cplx* un, const cplx* um, const double* Knat, double wf, acc_c* acc, cplx* W) {
    typedef FusedCfg<R1> C;
    constexpr int N = 8 * R1, U = C::U1, NT13 = C::NT1, U3 = C::U3, NT3 = C::NT3, Z = C::Z, NT2 = C::NT2;
    constexpr bool TWREG = C::TWREG, ACCREG = C::ACCREG, STAGE3 = C::STAGE3 >= 1, STAGEU = C::STAGE3 >= 2;
    std::vector<double> Kp((size_t)N * N * N);
    permute_ktable(R1, Z, KVW, Knat, Kp.data());
    std::vector<acc_c> A((size_t)U3 * R1 * N);
    std::vector<cplx> S((size_t)(U > U3 ? U : U3) * R1 * N), T(R1 * 8), S2((size_t)N * P2Geo<Z>::PX);
    for (int k = 0; k < R1; k++)
        for (int j = 0; j < 8; j++) T[tidx(k, j)] = EXX_TW(R1, j * k);
    // pass A
    for (int x = 0; x < N; x++)
        for (int yb = 0; yb < 8 / U; yb++) {
            for (int t = 0; t < NT13; t++) p1_z1<R1, U, NT13>(t, un, um, x, yb, S.data());
            for (int t = 0; t < NT13; t++) {
                cplx twr[8];
                load_twr<R1>(t, twr);
                p13_z8<R1, U, NT13, -1, TWREG>(t, S.data(), T.data(), twr);
            }
            for (int t = 0; t < NT13; t++) p1_y1<R1, U, NT13>(t, S.data(), W, x, yb);
        }
    // pass B
    for (int k1y = 0; k1y < R1; k1y++)
        for (int zb = 0; zb < N / Z; zb++) {
            const double* Kt = Kp.data() + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            cplx* Wt = W + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            p2_copy_rows<R1, Z>(S2.data(), Wt, true);
            for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, -1>(t, S2.data(), k1y);
            for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, -1>(t, S2.data());
            for (int t = 0; t < NT2; t++) p2_x8<R1, Z, NT2>(t, S2.data(), Kt);
            for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, +1>(t, S2.data());
            for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, +1>(t, S2.data(), k1y);
            p2_copy_rows<R1, Z>(S2.data(), Wt, false);
        }
    // pass C (one m)
    constexpr int IT3 = (U3 * R1 * 8 + NT3 - 1) / NT3;
    std::vector<acc_c> accr((size_t)NT3 * IT3 * R1);
    for (int x = 0; x < N; x++)
        for (int yb = 0; yb < 8 / U3; yb++) {
            for (auto& a : accr) a = mka(0.0, 0.0);
            std::vector<cplx> G2((size_t)Slots<R1, U3, NT3>::COUNT);
            if (STAGE3) {  // per-thread staging slots, as pass_c_kernel uses them
                std::vector<cplx> G((size_t)Slots<R1, U3, NT3>::COUNT);
                for (int t = 0; t < NT3; t++) p3_stage<R1, U3, NT3>(t, W, x, yb, G.data());
                for (int t = 0; t < NT3; t++) p3_y2inv_staged<R1, U3, NT3>(t, G.data(), S.data());
                if (STAGEU)
                    for (int t = 0; t < NT3; t++) p3_stage_u<R1, U3, NT3>(t, um, x, yb, G2.data());
            } else {
                for (int t = 0; t < NT3; t++) p3_y2inv<R1, U3, NT3>(t, W, x, yb, S.data());
            }
            for (int t = 0; t < NT3; t++) {
                cplx twr[8];
                load_twr<R1>(t, twr);
                p13_z8<R1, U3, NT3, +1, TWREG>(t, S.data(), T.data(), twr);
            }
            for (int t = 0; t < NT3; t++) {
                if (ACCREG)
                    p3_zinv2_reg<R1, U3, NT3, STAGEU>(t, S.data(), um, wf, x, yb, accr.data() + (size_t)t * IT3 * R1, false, G2.data());
                else
                    p3_zinv2<R1, U3, NT3, STAGEU>(t, S.data(), um, wf, x, yb, A.data(), true, false, G2.data());
            }
            for (int t = 0; t < NT3; t++) {
                if (ACCREG)
                    p3_flush_reg<R1, U3, NT3>(t, accr.data() + (size_t)t * IT3 * R1, acc, x, yb);
                else
                    p3_flush<R1, U3, NT3>(t, A.data(), acc, x, yb);
            }
        }
}


// passes A and B of one pair into its work box W (Kp: permuted table)
template <int R1>
static void emu_ab(const cplx* un, const cplx* um, const double* Kp, cplx* W) {
    typedef FusedCfg<R1> C;
    constexpr int N = 8 * R1, U = C::U1, NT13 = C::NT1, Z = C::Z, NT2 = C::NT2;
    constexpr bool TWREG = C::TWREG;
    std::vector<cplx> S((size_t)U * R1 * N), T(R1 * 8), S2((size_t)N * P2Geo<Z>::PX);
    for (int k = 0; k < R1; k++)
        for (int j = 0; j < 8; j++) T[tidx(k, j)] = EXX_TW(R1, j * k);
    for (int x = 0; x < N; x++)
        for (int yb = 0; yb < 8 / U; yb++) {
            for (int t = 0; t < NT13; t++) p1_z1<R1, U, NT13>(t, un, um, x, yb, S.data());
            for (int t = 0; t < NT13; t++) {
                cplx twr[8];
                load_twr<R1>(t, twr);
                p13_z8<R1, U, NT13, -1, TWREG>(t, S.data(), T.data(), twr);
            }
            for (int t = 0; t < NT13; t++) p1_y1<R1, U, NT13>(t, S.data(), W, x, yb);
        }
    for (int k1y = 0; k1y < R1; k1y++)
        for (int zb = 0; zb < N / Z; zb++) {
            const double* Kt = Kp + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            cplx* Wt = W + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            p2_copy_rows<R1, Z>(S2.data(), Wt, true);
            for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, -1>(t, S2.data(), k1y);
            for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, -1>(t, S2.data());
            for (int t = 0; t < NT2; t++) p2_x8<R1, Z, NT2>(t, S2.data(), Kt);
            for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, +1>(t, S2.data());
            for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, +1>(t, S2.data(), k1y);
            p2_copy_rows<R1, Z>(S2.data(), Wt, false);
        }
}

// The dual sweep of a ta x tb batch exactly as pass_c_dual_kernel + pass_r_kernel schedule it (RG warp groups per CTA, columns
// in lockstep, side a in per-thread accumulators, side b through the P tiles and one partial box per (row group, column)).
// ua: ta boxes, ub: tb boxes, ev/bside: per-row column masks, amask: columns with side a; acc_a: ta boxes, acc_b: tb boxes (+=).
template <int R1>
static void emu_dual(int ta, int tb, const cplx* ua, const cplx* ub, const double* Knat, const double* coef_a, const double* coef_b,
                     const unsigned* ev, const unsigned* bside, unsigned amask, acc_c* acc_a, acc_c* acc_b) {
    typedef FusedCfg<R1> C;
    constexpr int N = 8 * R1, U = C::U3, NT = C::NT3, Z = C::Z, RG = C::RG > 0 ? C::RG : 1;
    constexpr int TILE = U * R1 * N, ITU = (U * R1 * 8 + NT - 1) / NT, GS = Slots<R1, U, NT>::COUNT, US = GS;
    const size_t Ng = (size_t)N * N * N;
    std::vector<double> Kp(Ng);
    permute_ktable(R1, Z, KVW, Knat, Kp.data());
    std::vector<cplx> work((size_t)ta * tb * Ng);
    for (int i = 0; i < ta; i++)
        for (int j = 0; j < tb; j++)
            if (ev[i] >> j & 1u) emu_ab<R1>(ua + i * Ng, ub + j * Ng, Kp.data(), work.data() + ((size_t)i * tb + j) * Ng);
    const int nrg = (ta + RG - 1) / RG;
    std::vector<cplx> part((size_t)nrg * tb * Ng);
    std::vector<cplx> S((size_t)RG * TILE), G((size_t)RG * GS), UA((size_t)RG * US), G2(US), T(R1 * 8);
    std::vector<acc_c> accr((size_t)RG * NT * ITU * R1);
    for (int k = 0; k < R1; k++)
        for (int j = 0; j < 8; j++) T[tidx(k, j)] = EXX_TW(R1, j * k);
    for (int x = 0; x < N; x++)
        for (int yb = 0; yb < 8 / U; yb++)
            for (int g = 0; g < nrg; g++) {
                unsigned cta_ev = 0;
                for (int w = 0; w < RG; w++)
                    if (g * RG + w < ta) cta_ev |= ev[g * RG + w];
                for (auto& a : accr) a = mka(0.0, 0.0);
                for (int w = 0; w < RG; w++) {
                    const int row = g * RG + w;
                    if (row >= ta || !bside[row]) continue;
                    for (int t = 0; t < NT; t++) p3_stage_u<R1, U, NT>(t, ua + row * Ng, x, yb, UA.data() + w * US);
                    for (int t = 0; t < NT; t++) p3_scale_slots<R1, U, NT>(t, UA.data() + w * US, -coef_a[row]);
                }
                for (int c = 0; c < tb; c++) {
                    if (!(cta_ev >> c & 1u)) continue;
                    const bool col_a = amask >> c & 1u;
                    unsigned gm = 0;
                    for (int w = 0; w < RG; w++) {
                        const int row = g * RG + w;
                        const bool act = row < ta && (ev[row] >> c & 1u);
                        if (row < ta && (bside[row] >> c & 1u)) gm |= 1u << w;
                        if (act) {
                            const cplx* W = work.data() + ((size_t)row * tb + c) * Ng;
                            for (int t = 0; t < NT; t++) p3_stage<R1, U, NT>(t, W, x, yb, G.data() + w * GS);
                            for (int t = 0; t < NT; t++) p3_y2inv_staged<R1, U, NT>(t, G.data() + w * GS, S.data() + w * TILE);
                        }
                        if (col_a)
                            for (int t = 0; t < NT; t++) p3_stage_u_share<R1, U, NT, RG>(w, t, ub + c * Ng, x, yb, G2.data());
                    }
                    for (int w = 0; w < RG; w++) {
                        const int row = g * RG + w;
                        if (!(row < ta && (ev[row] >> c & 1u))) continue;
                        for (int t = 0; t < NT; t++) {
                            cplx twr[8];
                            p13_z8<R1, U, NT, +1, false>(t, S.data() + w * TILE, T.data(), twr);
                        }
                    }
                    for (int w = 0; w < RG; w++) {
                        const int row = g * RG + w;
                        if (!(row < ta && (ev[row] >> c & 1u))) continue;
                        for (int t = 0; t < NT; t++)
                            p3_zinv2_dual<R1, U, NT>(t, S.data() + w * TILE, G2.data(), UA.data() + w * US, coef_b[c], col_a, bside[row] >> c & 1u,
                                                     accr.data() + ((size_t)w * NT + t) * ITU * R1);
                    }
                    if (gm)
                        for (int w = 0; w < RG; w++)
                            for (int t = 0; t < NT; t++)
                                p3_reduce_b<R1, U, NT, RG>(w, t, S.data(), TILE, gm, part.data() + ((size_t)g * tb + c) * Ng, x, yb);
                }
                for (int w = 0; w < RG; w++) {
                    const int row = g * RG + w;
                    if (row < ta && (ev[row] & amask))
                        for (int t = 0; t < NT; t++) p3_flush_reg<R1, U, NT>(t, accr.data() + ((size_t)w * NT + t) * ITU * R1, acc_a + row * Ng, x, yb);
                }
            }
    for (int c = 0; c < tb; c++)  // pass R
        for (int g = 0; g < nrg; g++) {
            bool any = false;
            for (int w = 0; w < RG; w++)
                if (g * RG + w < ta && (bside[g * RG + w] >> c & 1u)) any = true;
            if (!any) continue;
            for (size_t p = 0; p < Ng; p++) {
                cplx v = part[((size_t)g * tb + c) * Ng + p];
                acc_b[c * Ng + p] = mka(acc_b[c * Ng + p].x + v.x, acc_b[c * Ng + p].y + v.y);
            }
        }
}

// energy route of one pair (pass A, the forward half of pass B, the K' |rho^|^2 sum of p2_x8_energy), tile partials added up
// in tile order as pair_sum_kernel would see them
template <int R1>
static double emu_pair_energy(const cplx* un, const cplx* um, const double* Knat, cplx* W) {
    typedef FusedCfg<R1> C;
    constexpr int N = 8 * R1, U = C::U1, NT13 = C::NT1, Z = C::Z, NT2 = C::NT2;
    constexpr bool TWREG = C::TWREG;
    std::vector<double> Kp((size_t)N * N * N);
    permute_ktable(R1, Z, KVW, Knat, Kp.data());
    std::vector<cplx> S((size_t)U * R1 * N), T(R1 * 8), S2((size_t)N * P2Geo<Z>::PX);
    for (int k = 0; k < R1; k++)
        for (int j = 0; j < 8; j++) T[tidx(k, j)] = EXX_TW(R1, j * k);
    for (int x = 0; x < N; x++)
        for (int yb = 0; yb < 8 / U; yb++) {
            for (int t = 0; t < NT13; t++) p1_z1<R1, U, NT13>(t, un, um, x, yb, S.data());
            for (int t = 0; t < NT13; t++) {
                cplx twr[8];
                load_twr<R1>(t, twr);
                p13_z8<R1, U, NT13, -1, TWREG>(t, S.data(), T.data(), twr);
            }
            for (int t = 0; t < NT13; t++) p1_y1<R1, U, NT13>(t, S.data(), W, x, yb);
        }
    double e = 0.0;
    for (int k1y = 0; k1y < R1; k1y++)
        for (int zb = 0; zb < N / Z; zb++) {
            const double* Kt = Kp.data() + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            cplx* Wt = W + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
            p2_copy_rows<R1, Z>(S2.data(), Wt, true);
            for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, -1>(t, S2.data(), k1y);
            for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, -1>(t, S2.data());
            double tile = 0.0;
            for (int t = 0; t < NT2; t++) tile += p2_x8_energy<R1, Z, NT2>(t, S2.data(), Kt);
            e += tile;
        }
    return e;
}

// plain 3-D transforms through the fused passes.  sign < 0: natural box `in` -> F-layout box `out`;
// sign > 0: F-layout box `in` (modified in place by the pass-B half) -> natural box `out`
template <int R1>
static void emu_fft(int sign, cplx* in, cplx* out) {
    typedef FusedCfg<R1> C;
    constexpr int N = 8 * R1, U = C::U1, NT13 = C::NT1, U3 = C::U3, NT3 = C::NT3, Z = C::Z, NT2 = C::NT2;
    constexpr bool TWREG = C::TWREG;
    std::vector<cplx> S((size_t)(U > U3 ? U : U3) * R1 * N), T(R1 * 8), S2((size_t)N * P2Geo<Z>::PX);
    for (int k = 0; k < R1; k++)
        for (int j = 0; j < 8; j++) T[tidx(k, j)] = EXX_TW(R1, j * k);
    if (sign < 0) {
        for (int x = 0; x < N; x++)
            for (int yb = 0; yb < 8 / U; yb++) {
                for (int t = 0; t < NT13; t++) p1_z1_single<R1, U, NT13>(t, in, x, yb, S.data());
                for (int t = 0; t < NT13; t++) {
                    cplx twr[8];
                    load_twr<R1>(t, twr);
                    p13_z8<R1, U, NT13, -1, TWREG>(t, S.data(), T.data(), twr);
                }
                for (int t = 0; t < NT13; t++) p1_y1<R1, U, NT13>(t, S.data(), out, x, yb);
            }
        for (int k1y = 0; k1y < R1; k1y++)
            for (int zb = 0; zb < N / Z; zb++) {
                cplx* Wt = out + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
                p2_copy_rows<R1, Z>(S2.data(), Wt, true);
                for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, -1>(t, S2.data(), k1y);
                for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, -1>(t, S2.data());
                for (int t = 0; t < NT2; t++) p2_x8_half<R1, Z, NT2, -1>(t, S2.data());
                p2_copy_rows<R1, Z>(S2.data(), Wt, false);
            }
    } else {
        for (int k1y = 0; k1y < R1; k1y++)
            for (int zb = 0; zb < N / Z; zb++) {
                cplx* Wt = in + ((size_t)k1y * (N / Z) + zb) * ((size_t)N * 8 * Z);
                p2_copy_rows<R1, Z>(S2.data(), Wt, true);
                for (int t = 0; t < NT2; t++) p2_x8_half<R1, Z, NT2, +1>(t, S2.data());
                for (int t = 0; t < NT2; t++) p2_xR<R1, Z, NT2, +1>(t, S2.data());
                for (int t = 0; t < NT2; t++) p2_y8<R1, Z, NT2, +1>(t, S2.data(), k1y);
                p2_copy_rows<R1, Z>(S2.data(), Wt, false);
            }
        for (int x = 0; x < N; x++)
            for (int yb = 0; yb < 8 / U3; yb++) {
                for (int t = 0; t < NT3; t++) p3_y2inv<R1, U3, NT3>(t, in, x, yb, S.data());
                for (int t = 0; t < NT3; t++) {
                    cplx twr[8];
                    load_twr<R1>(t, twr);
                    p13_z8<R1, U3, NT3, +1, TWREG>(t, S.data(), T.data(), twr);
                }
                for (int t = 0; t < NT3; t++) p3_zinv2_store<R1, U3, NT3>(t, S.data(), out, x, yb);
            }
    }
}
template <int R1>
static void emu_findex(int64_t* idx) {
    constexpr int N = 8 * R1;
    for (int kx = 0; kx < N; kx++)
        for (int ky = 0; ky < N; ky++)
            for (int kz = 0; kz < N; kz++) idx[((size_t)kx * N + ky) * N + kz] = (int64_t)findex<R1>(kx, ky, kz);
}
}  // namespace exx

using namespace exx;

extern "C" {
// in-register codelet: inout = R complex numbers, sign -1 forward / +1 unnormalised inverse
int exx_emu_dft(int R, int sign, double* inout) {
    cplx* v = (cplx*)inout;
#define CASE(r)                 \
    case r:                     \
        if (sign < 0)           \
            dft<r, -1>(v);      \
        else                    \
            dft<r, +1>(v);      \
        return 0;
    switch (R) {
        CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(8) CASE(9) CASE(10) CASE(12) CASE(16)
    default: return -1;
    }
#undef CASE
}

// one pair evaluation through the three fused passes on the CPU: acc += -wf * u_m * IFFT[K' FFT[conj(u_m) u_n]]
// (un, um, acc, work: N^3 complex each, 16-byte aligned; Knat: N^3 doubles in natural C order), N = 8 R1
int exx_emu_pair(int R1, const double* un, const double* um, const double* Knat, double wf, double* acc, double* work) {
    fill_tw();
    switch (R1) {
    case 2: emu_pair<2>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 4: emu_pair<4>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 5: emu_pair<5>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 10: emu_pair<10>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 6: emu_pair<6>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 8: emu_pair<8>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 9: emu_pair<9>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 12: emu_pair<12>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    case 16: emu_pair<16>((const cplx*)un, (const cplx*)um, Knat, wf, (acc_c*)acc, (cplx*)work); return 0;
    default: return -1;
    }
}

// the dual sweep of a ta x tb batch (see emu_dual); returns -2 where the grid has no dual kernel (RG = 0)
int exx_emu_dual(int R1, int ta, int tb, const double* ua, const double* ub, const double* Knat, const double* coef_a, const double* coef_b,
                 const unsigned* ev, const unsigned* bside, unsigned amask, double* acc_a, double* acc_b) {
    fill_tw();
    switch (R1) {
#define EXX_EMU_D(r)                                                                                                             \
    case r:                                                                                                                      \
        if (FusedCfg<r>::RG == 0) return -2;                                                                                     \
        emu_dual<r>(ta, tb, (const cplx*)ua, (const cplx*)ub, Knat, coef_a, coef_b, ev, bside, amask, (acc_c*)acc_a, (acc_c*)acc_b); \
        return 0;
        EXX_EMU_D(2) EXX_EMU_D(4) EXX_EMU_D(5) EXX_EMU_D(10) EXX_EMU_D(6) EXX_EMU_D(8) EXX_EMU_D(9) EXX_EMU_D(12) EXX_EMU_D(16)
#undef EXX_EMU_D
    default: return -1;
    }
}

// sum_g K(g) |FFT[conj(u_m) u_n](g)|^2 through the energy route's phases
int exx_emu_pair_energy(int R1, const double* un, const double* um, const double* Knat, double* work, double* e_out) {
    fill_tw();
    switch (R1) {
#define EXX_EMU_E(r) \
    case r: *e_out = emu_pair_energy<r>((const cplx*)un, (const cplx*)um, Knat, (cplx*)work); return 0;
        EXX_EMU_E(2) EXX_EMU_E(4) EXX_EMU_E(5) EXX_EMU_E(10) EXX_EMU_E(6) EXX_EMU_E(8) EXX_EMU_E(9) EXX_EMU_E(12) EXX_EMU_E(16)
#undef EXX_EMU_E
    default: return -1;
    }
}

// plain 3-D transform through the fused passes (see emu_fft); findex_out (optional, N^3 int64) receives the F-layout index of
// every natural frequency index
int exx_emu_fft(int R1, int sign, double* in, double* out, int64_t* findex_out) {
    fill_tw();
#define CASE(r)                                         \
    case r:                                             \
        emu_fft<r>(sign, (cplx*)in, (cplx*)out);        \
        if (findex_out) emu_findex<r>(findex_out);      \
        return 0;
    switch (R1) {
        CASE(2) CASE(4) CASE(5) CASE(10) CASE(6) CASE(8) CASE(9) CASE(12) CASE(16)
    default: return -1;
    }
#undef CASE
}
}
