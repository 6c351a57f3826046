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
            std::vector<cplx> G2((size_t)IT3 * R1 * NT3);
            if (STAGE3) {  // per-thread staging slots, as pass_c_kernel uses them
                std::vector<cplx> G((size_t)((U3 * N + NT3 - 1) / NT3) * R1 * NT3);
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
