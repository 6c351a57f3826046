// exx_dft.h — complex fp64 helpers and in-register DFT codelets (R = 2,3,4,5,6,8,9,10,12,16) used by the fused passes.
// Product code: shares nothing with oracle/.  Everything here is __host__ __device__ so that the same index and
// butterfly logic can be executed on the CPU by tests/test_fused_host_emulation.py (host logic test, no GPU).
//
// Convention: dft_fwd<R>(v) replaces v[0..R) by X[k] = sum_n v[n] exp(-2 pi i n k / R), natural order in and out
// (the forward sign of S3).  dft<R,+1> is the unnormalised inverse (S5), obtained by swapping
// real and imaginary parts around the forward codelet (register renaming, no arithmetic).
//
// The header is written against the scalar type `real` of the enclosing mode: it may be included once per mode, each time
// with EXX_NS (namespace) and EXX_REAL (double or float) defined — the fp64 product path uses exx / double; the mixed-precision
// pair pipeline includes it a second time as exx32 / float.
#ifndef EXX_HD
#if defined(__CUDACC__)
#define EXX_HD __host__ __device__ __forceinline__
#else
#define EXX_HD inline
#endif
#endif
#ifndef EXX_NS
#define EXX_NS exx
#define EXX_REAL double
#endif
#define EXX_RC(x) ((real)(x))

namespace EXX_NS {

typedef EXX_REAL real;
struct alignas(2 * sizeof(EXX_REAL)) cplx {
    real x, y;
};

EXX_HD cplx mk(real x, real y) {
    cplx r;
    r.x = x;
    r.y = y;
    return r;
}
EXX_HD cplx operator+(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
EXX_HD cplx operator-(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
EXX_HD cplx operator*(cplx a, cplx b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
EXX_HD cplx mul_conj_b(cplx a, cplx b) { return mk(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a * conj(b)
EXX_HD cplx conj_mul(cplx a, cplx b) { return mk(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }    // conj(a) * b
EXX_HD cplx scale(real s, cplx a) { return mk(s * a.x, s * a.y); }
EXX_HD cplx mul_mi(cplx a) { return mk(a.y, -a.x); }  // a * (-i)
EXX_HD cplx mul_pi(cplx a) { return mk(-a.y, a.x); }  // a * (+i)
EXX_HD cplx mulc(cplx a, real cr, real ci) { return mk(a.x * cr - a.y * ci, a.x * ci + a.y * cr); }  // a * (cr + i ci)

#ifndef EXX_HS3
#define EXX_HS3 0.86602540378443864676372317075294   /* sqrt(3)/2 */
#define EXX_RH2 0.70710678118654752440084436210485   /* sqrt(1/2) */
#define EXX_C16 0.92387953251128675612818318939679   /* cos(pi/8) */
#define EXX_S16 0.38268343236508977172845998403040   /* sin(pi/8) */
#define EXX_C9_1 0.76604444311897803520239265055542  /* cos(2 pi/9) */
#define EXX_S9_1 0.64278760968653932632264340990726  /* sin(2 pi/9) */
#define EXX_C9_2 0.17364817766693034885171662676931  /* cos(4 pi/9) */
#define EXX_S9_2 0.98480775301220805936674302458952  /* sin(4 pi/9) */
#define EXX_C9_4 (-0.93969262078590838405410927732473) /* cos(8 pi/9) */
#define EXX_S9_4 0.34202014332566873304409961468226  /* sin(8 pi/9) */
#endif

EXX_HD void bf2(cplx& a, cplx& b) {
    cplx t = a - b;
    a = a + b;
    b = t;
}
EXX_HD void bf3(cplx& a, cplx& b, cplx& c) {  // forward 3-point DFT
    cplx t1 = b + c, t2 = b - c;
    cplx m = mk(a.x - EXX_RC(0.5) * t1.x, a.y - EXX_RC(0.5) * t1.y);
    cplx r = mk(EXX_RC(EXX_HS3) * t2.y, -EXX_RC(EXX_HS3) * t2.x);  // (-i) (sqrt3/2) t2
    a = a + t1;
    b = m + r;
    c = m - r;
}
EXX_HD void bf4(cplx& a, cplx& b, cplx& c, cplx& d) {  // forward 4-point DFT
    cplx t0 = a + c, t1 = a - c, t2 = b + d, t3 = mul_mi(b - d);
    a = t0 + t2;
    c = t0 - t2;
    b = t1 + t3;
    d = t1 - t3;
}

template <int R>
struct Dft;  // Dft<R>::fwd(v): forward DFT of v[0..R), natural order

template <>
struct Dft<2> {
    static EXX_HD void fwd(cplx* v) { bf2(v[0], v[1]); }
};
template <>
struct Dft<3> {
    static EXX_HD void fwd(cplx* v) { bf3(v[0], v[1], v[2]); }
};
template <>
struct Dft<4> {
    static EXX_HD void fwd(cplx* v) { bf4(v[0], v[1], v[2], v[3]); }
};
template <>
struct Dft<5> {
    // prime size: p_n = x_n + x_{5-n}, m_n = x_n - x_{5-n};  X_k = x_0 + sum_n p_n cos(2 pi n k/5) - i sum_n m_n sin(2 pi n k/5),
    // X_{5-k} the same with + i
    static EXX_HD void fwd(cplx* v) {
        constexpr double C[5] = {1, 0.309016994374947451262869435595348477, -0.809016994374947340240566973079694435, -0.80901699437494756228517189811100252, 0.309016994374947229218264510564040393};
        constexpr double S[5] = {0, 0.95105651629515353118193843329208903, 0.587785252292473248125759255344746634, -0.58778525229247302608115433031343855, -0.951056516295153642204240895807743073};
        cplx p1 = v[1] + v[4], m1 = v[1] - v[4], p2 = v[2] + v[3], m2 = v[2] - v[3], x0 = v[0];
        v[0] = x0 + p1 + p2;
#pragma unroll
        for (int k = 1; k <= 2; k++) {
            const real c1 = (real)C[k % 5], c2 = (real)C[(2 * k) % 5], s1 = (real)S[k % 5], s2 = (real)S[(2 * k) % 5];
            cplx a = mk(x0.x + c1 * p1.x + c2 * p2.x, x0.y + c1 * p1.y + c2 * p2.y);
            cplx b = mk(s1 * m1.x + s2 * m2.x, s1 * m1.y + s2 * m2.y);
            v[k] = a + mul_mi(b);
            v[5 - k] = a - mul_mi(b);
        }
    }
};
template <>
struct Dft<6> {
    // n = 3 n1 + n2, k = k1 + 2 k2: 2-point over n1, twiddle W6^(n2 k1), 3-point over n2
    static EXX_HD void fwd(cplx* v) {
        bf2(v[0], v[3]);
        bf2(v[1], v[4]);
        bf2(v[2], v[5]);
        v[4] = mulc(v[4], 0.5, -EXX_HS3);
        v[5] = mulc(v[5], -0.5, -EXX_HS3);
        bf3(v[0], v[1], v[2]);  // k1 = 0: X[0], X[2], X[4]
        bf3(v[3], v[4], v[5]);  // k1 = 1: X[1], X[3], X[5]
        cplx x1 = v[3], x2 = v[1], x3 = v[4], x4 = v[2];
        v[1] = x1;
        v[2] = x2;
        v[3] = x3;
        v[4] = x4;
    }
};
template <>
struct Dft<8> {
    static EXX_HD void fwd(cplx* v) {
        bf4(v[0], v[2], v[4], v[6]);  // E[k] in v[0], v[2], v[4], v[6]
        bf4(v[1], v[3], v[5], v[7]);  // O[k] in v[1], v[3], v[5], v[7]
        cplx o1 = mk(EXX_RC(EXX_RH2) * (v[3].x + v[3].y), EXX_RC(EXX_RH2) * (v[3].y - v[3].x));   // O1 * W8^1
        cplx o2 = mul_mi(v[5]);                                                   // O2 * W8^2
        cplx o3 = mk(EXX_RC(EXX_RH2) * (v[7].y - v[7].x), -EXX_RC(EXX_RH2) * (v[7].x + v[7].y));  // O3 * W8^3
        cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
        v[0] = e0 + o0;
        v[4] = e0 - o0;
        v[1] = e1 + o1;
        v[5] = e1 - o1;
        v[2] = e2 + o2;
        v[6] = e2 - o2;
        v[3] = e3 + o3;
        v[7] = e3 - o3;
    }
};
template <>
struct Dft<9> {
    // n = 3 n1 + n2, k = k1 + 3 k2: 3-point over n1, twiddle W9^(n2 k1), 3-point over n2
    static EXX_HD void fwd(cplx* v) {
        bf3(v[0], v[3], v[6]);
        bf3(v[1], v[4], v[7]);
        bf3(v[2], v[5], v[8]);
        v[4] = mulc(v[4], EXX_C9_1, -EXX_S9_1);  // k1 = 1, n2 = 1: W9^1
        v[5] = mulc(v[5], EXX_C9_2, -EXX_S9_2);  // k1 = 1, n2 = 2: W9^2
        v[7] = mulc(v[7], EXX_C9_2, -EXX_S9_2);  // k1 = 2, n2 = 1: W9^2
        v[8] = mulc(v[8], EXX_C9_4, -EXX_S9_4);  // k1 = 2, n2 = 2: W9^4
        bf3(v[0], v[1], v[2]);  // k1 = 0: X[0], X[3], X[6]
        bf3(v[3], v[4], v[5]);  // k1 = 1: X[1], X[4], X[7]
        bf3(v[6], v[7], v[8]);  // k1 = 2: X[2], X[5], X[8]
        cplx t[9];
        for (int k1 = 0; k1 < 3; k1++)
            for (int k2 = 0; k2 < 3; k2++) t[k1 + 3 * k2] = v[3 * k1 + k2];
        for (int k = 0; k < 9; k++) v[k] = t[k];
    }
};
template <>
struct Dft<10> {
    // n = 5 n1 + n2, k = k1 + 2 k2: 2-point over n1, twiddle W10^(n2 k1), 5-point over n2
    static EXX_HD void fwd(cplx* v) {
        constexpr double C[5] = {1, 0.809016994374947451262869435595348477, 0.309016994374947451262869435595348477, -0.309016994374947340240566973079694435, -0.809016994374947340240566973079694435};
        constexpr double S[5] = {0, 0.587785252292473137103456792829092592, 0.95105651629515353118193843329208903, 0.951056516295153642204240895807743073, 0.587785252292473248125759255344746634};
#pragma unroll
        for (int n2 = 0; n2 < 5; n2++) bf2(v[n2], v[5 + n2]);
#pragma unroll
        for (int n2 = 1; n2 < 5; n2++) v[5 + n2] = mulc(v[5 + n2], (real)C[n2], (real)(-S[n2]));
        Dft<5>::fwd(v);      // k1 = 0: X[0], X[2], X[4], X[6], X[8]
        Dft<5>::fwd(v + 5);  // k1 = 1: X[1], X[3], X[5], X[7], X[9]
        cplx t[10];
#pragma unroll
        for (int k2 = 0; k2 < 5; k2++) {
            t[2 * k2] = v[k2];
            t[2 * k2 + 1] = v[5 + k2];
        }
#pragma unroll
        for (int k = 0; k < 10; k++) v[k] = t[k];
    }
};
template <>
struct Dft<12> {
    // n = 4 n1 + n2, k = k1 + 3 k2: 3-point over n1, twiddle W12^(n2 k1), 4-point over n2
    static EXX_HD void fwd(cplx* v) {
        bf3(v[0], v[4], v[8]);
        bf3(v[1], v[5], v[9]);
        bf3(v[2], v[6], v[10]);
        bf3(v[3], v[7], v[11]);
        v[5] = mulc(v[5], EXX_HS3, -0.5);     // k1 = 1: W12^1
        v[6] = mulc(v[6], 0.5, -EXX_HS3);     //         W12^2
        v[7] = mul_mi(v[7]);                  //         W12^3
        v[9] = mulc(v[9], 0.5, -EXX_HS3);     // k1 = 2: W12^2
        v[10] = mulc(v[10], -0.5, -EXX_HS3);  //         W12^4
        v[11] = mk(-v[11].x, -v[11].y);       //         W12^6
        bf4(v[0], v[1], v[2], v[3]);    // k1 = 0: X[0], X[3], X[6], X[9]
        bf4(v[4], v[5], v[6], v[7]);    // k1 = 1: X[1], X[4], X[7], X[10]
        bf4(v[8], v[9], v[10], v[11]);  // k1 = 2: X[2], X[5], X[8], X[11]
        cplx t[12];
        for (int k1 = 0; k1 < 3; k1++)
            for (int k2 = 0; k2 < 4; k2++) t[k1 + 3 * k2] = v[4 * k1 + k2];
        for (int k = 0; k < 12; k++) v[k] = t[k];
    }
};
template <>
struct Dft<16> {
    // n = 4 n1 + n2, k = k1 + 4 k2: 4-point over n1, twiddle W16^(n2 k1), 4-point over n2
    static EXX_HD void fwd(cplx* v) {
        bf4(v[0], v[4], v[8], v[12]);
        bf4(v[1], v[5], v[9], v[13]);
        bf4(v[2], v[6], v[10], v[14]);
        bf4(v[3], v[7], v[11], v[15]);
        v[5] = mulc(v[5], EXX_C16, -EXX_S16);                                                    // W16^1
        v[6] = mk(EXX_RC(EXX_RH2) * (v[6].x + v[6].y), EXX_RC(EXX_RH2) * (v[6].y - v[6].x));                     // W16^2
        v[7] = mulc(v[7], EXX_S16, -EXX_C16);                                                    // W16^3
        v[9] = mk(EXX_RC(EXX_RH2) * (v[9].x + v[9].y), EXX_RC(EXX_RH2) * (v[9].y - v[9].x));                     // W16^2
        v[10] = mul_mi(v[10]);                                                                   // W16^4
        v[11] = mk(EXX_RC(EXX_RH2) * (v[11].y - v[11].x), -EXX_RC(EXX_RH2) * (v[11].x + v[11].y));               // W16^6
        v[13] = mulc(v[13], EXX_S16, -EXX_C16);                                                  // W16^3
        v[14] = mk(EXX_RC(EXX_RH2) * (v[14].y - v[14].x), -EXX_RC(EXX_RH2) * (v[14].x + v[14].y));               // W16^6
        v[15] = mulc(v[15], -EXX_C16, EXX_S16);                                                  // W16^9
        bf4(v[0], v[1], v[2], v[3]);
        bf4(v[4], v[5], v[6], v[7]);
        bf4(v[8], v[9], v[10], v[11]);
        bf4(v[12], v[13], v[14], v[15]);
        cplx t[16];
        for (int k1 = 0; k1 < 4; k1++)
            for (int k2 = 0; k2 < 4; k2++) t[k1 + 4 * k2] = v[4 * k1 + k2];
        for (int k = 0; k < 16; k++) v[k] = t[k];
    }
};

// SIGN = -1: forward (e^{-i}); SIGN = +1: unnormalised inverse via the real/imaginary swap identity
template <int R, int SIGN>
EXX_HD void dft(cplx* v) {
    if (SIGN < 0) {
        Dft<R>::fwd(v);
    } else {
#pragma unroll
        for (int i = 0; i < R; i++) v[i] = mk(v[i].y, v[i].x);
        Dft<R>::fwd(v);
#pragma unroll
        for (int i = 0; i < R; i++) v[i] = mk(v[i].y, v[i].x);
    }
}

}  // namespace EXX_NS
