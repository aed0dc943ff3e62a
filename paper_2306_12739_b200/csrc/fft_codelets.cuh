// Register-resident small DFT codelets (forward sign, exp(-2 pi i jk/R)) for the x/z transforms of the
// 3/2-rule padded grid (PAPER.md:182, :225 `fft2_cuben`).
// Lengths M = 3N/2 in 16..128 are 2^a 3^b, handled as M = R1*R2 with R1, R2 in {3,4,6,8,9,12,16}: every
// thread runs one R-point codelet per pass entirely in registers; passes exchange through shared memory.
// Inverse transforms use the swap identity  IDFT(x) = swap(DFT(swap(x))), swap(a+ib) = b+ia, so only forward
// codelets and forward twiddles exist.
#pragma once
#include "fft_consts.h"

#define DNS_HD __host__ __device__ __forceinline__

namespace dnsfft {

DNS_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
DNS_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
DNS_HD double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
DNS_HD double2 cswap(double2 a) { return make_double2(a.y, a.x); }
DNS_HD double2 cconj(double2 a) { return make_double2(a.x, -a.y); }
DNS_HD double2 cscale(double2 a, double s) { return make_double2(a.x * s, a.y * s); }
DNS_HD double2 cmul_i(double2 a) { return make_double2(-a.y, a.x); }     // * (+i)
DNS_HD double2 cmul_mi(double2 a) { return make_double2(a.y, -a.x); }    // * (-i)

// cos / sin (2 pi k / R) from the generated literal tables; k is a compile-time constant after unrolling
template <int R> struct TW;
#define DNS_DEF_TW(R)                                                                                       \
    template <> struct TW<R> {                                                                              \
        DNS_HD static constexpr double c(int k) { constexpr double t[R] = DNS_TWC##R; return t[k]; }        \
        DNS_HD static constexpr double s(int k) { constexpr double t[R] = DNS_TWS##R; return t[k]; }        \
    };
DNS_DEF_TW(8)
DNS_DEF_TW(9)
DNS_DEF_TW(12)
DNS_DEF_TW(16)
DNS_DEF_TW(18)
DNS_DEF_TW(24)
DNS_DEF_TW(36)
template <> struct TW<6> {
    DNS_HD static constexpr double c(int k) { return TW<12>::c(2 * k); }
    DNS_HD static constexpr double s(int k) { return TW<12>::s(2 * k); }
};

// a * exp(-2 pi i k / R), trivial rotations folded at compile time
template <int R> DNS_HD double2 twmul(double2 a, int k) {
    k %= R;
    if (k == 0) return a;
    if (4 * k == R) return cmul_mi(a);
    if (2 * k == R) return make_double2(-a.x, -a.y);
    if (4 * k == 3 * R) return cmul_i(a);
    return cmul(a, make_double2(TW<R>::c(k), -TW<R>::s(k)));
}

template <int R> struct DFT;

template <> struct DFT<1> {
    DNS_HD static void run(double2 (&)[1]) {}
};
template <> struct DFT<2> {
    DNS_HD static void run(double2 (&x)[2]) {
        double2 a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
};
template <> struct DFT<3> {
    DNS_HD static void run(double2 (&x)[3]) {
        const double s3 = 0.86602540378443864676;
        double2 t1 = cadd(x[1], x[2]);
        double2 d = csub(x[1], x[2]);
        double2 m1 = make_double2(fma(-0.5, t1.x, x[0].x), fma(-0.5, t1.y, x[0].y));
        double2 m2 = make_double2(s3 * d.y, -s3 * d.x);          // -i (sqrt3/2) (x1 - x2)
        x[0] = cadd(x[0], t1);
        x[1] = cadd(m1, m2);
        x[2] = csub(m1, m2);
    }
};
template <> struct DFT<4> {
    DNS_HD static void run(double2 (&x)[4]) {
        double2 a = cadd(x[0], x[2]), b = csub(x[0], x[2]);
        double2 c = cadd(x[1], x[3]), d = cmul_mi(csub(x[1], x[3]));   // -i (x1 - x3)
        x[0] = cadd(a, c);
        x[1] = cadd(b, d);
        x[2] = csub(a, c);
        x[3] = csub(b, d);
    }
};

// Cooley-Tukey composite: i = i1 + R1 i2, k = k2 + R2 k1
template <int R1, int R2> DNS_HD void dft_ct(double2 (&x)[R1 * R2]) {
    constexpr int R = R1 * R2;
    double2 y[R];
#pragma unroll
    for (int i1 = 0; i1 < R1; ++i1) {
        double2 t[R2];
#pragma unroll
        for (int i2 = 0; i2 < R2; ++i2) t[i2] = x[i1 + R1 * i2];
        DFT<R2>::run(t);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) y[i1 * R2 + k2] = twmul<R>(t[k2], i1 * k2);
    }
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) {
        double2 t[R1];
#pragma unroll
        for (int i1 = 0; i1 < R1; ++i1) t[i1] = y[i1 * R2 + k2];
        DFT<R1>::run(t);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) x[k2 + R2 * k1] = t[k1];
    }
}
template <> struct DFT<6> { DNS_HD static void run(double2 (&x)[6]) { dft_ct<2, 3>(x); } };
template <> struct DFT<8> { DNS_HD static void run(double2 (&x)[8]) { dft_ct<2, 4>(x); } };
template <> struct DFT<9> { DNS_HD static void run(double2 (&x)[9]) { dft_ct<3, 3>(x); } };
template <> struct DFT<12> { DNS_HD static void run(double2 (&x)[12]) { dft_ct<3, 4>(x); } };
template <> struct DFT<16> { DNS_HD static void run(double2 (&x)[16]) { dft_ct<4, 4>(x); } };
// half lengths of the register-resident z transforms (kernels_fft.cu: two threads per line)
template <> struct DFT<18> { DNS_HD static void run(double2 (&x)[18]) { dft_ct<3, 6>(x); } };
template <> struct DFT<24> { DNS_HD static void run(double2 (&x)[24]) { dft_ct<3, 8>(x); } };
template <> struct DFT<36> { DNS_HD static void run(double2 (&x)[36]) { dft_ct<6, 6>(x); } };

}  // namespace dnsfft
