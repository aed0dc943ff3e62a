// Fused x-line kernel (SURVEY.md 8(a) rows a4 (x part), a5, a6 (x part); north_star subsystems (1) and (2)).
// One "line" = (plane j, z index q, member e).  For every line the kernel
//   * reads the 8 mixed (kx, z) fields u v w Du Dw uz vz wz written by k_zinv, each exactly once per retained kx,
//   * forms the 11 physical fields u, v, w, their x/z derivatives and Du, Dw with 6 Hermitian two-for-one complex
//     inverse FFTs along x (x-derivatives = i kx folded into the packing; dv/dy = -du/dx - dw/dz pointwise, which
//     holds exactly at interior rows for the u, w of Eq. 17-18),
//   * forms the convective products u.grad u_i and the x-sums of u v, w v (Eq. 6-7) in registers,
//   * returns (u.grad)u, (u.grad)v, (u.grad)w on the retained kx with 2 forward FFTs.
// Nothing in physical space ever reaches HBM.
//
// Thread mapping: a line is shared by SL "slots"; every slot owns R1 x-points of each physical field in registers.
// A CTA is one group of SL slots x TPS lanes (lanes = members, or members x lines when E < TPS), 32..96 threads,
// so the four-step exchanges need only a warp- or CTA-local barrier and many independent groups are resident per SM.
#include "dns_internal.h"
#include "fft_codelets.cuh"

using namespace dnsfft;

namespace {

template <int BT> __device__ __forceinline__ void group_sync() {
    if (BT == 32) __syncwarp(); else __syncthreads();
}

// row pitch (in double2) of an exchange buffer with `cols` columns of TPS lanes: for TPS = 4 two slots share a
// quarter-warp, so consecutive rows must start 64 B apart modulo 128 B to stay bank-conflict free
constexpr int line_pitch(int cols, int TPS) {
    return TPS >= 8 ? cols * TPS : cols * TPS + ((TPS - (cols * TPS) % 8 + 8) % 8);
}

// mode index loaded for padded position pos: n (positive side), M - pos (negative side, conjugated) or -1 (zero)
template <int M, int NKX> __device__ __forceinline__ int pos_mode(int pos) {
    return pos < NKX ? pos : (pos > M - NKX ? M - pos : -1);
}

// Field pairing of the six complex transforms Z = A + iB (A, B real in x):
//   C = 0: (v, dv/dx)   1: (u, du/dx)   2: (w, dw/dx)   3: (Du, du/dz)   4: (Dw, dw/dz)   5: (dv/dz, -)
// I8 field order: 0 u, 1 v, 2 w, 3 Du, 4 Dw, 5 uz, 6 vz, 7 wz.
template <int C> struct LinePair;
template <> struct LinePair<0> { static constexpr int fa = 1, fb = -1; };
template <> struct LinePair<1> { static constexpr int fa = 0, fb = -1; };
template <> struct LinePair<2> { static constexpr int fa = 2, fb = -1; };
template <> struct LinePair<3> { static constexpr int fa = 3, fb = 5; };
template <> struct LinePair<4> { static constexpr int fa = 4, fb = 7; };
template <> struct LinePair<5> { static constexpr int fa = 6, fb = -1; };

template <int C, int R1, int R2>
__device__ __forceinline__ void line_load(const double2* __restrict__ src, size_t fstride, int E, int sl, bool act,
                                          double2 (&ra)[R2], double2 (&rb)[R2]) {
    constexpr int M = R1 * R2, NKX = M / 3;
#pragma unroll
    for (int i2 = 0; i2 < R2; ++i2) {
        const int lo = R1 * i2, hi = R1 * i2 + R1 - 1;
        if (lo >= NKX && hi <= M - NKX) continue;               // statically zero padding
        const int n = pos_mode<M, NKX>(sl + R1 * i2);
        ra[i2] = make_double2(0.0, 0.0);
        if (LinePair<C>::fb >= 0) rb[i2] = make_double2(0.0, 0.0);
        if (act && n >= 0) {
            ra[i2] = __ldg(src + (size_t)LinePair<C>::fa * fstride + (size_t)n * E);
            if (LinePair<C>::fb >= 0) rb[i2] = __ldg(src + (size_t)LinePair<C>::fb * fstride + (size_t)n * E);
        }
    }
}

// inverse pass A: pack Z(pos), R2-point DFTs over pos = sl + R1*i2, twiddle, store row sl
template <int C, int R1, int R2, int TPS>
__device__ __forceinline__ void line_pass_a(const double2 (&ra)[R2], const double2 (&rb)[R2], const double* kxs,
                                            const double2* tws, double2* buf, int sl, int lis) {
    constexpr int M = R1 * R2, NKX = M / 3, PI = line_pitch(R2, TPS);
    double2 a[R2];
#pragma unroll
    for (int i2 = 0; i2 < R2; ++i2) {
        const int lo = R1 * i2, hi = R1 * i2 + R1 - 1;
        if (lo >= NKX && hi <= M - NKX) { a[i2] = make_double2(0.0, 0.0); continue; }
        const int pos = sl + R1 * i2;
        const int n = pos_mode<M, NKX>(pos);
        const bool neg = pos >= NKX;
        const double2 A = ra[i2];
        double2 z;
        if (LinePair<C>::fb >= 0) {
            const double2 B = rb[i2];
            // Z(n) = A + iB ; Z(0) = (Re A, Re B) ; Z(M - n) = conj(A) + i conj(B)
            z = neg ? make_double2(A.x + B.y, B.x - A.y)
                    : (pos == 0 ? make_double2(A.x, B.x) : make_double2(A.x - B.y, A.y + B.x));
        } else if (C < 3) {
            // B = i kx A:  Z(n) = (1 - kx) A ; Z(M - n) = (1 + kx) conj(A)
            const double kx = n >= 0 ? kxs[n] : 0.0;
            z = neg ? make_double2((1.0 + kx) * A.x, -(1.0 + kx) * A.y)
                    : (pos == 0 ? make_double2(A.x, 0.0) : make_double2((1.0 - kx) * A.x, (1.0 - kx) * A.y));
        } else {
            z = neg ? make_double2(A.x, -A.y) : (pos == 0 ? make_double2(A.x, 0.0) : A);
        }
        a[i2] = cswap(z);                                       // inverse transform by the swap identity
    }
    DFT<R2>::run(a);
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) buf[sl * PI + k2 * TPS + lis] = cmul(a[k2], tws[sl * k2]);
}

// ------------------------------------------------------------------------------------------------ the kernel
// grid = Ni * nblk_q * ntile_e ; block = SL * TPS
template <int R1, int R2, int SL, int TPS, int MINB>
__global__ void __launch_bounds__(SL * TPS, MINB) k_line(DnsDev d, int etlog, int LQ) {
    constexpr int M = R1 * R2, NKX = M / 3, BT = SL * TPS;
    constexpr int PI = line_pitch(R2, TPS), PF = line_pitch(R1, TPS);
    constexpr int BUF = (R1 * PI > R2 * PF) ? R1 * PI : R2 * PF;
    __shared__ double2 tws[M];
    __shared__ double kxs[NKX];
    __shared__ double2 buf[2][BUF];
    __shared__ double2 exch[NKX * TPS];
    __shared__ double2 red[SL * TPS];

    const int t = threadIdx.x, sl = t / TPS, lis = t % TPS;
    const int ET = 1 << etlog, el = lis & (ET - 1), lc = lis >> etlog, LC = TPS >> etlog;
    const int ntile_e = (d.E + ET - 1) >> etlog, nblk_q = (d.Mz + LC * LQ - 1) / (LC * LQ);
    int b = blockIdx.x;
    const int te = b % ntile_e; b /= ntile_e;
    const int bq = b % nblk_q;  b /= nblk_q;
    const int j = b + 1;                                    // interior planes only (wall planes give N = 0 exactly)
    const int e = te * ET + el;
    const bool eok = e < d.E;
    for (int i = t; i < M; i += BT) tws[i] = d.twx[i];
    for (int i = t; i < NKX; i += BT) kxs[i] = d.kx[i];
    __syncthreads();
    const size_t fstride = d.Isz;
    const int E = d.E;

    for (int qi = 0; qi < LQ; ++qi) {
        const int q = (bq * LQ + qi) * LC + lc;
        const bool lok = eok && q < d.Mz;
        const size_t base = (((size_t)j * d.Mz + (lok ? q : 0)) * NKX) * E + (eok ? e : 0);
        const double2* src = d.I8 + base;
        const bool act = lok && sl < R1;
        double u[R1], v[R1], w[R1], Nu[R1], Nv[R1], Nw[R1];
        double suv = 0.0, swv = 0.0;
        double2 ra[R2], rb[R2];

#define DNS_LINE_INV(C, BODY)                                                              \
        if (sl < R1) line_pass_a<C, R1, R2, TPS>(ra, rb, kxs, tws, buf[(C) & 1], sl, lis); \
        group_sync<BT>();                                                                  \
        if ((C) < 5) line_load<((C) < 5 ? (C) + 1 : 5), R1, R2>(src, fstride, E, sl, act, ra, rb); \
        if (sl < R2) {                                                                     \
            double2 x[R1];                                                                 \
            _Pragma("unroll")                                                              \
            for (int i1 = 0; i1 < R1; ++i1) x[i1] = buf[(C) & 1][i1 * PI + sl * TPS + lis]; \
            DFT<R1>::run(x);                                                               \
            _Pragma("unroll")                                                              \
            for (int k = 0; k < R1; ++k) {                                                 \
                const double fa = x[k].y, fb = x[k].x; (void)fb;                           \
                BODY                                                                       \
            }                                                                              \
        }

        line_load<0, R1, R2>(src, fstride, E, sl, act, ra, rb);
        DNS_LINE_INV(0, { v[k] = fa; Nv[k] = fb; })
        DNS_LINE_INV(1, { u[k] = fa; Nu[k] = fa * fb; Nv[k] = fa * Nv[k] - v[k] * fb; suv += fa * v[k]; })
        DNS_LINE_INV(2, { w[k] = fa; Nw[k] = u[k] * fb; swv += fa * v[k]; })
        DNS_LINE_INV(3, { Nu[k] += v[k] * fa; Nu[k] += w[k] * fb; })
        DNS_LINE_INV(4, { Nw[k] += v[k] * fa; Nw[k] += w[k] * fb; Nv[k] -= v[k] * fb; })
        DNS_LINE_INV(5, { Nv[k] += w[k] * fa; })
#undef DNS_LINE_INV

        // forward transforms of W1 = Nu + i Nv and W2 = Nw, factorisation (R2, R1): pass A on the registers
        group_sync<BT>();                                   // pass B of transform 5 has finished reading buf[1]
        if (sl < R2) {
            double2 a1[R1], a2[R1];
#pragma unroll
            for (int k = 0; k < R1; ++k) { a1[k] = make_double2(Nu[k], Nv[k]); a2[k] = make_double2(Nw[k], 0.0); }
            DFT<R1>::run(a1);
            DFT<R1>::run(a2);
#pragma unroll
            for (int k = 0; k < R1; ++k) {
                const double2 tw = tws[sl * k];
                buf[0][sl * PF + k * TPS + lis] = cmul(a1[k], tw);
                buf[1][sl * PF + k * TPS + lis] = cmul(a2[k], tw);
            }
            red[sl * TPS + lis] = make_double2(suv, swv);
        }
        group_sync<BT>();
        double2 x1[R2], x2[R2];
        if (sl < R1) {                                      // forward pass B: output n = sl + R1*k
#pragma unroll
            for (int i = 0; i < R2; ++i) { x1[i] = buf[0][i * PF + sl * TPS + lis]; x2[i] = buf[1][i * PF + sl * TPS + lis]; }
            DFT<R2>::run(x1);
            DFT<R2>::run(x2);
#pragma unroll
            for (int k = 0; k < R2; ++k) {                  // hand Z1(M - n) to the slot that owns n
                const int lo = R1 * k, hi = R1 * k + R1 - 1;
                if (hi <= M - NKX) continue;
                const int pos = sl + R1 * k;
                if (lo > M - NKX || pos > M - NKX) exch[(M - pos) * TPS + lis] = x1[k];
            }
        }
        group_sync<BT>();
        if (sl < R1 && lok) {
            double2* dst = d.I3 + base;
#pragma unroll
            for (int k = 0; k < R2; ++k) {
                const int lo = R1 * k;
                if (lo >= NKX) continue;
                const int n = sl + R1 * k;
                if (n < NKX) {
                    const double2 zp = x1[k], zm = n == 0 ? x1[k] : exch[n * TPS + lis];
                    // (u.grad)u = (Z(n) + conj Z(-n))/2 ; (u.grad)v = (Z(n) - conj Z(-n))/(2i) ; (u.grad)w = Z2(n)
                    dst[(size_t)n * E] = make_double2(0.5 * (zp.x + zm.x), 0.5 * (zp.y - zm.y));
                    dst[fstride + (size_t)n * E] = make_double2(0.5 * (zp.y + zm.y), 0.5 * (zm.x - zp.x));
                    dst[2 * fstride + (size_t)n * E] = n == 0 ? make_double2(x2[k].x, 0.0) : x2[k];
                }
            }
            if (sl == 0) {
                double sa = 0.0, sb = 0.0;
#pragma unroll
                for (int s = 0; s < R2; ++s) { sa += red[s * TPS + lis].x; sb += red[s * TPS + lis].y; }
                d.uvpart[((size_t)j * d.Mz + q) * E + e] = make_double2(sa, sb);
            }
        }
    }
}

template <int R1, int R2, int SL, int TPS, int MINB> void line_launch(dns_plan* p) {
    const DnsDev& d = p->d;
    int ET = 1;
    while (ET < TPS && ET < d.E) ET <<= 1;                  // members per group (power of two <= TPS)
    const int etlog = __builtin_ctz(ET), LC = TPS / ET;
    const int LQ = d.Mz % (LC * 4) == 0 ? 4 : (d.Mz % (LC * 3) == 0 ? 3 : 4);
    const int nblk_q = (d.Mz + LC * LQ - 1) / (LC * LQ);
    dim3 grid((unsigned)(d.Ni * nblk_q * ((d.E + ET - 1) / ET)));
    k_line<R1, R2, SL, TPS, MINB><<<grid, SL * TPS, 0, p->stream>>>(d, etlog, LQ);
}

}  // namespace

void launch_line(dns_plan* p) {
    switch (p->d.Mx) {
        case 18: line_launch<3, 6, 8, 4, 16>(p); break;
        case 24: line_launch<4, 6, 8, 4, 16>(p); break;
        case 27: line_launch<3, 9, 12, 8, 5>(p); break;
        case 36: line_launch<6, 6, 8, 4, 16>(p); break;
        case 48: line_launch<6, 8, 8, 4, 16>(p); break;
        case 54: line_launch<6, 9, 12, 8, 5>(p); break;
        case 72: line_launch<6, 12, 12, 8, 5>(p); break;
        case 81: line_launch<9, 9, 12, 8, 4>(p); break;
        case 96: line_launch<8, 12, 12, 8, 3>(p); break;
        case 108: line_launch<9, 12, 12, 8, 3>(p); break;
        default: break;
    }
}
