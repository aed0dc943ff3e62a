// Physical-space part of one stage (north_star subsystems (1) and (2)):
//   k_zinv : spectral (kx,kz) -> mixed (kx,z): zero-pad Nz -> Mz (3/2 rule), i kz multiply on load
//            for the z-derivatives, complex inverse FFT along z.
//   k_line : per (y, z) line and member: Hermitian two-for-one complex inverse FFTs along x of the 12 fields
//            u,v,w and their x,y,z derivatives (x-derivatives = i kx on load, dv/dy = -du/dx - dw/dz),
//            the convective products u.grad u_i and the plane sums of uv, wv (Eq. 6-7) in
//            registers, forward FFT along x of the three products; nothing physical ever reaches HBM.
//   k_zfwd : mixed -> spectral: forward FFT along z, truncation to the retained modes, 1/(Mx Mz).
// All FFTs are four-step M = R1*R2 with register codelets (fft_codelets.cuh); the ensemble index is the lane
// index, so every global access is a contiguous run of members (PAPER.md:167 turned into coalescing).
#include <cstdlib>

#include "dns_internal.h"
#include "fft_codelets.cuh"

using namespace dnsfft;

namespace {

__device__ __forceinline__ double2 ldg2(const double2* p) { return __ldg(p); }

// position in the padded length-M array -> index of the stored spanwise mode, or -1 (zero padding)
__device__ __forceinline__ int pos_to_mi(int pos, int M, int nzh, int nkz) {
    if (pos < nzh) return pos;
    if (pos > M - nzh) return pos - M + nkz;
    return -1;
}

// Input field f of the z-inverse transform.  Convective form: u, v, w, du/dy, dw/dy -- u, v, w also give
// their z-derivative (i kz on load), 8 mixed fields.  Rotational form (row f1): u, v, w, omega_x, omega_y = eta, omega_z,
// 6 mixed fields in that order, no derivative.
__device__ __forceinline__ const double2* zinv_src(const DnsDev& d, int f, const double2* vin, const double2* ein) {
    if (d.form == DNS_FORM_ROTATIONAL) return f == 0 ? d.uh : f == 1 ? vin : f == 2 ? d.wh : f == 3 ? d.dwh : f == 4 ? ein : d.duh;
    return f == 0 ? d.uh : f == 1 ? vin : f == 2 ? d.wh : f == 3 ? d.duh : d.dwh;
}

// ------------------------------------------------------------------------------------------------ z inverse
// grid.x = Ni * nblk_n * ntile_e, grid.y = input fields (5 convective, 6 rotational); block = 256
#ifndef DNS_FFT_MINB
#define DNS_FFT_MINB 2
#endif
template <int R1, int R2>
__global__ void __launch_bounds__(256, DNS_FFT_MINB) k_zinv(DnsDev d, const double2* __restrict__ vin, const double2* __restrict__ ein, int etlog, int NB) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = R1 * R2;
    extern __shared__ double2 sm[];
    const int ET = 1 << etlog, e_l = threadIdx.x & (ET - 1), slot = threadIdx.x >> etlog, nslots = blockDim.x >> etlog;
    const int ntile_e = (d.E + ET - 1) >> etlog, nblk_n = (d.nkx + NB - 1) / NB;
    int b = blockIdx.x;
    const int te = b % ntile_e; b /= ntile_e;
    const int bn = b % nblk_n;  b /= nblk_n;
    const int j = b + 1;                               // interior planes only: wall planes give N = 0 exactly
    const int f = blockIdx.y;
    const int e = te * ET + e_l, n0 = bn * NB;
    const bool eok = e < d.E;
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    const double2* src = zinv_src(d, f, vin, ein);
    const int nv = (!rot && f < 3) ? 2 : 1;            // convective: u, v, w also produce their z-derivative
    double2* tws = sm;                                 // [M] twiddles
    double2* buf = sm + M;                             // [NB*nv][M][ET]
    for (int i = threadIdx.x; i < M; i += blockDim.x) tws[i] = d.twz[i];
    __syncthreads();
    // pass A: R2-point DFTs over pos = i1 + R1*i2
    for (int item = slot; item < NB * R1; item += nslots) {
        const int nb = item / R1, i1 = item % R1, n = n0 + nb;
        double2 a[R2], az[R2];
#pragma unroll
        for (int i2 = 0; i2 < R2; ++i2) {
            const int mi = pos_to_mi(i1 + R1 * i2, M, d.nzh, d.nkz);
            double2 v = make_double2(0.0, 0.0);
            double kz = 0.0;
            if (mi >= 0 && n < d.nkx && eok) {
                v = ldg2(src + (((size_t)j * d.nkx + n) * d.nkz + mi) * d.E + e);
                kz = d.kz[mi];
            }
            a[i2] = cswap(v);                                          // inverse transform by the swap identity
            az[i2] = cswap(make_double2(-kz * v.y, kz * v.x));        // i kz v
        }
        DFT<R2>::run(a);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2)
            buf[((size_t)(nb * nv) * M + i1 * R2 + k2) * ET + e_l] = cmul(a[k2], tws[i1 * k2]);
        if (nv == 2) {
            DFT<R2>::run(az);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2)
                buf[((size_t)(nb * nv + 1) * M + i1 * R2 + k2) * ET + e_l] = cmul(az[k2], tws[i1 * k2]);
        }
    }
    __syncthreads();
    // pass B: R1-point DFTs, output q = k2 + R2*k1
    for (int item = slot; item < NB * nv * R2; item += nslots) {
        const int line = item / R2, k2 = item % R2, nb = line / nv, var = line % nv, n = n0 + nb;
        double2 x[R1];
#pragma unroll
        for (int i1 = 0; i1 < R1; ++i1) x[i1] = buf[((size_t)line * M + i1 * R2 + k2) * ET + e_l];
        DFT<R1>::run(x);
        if (n < d.nkx && eok) {
            const int fo = var ? 5 + f : f;
            double2* dst = d.I8 + (size_t)fo * d.Isz + dns_mix_off(d, j, 0, n, e);
            const size_t qs = ((size_t)d.ntl * d.nkx) << d.etl;
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) dst[(size_t)(k2 + R2 * k1) * qs] = cswap(x[k1]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ z forward
// grid.x = Ni * nblk_n * ntile_e, grid.y = 3 fields; block = 256
template <int R1, int R2>
__global__ void __launch_bounds__(256) k_zfwd(DnsDev d, int etlog, int NB) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = R1 * R2;
    extern __shared__ double2 sm[];
    const int ET = 1 << etlog, e_l = threadIdx.x & (ET - 1), slot = threadIdx.x >> etlog, nslots = blockDim.x >> etlog;
    const int ntile_e = (d.E + ET - 1) >> etlog, nblk_n = (d.nkx + NB - 1) / NB;
    int b = blockIdx.x;
    const int te = b % ntile_e; b /= ntile_e;
    const int bn = b % nblk_n;  b /= nblk_n;
    const int j = b + 1;
    const int f = blockIdx.y;
    const int e = te * ET + e_l, n0 = bn * NB;
    const bool eok = e < d.E;
    double2* tws = sm;
    double2* buf = sm + M;                             // [NB][M][ET]
    for (int i = threadIdx.x; i < M; i += blockDim.x) tws[i] = d.twz[i];
    __syncthreads();
    for (int item = slot; item < NB * R1; item += nslots) {
        const int nb = item / R1, i1 = item % R1, n = n0 + nb;
        double2 a[R2];
        const bool ok = n < d.nkx && eok;
        const double2* src = d.I3 + (size_t)f * d.Isz + dns_mix_off(d, j, 0, ok ? n : 0, ok ? e : 0);
        const size_t qs = ((size_t)d.ntl * d.nkx) << d.etl;
#pragma unroll
        for (int i2 = 0; i2 < R2; ++i2)
            a[i2] = ok ? src[(size_t)(i1 + R1 * i2) * qs] : make_double2(0.0, 0.0);
        DFT<R2>::run(a);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) buf[((size_t)nb * M + i1 * R2 + k2) * ET + e_l] = cmul(a[k2], tws[i1 * k2]);
    }
    __syncthreads();
    for (int item = slot; item < NB * R2; item += nslots) {
        const int nb = item / R2, k2 = item % R2, n = n0 + nb;
        double2 x[R1];
#pragma unroll
        for (int i1 = 0; i1 < R1; ++i1) x[i1] = buf[((size_t)nb * M + i1 * R2 + k2) * ET + e_l];
        DFT<R1>::run(x);
        if (n < d.nkx && eok) {
            double2* dst = d.Nh + (size_t)f * d.S + (((size_t)j * d.nkx + n) * d.nkz) * d.E + e;
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) {
                const int mi = pos_to_mi(k2 + R2 * k1, M, d.nzh, d.nkz);
                if (mi >= 0) dst[(size_t)mi * d.E] = cscale(x[k1], d.invMxMz);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ register versions
// For Mz = 2H <= 72 a whole z line fits the registers of TWO threads: the pair (lane, lane^1) splits the length-2H
// transform by one radix-2 step exchanged with warp shuffles, and each thread runs one H-point codelet on its
// half.  No shared memory, no barrier; every thread has H/1.5 independent 16-byte loads in flight, which is what
// keeps HBM busy.  Items (kx mode n, member e) of one plane are laid along the lanes, member fastest.
//   inverse (decimation in time):  thread h transforms the inputs at positions 2i+h;
//                                  x(k + H h) = E(k) +- w^k O(k), w = exp(-2 pi i / M) on swapped data (swap identity)
//   forward (decimation in frequency): thread h holds x(i + H h); a_h(i) = (x(i) +- x(i+H)) w^(h i); X(2m + h) = DFT_H(a_h)(m)
template <int H, bool TP>
__global__ void __launch_bounds__(128) k_zinv_r(DnsDev d, const double2* __restrict__ vin, const double2* __restrict__ ein, int pf) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = 2 * H, LO = H / 3, HI = 2 * H / 3;   // positions 2i+h < M/3 <=> i < LO ; > 2M/3 <=> i > HI (i == HI: h = 1 only)
    static_assert(H % 3 == 0, "padded length must be 3/2 of an even grid");
    const int h = threadIdx.x & 1;
    const int nper = d.nkx * d.E, nblk = (nper + 63) >> 6;
    const int j = blockIdx.x / nblk + 1;
    const int q = (blockIdx.x % nblk) * 64 + (threadIdx.x >> 1);
    const bool ok = q < nper;
    const int n = ok ? q / d.E : 0, e = ok ? q - n * d.E : 0;
    // TP (two passes): blockIdx.y = input field; u, v, w also give their z-derivative in a second pass over the same
    // inputs (now L1/L2 hits): 3 S less DRAM traffic, more registers.  Otherwise blockIdx.y = one of the 8 outputs.
    // Rotational form: blockIdx.y = one of the 6 fields, no derivative pass.
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    const int f = (TP || rot) ? blockIdx.y : (blockIdx.y < 5 ? blockIdx.y : blockIdx.y - 5);
    const double2* src = zinv_src(d, f, vin, ein) + ((size_t)j * d.nkx + n) * d.nkz * d.E + e;
#pragma unroll 1
    for (int pass = 0; pass < (TP && !rot && f < 3 ? 2 : 1); ++pass) {
    const bool deriv = rot ? false : (TP ? pass == 1 : blockIdx.y >= 5);
    const int var = rot ? f : (TP ? (deriv ? f + 5 : f) : blockIdx.y);
    // all loads first (independent, in flight together), then the i kz factor and the swap of the inverse transform
    double2 a[H];
    double kzv[H];
#pragma unroll
    for (int i = 0; i < H; ++i) {
        a[i] = make_double2(0.0, 0.0);
        kzv[i] = 0.0;
        if (i < LO || i >= HI) {
            const int mi = i < LO ? 2 * i + h : 2 * i + h - M / 3 - 1;
            if (ok && (i != HI || h == 1)) {
                a[i] = ldg2(src + (size_t)mi * d.E);
                if (deriv) kzv[i] = __ldg(d.kz + mi);
            }
        }
    }
    if (TP && pass == 0 && pf > 0) {
        // two-pass CTAs issue no loads during their second transform: keep the DRAM queue fed with the lines of the CTA
        // that will replace this one (pf blocks ahead in launch order), as L2 prefetches
        const unsigned bn = blockIdx.x + (unsigned)pf;
        if (bn < gridDim.x) {
            const int jn = bn / nblk + 1, qn = (bn % nblk) * 64 + (threadIdx.x >> 1);
            if (qn < nper) {
                const int nn = qn / d.E, en = qn - nn * d.E;
                const double2* sn = zinv_src(d, f, vin, ein) + ((size_t)jn * d.nkx + nn) * d.nkz * d.E + en;
                if ((en & 7) == 0) {                           // one prefetch per 128-byte line (8 members)
#pragma unroll
                    for (int i = 0; i < H; ++i)
                        if (i < LO || i >= HI) {
                            const int mi = i < LO ? 2 * i + h : 2 * i + h - M / 3 - 1;
                            if (i != HI || h == 1) asm volatile("prefetch.global.L2 [%0];" ::"l"(sn + (size_t)mi * d.E));
                        }
                }
            }
        }
    }
    if (deriv) {
#pragma unroll
        for (int i = 0; i < H; ++i)
            if (i < LO || i >= HI) a[i] = make_double2(kzv[i] * a[i].x, -kzv[i] * a[i].y);      // swap(i kz v)
    } else {
#pragma unroll
        for (int i = 0; i < H; ++i)
            if (i < LO || i >= HI) a[i] = cswap(a[i]);
    }
    DFT<H>::run(a);
    double2* dst = d.I8 + (size_t)var * d.Isz + dns_mix_off(d, j, 0, n, e) + (size_t)(H * h) * ((size_t)(d.ntl * d.nkx) << d.etl);
    const size_t qs = (size_t)(d.ntl * d.nkx) << d.etl;
    const double sg = h ? -1.0 : 1.0;
#pragma unroll
    for (int k = 0; k < H; ++k) {
        const double2 o = cmul(a[k], __ldg(d.twz + h * k));
        double2 r;
        r.x = __shfl_xor_sync(0xffffffffu, o.x, 1);
        r.y = __shfl_xor_sync(0xffffffffu, o.y, 1);
        const double2 x = make_double2(fma(sg, o.x, r.x), fma(sg, o.y, r.y));
        if (ok) dst[(size_t)k * qs] = cswap(x);
    }
    }
}

// H = 36 (Mz = 72): two CTAs per SM fit with any register count, so the allocator is left free (254 instead of its own
// 178 registers: every load of the line stays in flight; config 4: 477 -> 371 us per launch).  Shorter lines keep the
// allocator's choice (0 = unspecified): more registers would cost them a CTA per SM (measured slower for H = 24).
template <int H>
__global__ void __launch_bounds__(128, H == 36 ? 1 : 0) k_zfwd_r(DnsDev d) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = 2 * H, LO = H / 3, HI = 2 * H / 3;
    const int h = threadIdx.x & 1;
    const int nper = d.nkx * d.E, nblk = (nper + 63) >> 6;
    const int j = blockIdx.x / nblk + 1;
    const int q = (blockIdx.x % nblk) * 64 + (threadIdx.x >> 1);
    const bool ok = q < nper;
    const int n = ok ? q / d.E : 0, e = ok ? q - n * d.E : 0;
    const int f = blockIdx.y;
    const size_t qs = (size_t)(d.ntl * d.nkx) << d.etl;
    const double2* src = d.I3 + (size_t)f * d.Isz + dns_mix_off(d, j, 0, n, e) + (size_t)(H * h) * qs;
    const double sg = h ? -1.0 : 1.0;
    double2 a[H];
#pragma unroll
    for (int i = 0; i < H; ++i) a[i] = ok ? src[(size_t)i * qs] : make_double2(0.0, 0.0);
#pragma unroll
    for (int i = 0; i < H; ++i) {
        double2 r;
        r.x = __shfl_xor_sync(0xffffffffu, a[i].x, 1);
        r.y = __shfl_xor_sync(0xffffffffu, a[i].y, 1);
        const double2 t = make_double2(fma(sg, a[i].x, r.x), fma(sg, a[i].y, r.y));     // x(i) + x(i+H)  |  x(i) - x(i+H)
        a[i] = cmul(t, __ldg(d.twz + h * i));
    }
    DFT<H>::run(a);
    double2* dst = d.Nh + (size_t)f * d.S + ((size_t)j * d.nkx + n) * d.nkz * d.E + e;
#pragma unroll
    for (int m = 0; m < H; ++m) {
        if (m < LO || m >= HI) {
            const int mi = m < LO ? 2 * m + h : 2 * m + h - M / 3 - 1;
            if (ok && (m != HI || h == 1)) dst[(size_t)mi * d.E] = cscale(a[m], d.invMxMz);
        }
    }
}

// Four threads per line (Mz = 4H = 96): a radix-4 step across the lane quad, done as two radix-2 shuffle stages.
// Lane (l1, l0) of a quad enters with index 2 l1 + l0 and leaves with index l1 + 2 l0 (the network is its own
// transpose, so the same code serves the decimation-in-time inverse and the decimation-in-frequency forward).
__device__ __forceinline__ double2 quad_dft4(double2 z, int l1, int l0) {
    double2 r;
    r.x = __shfl_xor_sync(0xffffffffu, z.x, 2);
    r.y = __shfl_xor_sync(0xffffffffu, z.y, 2);
    const double s1 = l1 ? -1.0 : 1.0;
    double2 a = make_double2(fma(s1, z.x, r.x), fma(s1, z.y, r.y));          // l1 = 0: z + partner ; l1 = 1: partner - z
    if (l0 && l1) a = make_double2(a.y, -a.x);                                 // odd input of the second stage: * (-i)^l1
    r.x = __shfl_xor_sync(0xffffffffu, a.x, 1);
    r.y = __shfl_xor_sync(0xffffffffu, a.y, 1);
    const double s0 = l0 ? -1.0 : 1.0;
    return make_double2(fma(s0, a.x, r.x), fma(s0, a.y, r.y));
}

template <int H, bool TP>
__global__ void __launch_bounds__(128) k_zinv_r4(DnsDev d, const double2* __restrict__ vin, const double2* __restrict__ ein) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = 4 * H, LO = H / 3, HI = 2 * H / 3;   // positions 4i+r < M/3 <=> i < LO ; > 2M/3 <=> i > HI (i == HI: r >= 1)
    static_assert(H % 3 == 0, "padded length must be 3/2 of an even grid");
    const int l0 = threadIdx.x & 1, l1 = (threadIdx.x >> 1) & 1, r = 2 * l1 + l0, qo = l1 + 2 * l0;
    const int nper = d.nkx * d.E, nblk = (nper + 31) >> 5;
    const int j = blockIdx.x / nblk + 1;
    const int q = (blockIdx.x % nblk) * 32 + (threadIdx.x >> 2);
    const bool ok = q < nper;
    const int n = ok ? q / d.E : 0, e = ok ? q - n * d.E : 0;
    // TP (two passes): blockIdx.y = input field; u, v, w also give their z-derivative in a second pass over the same
    // inputs (now L1/L2 hits): 3 S less DRAM traffic, more registers.  Otherwise blockIdx.y = one of the 8 outputs.
    // Rotational form: blockIdx.y = one of the 6 fields, no derivative pass.
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    const int f = (TP || rot) ? blockIdx.y : (blockIdx.y < 5 ? blockIdx.y : blockIdx.y - 5);
    const double2* src = zinv_src(d, f, vin, ein) + ((size_t)j * d.nkx + n) * d.nkz * d.E + e;
#pragma unroll 1
    for (int pass = 0; pass < (TP && !rot && f < 3 ? 2 : 1); ++pass) {
    const bool deriv = rot ? false : (TP ? pass == 1 : blockIdx.y >= 5);
    const int var = rot ? f : (TP ? (deriv ? f + 5 : f) : blockIdx.y);
    double2 a[H];
    double kzv[H];
#pragma unroll
    for (int i = 0; i < H; ++i) {
        a[i] = make_double2(0.0, 0.0);
        kzv[i] = 0.0;
        if (i < LO || i >= HI) {
            const int mi = i < LO ? 4 * i + r : 4 * i + r - M / 3 - 1;
            if (ok && (i != HI || r >= 1)) {
                a[i] = ldg2(src + (size_t)mi * d.E);
                if (deriv) kzv[i] = __ldg(d.kz + mi);
            }
        }
    }
    if (deriv) {
#pragma unroll
        for (int i = 0; i < H; ++i)
            if (i < LO || i >= HI) a[i] = make_double2(kzv[i] * a[i].x, -kzv[i] * a[i].y);      // swap(i kz v)
    } else {
#pragma unroll
        for (int i = 0; i < H; ++i)
            if (i < LO || i >= HI) a[i] = cswap(a[i]);
    }
    DFT<H>::run(a);
    const size_t qs = (size_t)(d.ntl * d.nkx) << d.etl;
    double2* dst = d.I8 + (size_t)var * d.Isz + dns_mix_off(d, j, 0, n, e) + (size_t)(H * qo) * qs;
#pragma unroll
    for (int k = 0; k < H; ++k) {
        const double2 x = quad_dft4(cmul(a[k], __ldg(d.twz + r * k)), l1, l0);       // x(k + H qo) on swapped data
        if (ok) dst[(size_t)k * qs] = cswap(x);
    }
    }
}

template <int H>
__global__ void __launch_bounds__(128) k_zfwd_r4(DnsDev d) {
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    constexpr int M = 4 * H, LO = H / 3, HI = 2 * H / 3;
    const int l0 = threadIdx.x & 1, l1 = (threadIdx.x >> 1) & 1, qi = 2 * l1 + l0, r = l1 + 2 * l0;
    const int nper = d.nkx * d.E, nblk = (nper + 31) >> 5;
    const int j = blockIdx.x / nblk + 1;
    const int q = (blockIdx.x % nblk) * 32 + (threadIdx.x >> 2);
    const bool ok = q < nper;
    const int n = ok ? q / d.E : 0, e = ok ? q - n * d.E : 0;
    const int f = blockIdx.y;
    const size_t qs = (size_t)(d.ntl * d.nkx) << d.etl;
    const double2* src = d.I3 + (size_t)f * d.Isz + dns_mix_off(d, j, 0, n, e) + (size_t)(H * qi) * qs;
    double2 a[H];
#pragma unroll
    for (int i = 0; i < H; ++i) a[i] = ok ? src[(size_t)i * qs] : make_double2(0.0, 0.0);
#pragma unroll
    for (int i = 0; i < H; ++i) a[i] = cmul(quad_dft4(a[i], l1, l0), __ldg(d.twz + r * i));
    DFT<H>::run(a);                                                 // X(4m + r) = a[m]
    double2* dst = d.Nh + (size_t)f * d.S + ((size_t)j * d.nkx + n) * d.nkz * d.E + e;
#pragma unroll
    for (int m = 0; m < H; ++m) {
        if (m < LO || m >= HI) {
            const int mi = m < LO ? 4 * m + r : 4 * m + r - M / 3 - 1;
            if (ok && (m != HI || r >= 1)) dst[(size_t)mi * d.E] = cscale(a[m], d.invMxMz);
        }
    }
}

// Mz = 96: one pass per output field (the two-pass variant with the L2 prefetch of k_zinv_r measured no better: 198 against 195 us)
template <int H> void zinv_r4_launch(dns_plan* p, const double2* vin, const double2* ein) {
    const DnsDev& d = p->d;
    dim3 grid((unsigned)(d.Ni * ((d.nkx * d.E + 31) / 32)), d.form == DNS_FORM_ROTATIONAL ? 6 : 8);
    dns_launch(k_zinv_r4<H, false>, grid, dim3(128), 0, p->stream, d, vin, ein);
}
template <int H> void zfwd_r4_launch(dns_plan* p) {
    const DnsDev& d = p->d;
    dim3 grid((unsigned)(d.Ni * ((d.nkx * d.E + 31) / 32)), 3);
    dns_launch(k_zfwd_r4<H>, grid, dim3(128), 0, p->stream, d);
}

template <int H> void zinv_r_launch(dns_plan* p, const double2* vin, const double2* ein) {
    const DnsDev& d = p->d;
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    const unsigned nb = (unsigned)(d.Ni * ((d.nkx * d.E + 63) / 64));
    // Two passes (u, v, w also give their z-derivative from the same inputs: 3 S less DRAM traffic): always for Mz <= 48.
    // Mz = 72: alone it gains little (a thread in its second transform issues no loads and the DRAM queue runs shallow:
    // 985 -> 948 us on config 4), with the L2 prefetch of the lines of a CTA half a wave ahead it gives 915 us (flat for
    // distances of 74 .. 296 CTAs).  Option "zinv_tp" = 0: the one-pass kernel with 8 output fields.
    if constexpr (H == 36) {
        if (!rot && dns_option("zinv_tp") != 0) {
            dns_launch(k_zinv_r<H, true>, dim3(nb, 5), dim3(128), 0, p->stream, d, vin, ein, 148);
            return;
        }
    }
    constexpr bool TP = H <= 24;
    dim3 grid(nb, rot ? 6 : (TP ? 5 : 8));
    dns_launch(k_zinv_r<H, TP>, grid, dim3(128), 0, p->stream, d, vin, ein, (TP && !rot && dns_option("zinv_tp") != 0) ? 148 : 0);   // Mz = 48: 75.6 -> 73.2 us on config 2
}
template <int H> void zfwd_r_launch(dns_plan* p) {
    const DnsDev& d = p->d;
    dim3 grid((unsigned)(d.Ni * ((d.nkx * d.E + 63) / 64)), 3);
    dns_launch(k_zfwd_r<H>, grid, dim3(128), 0, p->stream, d);
}
bool use_zreg(int Mz) {
    return dns_option("zreg") != 0 && (Mz == 24 || Mz == 36 || Mz == 48 || Mz == 72 || Mz == 96);
}

// dynamic shared memory attributes are set once per kernel, device and size, not per launch (dns_grant_smem, dns_internal.h)

template <int R1, int R2> void zinv_launch(dns_plan* p, const double2* vin, const double2* ein) {
    const DnsDev& d = p->d;
    const int ET = p->ETf, etlog = __builtin_ctz(ET), M = R1 * R2;
    const int nslots = 256 / ET;
    int NB = (nslots + R1 - 1) / R1;                    // enough items to occupy every slot in pass A
    if (NB > d.nkx) NB = d.nkx;
    while (NB > 1 && (size_t)(M + (size_t)NB * 2 * M * ET) * sizeof(double2) > 96 * 1024) --NB;
    const size_t smem = (size_t)(M + (size_t)NB * 2 * M * ET) * sizeof(double2);
    auto kern = k_zinv<R1, R2>;
    static DnsSmemGrant grant;
    dns_grant_smem(kern, smem, grant, 0, true);
    dim3 grid((unsigned)(d.Ni * ((d.nkx + NB - 1) / NB) * ((d.E + ET - 1) / ET)), d.form == DNS_FORM_ROTATIONAL ? 6 : 5);
    dns_launch(kern, grid, dim3(256), smem, p->stream, d, vin, ein, etlog, NB);
}

template <int R1, int R2> void zfwd_launch(dns_plan* p) {
    const DnsDev& d = p->d;
    const int ET = p->ETf, etlog = __builtin_ctz(ET), M = R1 * R2;
    const int nslots = 256 / ET;
    int NB = (nslots + R1 - 1) / R1;
    if (NB > d.nkx) NB = d.nkx;
    while (NB > 1 && (size_t)(M + (size_t)NB * M * ET) * sizeof(double2) > 96 * 1024) --NB;
    const size_t smem = (size_t)(M + (size_t)NB * M * ET) * sizeof(double2);
    auto kern = k_zfwd<R1, R2>;
    static DnsSmemGrant grant;
    dns_grant_smem(kern, smem, grant, 0, true);
    dim3 grid((unsigned)(d.Ni * ((d.nkx + NB - 1) / NB) * ((d.E + ET - 1) / ET)), 3);
    dns_launch(kern, grid, dim3(256), smem, p->stream, d, etlog, NB);
}

}  // namespace

#define DNS_FFT_DISPATCH(M, CALL)                                         \
    switch (M) {                                                          \
        case 18: CALL(3, 6); break;                                       \
        case 24: CALL(4, 6); break;                                       \
        case 27: CALL(3, 9); break;                                       \
        case 36: CALL(6, 6); break;                                       \
        case 48: CALL(6, 8); break;                                       \
        case 54: CALL(6, 9); break;                                       \
        case 72: CALL(8, 9); break;                                       \
        case 81: CALL(9, 9); break;                                       \
        case 96: CALL(8, 12); break;                                      \
        case 108: CALL(9, 12); break;                                     \
        default: break;                                                   \
    }

void launch_zinv(dns_plan* p, const double2* vin, const double2* ein) {
    if (use_zreg(p->d.Mz)) {
        switch (p->d.Mz) {
            case 24: zinv_r_launch<12>(p, vin, ein); return;
            case 36: zinv_r_launch<18>(p, vin, ein); return;
            case 48: zinv_r_launch<24>(p, vin, ein); return;
            case 96: zinv_r4_launch<24>(p, vin, ein); return;
            default: zinv_r_launch<36>(p, vin, ein); return;
        }
    }
#define CALL(a, b) zinv_launch<a, b>(p, vin, ein)
    DNS_FFT_DISPATCH(p->d.Mz, CALL)
#undef CALL
}
void launch_zfwd(dns_plan* p) {
    if (use_zreg(p->d.Mz)) {
        switch (p->d.Mz) {
            case 24: zfwd_r_launch<12>(p); return;
            case 36: zfwd_r_launch<18>(p); return;
            case 48: zfwd_r_launch<24>(p); return;
            case 96: zfwd_r4_launch<24>(p); return;
            default: zfwd_r_launch<36>(p); return;
        }
    }
#define CALL(a, b) zfwd_launch<a, b>(p)
    DNS_FFT_DISPATCH(p->d.Mz, CALL)
#undef CALL
}
