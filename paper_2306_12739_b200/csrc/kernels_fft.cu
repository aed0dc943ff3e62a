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

// ------------------------------------------------------------------------------------------------ z inverse
// grid.x = Ni * nblk_n * ntile_e, grid.y = 5 input fields (u, v, w, Du, Dw); block = 256
template <int R1, int R2>
__global__ void __launch_bounds__(256) k_zinv(DnsDev d, const double2* __restrict__ vin, int etlog, int NB) {
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
    const double2* src = f == 0 ? d.uh : f == 1 ? vin : f == 2 ? d.wh : f == 3 ? d.duh : d.dwh;
    const int nv = f < 3 ? 2 : 1;                      // u, v, w also produce their z-derivative
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
            double2* dst = d.I8 + (((size_t)fo * d.Ny + j) * d.Mz) * d.nkx * d.E + (size_t)n * d.E + e;
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) dst[(size_t)(k2 + R2 * k1) * d.nkx * d.E] = cswap(x[k1]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ z forward
// grid.x = Ni * nblk_n * ntile_e, grid.y = 3 fields; block = 256
template <int R1, int R2>
__global__ void __launch_bounds__(256) k_zfwd(DnsDev d, int etlog, int NB) {
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
        const double2* src = d.I3 + (((size_t)f * d.Ny + j) * d.Mz) * d.nkx * d.E + (size_t)n * d.E + e;
#pragma unroll
        for (int i2 = 0; i2 < R2; ++i2)
            a[i2] = (n < d.nkx && eok) ? src[(size_t)(i1 + R1 * i2) * d.nkx * d.E] : make_double2(0.0, 0.0);
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

// ------------------------------------------------------------------------------------------------ x line kernel
// One "line" = (plane j, z index q, member e).  SL = max(R1,R2) thread slots cooperate on a line:
// inverse pass A runs on slots < R1 (slot = i1), inverse pass B on slots < R2 (slot = k2), after which slot k2
// holds the physical values at x = k2 + R2*k1, k1 < R1, in registers; the forward transform uses the mirrored
// factorisation (R2, R1) so that its pass A starts from exactly those registers.
template <int R1, int R2, int SL, int BT>
__global__ void __launch_bounds__(BT) k_line(DnsDev d, int etlog, int LC, int LQ) {
    constexpr int M = R1 * R2;
    extern __shared__ double2 sm[];
    const int ET = 1 << etlog, e_l = threadIdx.x & (ET - 1), slot = threadIdx.x >> etlog;
    const int sl = slot % SL, lc = slot / SL;
    const int ntile_e = (d.E + ET - 1) >> etlog, nblk_q = (d.Mz + LC * LQ - 1) / (LC * LQ);
    int b = blockIdx.x;
    const int te = b % ntile_e; b /= ntile_e;
    const int bq = b % nblk_q;  b /= nblk_q;
    const int j = b + 1;
    const int e = te * ET + e_l;
    const bool eok = e < d.E;
    const size_t LB = (size_t)M * ET;                   // one line buffer
    double2* tws = sm;                                  // [M]
    double2* B0 = sm + M + (size_t)lc * 4 * LB;         // four buffers per concurrent line
    double2* B1 = B0 + LB;
    double2* B2 = B1 + LB;
    double2* B3 = B2 + LB;
    double2* red = sm + M + (size_t)LC * 4 * LB + ((size_t)lc * SL) * ET;   // [LC][SL][ET]
    for (int i = threadIdx.x; i < M; i += blockDim.x) tws[i] = d.twx[i];
    __syncthreads();
    const size_t fstride = (size_t)d.Ny * d.Mz * d.nkx * d.E;
    const int nkx = d.nkx;

    for (int qi = 0; qi < LQ; ++qi) {
        const int q = (bq * LQ + qi) * LC + lc;
        const bool lok = eok && q < d.Mz && lc < LC;
        const size_t base = (((size_t)j * d.Mz + (lok ? q : 0)) * nkx) * d.E + e;
        auto ld = [&](int f, int n) -> double2 { return ldg2(d.I8 + f * fstride + base + (size_t)n * d.E); };
        // spectral value pair (A, B) of complex transform c at mode n:  Z = A + iB packs two real fields
        auto pairAB = [&](int c, int n, double2& A, double2& Bv) {
            const double kx = d.kx[n];
            switch (c) {
                case 0: A = ld(0, n); Bv = ld(1, n); break;                                        // u , v
                case 1: { A = ld(2, n); double2 u = ld(0, n); Bv = make_double2(-kx * u.y, kx * u.x); } break;   // w , du/dx
                case 2: A = ld(3, n); Bv = ld(5, n); break;                                        // du/dy , du/dz
                case 3: { A = ld(7, n); double2 w = ld(2, n); Bv = make_double2(-kx * w.y, kx * w.x); } break;   // dw/dz , dw/dx
                case 4: { double2 v = ld(1, n); A = make_double2(-kx * v.y, kx * v.x); Bv = ld(6, n); } break;   // dv/dx , dv/dz
                default: { A = ld(4, n); double2 u = ld(0, n), wz = ld(7, n);                     // dw/dy , dv/dy
                           Bv = make_double2(kx * u.y - wz.x, -kx * u.x - wz.y); } break;          // = -i kx u - dw/dz
            }
        };
        double u[R1], v[R1], w[R1], Nu[R1], Nv[R1], Nw[R1];
        double suv = 0.0, swv = 0.0;
#pragma unroll 1
        for (int c = 0; c < 6; ++c) {
            double2* buf = (c & 1) ? B1 : B0;
            if (sl < R1) {                                              // inverse pass A, i1 = sl
                double2 a[R2];
#pragma unroll
                for (int i2 = 0; i2 < R2; ++i2) {
                    const int pos = sl + R1 * i2;
                    double2 z = make_double2(0.0, 0.0);
                    if (lok) {
                        double2 A, Bv;
                        if (pos < nkx) {
                            pairAB(c, pos, A, Bv);
                            z = pos == 0 ? make_double2(A.x, Bv.x) : make_double2(A.x - Bv.y, A.y + Bv.x);
                        } else if (pos > M - nkx) {
                            pairAB(c, M - pos, A, Bv);
                            z = make_double2(A.x + Bv.y, Bv.x - A.y);   // conj(A) + i conj(B)
                        }
                    }
                    a[i2] = cswap(z);
                }
                DFT<R2>::run(a);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) buf[(size_t)(sl * R2 + k2) * ET + e_l] = cmul(a[k2], tws[sl * k2]);
            }
            __syncthreads();
            if (sl < R2) {                                              // inverse pass B, k2 = sl
                double2 x[R1];
#pragma unroll
                for (int i1 = 0; i1 < R1; ++i1) x[i1] = buf[(size_t)(i1 * R2 + sl) * ET + e_l];
                DFT<R1>::run(x);
                // physical pair: first field = x.y, second = x.x (swap identity)
#pragma unroll
                for (int k1 = 0; k1 < R1; ++k1) {
                    const double fa = x[k1].y, fb = x[k1].x;
                    switch (c) {
                        case 0: u[k1] = fa; v[k1] = fb; suv += fa * fb; break;
                        case 1: w[k1] = fa; Nu[k1] = u[k1] * fb; swv += fa * v[k1]; break;
                        case 2: Nu[k1] += v[k1] * fa; Nu[k1] += w[k1] * fb; break;
                        case 3: Nw[k1] = u[k1] * fb + w[k1] * fa; break;
                        case 4: Nv[k1] = u[k1] * fa + w[k1] * fb; break;
                        default: Nw[k1] += v[k1] * fa; Nv[k1] += v[k1] * fb; break;
                    }
                }
            }
        }
        // forward transforms of W1 = Nu + i Nv and W2 = Nw, factorisation (R2, R1): pass A on the registers
        __syncthreads();                                                // all reads of B0/B1 done
        if (sl < R2) {
            double2 a1[R1], a2[R1];
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) { a1[k1] = make_double2(Nu[k1], Nv[k1]); a2[k1] = make_double2(Nw[k1], 0.0); }
            DFT<R1>::run(a1);
            DFT<R1>::run(a2);
#pragma unroll
            for (int k = 0; k < R1; ++k) {
                B0[(size_t)(sl * R1 + k) * ET + e_l] = cmul(a1[k], tws[sl * k]);
                B1[(size_t)(sl * R1 + k) * ET + e_l] = cmul(a2[k], tws[sl * k]);
            }
            red[(size_t)sl * ET + e_l] = make_double2(suv, swv);
        }
        __syncthreads();
        if (sl < R1) {                                                  // forward pass B, k2' = sl, R2-point DFTs
            double2 x1[R2], x2[R2];
#pragma unroll
            for (int i = 0; i < R2; ++i) { x1[i] = B0[(size_t)(i * R1 + sl) * ET + e_l]; x2[i] = B1[(size_t)(i * R1 + sl) * ET + e_l]; }
            DFT<R2>::run(x1);
            DFT<R2>::run(x2);
#pragma unroll
            for (int k = 0; k < R2; ++k) {
                B2[(size_t)(sl + R1 * k) * ET + e_l] = x1[k];
                B3[(size_t)(sl + R1 * k) * ET + e_l] = x2[k];
            }
        }
        __syncthreads();
        // unpack the two-for-one spectra and store the retained modes (no scaling here; k_zfwd applies 1/(Mx Mz))
        if (lok) {
            const size_t ob = base;
            for (int n = sl; n < nkx; n += SL) {
                const double2 zp = B2[(size_t)n * ET + e_l], zm = B2[(size_t)((M - n) % M) * ET + e_l];
                const double2 wp = B3[(size_t)n * ET + e_l], wm = B3[(size_t)((M - n) % M) * ET + e_l];
                d.I3[0 * fstride + ob + (size_t)n * d.E] = make_double2(0.5 * (zp.x + zm.x), 0.5 * (zp.y - zm.y));   // (Z(n)+conj Z(-n))/2
                d.I3[1 * fstride + ob + (size_t)n * d.E] = make_double2(0.5 * (zp.y + zm.y), 0.5 * (zm.x - zp.x));   // (Z(n)-conj Z(-n))/(2i)
                d.I3[2 * fstride + ob + (size_t)n * d.E] = make_double2(0.5 * (wp.x + wm.x), 0.5 * (wp.y - wm.y));
            }
            if (sl == 0) {
                double a = 0.0, bsum = 0.0;
                for (int s = 0; s < R2; ++s) { a += red[(size_t)s * ET + e_l].x; bsum += red[(size_t)s * ET + e_l].y; }
                d.uvpart[((size_t)j * d.Mz + q) * d.E + e] = make_double2(a, bsum);
            }
        }
        __syncthreads();                                                // buffers reused by the next line
    }
}

template <int R1, int R2> void zinv_launch(dns_plan* p, const double2* vin) {
    const DnsDev& d = p->d;
    const int ET = p->ETf, etlog = __builtin_ctz(ET), M = R1 * R2;
    const int nslots = 256 / ET;
    int NB = (nslots + R1 - 1) / R1;                    // enough items to occupy every slot in pass A
    if (NB > d.nkx) NB = d.nkx;
    while (NB > 1 && (size_t)(M + (size_t)NB * 2 * M * ET) * sizeof(double2) > 96 * 1024) --NB;
    const size_t smem = (size_t)(M + (size_t)NB * 2 * M * ET) * sizeof(double2);
    auto kern = k_zinv<R1, R2>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    dim3 grid((unsigned)(d.Ni * ((d.nkx + NB - 1) / NB) * ((d.E + ET - 1) / ET)), 5);
    kern<<<grid, 256, smem, p->stream>>>(d, vin, etlog, NB);
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
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    dim3 grid((unsigned)(d.Ni * ((d.nkx + NB - 1) / NB) * ((d.E + ET - 1) / ET)), 3);
    kern<<<grid, 256, smem, p->stream>>>(d, etlog, NB);
}

template <int R1, int R2> void line_launch(dns_plan* p) {
    const DnsDev& d = p->d;
    constexpr int SL = R1 > R2 ? R1 : R2, M = R1 * R2;
    constexpr int TPS = SL <= 8 ? 32 : 16;              // lanes per slot: keeps the block at <= 256 threads
    constexpr int BT = SL * TPS;
    int ET = p->ETf < TPS ? p->ETf : TPS;
    const int etlog = __builtin_ctz(ET);
    const int LC = TPS / ET;                            // block = LC concurrent lines of SL*ET threads
    const int LQ = 4;
    const size_t smem = (size_t)(M + (size_t)LC * 4 * M * ET + (size_t)LC * SL * ET) * sizeof(double2);
    auto kern = k_line<R1, R2, SL, BT>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int nblk_q = (d.Mz + LC * LQ - 1) / (LC * LQ);
    dim3 grid((unsigned)(d.Ni * nblk_q * ((d.E + ET - 1) / ET)));
    kern<<<grid, BT, smem, p->stream>>>(d, etlog, LC, LQ);
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
#define DNS_LINE_DISPATCH(M, CALL)                                        \
    switch (M) {                                                          \
        case 18: CALL(3, 6); break;                                       \
        case 24: CALL(4, 6); break;                                       \
        case 27: CALL(3, 9); break;                                       \
        case 36: CALL(6, 6); break;                                       \
        case 48: CALL(6, 8); break;                                       \
        case 54: CALL(6, 9); break;                                       \
        case 72: CALL(6, 12); break;                                      \
        case 81: CALL(9, 9); break;                                       \
        case 96: CALL(6, 16); break;                                      \
        case 108: CALL(9, 12); break;                                     \
        default: break;                                                   \
    }

void launch_zinv(dns_plan* p, const double2* vin) {
#define CALL(a, b) zinv_launch<a, b>(p, vin)
    DNS_FFT_DISPATCH(p->d.Mz, CALL)
#undef CALL
}
void launch_zfwd(dns_plan* p) {
#define CALL(a, b) zfwd_launch<a, b>(p)
    DNS_FFT_DISPATCH(p->d.Mz, CALL)
#undef CALL
}
void launch_line(dns_plan* p) {
#define CALL(a, b) line_launch<a, b>(p)
    DNS_LINE_DISPATCH(p->d.Mx, CALL)
#undef CALL
}
