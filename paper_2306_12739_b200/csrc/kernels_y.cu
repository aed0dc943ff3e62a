// Wall-normal part of one stage (north_star subsystems (3), (4)).
//   k_ypair : one CTA per (kx,kz) pair and member tile.  Everything that couples only along y is chained in
//             shared memory: F,G assembly (Eq. 4-5), RK3 combination, the precomputed-inverse
//             solves of Eq. 12-13 for ALL members of the tile at once, dv/dy, the u,w
//             reconstruction of Eq. 17-18 and du/dy, dw/dy.  The contractions run on the fp64 tensor cores
//             (DMMA.8x8x4; the only fp64 MMA shape sm_100a executes natively) in the REFLECTION-PARITY basis:
//             with J the reversal y -> -y of the interior Gauss-Lobatto points, the Chebyshev matrix obeys
//             J D J = -D and every solve matrix J M J = M, so in the variables s = x + Jx, dd = x - Jx each
//             [Ni x Ni] product splits into two [Ni/2 x Ni/2] ones: half the flops and half the matrix bytes.
//             Inputs arrive as TMA tensor-map tiles (one per field: Ni rows x one member tile, landing in the padded
//             panel layout).
//   k_mean  : mean flow (row a10): U00, W00 of Eq. 14-15 with the wall lift f+-  and the mass-flux
//             pressure gamma solved so that the discrete bulk flux is held; api.cu runs it on a
//             side stream under the z-forward and per-pair kernels.
// plus layout conversion, input normalisation and diagnostics.
#include <cuda.h>

#include <cstdint>
#include <cstdlib>

#include "dns_internal.h"

namespace {

// weight of the third RK3 stage, (F0 + 4 F1 + F2)/6, as a multiplication: a double-precision division is a
// ~25-instruction sequence on the fp64 pipe, and the four per-element divisions of the stage-2 launch of k_ypair were 15 % of
// its instructions (ncu, profiles/r3_kernels.md).  x * SIXTH differs from x / 6 by at most one unit in the last place.
constexpr double SIXTH = 1.0 / 6.0;


__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one 2-D tile (box fixed by the tensor map: ld doubles x Ni rows) -> shared memory, completion on an mbarrier
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                     smem_u32(dst)),
                 "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}

// One k-sweep of two parity blocks at once (four independent accumulator chains per n-tile pair keep the DMMA
// pipe busy):  accS[nt] += AS[rows 8 mt..+7][:] * B_S[:][col0 + 8 nt..+7],  accD likewise with AD, B_D.
// AS, AD are parity blocks in DMMA fragment order (plan.cu: fold_block): a warp reads 512 contiguous bytes per
// pair of k-steps.  The B operands are parity panels in shared memory: row k of the s part is smem row k, row k
// of the dd part is smem row Ni-1-k (REV).
template <int NT, int KS2T, bool REVS, bool REVD>
__device__ __forceinline__ void gemm2(double (&accS)[NT][2], double (&accD)[NT][2], const double* __restrict__ AS,
                                      const double* __restrict__ AD, const double* BS, const double* BD, int KS2r,
                                      int mt, int lane, int ld, int Ni, int col0) {
    const int KS2 = KS2T ? KS2T : KS2r;
    const int g = lane >> 2, t = lane & 3;
    const double2* AfS = reinterpret_cast<const double2*>(AS) + (size_t)mt * KS2 * 32 + lane;
    const double2* AfD = reinterpret_cast<const double2*>(AD) + (size_t)mt * KS2 * 32 + lane;
    const double* BcS = BS + col0 + g;
    const double* BcD = BD + col0 + g;
    // Specialised sweep lengths (KS2T != 0: Kp = 16, 24, 32, 48) always have Kp <= Ni, so no row index ever needs the
    // clamp below: the row pointers are then one per-thread base plus compile-time multiples of ld (immediate offsets).
    const double* SF = BcS + t * ld;
    const double* SR = BcS + (Ni - 1 - t) * ld;
    const double* DF = BcD + t * ld;
    const double* DR = BcD + (Ni - 1 - t) * ld;
#pragma unroll
    for (int ks2 = 0; ks2 < KS2; ++ks2) {
        const double2 aS = __ldg(AfS + ks2 * 32), aD = __ldg(AfD + ks2 * 32);
        const double *s0, *s1, *d0, *d1;
        if constexpr (KS2T != 0) {
            s0 = REVS ? SR - (8 * ks2) * ld : SF + (8 * ks2) * ld;
            s1 = REVS ? SR - (8 * ks2 + 4) * ld : SF + (8 * ks2 + 4) * ld;
            d0 = REVD ? DR - (8 * ks2) * ld : DF + (8 * ks2) * ld;
            d1 = REVD ? DR - (8 * ks2 + 4) * ld : DF + (8 * ks2 + 4) * ld;
        } else {
            const int k = 8 * ks2 + t;
            const int f0 = min(k, Ni - 1), f1 = min(k + 4, Ni - 1), r0 = max(Ni - 1 - k, 0), r1 = max(Ni - 5 - k, 0);
            s0 = BcS + (REVS ? r0 : f0) * ld;
            s1 = BcS + (REVS ? r1 : f1) * ld;
            d0 = BcD + (REVD ? r0 : f0) * ld;
            d1 = BcD + (REVD ? r1 : f1) * ld;
        }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) { dmma(accS[nt], aS.x, s0[8 * nt]); dmma(accD[nt], aD.x, d0[8 * nt]); }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) { dmma(accS[nt], aS.y, s1[8 * nt]); dmma(accD[nt], aD.y, d1[8 * nt]); }
    }
}

template <int NT> __device__ __forceinline__ void zero_acc(double (&acc)[NT][2]) {
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
}

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double2 v) { *reinterpret_cast<double2*>(p) = v; }

// ------------------------------------------------------------------------------------------------ mean flow
// CTA-wide: tiles of 8 members x (blockDim/8) row slots; dynamic smem = 6 vectors [Ny][8]
// sa += sum_k M[k] xa[8 k + el], sb likewise with xb, k in [k0, k1) in ascending order.  The 8 member lanes of a row slot
// need the same matrix row: each loads one eighth of it (all loads of a 64-column chunk in flight at once) and the
// values are handed round with shuffles, so a row costs one memory round trip instead of one per four columns.
// Must be called by all 32 lanes with the same k0, k1 (Mrow may differ per row slot).
__device__ __forceinline__ void rowdot2(const double* __restrict__ Mrow, int k0, int k1, const double* xa, const double* xb,
                                        int el, int lane, double& sa, double& sb) {
    for (int base = k0; base < k1; base += 64) {
        double c[8];
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const int kk = base + 8 * m + el;
            c[m] = kk < k1 ? __ldg(Mrow + kk) : 0.0;
        }
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            if (base + 8 * m >= k1) break;
#pragma unroll
            for (int s8 = 0; s8 < 8; ++s8) {
                const double v = __shfl_sync(0xffffffffu, c[m], (lane & 24) + s8);
                const int k = base + 8 * m + s8;
                if (k < k1) { sa += v * xa[k * 8 + el]; sb += v * xb[k * 8 + el]; }
            }
        }
    }
}

__device__ void mean_body(const DnsDev& d, int stage, int derive_only, int tile, double* smm) {
    const int Ny = d.Ny, Ni = d.Ni, nrs = blockDim.x >> 3;
    const int el = threadIdx.x & 7, rs = threadIdx.x >> 3, e = tile * 8 + el, lane = threadIdx.x & 31;
    const bool eok = e < d.E;
    const int hi = stage == 0 ? 0 : 1;
    const double hdt = (stage == 0 ? 0.5 : 1.0) * d.dt;
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    double* uvc = smm;                  // [Ny][8] RK-combined plane mean of u v
    double* wvc = uvc + Ny * 8;
    double* ru = wvc + Ny * 8;          // rhs / new profile U
    double* rw = ru + Ny * 8;
    double* Un = rw + Ny * 8;
    double* Wn = Un + Ny * 8;
    __shared__ double gam[8];
    double* Uout = stage == 2 ? d.Ut : d.Us;
    double* Wout = stage == 2 ? d.Wt : d.Ws;
    if (!derive_only) {
        // plane means [uv]00, [wv]00 (Eq. 6-7): fixed-order sum of the per-line partial sums
        if (threadIdx.x < 16) { const int w = threadIdx.x >> 3; uvc[w * (Ny - 1) * 8 + el] = 0.0; wvc[w * (Ny - 1) * 8 + el] = 0.0; }   // wall rows
        for (int j = 1 + rs; j < Ny - 1; j += nrs) {
            double a = 0.0, b = 0.0;
            if (eok) {
                const double2* src = d.uvpart + (size_t)j * d.Mz * d.E + e;
                for (int q0 = 0; q0 < d.Mz; q0 += 16) {          // 16 loads in flight, summed in ascending q
                    double2 v[16];
#pragma unroll
                    for (int u = 0; u < 16; ++u) v[u] = q0 + u < d.Mz ? src[(size_t)(q0 + u) * d.E] : make_double2(0.0, 0.0);
#pragma unroll
                    for (int u = 0; u < 16; ++u) { a += v[u].x; b += v[u].y; }
                }
                a *= d.invMxMz; b *= d.invMxMz;
                // history: stage 0 stores S0, stage 1 replaces it by S0 + 4 S1
                const size_t gi = (size_t)j * d.E + e;
                if (stage == 0) d.uvc0[gi] = make_double2(a, b);
                else if (stage == 1) { const double2 s0 = d.uvc0[gi]; d.uvc0[gi] = make_double2(s0.x + 4.0 * a, s0.y + 4.0 * b); a = 2.0 * a - s0.x; b = 2.0 * b - s0.y; }
                else { const double2 s01 = d.uvc0[gi]; a = (s01.x + a) * SIXTH; b = (s01.y + b) * SIXTH; }
            }
            uvc[j * 8 + el] = a; wvc[j * 8 + el] = b;
        }
        __syncthreads();
        // rhs = 2 U_t - h dt D [uv] - 2 bc  (Eq. 14 with S0p = 2I - S0m and the wall columns on the rhs)
        for (int i0 = 0; i0 < Ni; i0 += nrs) {                    // all lanes run every round (shuffles inside rowdot2)
            const int i = i0 + rs < Ni ? i0 + rs : Ni - 1;
            double su = 0.0, sw = 0.0;
            // convective: S = d/dy of the plane mean of u v (Eq. 6-7, reading A9) ; rotational: S = plane mean of H_x itself
            if (rot) { su = uvc[(i + 1) * 8 + el]; sw = wvc[(i + 1) * 8 + el]; }
            else rowdot2(d.Dfull + (size_t)(i + 1) * Ny, 1, Ny - 1, uvc, wvc, el, lane, su, sw);
            const double ut = eok ? d.Ut[(size_t)(i + 1) * d.E + e] : 0.0, wt = eok ? d.Wt[(size_t)(i + 1) * d.E + e] : 0.0;
            if (i0 + rs < Ni) {
                ru[i * 8 + el] = 2.0 * ut - hdt * su - 2.0 * d.bc[hi * Ni + i];
                rw[i * 8 + el] = 2.0 * wt - hdt * sw;
            }
        }
        __syncthreads();
        for (int i0 = 0; i0 < Ni; i0 += nrs) {
            const int i = i0 + rs < Ni ? i0 + rs : Ni - 1;
            double su = 0.0, sw = 0.0;
            rowdot2(d.S0inv + (size_t)hi * Ni * Ni + (size_t)i * Ni, 0, Ni, ru, rw, el, lane, su, sw);
            const double ut = eok ? d.Ut[(size_t)(i + 1) * d.E + e] : 0.0, wt = eok ? d.Wt[(size_t)(i + 1) * d.E + e] : 0.0;
            if (i0 + rs < Ni) {
                Un[(i + 1) * 8 + el] = su - ut;
                Wn[(i + 1) * 8 + el] = sw - wt;
            }
        }
        if (rs == 0) { Un[el] = -d.Uw; Un[(Ny - 1) * 8 + el] = d.Uw; Wn[el] = 0.0; Wn[(Ny - 1) * 8 + el] = 0.0; }
        __syncthreads();
        if (rs == 0) {
            double gm = 0.0;
            if (d.flow == DNS_POISEUILLE_CMF && eok) {
                double q = 0.0;
                for (int j = 0; j < Ny; ++j) q += d.w[j] * Un[j * 8 + el];
                gm = (d.Qstar[e] - 0.5 * q) / d.wUg[hi];      // hold the bulk flux
            }
            gam[el] = gm;
            if (eok) d.gamma[e] = gm;
        }
        __syncthreads();
        for (int j = rs; j < Ny; j += nrs) {
            double un = Un[j * 8 + el];
            if (j > 0 && j < Ny - 1) un += gam[el] * d.Ugam[hi * Ni + j - 1];
            Un[j * 8 + el] = un;
            if (eok) { Uout[(size_t)j * d.E + e] = un; Wout[(size_t)j * d.E + e] = Wn[j * 8 + el]; }
        }
        __syncthreads();
    } else {
        for (int j = rs; j < Ny; j += nrs) {
            Un[j * 8 + el] = eok ? d.Ut[(size_t)j * d.E + e] : 0.0;
            Wn[j * 8 + el] = eok ? d.Wt[(size_t)j * d.E + e] : 0.0;
        }
        __syncthreads();
    }
    // (0,0) column of the transform inputs: u = U00, w = W00, du/dy = D U00, dw/dy = D W00
    for (int j0 = 0; j0 < Ny; j0 += nrs) {
        const int j = j0 + rs < Ny ? j0 + rs : Ny - 1;
        double du = 0.0, dw = 0.0;
        rowdot2(d.Dfull + (size_t)j * Ny, 0, Ny, Un, Wn, el, lane, du, dw);
        if (eok && j0 + rs < Ny) {
            const size_t gi = ((size_t)j * d.P) * d.E + e;
            d.uh[gi] = make_double2(Un[j * 8 + el], 0.0);
            d.wh[gi] = make_double2(Wn[j * 8 + el], 0.0);
            d.duh[gi] = make_double2(rot ? -du : du, 0.0);      // rotational: omega_z = -dU/dy, omega_x = dW/dy at (0,0)
            d.dwh[gi] = make_double2(dw, 0.0);
        }
    }
}

// ------------------------------------------------------------------------------------------------ per-pair chain
// grid = nmean + (P-1) * ntile_e ; block = 32 * (Kp/8) * NWN ; dynamic smem = 5 panels of Ni x ld doubles.
// A warp owns m-tile mt (rows 8 mt..+7 of BOTH parities) and NT n-tiles (members 4 NT wn .. of the tile).
#ifndef DNS_YP_REGCAP
#define DNS_YP_REGCAP 128
#endif
// CTAs per SM the register allocation is asked to allow: as many as fit with DNS_YP_REGCAP registers per thread
constexpr int ypair_minb(int threads) {
    return threads == 0 ? 1 : (65536 / (threads * DNS_YP_REGCAP) > 0 ? 65536 / (threads * DNS_YP_REGCAP) : 1);
}

template <int NT, int NWNT, int KS2T>
__global__ void __launch_bounds__(KS2T ? 32 * KS2T * NWNT : 1024, ypair_minb(32 * KS2T * NWNT))
k_ypair(DnsDev d, const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmV,
        const __grid_constant__ CUtensorMap tmE, int stage, int derive_only) {
    DNS_PDL_TRIGGER();
    extern __shared__ __align__(128) double smy[];
    __shared__ uint64_t bar;
    const int bid = blockIdx.x;
    const int Ni = d.Ni, KS2 = KS2T ? KS2T : (d.Kp >> 3), Kp = 8 * KS2, Kh = (Ni + 1) >> 1, Kho = Ni >> 1;
    constexpr int NWN = NWNT, NC = 8 * NT * NWN, ET = NC >> 1, ld = NC + 4;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int mt = warp % KS2, wn = warp / KS2;
    // DNS plan: pair p = (n, mi) != (0, 0), member tiles over all E.  Linearised ensemble (row f3): the arrays hold one
    // streamwise mode per member, p = mi, and a member tile lies inside one kx group (members g Eg .. (g+1) Eg - 1 share n)
    int p, e0, eend, n, mi;
    if (d.lin) {
        const int ntile_g = (d.Eg + ET - 1) / ET, ntile_e = d.nmodes * ntile_g, tile = bid % ntile_e, g = tile / ntile_g;
        p = bid / ntile_e;
        e0 = g * d.Eg + (tile % ntile_g) * ET;
        eend = (g + 1) * d.Eg;
        n = d.nlist[g];
        mi = p;
    } else {
        const int ntile_e = (d.E + ET - 1) / ET;
        p = 1 + bid / ntile_e;
        e0 = (bid % ntile_e) * ET;
        eend = d.E;
        n = p / d.nkz;
        mi = p % d.nkz;
    }
    const int mabs = mi < d.nzh ? mi : d.nkz - mi;
    const double kx = d.kx[n], kz = d.kz[mi], alpha = kx * kx + kz * kz, ialpha = 1.0 / alpha;
    const int hi = stage == 0 ? 0 : 1;
    const double hdt = (stage == 0 ? 0.5 : 1.0) * d.dt;
    const size_t BB = (size_t)Kp * Kp;
    const double* mA = d.matsP + (((size_t)hi * d.nkxm * d.nzh + (size_t)n * d.nzh + mabs) * 6) * BB;
    const double* Dsd = d.Dfrag;            // dd -> s
    const double* Dds = d.Dfrag + BB;       // s -> dd
    const size_t PS = ((size_t)Ni * ld + 15) & ~(size_t)15;      // panel pitch: a multiple of 128 B (TMA destination)
    double* P0 = smy;
    double* P1 = P0 + PS;
    double* P2 = P1 + PS;
    double* P3 = P2 + PS;
    double* P4 = P3 + PS;
    const size_t rowstride = (size_t)d.P * d.E;             // complex elements between consecutive y rows
    const size_t pbase = (size_t)p * d.E + e0;              // + (row + 1) * rowstride + member
    double2* vout = stage == 2 ? d.vt : d.vs;
    const bool rot = d.form == DNS_FORM_ROTATIONAL;
    double2* eout = stage == 2 ? d.et : (rot ? d.es : nullptr);     // omega_y = eta is a transform input of omega x u

    // ---- stage the inputs: one TMA tile per field (box = Ni rows x ld doubles, landing in the padded panel layout;
    //      the 4 pad columns of every row are the first two members of the neighbouring tile: never used)
    const int nvalid = eend - e0 < ET ? eend - e0 : ET;
    DNS_PDL_WAIT();                                          // the index arithmetic above overlaps the z-forward kernel's tail
    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const int c0 = 2 * (p * d.E + e0);
        mbar_arrive_expect_tx(&bar, (uint32_t)((derive_only ? 2 : 5) * Ni * ld * 8));
        if (derive_only) {
            tma_load_2d(P0, &tmV, c0, 1, &bar);
            tma_load_2d(P4, &tmE, c0, 1, &bar);
        } else {
            tma_load_2d(P0, &tmN, c0, 1, &bar);                  // (u.grad)u
            tma_load_2d(P1, &tmN, c0, 2 * d.Ny + 1, &bar);      // (u.grad)w
            tma_load_2d(P2, &tmN, c0, d.Ny + 1, &bar);          // (u.grad)v
            tma_load_2d(P3, &tmV, c0, 1, &bar);                 // v_t
            tma_load_2d(P4, &tmE, c0, 1, &bar);                 // eta_t
        }
    }
    __syncthreads();                                         // the barrier is initialised before anyone waits on it

    // ---- own fragment elements: row i = 8 mt + g of both parities, columns col0 + 8 nt + 2t, +1 (one member)
    const int i = 8 * mt + g, Ji = Ni - 1 - i;
    const bool sok = i < Kh, dok = i < Kho;
    const int col0 = 8 * NT * wn;
    const int offS = (sok ? i : 0) * ld + col0 + 2 * t, offD = (dok ? Ji : 0) * ld + col0 + 2 * t;
    auto eokf = [&](int nt) { return (e0 + (col0 >> 1) + 4 * nt + t) < eend; };
    const size_t gS = pbase + (size_t)(i + 1) * rowstride + (col0 >> 1) + t;      // + 4 nt : natural row i
    const size_t gD = pbase + (size_t)(Ji + 1) * rowstride + (col0 >> 1) + t;     // natural row J i

    // ---- history of the nonlinear terms: hist = N0 after stage 0, N0 + 4 N1 after stage 1
    double2 fhS[NT], fhD[NT], ghA[NT], ghB[NT];
    if (!derive_only && stage > 0) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            fhS[nt] = fhD[nt] = make_double2(0.0, 0.0);
            if (eokf(nt)) {
                if (sok) fhS[nt] = d.F0[gS + 4 * nt];
                if (dok) fhD[nt] = d.F0[gD + 4 * nt];
            }
        }
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            const int q = threadIdx.x + k * blockDim.x, ia = q / ET, e = q - ia * ET;
            ghA[k] = ghB[k] = make_double2(0.0, 0.0);
            if (ia < Kh && e < nvalid) {
                ghA[k] = d.G0[pbase + (size_t)(ia + 1) * rowstride + e];
                ghB[k] = d.G0[pbase + (size_t)(Ni - ia) * rowstride + e];
            }
        }
    }
    mbar_wait(&bar, 0);

    double accS[NT][2], accD[NT][2];
    if (!derive_only) {
        // ---- A (element-wise, in place): natural rows (ia, J ia) -> parity rows; H = i kx Nu + i kz Nw -> P0,
        //      G = i kz Nu - i kx Nw (Eq. 5), RK3 combination, 2 eta_t - h dt Gc -> P1, 2 v_t -> P3; (u.grad)v (P2) and
        //      eta_t (P4) stay in natural rows for the epilogues of B and C, which own them element by element
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            const int q = threadIdx.x + k * blockDim.x, ia = q / ET, e = q - ia * ET;
            if (ia >= Kh) continue;
            const int ib = Ni - 1 - ia;
            double* a0 = P0 + ia * ld + 2 * e;
            double* b0 = P0 + ib * ld + 2 * e;
            const double2 nuA = ld2(a0), nuB = ld2(b0), nwA = ld2(a0 + PS), nwB = ld2(b0 + PS);
            const double2 vtA = ld2(a0 + 3 * PS), vtB = ld2(b0 + 3 * PS);
            const double2 etA = ld2(a0 + 4 * PS), etB = ld2(b0 + 4 * PS);
            const double2 HA = make_double2(-kx * nuA.y - kz * nwA.y, kx * nuA.x + kz * nwA.x);
            const double2 HB = make_double2(-kx * nuB.y - kz * nwB.y, kx * nuB.x + kz * nwB.x);
            const double2 GA = make_double2(-kz * nuA.y + kx * nwA.y, kz * nuA.x - kx * nwA.x);
            const double2 GB = make_double2(-kz * nuB.y + kx * nwB.y, kz * nuB.x - kx * nwB.x);
            double2 GcA, GcB;
            const bool eok = e < nvalid;
            const size_t giA = pbase + (size_t)(ia + 1) * rowstride + e, giB = pbase + (size_t)(ib + 1) * rowstride + e;
            if (stage == 0) {
                GcA = GA; GcB = GB;
                if (eok) { d.G0[giA] = GA; d.G0[giB] = GB; }
            } else if (stage == 1) {
                GcA = make_double2(2.0 * GA.x - ghA[k].x, 2.0 * GA.y - ghA[k].y);
                GcB = make_double2(2.0 * GB.x - ghB[k].x, 2.0 * GB.y - ghB[k].y);
                if (eok) {
                    d.G0[giA] = make_double2(ghA[k].x + 4.0 * GA.x, ghA[k].y + 4.0 * GA.y);
                    d.G0[giB] = make_double2(ghB[k].x + 4.0 * GB.x, ghB[k].y + 4.0 * GB.y);
                }
            } else {
                GcA = make_double2((ghA[k].x + GA.x) * SIXTH, (ghA[k].y + GA.y) * SIXTH);
                GcB = make_double2((ghB[k].x + GB.x) * SIXTH, (ghB[k].y + GB.y) * SIXTH);
            }
            const double2 rA = make_double2(2.0 * etA.x - hdt * GcA.x, 2.0 * etA.y - hdt * GcA.y);
            const double2 rB = make_double2(2.0 * etB.x - hdt * GcB.x, 2.0 * etB.y - hdt * GcB.y);
            st2(a0, make_double2(HA.x + HB.x, HA.y + HB.y));
            st2(a0 + PS, make_double2(rA.x + rB.x, rA.y + rB.y));
            st2(a0 + 3 * PS, make_double2(2.0 * (vtA.x + vtB.x), 2.0 * (vtA.y + vtB.y)));
            if (ib != ia) {
                st2(b0, make_double2(HA.x - HB.x, HA.y - HB.y));
                st2(b0 + PS, make_double2(rA.x - rB.x, rA.y - rB.y));
                st2(b0 + 3 * PS, make_double2(2.0 * (vtA.x - vtB.x), 2.0 * (vtA.y - vtB.y)));
            }
        }
        __syncthreads();
        // ---- B: F = -alpha Nv - D H (Eq. 4 with Eq. 10's sign), RK3 combination; -h dt Fc -> P2
        zero_acc<NT>(accS); zero_acc<NT>(accD);
        gemm2<NT, KS2T, true, false>(accS, accD, Dsd, Dds, P0, P0, KS2, mt, lane, ld, Ni, col0);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            double2 FS = make_double2(0.0, 0.0), FD = make_double2(0.0, 0.0);
            // (u.grad)v is still in natural rows (i at offS, J i at offD): its parity parts are formed here, in registers
            if (sok) {
                const double2 na = ld2(P2 + offS + 8 * nt), nb = dok ? ld2(P2 + offD + 8 * nt) : na;
                FS = make_double2(-alpha * (na.x + nb.x) - accS[nt][0], -alpha * (na.y + nb.y) - accS[nt][1]);
                if (dok) FD = make_double2(-alpha * (na.x - nb.x) - accD[nt][0], -alpha * (na.y - nb.y) - accD[nt][1]);
            }
            // natural rows: F(i) = (FS + FD)/2, F(Ji) = (FS - FD)/2
            const double2 FA = make_double2(0.5 * (FS.x + FD.x), 0.5 * (FS.y + FD.y));
            const double2 FB = make_double2(0.5 * (FS.x - FD.x), 0.5 * (FS.y - FD.y));
            double2 cA, cB;
            const bool eok = eokf(nt);
            if (stage == 0) {
                cA = FA; cB = FB;
                if (eok && sok) d.F0[gS + 4 * nt] = FA;
                if (eok && dok) d.F0[gD + 4 * nt] = FB;
            } else if (stage == 1) {
                cA = make_double2(2.0 * FA.x - fhS[nt].x, 2.0 * FA.y - fhS[nt].y);
                cB = make_double2(2.0 * FB.x - fhD[nt].x, 2.0 * FB.y - fhD[nt].y);
                if (eok && sok) d.F0[gS + 4 * nt] = make_double2(fhS[nt].x + 4.0 * FA.x, fhS[nt].y + 4.0 * FA.y);
                if (eok && dok) d.F0[gD + 4 * nt] = make_double2(fhD[nt].x + 4.0 * FB.x, fhD[nt].y + 4.0 * FB.y);
            } else {
                cA = make_double2((fhS[nt].x + FA.x) * SIXTH, (fhS[nt].y + FA.y) * SIXTH);
                cB = make_double2((fhD[nt].x + FB.x) * SIXTH, (fhD[nt].y + FB.y) * SIXTH);
            }
            if (!dok) cB = cA;                              // middle row of an odd Ni: s = 2 x
            if (sok) st2(P2 + offS + 8 * nt, make_double2(-hdt * (cA.x + cB.x), -hdt * (cA.y + cB.y)));
            if (dok) st2(P2 + offD + 8 * nt, make_double2(-hdt * (cA.x - cB.x), -hdt * (cA.y - cB.y)));
        }
        __syncthreads();
        // ---- C: v' = Ainv (2 v_t) + AD (-h dt Fc) - v_t (Eq. 12) -> global, P0 ; eta' = Sinv P1 - eta_t (Eq. 13) -> P4
        zero_acc<NT>(accS); zero_acc<NT>(accD);
        gemm2<NT, KS2T, false, true>(accS, accD, mA, mA + BB, P3, P3, KS2, mt, lane, ld, Ni, col0);
        gemm2<NT, KS2T, false, true>(accS, accD, mA + 2 * BB, mA + 3 * BB, P2, P2, KS2, mt, lane, ld, Ni, col0);
        double acc2S[NT][2], acc2D[NT][2];
        zero_acc<NT>(acc2S); zero_acc<NT>(acc2D);
        gemm2<NT, KS2T, false, true>(acc2S, acc2D, mA + 4 * BB, mA + 5 * BB, P1, P1, KS2, mt, lane, ld, Ni, col0);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            double2 vS = make_double2(0.0, 0.0), vD = vS, eS = vS, eD = vS;
            // eta_t is still in natural rows (i at offS, J i at offD); eta' replaces it in parity form
            double2 ea = make_double2(0.0, 0.0), eb = ea;
            if (sok) { ea = ld2(P4 + offS + 8 * nt); eb = dok ? ld2(P4 + offD + 8 * nt) : ea; }
            if (sok) {
                const double2 v2 = ld2(P3 + offS + 8 * nt);
                vS = make_double2(accS[nt][0] - 0.5 * v2.x, accS[nt][1] - 0.5 * v2.y);
                eS = make_double2(acc2S[nt][0] - (ea.x + eb.x), acc2S[nt][1] - (ea.y + eb.y));
                st2(P0 + offS + 8 * nt, vS);
                st2(P4 + offS + 8 * nt, eS);
            }
            if (dok) {
                const double2 v2 = ld2(P3 + offD + 8 * nt);
                vD = make_double2(accD[nt][0] - 0.5 * v2.x, accD[nt][1] - 0.5 * v2.y);
                eD = make_double2(acc2D[nt][0] - (ea.x - eb.x), acc2D[nt][1] - (ea.y - eb.y));
                st2(P0 + offD + 8 * nt, vD);
                st2(P4 + offD + 8 * nt, eD);
            }
            if (eokf(nt)) {
                if (sok) {
                    vout[gS + 4 * nt] = make_double2(0.5 * (vS.x + vD.x), 0.5 * (vS.y + vD.y));
                    if (eout) eout[gS + 4 * nt] = make_double2(0.5 * (eS.x + eD.x), 0.5 * (eS.y + eD.y));
                }
                if (dok) {
                    vout[gD + 4 * nt] = make_double2(0.5 * (vS.x - vD.x), 0.5 * (vS.y - vD.y));
                    if (eout) eout[gD + 4 * nt] = make_double2(0.5 * (eS.x - eD.x), 0.5 * (eS.y - eD.y));
                }
            }
        }
        __syncthreads();
    } else {
        // parity transform of v_t (P0) and eta_t (P4) in place
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            const int q = threadIdx.x + k * blockDim.x, ia = q / ET, e = q - ia * ET;
            if (ia >= Kh) continue;
            const int ib = Ni - 1 - ia;
            double* a0 = P0 + ia * ld + 2 * e;
            double* b0 = P0 + ib * ld + 2 * e;
            const double2 vA = ld2(a0), vB = ld2(b0), eA = ld2(a0 + 4 * PS), eB = ld2(b0 + 4 * PS);
            st2(a0, make_double2(vA.x + vB.x, vA.y + vB.y));
            st2(a0 + 4 * PS, make_double2(eA.x + eB.x, eA.y + eB.y));
            if (ib != ia) {
                st2(b0, make_double2(vA.x - vB.x, vA.y - vB.y));
                st2(b0 + 4 * PS, make_double2(eA.x - eB.x, eA.y - eB.y));
            }
        }
        __syncthreads();
    }
    // ---- D: dv/dy = D v' ; u = (i kx Dv - i kz eta)/alpha, w = (i kz Dv + i kx eta)/alpha (Eq. 17-18) -> global, P2, P3
    zero_acc<NT>(accS); zero_acc<NT>(accD);
    gemm2<NT, KS2T, true, false>(accS, accD, Dsd, Dds, P0, P0, KS2, mt, lane, ld, Ni, col0);
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        double2 uS = make_double2(0.0, 0.0), uD = uS, wS = uS, wD = uS;
        if (sok) {
            const double2 en = ld2(P4 + offS + 8 * nt);
            uS = make_double2((-kx * accS[nt][1] + kz * en.y) * ialpha, (kx * accS[nt][0] - kz * en.x) * ialpha);
            wS = make_double2((-kz * accS[nt][1] - kx * en.y) * ialpha, (kz * accS[nt][0] + kx * en.x) * ialpha);
            st2(P2 + offS + 8 * nt, uS);
            st2(P3 + offS + 8 * nt, wS);
        }
        if (dok) {
            const double2 en = ld2(P4 + offD + 8 * nt);
            uD = make_double2((-kx * accD[nt][1] + kz * en.y) * ialpha, (kx * accD[nt][0] - kz * en.x) * ialpha);
            wD = make_double2((-kz * accD[nt][1] - kx * en.y) * ialpha, (kz * accD[nt][0] + kx * en.x) * ialpha);
            st2(P2 + offD + 8 * nt, uD);
            st2(P3 + offD + 8 * nt, wD);
        }
        if (eokf(nt)) {
            if (sok) {
                d.uh[gS + 4 * nt] = make_double2(0.5 * (uS.x + uD.x), 0.5 * (uS.y + uD.y));
                d.wh[gS + 4 * nt] = make_double2(0.5 * (wS.x + wD.x), 0.5 * (wS.y + wD.y));
            }
            if (dok) {
                d.uh[gD + 4 * nt] = make_double2(0.5 * (uS.x - uD.x), 0.5 * (uS.y - uD.y));
                d.wh[gD + 4 * nt] = make_double2(0.5 * (wS.x - wD.x), 0.5 * (wS.y - wD.y));
            }
        }
    }
    __syncthreads();
    // ---- E: du/dy, dw/dy
    {
        double a2S[NT][2], a2D[NT][2];
        zero_acc<NT>(accS); zero_acc<NT>(accD); zero_acc<NT>(a2S); zero_acc<NT>(a2D);
        gemm2<NT, KS2T, true, false>(accS, accD, Dsd, Dds, P2, P2, KS2, mt, lane, ld, Ni, col0);
        gemm2<NT, KS2T, true, false>(a2S, a2D, Dsd, Dds, P3, P3, KS2, mt, lane, ld, Ni, col0);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (!eokf(nt)) continue;
            double2 aS = make_double2(accS[nt][0], accS[nt][1]), aD = make_double2(accD[nt][0], accD[nt][1]);
            double2 bS = make_double2(a2S[nt][0], a2S[nt][1]), bD = make_double2(a2D[nt][0], a2D[nt][1]);
            if (rot) {
                // omega_z = i kx v - du/dy, omega_x = dw/dy - i kz v (row f1): linear, so formed on the parity parts of
                // v' (still in P0) and of the two derivatives
                const double2 vS = sok ? ld2(P0 + offS + 8 * nt) : make_double2(0.0, 0.0);
                const double2 vD = dok ? ld2(P0 + offD + 8 * nt) : make_double2(0.0, 0.0);
                aS = make_double2(-kx * vS.y - aS.x, kx * vS.x - aS.y);
                aD = make_double2(-kx * vD.y - aD.x, kx * vD.x - aD.y);
                bS = make_double2(bS.x + kz * vS.y, bS.y - kz * vS.x);
                bD = make_double2(bD.x + kz * vD.y, bD.y - kz * vD.x);
            }
            if (sok) {
                d.duh[gS + 4 * nt] = make_double2(0.5 * (aS.x + aD.x), 0.5 * (aS.y + aD.y));
                d.dwh[gS + 4 * nt] = make_double2(0.5 * (bS.x + bD.x), 0.5 * (bS.y + bD.y));
            }
            if (dok) {
                d.duh[gD + 4 * nt] = make_double2(0.5 * (aS.x - aD.x), 0.5 * (aS.y - aD.y));
                d.dwh[gD + 4 * nt] = make_double2(0.5 * (bS.x - bD.x), 0.5 * (bS.y - bD.y));
            }
        }
    }
}

// mean flow as its own small launch (8 members per CTA); api.cu runs it on a side stream under the z-forward and
// per-pair kernels: it needs only the plane sums written by the line kernel
__global__ void __launch_bounds__(512) k_mean(DnsDev d, int stage, int derive_only) {
    extern __shared__ __align__(128) double smm[];
    DNS_PDL_TRIGGER();
    DNS_PDL_WAIT();
    mean_body(d, stage, derive_only, blockIdx.x, smm);
}

// ------------------------------------------------------------------------------------------------ layout / IO
// ABI [E][P][Ny] <-> internal [Ny][P][E]; grid = (P, ceil(E/32), ceil(Ny/32)), block = (32, 8)
__global__ void k_abi_to_internal(const double2* __restrict__ src, double2* __restrict__ dst, int Ny, int P, int E, int acc) {
    __shared__ double2 tile[32][33];
    const int p = blockIdx.x, e0 = blockIdx.y * 32, j0 = blockIdx.z * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int e = e0 + k, j = j0 + threadIdx.x;
        if (e < E && j < Ny) tile[k][threadIdx.x] = src[((size_t)e * P + p) * Ny + j];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int j = j0 + k, e = e0 + threadIdx.x;
        if (e < E && j < Ny) {
            double2* o = dst + ((size_t)j * P + p) * E + e;
            const double2 a = tile[threadIdx.x][k];
            *o = acc ? make_double2(o->x + a.x, o->y + a.y) : a;
        }
    }
}
__global__ void k_internal_to_abi(const double2* __restrict__ src, double2* __restrict__ dst, int Ny, int P, int E) {
    __shared__ double2 tile[32][33];
    const int p = blockIdx.x, e0 = blockIdx.y * 32, j0 = blockIdx.z * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int j = j0 + k, e = e0 + threadIdx.x;
        if (e < E && j < Ny) tile[k][threadIdx.x] = src[((size_t)j * P + p) * E + e];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int e = e0 + k, j = j0 + threadIdx.x;
        if (e < E && j < Ny) dst[((size_t)e * P + p) * Ny + j] = tile[threadIdx.x][k];
    }
}

// input normalisation (include/dns.h dns_set_state): walls, (0,0) column, Hermitian n = 0 plane
__global__ void k_normalise(DnsDev d) {
    const size_t tot = (size_t)d.Ny * d.nkz * d.E;      // the n = 0 plane and all wall rows
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < d.S; i += (size_t)gridDim.x * blockDim.x) {
        const int e = (int)(i % d.E);
        const size_t pe = i / d.E;
        const int p = (int)(pe % d.P), j = (int)(pe / d.P);
        const int n = p / d.nkz, mi = p % d.nkz;
        if (j == 0 || j == d.Ny - 1 || p == 0) { d.vt[i] = make_double2(0.0, 0.0); d.et[i] = make_double2(0.0, 0.0); }
        else if (n == 0 && mi >= d.nzh) {
            const size_t src = ((size_t)j * d.P + (d.nkz - mi)) * d.E + e;
            const double2 a = d.vt[src], b = d.et[src];
            d.vt[i] = make_double2(a.x, -a.y);
            d.et[i] = make_double2(b.x, -b.y);
        }
    }
    (void)tot;
}

// U_abi [E][Ny] -> Ut [Ny][E] with wall values imposed (Eq. 9); Qstar = (1/2) w^T U
__global__ void k_mean_in(DnsDev d, const double* __restrict__ U, const double* __restrict__ W) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= d.E) return;
    double q = 0.0;
    for (int j = 0; j < d.Ny; ++j) {
        double u = U[(size_t)e * d.Ny + j], w = W[(size_t)e * d.Ny + j];
        if (j == 0) { u = -d.Uw; w = 0.0; }
        if (j == d.Ny - 1) { u = d.Uw; w = 0.0; }
        d.Ut[(size_t)j * d.E + e] = u;
        d.Wt[(size_t)j * d.E + e] = w;
        q += d.w[j] * u;
    }
    d.Qstar[e] = 0.5 * q;
    d.gamma[e] = 0.0;
}
__global__ void k_mean_out(DnsDev d, double* __restrict__ U, double* __restrict__ W) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= d.E) return;
    for (int j = 0; j < d.Ny; ++j) {
        if (U) U[(size_t)e * d.Ny + j] = d.Ut[(size_t)j * d.E + e];
        if (W) W[(size_t)e * d.Ny + j] = d.Wt[(size_t)j * d.E + e];
    }
}

// Sums over the retained modes of one wall-normal plane, per member, for the diagnostics: the 256 threads of a CTA are
// EB member lanes x (256 / EB) mode slots; every slot walks the pairs p = slot, slot + nslot, ... and the slots are then
// added in ascending order (fixed order: deterministic).  f(p, gi, acc) adds the contribution of pair p.
template <int NS, class F> __device__ __forceinline__ void plane_mode_sums(const DnsDev& d, int j, int p0, double* sm, F f, double (&out)[NS], int e0, int EB) {
    const int el = threadIdx.x % EB, slot = threadIdx.x / EB, nslot = blockDim.x / EB, e = e0 + el;
    double acc[NS];
#pragma unroll
    for (int k = 0; k < NS; ++k) acc[k] = 0.0;
    if (e < d.E)
        for (int p = p0 + slot; p < d.P; p += nslot) f(p, ((size_t)j * d.P + p) * d.E + e, acc);
#pragma unroll
    for (int k = 0; k < NS; ++k) sm[(k * nslot + slot) * EB + el] = acc[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        double t = 0.0;
        if (slot == 0)
            for (int q = 0; q < nslot; ++q) t += sm[(k * nslot + q) * EB + el];
        out[k] = t;
    }
    __syncthreads();
}
__device__ __forceinline__ int member_block(int E) { int b = 1; while (b < E && b < 256) b <<= 1; return b; }

// diagnostics: energy partial sums per (j, e), then the per-member rows
__global__ void __launch_bounds__(256) k_diag_energy(DnsDev d, double* __restrict__ part) {
    __shared__ double sm[256];
    const int j = blockIdx.x, EB = member_block(d.E);
    for (int e0 = 0; e0 < d.E; e0 += EB) {
        double s[1];
        plane_mode_sums<1>(d, j, 0, sm, [&](int p, size_t gi, double* a) {
            const double2 u = d.uh[gi], v = d.vt[gi], w = d.wh[gi];
            const double cn = (!d.lin && (p / d.nkz) == 0) ? 1.0 : 2.0;     // a stored mode with kx > 0 stands for +-kx
            a[0] += cn * (u.x * u.x + u.y * u.y + v.x * v.x + v.y * v.y + w.x * w.x + w.y * w.y);
        }, s, e0, EB);
        const int e = e0 + threadIdx.x;
        if (threadIdx.x < EB && e < d.E) part[(size_t)j * d.E + e] = 0.25 * d.w[j] * s[0];
    }
}
__global__ void k_diag_rows(DnsDev d, const double* __restrict__ part, double t) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= d.E) return;
    double en = 0.0, dlo = 0.0, dhi = 0.0, q = 0.0;
    for (int j = 0; j < d.Ny; ++j) {
        const double u = d.Ut[(size_t)j * d.E + e];
        en += part[(size_t)j * d.E + e];
        dlo += d.Dfull[j] * u;
        dhi += d.Dfull[(size_t)(d.Ny - 1) * d.Ny + j] * u;
        q += d.w[j] * u;
    }
    double* o = d.diag + (size_t)e * 6;
    o[0] = en; o[1] = dlo; o[2] = dhi; o[3] = 0.5 * q; o[4] = d.gamma[e]; o[5] = t;
}

// one-point statistics of the current state (row f4): Parseval sums over the retained modes, added to the running sums
// grid = (Ny, ceil(E / EB)) with EB = 32 member lanes at most: 8 mode slots per member block and enough CTAs to fill the GPU
// (one CTA per plane walked all P modes of 256 members with one slot: 65 CTAs, 0.20 of the HBM roofline on config 4)
__global__ void __launch_bounds__(256) k_stats(DnsDev d) {
    __shared__ double sm[4 * 256];
    const int j = blockIdx.x, EB = min(member_block(d.E), 32);
    const size_t NE = (size_t)d.Ny * d.E;
    {
        const int e0 = blockIdx.y * EB;
        double s[4];
        plane_mode_sums<4>(d, j, 1, sm, [&](int p, size_t gi, double* a) {
            const double2 u = d.uh[gi], v = d.vt[gi], w = d.wh[gi];
            const double cn = (p / d.nkz) == 0 ? 1.0 : 2.0;      // the n = 0 plane stores both +-m, n > 0 stands for +-n
            a[0] += cn * (u.x * u.x + u.y * u.y);
            a[1] += cn * (v.x * v.x + v.y * v.y);
            a[2] += cn * (w.x * w.x + w.y * w.y);
            a[3] += cn * (u.x * v.x + u.y * v.y);
        }, s, e0, EB);
        const int e = e0 + threadIdx.x;
        if (threadIdx.x < EB && e < d.E) {
            const size_t o = (size_t)j * d.E + e;
            d.stat[o] += d.Ut[o];
            d.stat[NE + o] += s[0];
            d.stat[2 * NE + o] += s[1];
            d.stat[3 * NE + o] += s[2];
            d.stat[4 * NE + o] += s[3];
        }
    }
}

// ------------------------------------------------------------------------------------------------ coupled ensemble (row f2)
// the members share their streamwise-mean flow, which is forced by the Reynolds stresses averaged over
// the members.  One warp per item = one run of E member values: the kx = 0 plane of the three components of the
// nonlinear vector in spectral space ([3][Ni][nkz] items) and the per-z-line plane sums of the mean-flow sources
// ([Ni][Mz] items).  phase 0: fixed-order sum over the members of this GPU -> d.ens (the exchange buffer);
// phase 1: d.ens / E_total -> every member; phase 2: both at once (one GPU).
__global__ void __launch_bounds__(256) k_ens(DnsDev d, int phase) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int nN = 3 * d.Ni * d.nkz, nUV = d.Ni * d.Mz;
    if (warp >= nN + nUV) return;
    double2* run;
    size_t slot;
    if (warp < nN) {
        const int f = warp / (d.Ni * d.nkz), r = warp % (d.Ni * d.nkz), j = r / d.nkz + 1, mi = r % d.nkz;
        run = d.Nh + (size_t)f * d.S + ((size_t)j * d.P + mi) * d.E;
        slot = ((size_t)f * d.Ny + j) * d.nkz + mi;
    } else {
        const int r = warp - nN, j = r / d.Mz + 1, q = r % d.Mz;
        run = d.uvpart + ((size_t)j * d.Mz + q) * d.E;
        slot = (size_t)3 * d.Ny * d.nkz + (size_t)j * d.Mz + q;
    }
    double2 t = make_double2(0.0, 0.0);
    if (phase != 1) {
        for (int e = lane; e < d.E; e += 32) { const double2 a = run[e]; t.x += a.x; t.y += a.y; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {          // xor tree: the same order on every lane, every launch
            t.x += __shfl_xor_sync(0xffffffffu, t.x, o);
            t.y += __shfl_xor_sync(0xffffffffu, t.y, o);
        }
        if (phase == 0) { if (lane == 0) d.ens[slot] = t; return; }
    } else {
        t = d.ens[slot];
    }
    t.x *= d.invEtot; t.y *= d.invEtot;
    for (int e = lane; e < d.E; e += 32) run[e] = t;
}

}  // namespace

size_t dns_ypair_smem(int Ni, int Ny, int ET) {
    (void)Ny;
    return 5 * ((((size_t)Ni * (2 * ET + 4) + 15) & ~(size_t)15) * sizeof(double));
}

// TMA descriptors of the per-pair kernel's inputs: 2-D views [rows][2 P E doubles] of the spectral arrays with a
// box of Ni rows x (2 ET + 4) doubles, i.e. exactly one padded shared-memory panel.  Encoded at dns_plan_bind.
int dns_ypair_encode_maps(dns_plan* p) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static const encode_fn encode = [] {       // looked up once; the initialisation of a local static is thread-safe
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess) fn = nullptr;
        return reinterpret_cast<encode_fn>(fn);
    }();
    if (!encode) return DNS_ECUDA;
    const DnsDev& d = p->d;
    static_assert(sizeof(CUtensorMap) == sizeof(p->tmaps[0]), "tensor map storage");
    struct Src { void* ptr; cuuint64_t rows; } src[3] = {{d.Nh, (cuuint64_t)3 * d.Ny}, {d.vt, (cuuint64_t)d.Ny}, {d.et, (cuuint64_t)d.Ny}};
    for (int i = 0; i < 3; ++i) {
        const cuuint64_t dims[2] = {(cuuint64_t)2 * d.P * d.E, src[i].rows};
        const cuuint64_t strides[1] = {(cuuint64_t)d.P * d.E * sizeof(double2)};
        const cuuint32_t box[2] = {(cuuint32_t)(2 * p->ETy + 4), (cuuint32_t)d.Ni};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = encode(reinterpret_cast<CUtensorMap*>(&p->tmaps[i]), CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, src[i].ptr, dims,
                            strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return DNS_ECUDA;
    }
    return DNS_OK;
}

template <int NT, int NWN> static void ypair_launch(dns_plan* p, int stage, int derive_only) {
    const DnsDev& d = p->d;
    const int KS2 = d.Kp >> 3, ET = 4 * NT * NWN;
    const unsigned grid = d.lin ? (unsigned)(d.nkz * d.nmodes * ((d.Eg + ET - 1) / ET))
                                : (unsigned)((d.P - 1) * ((d.E + ET - 1) / ET));
    const size_t smem = dns_ypair_smem(d.Ni, d.Ny, ET);
#define LAUNCH(K)                                                                                     \
    {                                                                                                 \
        auto kern = k_ypair<NT, NWN, K>;                                                              \
        static DnsSmemGrant grant;            /* the attributes are set once per instantiation, device and size, not per launch */ \
        dns_grant_smem(kern, smem, grant, 0, true);                                                   \
        const CUtensorMap* tm = reinterpret_cast<const CUtensorMap*>(p->tmaps);                       \
        dns_launch(kern, dim3(grid), dim3(32 * KS2 * NWN), smem, p->stream, d, tm[0], tm[1], tm[2], stage, derive_only); \
    }
    switch (KS2) {
        case 2: LAUNCH(2) break;
        case 3: LAUNCH(3) break;
        case 4: LAUNCH(4) break;
        case 6: LAUNCH(6) break;
        default: LAUNCH(0) break;
    }
#undef LAUNCH
}

void launch_ypair(dns_plan* p, int stage, int derive_only) {
    const int NT = p->NTy, NWN = p->ETy / (4 * NT);
    if (NT == 1 && NWN == 1) ypair_launch<1, 1>(p, stage, derive_only);
    else if (NT == 2 && NWN == 1) ypair_launch<2, 1>(p, stage, derive_only);
    else if (NT == 1 && NWN == 2) ypair_launch<1, 2>(p, stage, derive_only);
    else if (NT == 2 && NWN == 2) ypair_launch<2, 2>(p, stage, derive_only);
    else if (NT == 4 && NWN == 1) ypair_launch<4, 1>(p, stage, derive_only);
    else ypair_launch<1, 4>(p, stage, derive_only);
}

void launch_mean(dns_plan* p, int stage, int derive_only, cudaStream_t stream) {
    const DnsDev& d = p->d;
    const size_t smem = (size_t)6 * d.Ny * 8 * sizeof(double);
    static DnsSmemGrant grant;
    dns_grant_smem(k_mean, smem, grant, 48 * 1024, false);      // Ny >= 129
    // small ensembles: the kernel is one or a few CTAs whose serial rounds over the rows ARE its duration (and, below about
    // 16 members, longer than the z-forward + per-pair kernels it runs beside): 64 row slots finish Ny <= 66 in one round
    const int threads = (d.E <= 8 && d.Ni > 32) ? 512 : 256;
    k_mean<<<(d.E + 7) / 8, threads, smem, stream>>>(d, stage, derive_only);
}

void launch_abi_to_internal(dns_plan* p, const double2* src, double2* dst, int accumulate) {
    const DnsDev& d = p->d;
    dim3 grid(d.P, (d.E + 31) / 32, (d.Ny + 31) / 32), block(32, 8);
    k_abi_to_internal<<<grid, block, 0, p->stream>>>(src, dst, d.Ny, d.P, d.E, accumulate);
}
void launch_internal_to_abi(dns_plan* p, const double2* src, double2* dst) {
    const DnsDev& d = p->d;
    dim3 grid(d.P, (d.E + 31) / 32, (d.Ny + 31) / 32), block(32, 8);
    k_internal_to_abi<<<grid, block, 0, p->stream>>>(src, dst, d.Ny, d.P, d.E);
}
void launch_normalise_state(dns_plan* p) { k_normalise<<<148 * 4, 256, 0, p->stream>>>(p->d); }
void launch_mean_in(dns_plan* p, const double* U, const double* W) {
    k_mean_in<<<(p->d.E + 127) / 128, 128, 0, p->stream>>>(p->d, U, W);
}
void launch_mean_out(dns_plan* p, double* U, double* W) {
    k_mean_out<<<(p->d.E + 127) / 128, 128, 0, p->stream>>>(p->d, U, W);
}
void launch_stats(dns_plan* p) {
    int EB = 1;
    while (EB < p->d.E && EB < 32) EB <<= 1;
    k_stats<<<dim3(p->d.Ny, (p->d.E + EB - 1) / EB), 256, 0, p->stream>>>(p->d);
}

size_t dns_ens_count(const DnsDev& d) { return 2 * ((size_t)3 * d.Ny * d.nkz + (size_t)d.Ny * d.Mz); }
void launch_ens(dns_plan* p, int phase) {
    const DnsDev& d = p->d;
    const int nwarps = 3 * d.Ni * d.nkz + d.Ni * d.Mz;
    k_ens<<<(nwarps + 7) / 8, 256, 0, p->stream>>>(d, phase);
}
void launch_diag_energy_part(dns_plan* p, double* part) { k_diag_energy<<<p->d.Ny, 256, 0, p->stream>>>(p->d, part); }
void launch_diag(dns_plan* p, double t) {
    const DnsDev& d = p->d;
    double* part = d.diag + (size_t)d.E * 6;
    k_diag_energy<<<d.Ny, 256, 0, p->stream>>>(d, part);
    k_diag_rows<<<(d.E + 127) / 128, 128, 0, p->stream>>>(d, part, t);
}
