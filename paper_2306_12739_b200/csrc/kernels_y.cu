// Wall-normal part of one stage (north_star subsystems (3), (4)).
//   k_ypair : one CTA per (kx,kz) pair and member tile.  Everything that couples only along y is chained in
//             shared memory: F,G assembly (Eq. 4-5), RK3 combination, the precomputed-inverse
//             solves of Eq. 12-13 for ALL members of the tile at once, dv/dy, the u,w
//             reconstruction of Eq. 17-18 and du/dy, dw/dy.  The contractions are [Ni x Ni] x [Ni x 2 ET] fp64
//             tensor-core MMAs (DMMA.8x8x4; the only fp64 MMA shape sm_100a executes natively).
//   k_mean  : mean profiles U00, W00 (Eq. 14-15) with the wall lift f+-  and the mass-flux
//             pressure gamma solved so that the discrete bulk flux is held.
// plus layout conversion, input normalisation and diagnostics.
#include "dns_internal.h"

namespace {

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}

// acc[nt] += A[rows 8w..8w+7][0..Ni) * Bs[0..K)[8nt..8nt+7];  A row-major in global memory (ld = Ni), Bs in
// shared memory with leading dimension ld (rows >= Ni are zero).
template <int NT>
__device__ __forceinline__ void gemm_acc(double (&acc)[NT][2], const double* __restrict__ A, const double* Bs,
                                         int Ni, int K, int ld, int r, int t, int g) {
    const bool rok = r < Ni;
    const double* Ar = A + (size_t)(rok ? r : 0) * Ni;
#pragma unroll 4
    for (int k0 = 0; k0 < K; k0 += 4) {
        const int k = k0 + t;
        const double a = (rok && k < Ni) ? __ldg(Ar + k) : 0.0;
        const double* bp = Bs + (size_t)k * ld + g;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) dmma(acc[nt], a, bp[8 * nt]);
    }
}

template <int NT> __device__ __forceinline__ void zero_acc(double (&acc)[NT][2]) {
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
}

// grid = (P-1) * ntile_e ; block = 32 * MT, MT = ceil(Ni/8); dynamic smem = 5 panels of K x ld doubles
template <int NT>
__global__ void k_ypair(DnsDev d, int stage, int derive_only) {
    extern __shared__ double smy[];
    constexpr int NC = 8 * NT, ET = 4 * NT;
    constexpr int ld = (NC % 16 == 0) ? NC + 8 : NC;    // row stride = 64 B mod 128 B: conflict-free B fragments
    const int Ni = d.Ni, MT = blockDim.x >> 5, K = MT * 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int ntile_e = (d.E + ET - 1) / ET;
    const int p = 1 + blockIdx.x / ntile_e, e0 = (blockIdx.x % ntile_e) * ET;
    const int n = p / d.nkz, mi = p % d.nkz;
    const int mabs = mi < d.nzh ? mi : d.nkz - mi;
    const double kx = d.kx[n], kz = d.kz[mi], alpha = kx * kx + kz * kz;
    const int hi = stage == 0 ? 0 : 1;
    const double hdt = (stage == 0 ? 0.5 : 1.0) * d.dt;
    const size_t NN = (size_t)Ni * Ni;
    const double* mAinv = d.mats + (((size_t)hi * d.nkx * d.nzh + (size_t)n * d.nzh + mabs) * 3) * NN;
    const double* mAD = mAinv + NN;
    const double* mSinv = mAD + NN;
    const size_t PS = (size_t)K * ld;
    double* P0 = smy;
    double* P1 = P0 + PS;
    double* P2 = P1 + PS;
    double* P3 = P2 + PS;
    double* P4 = P3 + PS;
    const int r = 8 * warp + g;                         // interior row owned in every fragment
    const bool rok = r < Ni;
    // global offset of element (row r, pair p, member e0 + 4nt + t)
    const size_t gbase = ((size_t)(r + 1) * d.P + p) * d.E + e0 + t;
    auto eok = [&](int nt) { return rok && (e0 + 4 * nt + t) < d.E; };
    auto sidx = [&](int nt) { return (size_t)r * ld + 8 * nt + 2 * t; };
    const double2 Z2 = make_double2(0.0, 0.0);
    double2* vout = stage == 2 ? d.vt : d.vs;

    // zero every panel once (padding rows >= Ni and padding columns must hold finite zeros)
    for (size_t i = threadIdx.x; i < 5 * PS; i += blockDim.x) smy[i] = 0.0;
    __syncthreads();

    double acc[NT][2];
    if (!derive_only) {
        // ---- A: H = i kx Nu + i kz Nw -> P0 ; G = i kz Nu - i kx Nw, RK3 combination, eta rhs -> P1
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (!eok(nt)) continue;
            const size_t gi = gbase + 4 * nt;
            const double2 nu = d.Nh[gi], nw = d.Nh[2 * d.S + gi];
            const double2 H = make_double2(-kx * nu.y - kz * nw.y, kx * nu.x + kz * nw.x);
            double2 G = make_double2(-kz * nu.y + kx * nw.y, kz * nu.x - kx * nw.x);      // Eq. 5
            double2 Gc;
            if (stage == 0) { d.G0[gi] = G; Gc = G; }
            else if (stage == 1) { const double2 g0 = d.G0[gi]; d.G1[gi] = G; Gc = make_double2(2.0 * G.x - g0.x, 2.0 * G.y - g0.y); }
            else { const double2 g0 = d.G0[gi], g1 = d.G1[gi];
                   Gc = make_double2((g0.x + 4.0 * g1.x + G.x) / 6.0, (g0.y + 4.0 * g1.y + G.y) / 6.0); }
            const double2 et = d.et[gi];
            P0[sidx(nt)] = H.x; P0[sidx(nt) + 1] = H.y;
            P1[sidx(nt)] = 2.0 * et.x - hdt * Gc.x; P1[sidx(nt) + 1] = 2.0 * et.y - hdt * Gc.y;
        }
        __syncthreads();
        // ---- B: F = -alpha Nv - D H (Eq. 4 with Eq. 10's sign), RK3 combination; -h dt Fc -> P2 ; 2 v_t -> P3
        zero_acc<NT>(acc);
        gemm_acc<NT>(acc, d.Dii, P0, Ni, K, ld, r, t, g);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (!eok(nt)) continue;
            const size_t gi = gbase + 4 * nt;
            const double2 nv = d.Nh[d.S + gi];
            const double2 F = make_double2(-alpha * nv.x - acc[nt][0], -alpha * nv.y - acc[nt][1]);
            double2 Fc;
            if (stage == 0) { d.F0[gi] = F; Fc = F; }
            else if (stage == 1) { const double2 f0 = d.F0[gi]; d.F1[gi] = F; Fc = make_double2(2.0 * F.x - f0.x, 2.0 * F.y - f0.y); }
            else { const double2 f0 = d.F0[gi], f1 = d.F1[gi];
                   Fc = make_double2((f0.x + 4.0 * f1.x + F.x) / 6.0, (f0.y + 4.0 * f1.y + F.y) / 6.0); }
            const double2 vt = d.vt[gi];
            P2[sidx(nt)] = -hdt * Fc.x; P2[sidx(nt) + 1] = -hdt * Fc.y;
            P3[sidx(nt)] = 2.0 * vt.x;  P3[sidx(nt) + 1] = 2.0 * vt.y;
        }
        __syncthreads();
        // ---- C: v' = Ainv (2 v_t) + AD (-h dt Fc) - v_t (Eq. 12) -> global, P0 ; eta' = Sinv P1 - eta_t (Eq. 13) -> P4
        zero_acc<NT>(acc);
        gemm_acc<NT>(acc, mAinv, P3, Ni, K, ld, r, t, g);
        gemm_acc<NT>(acc, mAD, P2, Ni, K, ld, r, t, g);
        double acc2[NT][2];
        zero_acc<NT>(acc2);
        gemm_acc<NT>(acc2, mSinv, P1, Ni, K, ld, r, t, g);
        __syncthreads();                                 // every warp has finished reading P0..P3
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (!eok(nt)) continue;
            const size_t gi = gbase + 4 * nt;
            const double2 vn = make_double2(acc[nt][0] - 0.5 * P3[sidx(nt)], acc[nt][1] - 0.5 * P3[sidx(nt) + 1]);
            const double2 et = d.et[gi];
            const double2 en = make_double2(acc2[nt][0] - et.x, acc2[nt][1] - et.y);
            vout[gi] = vn;
            if (stage == 2) d.et[gi] = en;
            P0[sidx(nt)] = vn.x; P0[sidx(nt) + 1] = vn.y;
            P4[sidx(nt)] = en.x; P4[sidx(nt) + 1] = en.y;
        }
        __syncthreads();
    } else {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            if (!eok(nt)) continue;
            const size_t gi = gbase + 4 * nt;
            const double2 vt = d.vt[gi], et = d.et[gi];
            P0[sidx(nt)] = vt.x; P0[sidx(nt) + 1] = vt.y;
            P4[sidx(nt)] = et.x; P4[sidx(nt) + 1] = et.y;
        }
        __syncthreads();
    }
    // ---- D: dv/dy = D v' ; u = (i kx Dv - i kz eta)/alpha, w = (i kz Dv + i kx eta)/alpha (Eq. 17-18) -> global, P2, P3
    zero_acc<NT>(acc);
    gemm_acc<NT>(acc, d.Dii, P0, Ni, K, ld, r, t, g);
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        if (!eok(nt)) continue;
        const size_t gi = gbase + 4 * nt;
        const double2 dv = make_double2(acc[nt][0], acc[nt][1]);
        const double2 en = make_double2(P4[sidx(nt)], P4[sidx(nt) + 1]);
        const double2 u = make_double2((-kx * dv.y + kz * en.y) / alpha, (kx * dv.x - kz * en.x) / alpha);
        const double2 w = make_double2((-kz * dv.y - kx * en.y) / alpha, (kz * dv.x + kx * en.x) / alpha);
        d.uh[gi] = u;
        d.wh[gi] = w;
        P2[sidx(nt)] = u.x; P2[sidx(nt) + 1] = u.y;
        P3[sidx(nt)] = w.x; P3[sidx(nt) + 1] = w.y;
    }
    __syncthreads();
    // ---- E: du/dy, dw/dy
    zero_acc<NT>(acc);
    gemm_acc<NT>(acc, d.Dii, P2, Ni, K, ld, r, t, g);
    double acc2[NT][2];
    zero_acc<NT>(acc2);
    gemm_acc<NT>(acc2, d.Dii, P3, Ni, K, ld, r, t, g);
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        if (!eok(nt)) continue;
        const size_t gi = gbase + 4 * nt;
        d.duh[gi] = make_double2(acc[nt][0], acc[nt][1]);
        d.dwh[gi] = make_double2(acc2[nt][0], acc2[nt][1]);
    }
    (void)Z2;
}

// ------------------------------------------------------------------------------------------------ mean flow
// grid = ceil(E/8); block = 256 = 32 row slots x 8 members; dynamic smem = 6 vectors [Ny][8]
__global__ void __launch_bounds__(256) k_mean(DnsDev d, int stage, int derive_only) {
    extern __shared__ double smm[];
    const int Ny = d.Ny, Ni = d.Ni;
    const int el = threadIdx.x & 7, rs = threadIdx.x >> 3, e = blockIdx.x * 8 + el;
    const bool eok = e < d.E;
    const int hi = stage == 0 ? 0 : 1;
    const double hdt = (stage == 0 ? 0.5 : 1.0) * d.dt;
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
        for (int j = rs; j < Ny; j += 32) {
            double a = 0.0, b = 0.0;
            if (eok && j > 0 && j < Ny - 1) {
                for (int q = 0; q < d.Mz; ++q) {
                    const double2 v = d.uvpart[((size_t)j * d.Mz + q) * d.E + e];
                    a += v.x; b += v.y;
                }
                a *= d.invMxMz; b *= d.invMxMz;
                const size_t gi = (size_t)j * d.E + e;
                if (stage == 0) d.uvc0[gi] = make_double2(a, b);
                else if (stage == 1) { const double2 s0 = d.uvc0[gi]; d.uvc1[gi] = make_double2(a, b); a = 2.0 * a - s0.x; b = 2.0 * b - s0.y; }
                else { const double2 s0 = d.uvc0[gi], s1 = d.uvc1[gi]; a = (s0.x + 4.0 * s1.x + a) / 6.0; b = (s0.y + 4.0 * s1.y + b) / 6.0; }
            }
            uvc[j * 8 + el] = a; wvc[j * 8 + el] = b;
        }
        __syncthreads();
        // rhs = 2 U_t - h dt D [uv] - 2 bc  (Eq. 14 with S0p = 2I - S0m and the wall columns on the rhs)
        for (int i = rs; i < Ni; i += 32) {
            double su = 0.0, sw = 0.0;
            const double* Dr = d.Dfull + (size_t)(i + 1) * Ny;
            for (int j = 1; j < Ny - 1; ++j) { su += Dr[j] * uvc[j * 8 + el]; sw += Dr[j] * wvc[j * 8 + el]; }
            const double ut = eok ? d.Ut[(size_t)(i + 1) * d.E + e] : 0.0, wt = eok ? d.Wt[(size_t)(i + 1) * d.E + e] : 0.0;
            ru[i * 8 + el] = 2.0 * ut - hdt * su - 2.0 * d.bc[hi * Ni + i];
            rw[i * 8 + el] = 2.0 * wt - hdt * sw;
        }
        __syncthreads();
        for (int i = rs; i < Ni; i += 32) {
            double su = 0.0, sw = 0.0;
            const double* Sr = d.S0inv + (size_t)hi * Ni * Ni + (size_t)i * Ni;
            for (int k = 0; k < Ni; ++k) { su += Sr[k] * ru[k * 8 + el]; sw += Sr[k] * rw[k * 8 + el]; }
            const double ut = eok ? d.Ut[(size_t)(i + 1) * d.E + e] : 0.0, wt = eok ? d.Wt[(size_t)(i + 1) * d.E + e] : 0.0;
            Un[(i + 1) * 8 + el] = su - ut;
            Wn[(i + 1) * 8 + el] = sw - wt;
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
        for (int j = rs; j < Ny; j += 32) {
            double un = Un[j * 8 + el];
            if (j > 0 && j < Ny - 1) un += gam[el] * d.Ugam[hi * Ni + j - 1];
            Un[j * 8 + el] = un;
            if (eok) { Uout[(size_t)j * d.E + e] = un; Wout[(size_t)j * d.E + e] = Wn[j * 8 + el]; }
        }
        __syncthreads();
    } else {
        for (int j = rs; j < Ny; j += 32) {
            Un[j * 8 + el] = eok ? d.Ut[(size_t)j * d.E + e] : 0.0;
            Wn[j * 8 + el] = eok ? d.Wt[(size_t)j * d.E + e] : 0.0;
        }
        __syncthreads();
    }
    // (0,0) column of the transform inputs: u = U00, w = W00, du/dy = D U00, dw/dy = D W00
    for (int j = rs; j < Ny; j += 32) {
        double du = 0.0, dw = 0.0;
        const double* Dr = d.Dfull + (size_t)j * Ny;
        for (int k = 0; k < Ny; ++k) { du += Dr[k] * Un[k * 8 + el]; dw += Dr[k] * Wn[k * 8 + el]; }
        if (eok) {
            const size_t gi = ((size_t)j * d.P) * d.E + e;
            d.uh[gi] = make_double2(Un[j * 8 + el], 0.0);
            d.wh[gi] = make_double2(Wn[j * 8 + el], 0.0);
            d.duh[gi] = make_double2(du, 0.0);
            d.dwh[gi] = make_double2(dw, 0.0);
        }
    }
}

// ------------------------------------------------------------------------------------------------ layout / IO
// ABI [E][P][Ny] <-> internal [Ny][P][E]; grid = (P, ceil(E/32), ceil(Ny/32)), block = (32, 8)
__global__ void k_abi_to_internal(const double2* __restrict__ src, double2* __restrict__ dst, int Ny, int P, int E) {
    __shared__ double2 tile[32][33];
    const int p = blockIdx.x, e0 = blockIdx.y * 32, j0 = blockIdx.z * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int e = e0 + k, j = j0 + threadIdx.x;
        if (e < E && j < Ny) tile[k][threadIdx.x] = src[((size_t)e * P + p) * Ny + j];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int j = j0 + k, e = e0 + threadIdx.x;
        if (e < E && j < Ny) dst[((size_t)j * P + p) * E + e] = tile[threadIdx.x][k];
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

// diagnostics: energy partial sums per (j, e), then the per-member rows
__global__ void k_diag_energy(DnsDev d, double* __restrict__ part) {
    const int j = blockIdx.x;
    for (int e = threadIdx.x; e < d.E; e += blockDim.x) {
        double s = 0.0;
        for (int p = 0; p < d.P; ++p) {
            const size_t gi = ((size_t)j * d.P + p) * d.E + e;
            const double2 u = d.uh[gi], v = d.vt[gi], w = d.wh[gi];
            const double cn = (p / d.nkz) == 0 ? 1.0 : 2.0;
            s += cn * (u.x * u.x + u.y * u.y + v.x * v.x + v.y * v.y + w.x * w.x + w.y * w.y);
        }
        part[(size_t)j * d.E + e] = 0.25 * d.w[j] * s;
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

}  // namespace

static size_t ypair_smem(int Ni, int NT) {
    const int NC = 8 * NT, ld = (NC % 16 == 0) ? NC + 8 : NC, K = ((Ni + 7) / 8) * 8;
    return (size_t)5 * K * ld * sizeof(double);
}

void launch_ypair(dns_plan* p, int stage, int derive_only) {
    const DnsDev& d = p->d;
    const int MT = (d.Ni + 7) / 8, ET = p->ETy, NT = ET / 4;
    const unsigned grid = (unsigned)((d.P - 1) * ((d.E + ET - 1) / ET));
    const size_t smem = ypair_smem(d.Ni, NT);
#define LAUNCH(NTv)                                                                                   \
    {                                                                                                 \
        auto kern = k_ypair<NTv>;                                                                     \
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);           \
        kern<<<grid, 32 * MT, smem, p->stream>>>(d, stage, derive_only);                              \
    }
    switch (NT) {
        case 1: LAUNCH(1) break;
        case 2: LAUNCH(2) break;
        case 4: LAUNCH(4) break;
        default: LAUNCH(8) break;
    }
#undef LAUNCH
}

void launch_mean(dns_plan* p, int stage, int derive_only) {
    const DnsDev& d = p->d;
    const size_t smem = (size_t)6 * d.Ny * 8 * sizeof(double);
    k_mean<<<(d.E + 7) / 8, 256, smem, p->stream>>>(d, stage, derive_only);
}

void launch_abi_to_internal(dns_plan* p, const double2* src, double2* dst) {
    const DnsDev& d = p->d;
    dim3 grid(d.P, (d.E + 31) / 32, (d.Ny + 31) / 32), block(32, 8);
    k_abi_to_internal<<<grid, block, 0, p->stream>>>(src, dst, d.Ny, d.P, d.E);
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
void launch_diag(dns_plan* p, double t) {
    const DnsDev& d = p->d;
    double* part = d.diag + (size_t)d.E * 6;
    k_diag_energy<<<d.Ny, 256, 0, p->stream>>>(d, part);
    k_diag_rows<<<(d.E + 127) / 128, 128, 0, p->stream>>>(d, part, t);
}
