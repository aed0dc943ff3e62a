// Linearised forward / adjoint ensemble (PAPER.md:296-317 and Appendix B, Eq. B.1-B.6 :390-417).
// Every member is a disturbance with ONE streamwise wavenumber on a frozen streamwise-mean base flow (U, V, W)(y, z), so x is
// analytic (d/dx = i kx) and only z is transformed.  A stage reuses the DNS kernels on arrays with a single kx row
// (k_zinv* -> 8 mixed fields, k_zfwd*, k_ypair with the member's own single-kx matrices, "also valid for the adjoint
// equations", :304); this file holds what is specific to the linear problem:
//   k_lin_products : the linear vector that takes the place of u.grad u in Eq. 4-5, formed pointwise on the padded z grid
//                    forward (B.2)  N_i = (U.grad) u_i + (u.grad) U_i
//                    adjoint (B.5, reversed time, reading L1)  N_i = -(U.grad) lam_i - U_j d_i lam_j
//   k_lin_base     : copies the kx = 0 column of one member of a DNS plan's mixed arrays = the base flow and its gradient
//   k_lin_energy   : E_e = (1/2) sum_m sum_j w_j (|u|^2 + |v|^2 + |w|^2)                                  (B.1)
//   k_lin_gs_*     : modified Gram-Schmidt in member order within each kx group, energy inner product     (:417)
#include "dns_internal.h"

namespace {

__device__ __forceinline__ double2 cscale(double s, double2 a) { return make_double2(s * a.x, s * a.y); }
__device__ __forceinline__ double2 cmuli(double s, double2 a) { return make_double2(-s * a.y, s * a.x); }      // (i s) a
__device__ __forceinline__ double2 cadd3(double2 a, double2 b, double2 c) { return make_double2(a.x + b.x + c.x, a.y + b.y + c.y); }

// grid = (ceil(E / 128), Mz, Ni); mixed arrays with one kx row are [Ny][Mz][Epad], Epad = ntl << etl
__global__ void __launch_bounds__(128) k_lin_products(DnsDev d, int adjoint) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y, j = blockIdx.z + 1;
    if (e >= d.E) return;
    const size_t Epad = (size_t)d.ntl << d.etl, gi = ((size_t)j * d.Mz + q) * Epad + e, fs = d.Isz;
    const size_t bi = (size_t)j * d.Mz + q, bs = (size_t)d.Ny * d.Mz;
    const double kx = d.kx[d.nlist[e / d.Eg]];
    const double U = d.base[bi], V = d.base[bs + bi], W = d.base[2 * bs + bi];
    const double2 u = d.I8[gi], v = d.I8[fs + gi], w = d.I8[2 * fs + gi];
    const double2 uy = d.I8[3 * fs + gi], wy = d.I8[4 * fs + gi];
    const double2 uz = d.I8[5 * fs + gi], vz = d.I8[6 * fs + gi], wz = d.I8[7 * fs + gi];
    const double2 ux = cmuli(kx, u), vx = cmuli(kx, v), wx = cmuli(kx, w);
    const double2 vy = make_double2(-ux.x - wz.x, -ux.y - wz.y);      // continuity: dv/dy = -du/dx - dw/dz (interior rows)
    // (U.grad) f for f = u, v, w
    const double2 au = cadd3(cscale(U, ux), cscale(V, uy), cscale(W, uz));
    const double2 av = cadd3(cscale(U, vx), cscale(V, vy), cscale(W, vz));
    const double2 aw = cadd3(cscale(U, wx), cscale(V, wy), cscale(W, wz));
    double2 Nu, Nv, Nw;
    if (!adjoint) {
        const double Uy = d.base[3 * bs + bi], Vy = d.base[4 * bs + bi], Wy = d.base[5 * bs + bi];
        const double Uz = d.base[6 * bs + bi], Vz = d.base[7 * bs + bi], Wz = d.base[8 * bs + bi];
        Nu = cadd3(au, cscale(Uy, v), cscale(Uz, w));                 // + (u.grad) U, dU/dx = 0
        Nv = cadd3(av, cscale(Vy, v), cscale(Vz, w));
        Nw = cadd3(aw, cscale(Wy, v), cscale(Wz, w));
    } else {
        const double2 bx = cadd3(cscale(U, ux), cscale(V, vx), cscale(W, wx));      // U_j d lam_j / dx
        const double2 by = cadd3(cscale(U, uy), cscale(V, vy), cscale(W, wy));
        const double2 bz = cadd3(cscale(U, uz), cscale(V, vz), cscale(W, wz));
        Nu = make_double2(-au.x - bx.x, -au.y - bx.y);
        Nv = make_double2(-av.x - by.x, -av.y - by.y);
        Nw = make_double2(-aw.x - bz.x, -aw.y - bz.y);
    }
    d.I3[gi] = Nu;
    d.I3[fs + gi] = Nv;
    d.I3[2 * fs + gi] = Nw;
}

// base flow of the linear plan from the mixed arrays of a DNS plan (convective form: u v w Du Dw uz vz wz), kx = 0 column
// of `member`, which is a real function of (y, z).  grid = (ceil(Mz / 64), Ni), block = 64
__global__ void k_lin_base(DnsDev lin, DnsDev dns, int member) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y + 1;
    if (q >= dns.Mz) return;
    const size_t src = dns_mix_off(dns, j, q, 0, member), fs = dns.Isz;
    const size_t bi = (size_t)j * lin.Mz + q, bs = (size_t)lin.Ny * lin.Mz;
    const double U = dns.I8[src].x, V = dns.I8[fs + src].x, W = dns.I8[2 * fs + src].x;
    const double Uy = dns.I8[3 * fs + src].x, Wy = dns.I8[4 * fs + src].x;
    const double Uz = dns.I8[5 * fs + src].x, Vz = dns.I8[6 * fs + src].x, Wz = dns.I8[7 * fs + src].x;
    lin.base[bi] = U; lin.base[bs + bi] = V; lin.base[2 * bs + bi] = W;
    lin.base[3 * bs + bi] = Uy; lin.base[4 * bs + bi] = -Wz; lin.base[5 * bs + bi] = Wy;      // dV/dy = -dW/dz at kx = 0
    lin.base[6 * bs + bi] = Uz; lin.base[7 * bs + bi] = Vz; lin.base[8 * bs + bi] = Wz;
}

// wall rows of the state are zero (Eq. 8); every (n, m) is a valid mode here (n >= 1)
__global__ void k_lin_normalise(DnsDev d) {
    const size_t row = (size_t)d.P * d.E;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < row; i += (size_t)gridDim.x * blockDim.x) {
        const double2 z = make_double2(0.0, 0.0);
        d.vt[i] = z; d.et[i] = z;
        d.vt[(size_t)(d.Ny - 1) * row + i] = z; d.et[(size_t)(d.Ny - 1) * row + i] = z;
    }
}

// out[e] = sum_j part[j][e] in ascending j (part = the per-plane sums of k_diag_energy, already weighted)
__global__ void k_lin_energy_rows(DnsDev d, const double* __restrict__ part, double* __restrict__ out) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= d.E) return;
    double s = 0.0;
    for (int j = 0; j < d.Ny; ++j) s += part[(size_t)j * d.E + e];
    out[e] = s;
}

// ---- modified Gram-Schmidt (reading L4) in member order within each kx group.  The vectors are (v, eta) with
// their u, w (linear in the state); the inner product is (1/2) sum_{m,j} w_j (conj(u_a) u_b + conj(v_a) v_b + conj(w_a) w_b).
// The loop over a is serial by nature; everything inside one a is not: the products of member a with itself and with all
// later members b of its group are independent, and so are their updates.  Two launches per a over a grid of
// (kx groups) x (NCH chunks of the Ny P elements of a vector):
//   k_lin_gs_dots   : part[g][chunk][b] = sum over the chunk of w_j conj(x_a) . x_b for b = a .. Eg-1 (b = a: the norm)
//   k_lin_gs_update : every CTA adds the chunk sums in ascending order (the same numbers in every CTA), then in its own chunk
//                     x_b -= (<x_a, x_b> / <x_a, x_a>) x_a for b > a and, once all of those have read x_a, x_a /= |x_a|
// which is the modified Gram-Schmidt step with the division by |x_a| moved out of the inner product.  Threads = EB member
// lanes x (256 / EB) element slots; slot and chunk sums are added in fixed ascending order (deterministic).  A member with
// exactly zero (or non-finite) energy has no direction: it is set to zero instead of being divided by zero, so that it cannot
// turn the later members of its group into NaN; its energy then reads 0.
// (Until round 3 this was one 1024-thread CTA per kx group: 2.08 ms for 3 x 15 vectors at 48 x 65 x 48 on 3 of 148 SMs.)
constexpr int GS_THREADS = 256;
__device__ __forceinline__ int gs_lanes(int Eg) { int b = 1; while (b < Eg && b < 32) b <<= 1; return b; }

__global__ void __launch_bounds__(GS_THREADS) k_lin_gs_dots(DnsDev d, int a, int NCH, double2* __restrict__ part) {
    __shared__ double2 red[GS_THREADS];
    const int g = blockIdx.x, ch = blockIdx.y, EB = gs_lanes(d.Eg), nslot = GS_THREADS / EB;
    const int bl = threadIdx.x % EB, slot = threadIdx.x / EB;
    const int L = d.Ny * d.P, CL = (L + NCH - 1) / NCH, i0 = ch * CL, i1 = min(L, i0 + CL);
    const int e_first = g * d.Eg, ea = e_first + a;
    for (int b0 = a; b0 < d.Eg; b0 += EB) {
        const int b = b0 + bl, eb = e_first + b;
        double2 acc = make_double2(0.0, 0.0);
        if (b < d.Eg)
            for (int i = i0 + slot; i < i1; i += nslot) {
                const size_t ga = (size_t)i * d.E + ea, gb = (size_t)i * d.E + eb;
                const double wj = d.w[i / d.P];
                const double2 ua = d.uh[ga], va = d.vt[ga], wa = d.wh[ga], ub = d.uh[gb], vb = d.vt[gb], wb = d.wh[gb];
                acc.x += wj * (ua.x * ub.x + ua.y * ub.y + va.x * vb.x + va.y * vb.y + wa.x * wb.x + wa.y * wb.y);      // conj(a) b
                acc.y += wj * (ua.x * ub.y - ua.y * ub.x + va.x * vb.y - va.y * vb.x + wa.x * wb.y - wa.y * wb.x);
            }
        red[slot * EB + bl] = acc;
        __syncthreads();
        if (slot == 0 && b < d.Eg) {
            double2 t = make_double2(0.0, 0.0);
            for (int k = 0; k < nslot; ++k) { t.x += red[k * EB + bl].x; t.y += red[k * EB + bl].y; }
            part[((size_t)g * NCH + ch) * d.Eg + b] = t;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(GS_THREADS) k_lin_gs_update(DnsDev d, int a, int NCH, const double2* __restrict__ part) {
    const int g = blockIdx.x, ch = blockIdx.y, EB = gs_lanes(d.Eg), nslot = GS_THREADS / EB;
    const int bl = threadIdx.x % EB, slot = threadIdx.x / EB;
    const int L = d.Ny * d.P, CL = (L + NCH - 1) / NCH, i0 = ch * CL, i1 = min(L, i0 + CL);
    const int e_first = g * d.Eg, ea = e_first + a;
    double2* X[4] = {d.vt, d.et, d.uh, d.wh};
    double saa = 0.0;
    for (int k = 0; k < NCH; ++k) saa += part[((size_t)g * NCH + k) * d.Eg + a].x;
    const double en = 0.5 * saa;                              // energy of x_a (B.1)
    const bool ok = en > 0.0 && en < 1.0e300;
    for (int b0 = a + 1; b0 < d.Eg; b0 += EB) {
        const int b = b0 + bl, eb = e_first + b;
        if (b >= d.Eg || !ok) continue;
        double2 sab = make_double2(0.0, 0.0);
        for (int k = 0; k < NCH; ++k) { const double2 t = part[((size_t)g * NCH + k) * d.Eg + b]; sab.x += t.x; sab.y += t.y; }
        const double2 c = make_double2(sab.x / saa, sab.y / saa);          // <x_a, x_b> / <x_a, x_a>
        for (int i = i0 + slot; i < i1; i += nslot) {
            const size_t ga = (size_t)i * d.E + ea, gb = (size_t)i * d.E + eb;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const double2 xa = X[f][ga];
                double2 xb = X[f][gb];
                xb.x -= c.x * xa.x - c.y * xa.y;
                xb.y -= c.x * xa.y + c.y * xa.x;
                X[f][gb] = xb;
            }
        }
    }
    __syncthreads();                                          // every read of x_a in this chunk is done
    const double sc = ok ? 1.0 / sqrt(en) : 0.0;
    for (int i = i0 + threadIdx.x; i < i1; i += GS_THREADS) {
        const size_t ga = (size_t)i * d.E + ea;
#pragma unroll
        for (int f = 0; f < 4; ++f) X[f][ga] = cscale(sc, X[f][ga]);
    }
}

}  // namespace

void launch_lin_products(dns_plan* p, int adjoint) {
    const DnsDev& d = p->d;
    dim3 grid((d.E + 127) / 128, d.Mz, d.Ni);
    k_lin_products<<<grid, 128, 0, p->stream>>>(d, adjoint);
}
void launch_lin_base(dns_plan* lin, const dns_plan* dns, int member, cudaStream_t stream) {
    dim3 grid((dns->d.Mz + 63) / 64, dns->d.Ni);
    k_lin_base<<<grid, 64, 0, stream>>>(lin->d, dns->d, member);
}
void launch_lin_normalise(dns_plan* p) { k_lin_normalise<<<148, 256, 0, p->stream>>>(p->d); }
void launch_lin_energy(dns_plan* p, double* out_dev) {
    const DnsDev& d = p->d;
    double* part = d.lin_scr + 2 * (size_t)d.E;
    launch_diag_energy_part(p, part);
    k_lin_energy_rows<<<(d.E + 127) / 128, 128, 0, p->stream>>>(d, part, out_dev);
}
void launch_lin_gs(dns_plan* p) {
    const DnsDev& d = p->d;
    // chunk sums live in the [Ny][E] part of lin_scr (shared with the energy's plane sums, same stream): E NCH complex
    int NCH = d.Ny / 2;
    if (NCH > 32) NCH = 32;
    if (NCH < 1) NCH = 1;
    double2* part = reinterpret_cast<double2*>(d.lin_scr + 2 * (size_t)d.E);
    const dim3 grid(d.nmodes, NCH);
    for (int a = 0; a < d.Eg; ++a) {
        k_lin_gs_dots<<<grid, GS_THREADS, 0, p->stream>>>(d, a, NCH, part);
        k_lin_gs_update<<<grid, GS_THREADS, 0, p->stream>>>(d, a, NCH, part);
    }
}
