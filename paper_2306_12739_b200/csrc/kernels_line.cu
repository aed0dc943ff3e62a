// Fused x-line kernel (SURVEY.md 8(a) rows a4 (x part), a5, a6 (x part); north_star subsystems (1) and (2)).
// One "line" = (plane j, z index q, member e).  For every line the kernel
//   * reads the 8 mixed (kx, z) fields u v w Du Dw uz vz wz written by k_zinv, each exactly once,
//   * forms the 11 physical fields u, v, w, their x/z derivatives and Du, Dw with 6 Hermitian two-for-one complex
//     inverse FFTs along x (x-derivatives = i kx folded into the packing; dv/dy = -du/dx - dw/dz pointwise, which
//     holds exactly at interior rows for the u, w of Eq. 17-18),
//   * forms the convective products u.grad u_i and the x-sums of u v, w v (Eq. 6-7) in registers,
//   * returns (u.grad)u, (u.grad)v, (u.grad)w on the retained kx with 2 forward FFTs.
// Rotational form (row f1, template parameter ROT): the 6 mixed fields u v w omega_x omega_y omega_z give the 6 physical
// fields with 3 two-for-one inverse FFTs, H = omega x u and the x-sums of H_x, H_z are formed in registers, and the same
// 2 forward FFTs return H on the retained kx.
// Nothing in physical space ever reaches HBM.
//
// Thread mapping: a line is shared by SL "slots"; every slot owns R1 x-points of each physical field in registers.
// A "group" = SL slots x TPS lanes (lanes = members, or members x lines when E < TPS; TPS = 4, 8 or 16 by ensemble
// size) = 1..6 warps; the four-step exchanges need only a group-local barrier.  The four-step twiddles are powers of
// one per-slot register value, and the thread that issues the bulk copies sits in a warp that idles in the first pass.  Groups are persistent: each walks over work items (j, q-group, member
// tile).  The mixed arrays are stored tile-major ([j][q][tile][kx][ET]) so that the input of one item and one field
// is ONE contiguous block, fetched by a single TMA bulk copy (cp.async.bulk + mbarrier) into a ring of field slots
// one item ahead of the arithmetic: global latency never touches the register file or the LSU pipe.
#include <cstdint>
#include <cstdlib>

#include "dns_internal.h"
#include "fft_codelets.cuh"

using namespace dnsfft;

namespace {

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
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

template <int GT> __device__ __forceinline__ void group_sync(int grp) {
    if (GT == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(GT) : "memory");
}

// row pitch (in double2) of an exchange buffer with `cols` columns of TPS lanes: for TPS = 4 two slots share a
// quarter-warp, so consecutive rows must start 64 B apart modulo 128 B to stay bank-conflict free
constexpr int line_pitch(int cols, int TPS) {
    return TPS >= 8 ? cols * TPS : cols * TPS + ((TPS - (cols * TPS) % 8 + 8) % 8);
}

// mode index read for padded position pos: n (positive side), M - pos (negative side, conjugated) or -1 (zero)
template <int M, int NKX> __device__ __forceinline__ int pos_mode(int pos) {
    return pos < NKX ? pos : (pos > M - NKX ? M - pos : -1);
}

// Order in which the 8 mixed fields are consumed (sequence s -> field of I8: 0 u, 1 v, 2 w, 3 Du, 4 Dw, 5 uz, 6 vz,
// 7 wz) by the six complex transforms Z = A + iB (A, B real in x):
//   C = 0: (v, dv/dx)  1: (u, du/dx)  2: (w, dw/dx)  3: (Du, du/dz)  4: (Dw, dw/dz)  5: (dv/dz, -)
// Rotational form: sequence s = field s of I8 (u v w omega_x omega_y omega_z), three transforms of two fields each:
//   C = 0: (u, v)  1: (w, omega_x)  2: (omega_y, omega_z)
__device__ __forceinline__ constexpr int seq_field(int s, bool rot) {
    return rot ? s : (s == 0 ? 1 : s == 1 ? 0 : s == 2 ? 2 : s == 3 ? 3 : s == 4 ? 5 : s == 5 ? 4 : s == 6 ? 7 : 6);
}
// first sequence of transform C and how its second field is made: 0 = a second stored field, 1 = i kx times the first,
// 2 = none
template <int C, bool ROT> struct LineSeq {
    static constexpr int sa = ROT ? 2 * C : (C < 3 ? C : (C == 3 ? 3 : (C == 4 ? 5 : 7)));
    static constexpr int mode = ROT ? 0 : ((C == 3 || C == 4) ? 0 : (C < 3 ? 1 : 2));
};

struct LineSmem {                     // byte offsets inside the dynamic shared memory of a CTA
    int kxs, group0, group_bytes, ring, buf, exch, red, bars, total;
};
__host__ __device__ inline LineSmem line_smem(int R1, int R2, int SL, int TPS, int NG, int NST, int NBUF = 2) {
    const int M = R1 * R2, NKX = M / 3;
    const int PI = line_pitch(R2, TPS), PF = line_pitch(R1, TPS);
    const int BUF = (R1 * PI > R2 * PF) ? R1 * PI : R2 * PF;
    LineSmem s{};
    int off = 0;
    auto take = [&](int bytes) { int o = off; off += (bytes + 127) & ~127; return o; };
    s.kxs = take(NKX * 8);
    s.group0 = off;
    off = 0;
    s.ring = take(NST * NKX * TPS * 16);
    s.buf = take(NBUF * BUF * 16);
    s.exch = NBUF == 4 ? s.buf : take(NKX * TPS * 16);   // four buffers: the handoff area lives in the pair that is free
    s.red = take(SL * TPS * 16);
    s.bars = take(NST * 8);
    s.group_bytes = off;
    s.total = s.group0 + NG * s.group_bytes;
    return s;
}

// ------------------------------------------------------------------------------------------------ the kernel
// grid = persistent CTAs ; block = NG groups of SL * TPS threads
// PAIR (needs SL >= 2 R1): two transforms share every round -- in the first pass of the inverse transforms slots < R1
// work on one transform and slots R1 .. 2 R1 - 1 on the next (without it those slots idle: 6 of 12 for Mx = 72), in the
// second pass every slot finishes both; the second pass of the two forward transforms is split the same way.
// NBUF = 4 (PAIR only): consecutive rounds use different pairs of exchange buffers, so no round needs a second barrier.
// FULL: the member tile fills the lanes of a slot (ET = TPS, every ensemble with E >= TPS): one line per item, the tile
// size is a compile-time constant (all ring / store offsets become immediates) and the item's block offset is linear in
// the item number, so that no integer division is left in the item loop.
template <int R1, int R2, int SL, int TPS, int NG, int NST, int MINB, bool ROT, bool PAIR, int NBUF = 2, bool FULL = false>
__global__ void __launch_bounds__(SL * TPS * NG, MINB) k_line(DnsDev d, int nitems) {
    static_assert(NBUF == 2 || (NBUF == 4 && PAIR), "four exchange buffers belong to the paired rounds");
    static_assert(!PAIR || SL >= 2 * R1, "paired rounds need two sets of first-pass slots");
    constexpr int M = R1 * R2, NKX = M / 3, GT = SL * TPS;
    constexpr int NSEQ = ROT ? 6 : 8;                        // input fields per item = sequence numbers of the ring
    constexpr bool HALF = 2 * NST == NSEQ;                   // ring of half an item: every slot is used twice per item
    // ring of 6 slots for the 8 fields of the convective form: fields 6, 7 reuse the slots of fields 0, 1 (free after the
    // first round), the other four slots take one field per item -- every field is requested at least one whole round
    // before it is needed, which a half ring cannot do once two transforms share a round
    constexpr bool SIX8 = NST == 6 && NSEQ == 8;
    constexpr int PI = line_pitch(R2, TPS), PF = line_pitch(R1, TPS);
    constexpr int BUF = (R1 * PI > R2 * PF) ? R1 * PI : R2 * PF;
    constexpr int SLOT = NKX * TPS;                          // double2 per ring slot
    static_assert(NST == NSEQ || 2 * NST == NSEQ || SIX8, "ring depth");
    DNS_PDL_TRIGGER();
    extern __shared__ __align__(128) unsigned char smraw[];
    const LineSmem L = line_smem(R1, R2, SL, TPS, NG, NST, NBUF);
    double* kxs = reinterpret_cast<double*>(smraw + L.kxs);
    const int grp = threadIdx.x / GT, t = threadIdx.x % GT;
    unsigned char* gs = smraw + L.group0 + grp * L.group_bytes;
    double2* ring = reinterpret_cast<double2*>(gs + L.ring);
    double2* buf0 = reinterpret_cast<double2*>(gs + L.buf);
    double2* buf1 = buf0 + BUF;
    double2* exch_own = reinterpret_cast<double2*>(gs + L.exch);
    double2* red = reinterpret_cast<double2*>(gs + L.red);
    uint64_t* bars = reinterpret_cast<uint64_t*>(gs + L.bars);

    const int sl = t / TPS, lis = t % TPS;
    const double2 om = d.twx[sl % M];                        // w_M^sl
    constexpr int TPSLOG = TPS == 4 ? 2 : (TPS == 8 ? 3 : (TPS == 16 ? 4 : 5));
    const int etlog = FULL ? TPSLOG : d.etl, ET = 1 << etlog, el = lis & (ET - 1), lc = lis >> etlog, LC = TPS >> etlog;
    const int ntile = d.ntl, nqg = (d.Mz + LC - 1) / LC;
    for (int i = threadIdx.x; i < NKX; i += blockDim.x) kxs[i] = d.kx[i];
    if (t == 0) {
        for (int s = 0; s < NST; ++s) mbar_init(bars + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    DNS_PDL_WAIT();                                          // the mixed fields of k_zinv are complete from here on

    const size_t fstride = d.Isz;
    const int E = d.E;
    const int stride = gridDim.x * NG;
    const int lidx = (lc * NKX) * ET + el;                   // + n * ET : element of this lane inside a slot / item block
    // item -> offset of its block inside one mixed field, number of valid lines
    auto item_off = [&](int it, int& nl) -> size_t {
        if constexpr (FULL) { nl = 1; return (size_t)(it + d.Mz * ntile) * SLOT; }   // ((j Mz + q) ntile + te) = it + Mz ntile
        const int te = it % ntile, qg = (it / ntile) % nqg, jj = it / (ntile * nqg) + 1;
        nl = d.Mz - qg * LC < LC ? d.Mz - qg * LC : LC;
        return ((((size_t)jj * d.Mz + (size_t)qg * LC) * ntile + te) * NKX) << etlog;
    };
    // lines q, q+1, .. of one member tile are contiguous in the mixed arrays only when there is a single tile
    const size_t gline = ((size_t)ntile * NKX) << etlog;      // elements between consecutive z lines of one tile
    // leader only: fetch sequence s of the item whose block starts at element `off` and holds nl lines (the item
    // offsets are computed once per item by every thread, never by the issuing lane alone: its warp is on the group's
    // critical path to the next barrier)
    auto issue = [&](size_t off, int nl, int s) {
        const uint32_t bytes = (uint32_t)(nl * NKX * ET * 16);
        uint64_t* bar = bars + (s % NST);
        mbar_arrive_expect_tx(bar, bytes);
        const double2* src = d.I8 + (size_t)seq_field(s, ROT) * fstride + off;
        if (FULL || ntile == 1) bulk_g2s(ring + (s % NST) * SLOT, src, bytes, bar);
        else
            for (int l = 0; l < nl; ++l) bulk_g2s(ring + (s % NST) * SLOT + l * NKX * ET, src + l * gline, bytes / nl, bar);
        static_assert(!SIX8 || NST == 6, "fields 6, 7 share the slots 0, 1: s % NST");
    };

    int it = blockIdx.x * NG + grp;
    // the thread that issues the bulk copies sits in a warp whose slots are idle in the first pass of the inverse
    // transforms (slots >= R1), when there is one: the refills then delay nobody on the way to the next group barrier
    constexpr int LEADER = (TPS * (SL - R1) >= 32 && GT > 32) ? GT - 32 : 0;
    int nl = 0, nnl = 0;
    size_t ioff = it < nitems ? item_off(it, nl) : 0, noff = 0;
    if (t == LEADER && it < nitems)
        for (int s = 0; s < NST; ++s) issue(ioff, nl, s);
    uint32_t itc = 0;                                        // items done by this group
    // FULL: plane-line number jq = it / ntile (+ Mz: interior planes start at j = 1) and member tile te = it % ntile, kept
    // by increments (one division per kernel, none per item)
    const int sjq = stride / ntile, ste = stride - sjq * ntile;
    int jq = it / ntile, tef = it - jq * ntile;

    for (; it < nitems; it += stride, ++itc, ioff = noff, nl = nnl) {
        const int nxt = it + stride;
        if (nxt < nitems) noff = item_off(nxt, nnl);
        int te, qg, j, q, e;
        if constexpr (FULL) {
            te = tef; e = te * TPS + lis; j = 0; q = jq + d.Mz; qg = 0;     // q holds j Mz + q, the only use of (j, q)
            tef += ste; jq += sjq;
            if (tef >= ntile) { tef -= ntile; ++jq; }
        } else {
            te = it % ntile; qg = (it / ntile) % nqg; j = it / (ntile * nqg) + 1;
            q = qg * LC + lc; e = te * ET + el;
        }
        (void)qg;
        const bool lok = e < E && lc < nl;
        double u[R1], v[R1], w[R1], Nu[R1], Nv[R1], Nw[R1];
        double suv = 0.0, swv = 0.0;
        // four exchange buffers: round r of this item uses pair (r ^ par); the forward passes use the pair the last round
        // did not, and their handoff area `exch` lives in the other one.  The convective form has three rounds, so the
        // roles swap from item to item (par): the pair that holds `exch`, read after the item's last barrier, is then not
        // written before the first barrier of the next item.
        const int par = (NBUF == 4 && !ROT) ? (int)(itc & 1) : 0;
        constexpr int FPAIR = (ROT ? 2 : 3) & 1;
        double2* exch = NBUF == 4 ? buf0 + ((1 - FPAIR) ^ par) * 2 * BUF : exch_own;
        // four-step twiddles w_M^(i sl), i < R1: powers of this slot's om = w_M^sl, rebuilt per item from one
        // register pair instead of R1 + R2 shared-memory reads per transform (the LSU pipe is this kernel's limit)
        double2 Wp[R1];
        Wp[0] = make_double2(1.0, 0.0);
#pragma unroll
        for (int i = 1; i < R1; ++i) Wp[i] = i == 1 ? om : cmul(Wp[i - 1], om);

        // wait for sequence s of this item; refill slot after use with sequence s + NST (this or the next item)
        auto wait_seq = [&](int s) {
            const uint32_t use = (HALF || (SIX8 && s % NST < 2)) ? 2 * itc + (s >= NST ? 1 : 0) : itc;
            mbar_wait(bars + (s % NST), use & 1);
        };
        auto refill = [&](int s) {
            if (t != LEADER) return;
            if ((HALF && s < NST) || (SIX8 && s < 2)) issue(ioff, nl, s + NST);
            else if (nxt < nitems) issue(noff, nnl, (HALF || (SIX8 && s >= NST)) ? s - NST : s);
        };

#define DNS_LINE_PASS_A(C, SLA, BUFC)                                                                 \
        {                                                                                             \
            constexpr int sa = LineSeq<C, ROT>::sa, two = LineSeq<C, ROT>::mode == 0, ikx = LineSeq<C, ROT>::mode == 1; \
            const double2* fa_s = ring + (sa % NST) * SLOT + lidx;                                    \
            const double2* fb_s = ring + ((sa + 1) % NST) * SLOT + lidx;                              \
            double2 a[R2];                                                                            \
            _Pragma("unroll")                                                                         \
            for (int i2 = 0; i2 < R2; ++i2) {                                                         \
                const int lo = R1 * i2, hi = R1 * i2 + R1 - 1;                                        \
                if (lo >= NKX && hi <= M - NKX) { a[i2] = make_double2(0.0, 0.0); continue; }         \
                const int pos = (SLA) + R1 * i2;                                                      \
                const int n = pos_mode<M, NKX>(pos);                                                  \
                const bool neg = pos >= NKX;                                                          \
                double2 z = make_double2(0.0, 0.0);                                                   \
                if (n >= 0) {                                                                         \
                    const double2 A = fa_s[n << etlog];                                               \
                    if (two) {                                                                        \
                        const double2 B = fb_s[n << etlog];                                           \
                        z = neg ? make_double2(A.x + B.y, B.x - A.y)                                  \
                                : (pos == 0 ? make_double2(A.x, B.x) : make_double2(A.x - B.y, A.y + B.x)); \
                    } else if (ikx) {                                                                 \
                        const double kx = kxs[n];                                                     \
                        z = neg ? make_double2((1.0 + kx) * A.x, -(1.0 + kx) * A.y)                   \
                                : (pos == 0 ? make_double2(A.x, 0.0) : make_double2((1.0 - kx) * A.x, (1.0 - kx) * A.y)); \
                    } else {                                                                          \
                        z = neg ? make_double2(A.x, -A.y) : (pos == 0 ? make_double2(A.x, 0.0) : A);  \
                    }                                                                                 \
                }                                                                                     \
                a[i2] = cswap(z);                                                                     \
            }                                                                                         \
            DFT<R2>::run(a);                                                                          \
            _Pragma("unroll")                                                                         \
            for (int k2 = 0; k2 < R2; ++k2) (BUFC)[(SLA) * PI + k2 * TPS + lis] = a[k2];              \
        }
#define DNS_LINE_PASS_B(BUFC, BODY)                                                                   \
        {                                                                                             \
            double2 x[R1];                                                                            \
            _Pragma("unroll")                                                                         \
            for (int i1 = 0; i1 < R1; ++i1)                                                           \
                x[i1] = i1 ? cmul((BUFC)[i1 * PI + sl * TPS + lis], Wp[i1]) : (BUFC)[sl * TPS + lis]; \
            DFT<R1>::run(x);                                                                          \
            _Pragma("unroll")                                                                         \
            for (int k = 0; k < R1; ++k) {                                                            \
                const double fa = x[k].y, fb = x[k].x; (void)fb;                                      \
                BODY                                                                                  \
            }                                                                                         \
        }
#define DNS_LINE_WAIT(C)                                                                              \
        { wait_seq(LineSeq<C, ROT>::sa); if (LineSeq<C, ROT>::mode == 0) wait_seq(LineSeq<C, ROT>::sa + 1); }
#define DNS_LINE_REFILL(C)                                                                            \
        { refill(LineSeq<C, ROT>::sa); if (LineSeq<C, ROT>::mode == 0) refill(LineSeq<C, ROT>::sa + 1); }
        // one transform per round: the two exchange buffers alternate, one group barrier per transform
#define DNS_LINE_INV(C, BODY)                                                                         \
        {                                                                                             \
            DNS_LINE_WAIT(C)                                                                          \
            double2* bufc = ((C) & 1) ? buf1 : buf0;                                                  \
            if (sl < R1) DNS_LINE_PASS_A(C, sl, bufc)                                                 \
            group_sync<GT>(grp);                                                                      \
            DNS_LINE_REFILL(C)                                                                        \
            if (sl < R2) DNS_LINE_PASS_B(bufc, BODY)                                                  \
        }
        // two transforms per round (PAIR); MORE: another round follows and will overwrite the buffers
#define DNS_LINE_INV2(CA, CB, PR, MORE, BODYA, BODYB)                                                 \
        {                                                                                             \
            double2* bA = buf0 + (NBUF == 4 ? ((PR) ^ par) * 2 * BUF : 0);                            \
            double2* bB = bA + BUF;                                                                   \
            DNS_LINE_WAIT(CA)                                                                         \
            DNS_LINE_WAIT(CB)                                                                         \
            if (sl < R1) DNS_LINE_PASS_A(CA, sl, bA)                                                  \
            else if (sl < 2 * R1) DNS_LINE_PASS_A(CB, sl - R1, bB)                                    \
            group_sync<GT>(grp);                                                                      \
            DNS_LINE_REFILL(CA)                                                                       \
            DNS_LINE_REFILL(CB)                                                                       \
            if (sl < R2) {                                                                            \
                DNS_LINE_PASS_B(bA, BODYA)                                                            \
                DNS_LINE_PASS_B(bB, BODYB)                                                            \
            }                                                                                         \
            if (MORE && NBUF != 4) group_sync<GT>(grp);                                               \
        }
        // a single transform inside a paired kernel
#define DNS_LINE_INV1(C, PR, MORE, BODY)                                                              \
        {                                                                                             \
            double2* bA = buf0 + (NBUF == 4 ? ((PR) ^ par) * 2 * BUF : 0);                            \
            DNS_LINE_WAIT(C)                                                                          \
            if (sl < R1) DNS_LINE_PASS_A(C, sl, bA)                                                   \
            group_sync<GT>(grp);                                                                      \
            DNS_LINE_REFILL(C)                                                                        \
            if (sl < R2) DNS_LINE_PASS_B(bA, BODY)                                                    \
            if (MORE && NBUF != 4) group_sync<GT>(grp);                                               \
        }

        // Z = A + iB:  Z(n) = A + iB, Z(0) = (Re A, Re B), Z(M - n) = conj(A) + i conj(B); with B = i kx A this is
        // Z(n) = (1 - kx) A, Z(M - n) = (1 + kx) conj(A).  Inverse transform by the swap identity: after the two
        // passes the first field is x.y and the second x.x.
#define B0 { v[k] = fa; Nv[k] = fb; }
#define B1 { u[k] = fa; Nu[k] = fa * fb; Nv[k] = fa * Nv[k] - v[k] * fb; suv += fa * v[k]; }
#define B2 { w[k] = fa; Nw[k] = u[k] * fb; swv += fa * v[k]; }
#define B3 { Nu[k] += v[k] * fa; Nu[k] += w[k] * fb; }
#define B4 { Nw[k] += v[k] * fa; Nw[k] += w[k] * fb; Nv[k] -= v[k] * fb; }
#define B5 { Nv[k] += w[k] * fa; }
        // H = omega x u: H_x = oy w - oz v, H_y = oz u - ox w, H_z = ox v - oy u; x-sums of H_x and H_z (Eq. 6-7)
#define R0 { u[k] = fa; v[k] = fb; }
#define R1B { w[k] = fa; Nv[k] = -(fb * fa); Nw[k] = fb * v[k]; }
#define R2B { Nu[k] = fa * w[k] - fb * v[k]; Nv[k] += fb * u[k]; Nw[k] -= fa * u[k]; suv += Nu[k]; swv += Nw[k]; }
        if constexpr (!ROT && !PAIR) {
            DNS_LINE_INV(0, B0) DNS_LINE_INV(1, B1) DNS_LINE_INV(2, B2) DNS_LINE_INV(3, B3) DNS_LINE_INV(4, B4) DNS_LINE_INV(5, B5)
        } else if constexpr (!ROT) {
            DNS_LINE_INV2(0, 1, 0, true, B0, B1) DNS_LINE_INV2(2, 3, 1, true, B2, B3) DNS_LINE_INV2(4, 5, 0, false, B4, B5)
        } else if constexpr (!PAIR) {
            DNS_LINE_INV(0, R0) DNS_LINE_INV(1, R1B) DNS_LINE_INV(2, R2B)
        } else {
            DNS_LINE_INV2(0, 1, 0, true, R0, R1B) DNS_LINE_INV1(2, 1, false, R2B)
        }
#undef B0
#undef B1
#undef B2
#undef B3
#undef B4
#undef B5
#undef R0
#undef R1B
#undef R2B
#undef DNS_LINE_INV2
#undef DNS_LINE_INV1
#undef DNS_LINE_PASS_A
#undef DNS_LINE_PASS_B
#undef DNS_LINE_WAIT
#undef DNS_LINE_REFILL
#undef DNS_LINE_INV

        // forward transforms of W1 = Nu + i Nv and W2 = Nw, factorisation (R2, R1): pass A on the registers
        // forward exchange buffers: with four buffers the pair the last round did not use (its barrier has ordered this
        // write after the reads of the round before); with two, wait until pass B of the last inverse has read them
        double2* bf0 = buf0 + (NBUF == 4 ? (FPAIR ^ par) * 2 * BUF : 0);
        double2* bf1 = bf0 + BUF;
        if (NBUF != 4) group_sync<GT>(grp);
        if (sl < R2) {
            double2 a1[R1], a2[R1];
#pragma unroll
            for (int k = 0; k < R1; ++k) { a1[k] = make_double2(Nu[k], Nv[k]); a2[k] = make_double2(Nw[k], 0.0); }
            DFT<R1>::run(a1);
            DFT<R1>::run(a2);
#pragma unroll
            for (int k = 0; k < R1; ++k) {
                bf0[sl * PF + k * TPS + lis] = k ? cmul(a1[k], Wp[k]) : a1[k];
                bf1[sl * PF + k * TPS + lis] = k ? cmul(a2[k], Wp[k]) : a2[k];
            }
            red[sl * TPS + lis] = make_double2(suv, swv);
        }
        group_sync<GT>(grp);
        double2 x1[R2], x2[R2];
        // PAIR: slots < R1 finish W1, slots R1 .. 2 R1 - 1 finish W2 (slf = output column n mod R1 of either)
        const bool second = PAIR && sl >= R1;
        const int slf = second ? sl - R1 : sl;
        if (sl < R1 || (second && sl < 2 * R1)) {           // forward pass B: output n = slf + R1*k
            if constexpr (PAIR) {
                const double2* src = second ? bf1 : bf0;
#pragma unroll
                for (int i = 0; i < R2; ++i) x1[i] = src[i * PF + slf * TPS + lis];
                DFT<R2>::run(x1);
            } else {
#pragma unroll
                for (int i = 0; i < R2; ++i) { x1[i] = bf0[i * PF + sl * TPS + lis]; x2[i] = bf1[i * PF + sl * TPS + lis]; }
                DFT<R2>::run(x1);
                DFT<R2>::run(x2);
            }
            if (!second) {
#pragma unroll
                for (int k = 0; k < R2; ++k) {              // hand Z1(M - n) to the slot that owns n
                    const int lo = R1 * k, hi = R1 * k + R1 - 1;
                    if (hi <= M - NKX) continue;
                    const int pos = sl + R1 * k;
                    if (lo > M - NKX || pos > M - NKX) exch[(M - pos) * TPS + lis] = x1[k];
                }
            }
        }
        group_sync<GT>(grp);
        if ((sl < R1 || (second && sl < 2 * R1)) && lok) {
            double2* dst = d.I3 + ioff + (size_t)lc * gline + el;
#pragma unroll
            for (int k = 0; k < R2; ++k) {
                const int lo = R1 * k;
                if (lo >= NKX) continue;
                const int n = slf + R1 * k;
                if (n < NKX) {
                    if (!second) {
                        const double2 zp = x1[k], zm = n == 0 ? x1[k] : exch[n * TPS + lis];
                        // (u.grad)u = (Z(n) + conj Z(-n))/2 ; (u.grad)v = (Z(n) - conj Z(-n))/(2i) ; (u.grad)w = Z2(n)
                        dst[n << etlog] = make_double2(0.5 * (zp.x + zm.x), 0.5 * (zp.y - zm.y));
                        dst[fstride + (n << etlog)] = make_double2(0.5 * (zp.y + zm.y), 0.5 * (zm.x - zp.x));
                    }
                    if constexpr (PAIR) {
                        if (second) dst[2 * fstride + (n << etlog)] = n == 0 ? make_double2(x1[k].x, 0.0) : x1[k];
                    } else {
                        dst[2 * fstride + (n << etlog)] = n == 0 ? make_double2(x2[k].x, 0.0) : x2[k];
                    }
                }
            }
        }
        if (sl == SL - 1 && lok) {                           // plane sums: by the last slot, idle in this pass when SL > R1
            double sa = 0.0, sb = 0.0;
#pragma unroll
            for (int s = 0; s < R2; ++s) { sa += red[s * TPS + lis].x; sb += red[s * TPS + lis].y; }
            d.uvpart[(FULL ? (size_t)q : (size_t)j * d.Mz + q) * E + e] = make_double2(sa, sb);
        }
    }
}

template <int R1, int R2, int SL, int TPS, int NG, int NST8, int MINB, bool ROT, bool PAIR, int NBUF, bool FULL> void line_launch_full(dns_plan* p) {
    const DnsDev& d = p->d;
    // ring depth: a whole item (8 | 6 fields), half of one, or 6 slots for 8 fields (convective form only)
    constexpr int NST = ROT ? (NST8 == 4 ? 3 : 6) : NST8;
    const LineSmem L = line_smem(R1, R2, SL, TPS, NG, NST, NBUF);
    auto kern = k_line<R1, R2, SL, TPS, NG, NST, MINB, ROT, PAIR, NBUF, FULL>;
    const int LC = TPS >> d.etl;
    const int nitems = d.Ni * ((d.Mz + LC - 1) / LC) * d.ntl;
    const int variant = (int)ROT + 2 * (int)PAIR + 4 * NST8 + 64 * NG + 256 * MINB + 4096 * NBUF + 65536 * (int)FULL;
    if (p->line_grid == 0 || p->line_grid_form != variant) {
        p->line_grid_form = variant;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L.total);
        cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        int nb = 0, nsm = 0, dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, SL * TPS * NG, L.total);
        if (nb < 1) nb = 1;
        p->line_grid = nsm * nb;
    }
    int grid = (nitems + NG - 1) / NG;
    if (grid > p->line_grid) grid = p->line_grid;
    dns_launch(kern, dim3(grid), dim3(SL * TPS * NG), (size_t)L.total, p->stream, d, nitems);
}
template <int R1, int R2, int SL, int TPS, int NG, int NST8, int MINB, bool ROT, bool PAIR, int NBUF> void line_launch_form(dns_plan* p) {
    // full member tiles (ET = TPS): always with 16 lanes (chosen for E >= 16 only), with 8 lanes when E >= 8
    if constexpr (TPS == 16) line_launch_full<R1, R2, SL, TPS, NG, NST8, MINB, ROT, PAIR, NBUF, true>(p);
    else if (TPS == 8 && (1 << p->d.etl) == TPS) line_launch_full<R1, R2, SL, TPS, NG, NST8, MINB, ROT, PAIR, NBUF, TPS == 8>(p);
    else line_launch_full<R1, R2, SL, TPS, NG, NST8, MINB, ROT, PAIR, NBUF, false>(p);
}
template <int R1, int R2, int SL, int TPS, int NG, int NST8, int MINB, bool PAIR = false, int NBUF = 2> void line_launch(dns_plan* p) {
    if (p->d.form == DNS_FORM_ROTATIONAL) line_launch_form<R1, R2, SL, TPS, NG, NST8, MINB, true, PAIR, NBUF>(p);
    else line_launch_form<R1, R2, SL, TPS, NG, NST8, MINB, false, PAIR, NBUF>(p);
}

}  // namespace

// Lanes per slot of the line kernel (= member tile of the mixed-array layout) for padded length Mx and ensemble
// size E.  Wider tiles amortise the per-item bookkeeping over more members and give the z-transform kernels longer
// contiguous runs (measured on config 2: 200 / 181 / 155 us per launch with 4 / 8 / 16 lanes).
int dns_line_tps(int Mx, int E) {
    const bool small = (Mx == 18 || Mx == 24 || Mx == 36 || Mx == 48);
    int tps = E >= 16 ? 16 : (E >= 8 ? 8 : (small ? 4 : 8));
    { const int v = dns_option("line_tps"); if (v == 8 || v == 16 || (v == 4 && small)) tps = v; }
    return tps;
}

// <R1, R2, SL> per padded length; NG groups per CTA, ring depth NST and MINB follow from the group size
template <int R1, int R2, int SL> static void line_launch_tps(dns_plan* p) {
    constexpr bool big = R1 * R2 > 72;                           // ring depth 4 keeps the long lengths inside shared memory
    switch (p->line_tps) {
        case 4:
            if constexpr (SL == 8) { line_launch<R1, R2, SL, 4, 4, 8, 3>(p); break; }
        case 8: line_launch<R1, R2, SL, 8, SL == 8 ? 2 : 1, big ? 4 : 8, SL == 8 ? 3 : (big ? 3 : 4)>(p); break;
        default:
            // small family: ring depth 4 measured best on config 2 (155 -> 141 us); 3 CTAs per SM without spills
            // ring depth: half an item for the convective form (measured best on config 2: 155 -> 141 us; a whole item
            // changes nothing), a whole item for the rotational form, where three transforms drain six fields too fast
            // for a half ring (config 4: 1381 -> 1281 us, config 2: 109 -> 96 us).  Option "line_ring": 0 half, 1 whole.
            {
                const int ring = dns_option("line_ring");
                const bool whole = !big && (ring < 0 ? p->d.form == DNS_FORM_ROTATIONAL : ring == 1);
                constexpr int MB = SL == 8 ? 3 : 2;
                // paired rounds where half of the slots would idle in the first pass (SL = 2 R1: Mx = 54, 72).  Config 4,
                // convective: 1732 us one transform per round, 1565 us paired with two exchange buffers, 1519 us with four and a
                // half ring, 1452 us with four and the 6-slot ring (default); rotational: 1063 -> 998 us (whole ring, four
                // buffers).  Option "line_pair": 0 off, 1 two buffers (convective), 5 four buffers + half ring (convective)
                if constexpr (SL == 2 * R1 && !big) {
                    const int pair = dns_option("line_pair");
                    const bool rotf = p->d.form == DNS_FORM_ROTATIONAL;
                    if (pair == 1 && !rotf) { line_launch<R1, R2, SL, 16, 1, 4, MB, true>(p); break; }
                    if (pair == 5 && !rotf) { line_launch<R1, R2, SL, 16, 1, 4, MB, true, 4>(p); break; }
                    if (pair != 0) { line_launch<R1, R2, SL, 16, 1, 6, MB, true, 4>(p); break; }
                }
                if constexpr (!big) {
                    if (whole) { line_launch<R1, R2, SL, 16, 1, 8, MB>(p); break; }
                }
                line_launch<R1, R2, SL, 16, 1, 4, MB>(p);
            }
            break;
    }
}

void launch_line(dns_plan* p) {
    switch (p->d.Mx) {
        case 18: line_launch_tps<3, 6, 8>(p); break;
        case 24: line_launch_tps<4, 6, 8>(p); break;
        case 27: line_launch_tps<3, 9, 12>(p); break;
        case 36: line_launch_tps<6, 6, 8>(p); break;
        case 48: line_launch_tps<6, 8, 8>(p); break;
        case 54: line_launch_tps<6, 9, 12>(p); break;
        case 72:
            // option "line_alt" = 1: 72 = 8 x 9 on 9 slots of one warp each (32 lanes = 2 lines x 16 members): 8 of 9 slots
            // work in the first pass and all 9 in the second, against 6 of 12 with 6 x 12 -- but only 9 warps per SM fit
            // (140 KB, 168 registers); measured on config 4: 2128 us against 2010 us, so it is not the default
            if (p->line_tps == 16 && dns_option("line_alt") == 1) line_launch<8, 9, 9, 32, 1, 4, 1>(p);
            else line_launch_tps<6, 12, 12>(p);
            break;
        case 81: line_launch_tps<9, 9, 12>(p); break;
        case 96: line_launch_tps<8, 12, 12>(p); break;
        case 108: line_launch_tps<9, 12, 12>(p); break;
        default: break;
    }
}
