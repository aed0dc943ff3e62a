// Host-side precompute of everything that is constant for a fixed dt: Chebyshev matrices
// (Listing 1), the clamped fourth derivative, and per distinct alpha = kx^2+kz^2
// and per h in {1/2, 1} the inverses of Eq. 12-13 (Listing 3) and of Eq. 14-15.
// Arithmetic is long double (x87 64-bit mantissa) and rounded once to fp64, so that the stored maps are
// accurate to fp64 round-off although d^4/dy^4 has entries ~ Ny^8.
//
// What is stored per (alpha, h), with g = h dt/(2 Re), Delta = D2 - alpha I, T = Delta^-1 (D4c - 2 alpha D2 + alpha^2 I):
//   Ainv = (I - g T)^-1,   AD = Ainv Delta^-1,   Sinv = (I - g Delta)^-1
// and the stage update is applied as (identities (I-gT)^-1 (I+gT) = 2 Ainv - I, same for S):
//   v'   = Ainv (2 v_t) + AD (-h dt F) - v_t          (Eq. 12)
//   eta' = Sinv (2 eta_t - h dt G) - eta_t            (Eq. 13)
// i.e. three matrices per pair instead of the paper's four (ICg, ICgCg and their v counterparts).
//
// Reflection parity.  With J the reversal of the interior Gauss-Lobatto points (y -> -y), D is centro-antisymmetric
// (J D J = -D) and Ainv, AD, Sinv are centrosymmetric (J M J = M).  In the variables s = x + Jx, dd = x - Jx (first
// half of the rows; the middle row of an odd Ni carries s = 2x, dd = 0) a product y = M x becomes
//   ys = Ms s,  yd = Md dd,   Ms(i,j) = M(i,j) + M(i,Jj),  Md(i,j) = M(i,j) - M(i,Jj)      (centrosymmetric)
//   ys = Dsd dd, yd = Dds s,  Dsd(i,j) = D(i,j) - D(i,Jj), Dds(i,j) = D(i,j) + D(i,Jj)     (centro-antisymmetric)
// (the middle column is not doubled).  Only these half-size blocks are stored, in the order the DMMA.8x8x4 A
// fragments consume them, so the per-pair kernel does half the flops on half the matrix bytes.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "dns_internal.h"

typedef long double real;
typedef std::vector<real> Mat;   // row-major n x n

static const real PI_L = 3.141592653589793238462643383279502884L;

static void matmul(const Mat& A, const Mat& B, Mat& C, int n) {
    C.assign((size_t)n * n, 0.0L);
    for (int i = 0; i < n; ++i)
        for (int k = 0; k < n; ++k) {
            real a = A[(size_t)i * n + k];
            if (a == 0.0L) continue;
            const real* b = &B[(size_t)k * n];
            real* c = &C[(size_t)i * n];
            for (int j = 0; j < n; ++j) c[j] += a * b[j];
        }
}

// LU with partial pivoting, in place; returns false if singular
static bool lu_factor(Mat& A, std::vector<int>& piv, int n) {
    piv.resize(n);
    for (int k = 0; k < n; ++k) {
        int p = k;
        real best = fabsl(A[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i) {
            real v = fabsl(A[(size_t)i * n + k]);
            if (v > best) { best = v; p = i; }
        }
        if (best == 0.0L) return false;
        piv[k] = p;
        if (p != k)
            for (int j = 0; j < n; ++j) std::swap(A[(size_t)k * n + j], A[(size_t)p * n + j]);
        real inv = 1.0L / A[(size_t)k * n + k];
        for (int i = k + 1; i < n; ++i) {
            real l = A[(size_t)i * n + k] * inv;
            A[(size_t)i * n + k] = l;
            if (l == 0.0L) continue;
            const real* rk = &A[(size_t)k * n];
            real* ri = &A[(size_t)i * n];
            for (int j = k + 1; j < n; ++j) ri[j] -= l * rk[j];
        }
    }
    return true;
}

// solve LU X = B for an n x n right-hand side, in place in B (row-major)
static void lu_solve(const Mat& LU, const std::vector<int>& piv, Mat& B, int n) {
    for (int k = 0; k < n; ++k)
        if (piv[k] != k)
            for (int j = 0; j < n; ++j) std::swap(B[(size_t)k * n + j], B[(size_t)piv[k] * n + j]);
    for (int k = 0; k < n; ++k) {
        const real* bk = &B[(size_t)k * n];
        for (int i = k + 1; i < n; ++i) {
            real l = LU[(size_t)i * n + k];
            if (l == 0.0L) continue;
            real* bi = &B[(size_t)i * n];
            for (int j = 0; j < n; ++j) bi[j] -= l * bk[j];
        }
    }
    for (int k = n - 1; k >= 0; --k) {
        real inv = 1.0L / LU[(size_t)k * n + k];
        real* bk = &B[(size_t)k * n];
        for (int j = 0; j < n; ++j) bk[j] *= inv;
        for (int i = 0; i < k; ++i) {
            real u = LU[(size_t)i * n + k];
            if (u == 0.0L) continue;
            real* bi = &B[(size_t)i * n];
            for (int j = 0; j < n; ++j) bi[j] -= u * bk[j];
        }
    }
}

static bool invert(const Mat& A, Mat& Ainv, int n) {
    Mat LU = A;
    std::vector<int> piv;
    if (!lu_factor(LU, piv, n)) return false;
    Ainv.assign((size_t)n * n, 0.0L);
    for (int i = 0; i < n; ++i) Ainv[(size_t)i * n + i] = 1.0L;
    lu_solve(LU, piv, Ainv, n);
    return true;
}

// Kp x Kp parity block of the Ni x Ni matrix M in DMMA fragment order: element (i, j) of m-tile i/8 and k-step
// pair j/8 sits at (((i/8) (Kp/8) + j/8) 32 + 4 (i%8) + j%4) 2 + (j/4)%2.  sign = +1: columns j < ceil(Ni/2);
// sign = -1: columns j < floor(Ni/2).  Rows >= nrows and unused columns stay zero.
static void fold_block(const Mat& M, int Ni, int Kp, int sign, int nrows, double* out) {
    const int ncols = sign > 0 ? (Ni + 1) / 2 : Ni / 2, KS2 = Kp / 8;
    for (int i = 0; i < nrows; ++i)
        for (int j = 0; j < ncols; ++j) {
            const int Jj = Ni - 1 - j;
            real v = M[(size_t)i * Ni + j];
            if (Jj != j) v += sign * M[(size_t)i * Ni + Jj];
            const size_t idx = ((((size_t)(i >> 3) * KS2 + (j >> 3)) * 32 + 4 * (i & 7) + (j & 3)) << 1) + ((j >> 2) & 1);
            out[idx] = (double)v;
        }
}

bool dns_factor_len(int M, int* R1, int* R2) {
    // M = R1*R2, R1 (points a thread keeps in registers in the line kernel) as small as the codelet set allows
    static const int tab[][3] = {{18, 3, 6},  {24, 4, 6},  {27, 3, 9},  {36, 6, 6},  {48, 6, 8},  {54, 6, 9},
                                 {72, 6, 12}, {81, 9, 9},  {96, 6, 16}, {108, 9, 12}, {64, 8, 8},  {32, 4, 8},
                                 {16, 4, 4},  {128, 8, 16}};
    for (auto& t : tab)
        if (t[0] == M) { *R1 = t[1]; *R2 = t[2]; return true; }
    return false;
}

template <class T> static T* upload(dns_plan* p, const std::vector<T>& h, cudaError_t* err) {
    T* d = nullptr;
    if (*err != cudaSuccess) return nullptr;
    *err = cudaMalloc((void**)&d, h.size() * sizeof(T));
    if (*err != cudaSuccess) return nullptr;
    p->owned.push_back(d);
    *err = cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
    return d;
}

int dns_host_precompute(dns_plan* p) {
    DnsDev& d = p->d;
    const int Ny = d.Ny, Ni = d.Ni, N = Ny - 1;
    // ---- Chebyshev-Gauss-Lobatto grid ascending from the lower wall and D
    std::vector<real> y(Ny);
    for (int j = 0; j < Ny; ++j) y[j] = -cosl(PI_L * j / N);
    Mat D((size_t)Ny * Ny, 0.0L);
    for (int i = 0; i < Ny; ++i) {
        real ci = (i == 0 || i == N) ? 2.0L : 1.0L;
        for (int j = 0; j < Ny; ++j) {
            if (i == j) continue;
            real cj = (j == 0 || j == N) ? 2.0L : 1.0L;
            // y_i - y_j = 2 sin(pi (i+j)/(2N)) sin(pi (i-j)/(2N)): no cancellation near the walls
            real dy = 2.0L * sinl(PI_L * (i + j) / (2.0L * N)) * sinl(PI_L * (i - j) / (2.0L * N));
            D[(size_t)i * Ny + j] = (ci / cj) * (((i + j) & 1) ? -1.0L : 1.0L) / dy;
        }
    }
    for (int i = 0; i < Ny; ++i) {   // negative-sum trick for the diagonal
        real s = 0.0L;
        for (int j = 0; j < Ny; ++j)
            if (j != i) s += D[(size_t)i * Ny + j];
        D[(size_t)i * Ny + i] = -s;
    }
    Mat D2F, D3F, D4F;
    matmul(D, D, D2F, Ny);      // PAPER.md:96 D2F = DYF*DYF
    matmul(D2F, D, D3F, Ny);
    matmul(D3F, D, D4F, Ny);
    // interior blocks; clamped 4th derivative from p = (1-y^2) q: p'''' = (1-y^2) q'''' - 8 y q''' - 12 q''
    Mat D2((size_t)Ni * Ni), D4c((size_t)Ni * Ni), Dii((size_t)Ni * Ni);
    for (int i = 0; i < Ni; ++i)
        for (int j = 0; j < Ni; ++j) {
            size_t f = (size_t)(i + 1) * Ny + (j + 1);
            real yi = y[i + 1], yj = y[j + 1];
            D2[(size_t)i * Ni + j] = D2F[f];
            Dii[(size_t)i * Ni + j] = D[f];
            D4c[(size_t)i * Ni + j] = ((1.0L - yi * yi) * D4F[f] - 8.0L * yi * D3F[f] - 12.0L * D2F[f]) / (1.0L - yj * yj);
        }
    // ---- Clenshaw-Curtis weights (closed form for the Gauss-Lobatto points)
    std::vector<double> w(Ny);
    {
        std::vector<real> v(Ny, 1.0L);
        real wend;
        if (N % 2 == 0) {
            wend = 1.0L / ((real)N * N - 1.0L);
            for (int j = 1; j < N; ++j) {
                real th = PI_L * j / N;
                for (int k = 1; k < N / 2; ++k) v[j] -= 2.0L * cosl(2.0L * k * th) / (4.0L * k * k - 1.0L);
                v[j] -= cosl((real)N * th) / ((real)N * N - 1.0L);
            }
        } else {
            wend = 1.0L / ((real)N * N);
            for (int j = 1; j < N; ++j) {
                real th = PI_L * j / N;
                for (int k = 1; k <= (N - 1) / 2; ++k) v[j] -= 2.0L * cosl(2.0L * k * th) / (4.0L * k * k - 1.0L);
            }
        }
        w[0] = w[N] = (double)wend;
        for (int j = 1; j < N; ++j) w[j] = (double)(2.0L * v[j] / N);
    }
    // ---- wavenumbers and FFT twiddles
    std::vector<double> kx(d.nkxm), kz(d.nkz);
    const real LX = p->Lx, LZ = p->Lz;
    for (int n = 0; n < d.nkxm; ++n) kx[n] = (double)(2.0L * PI_L * n / LX);
    for (int i = 0; i < d.nkz; ++i) {
        int m = (i < d.nzh) ? i : i - d.nkz;     // 0..Nz/2-1, -(Nz/2-1)..-1
        kz[i] = (double)(2.0L * PI_L * m / LZ);
    }
    auto twiddles = [](int M) {
        std::vector<double2> t(M);
        for (int k = 0; k < M; ++k) {
            real a = 2.0L * PI_L * k / M;
            t[k] = make_double2((double)cosl(a), (double)(-sinl(a)));
            if (4 * k == M) t[k] = make_double2(0.0, -1.0);
            if (2 * k == M) t[k] = make_double2(-1.0, 0.0);
            if (4 * k == 3 * M) t[k] = make_double2(0.0, 1.0);
        }
        return t;
    };
    // ---- per-(alpha, h) inverses (Listing 1 + Listing 3, Eq. 12-13)
    const int nA = d.nkxm * d.nzh;
    const size_t NN = (size_t)Ni * Ni;
    const int Kp = d.Kp, Kh = (Ni + 1) / 2, Kho = Ni / 2;
    const size_t BB = (size_t)Kp * Kp;
    std::vector<double> mats((size_t)2 * nA * 6 * BB, 0.0);
    int fail = 0, nomem = 0;
    const real dt = d.dt, Re = d.Re;
    // an exception may not leave an OpenMP region (it would terminate the process, and nothing may abort across the ABI):
    // allocation failures inside the loop body are caught per iteration and reported after the loop
#pragma omp parallel for schedule(dynamic, 1) reduction(| : fail, nomem)
    for (int a = 1; a < nA; ++a) {
        try {
        int n = a / d.nzh, m = a % d.nzh;
        // the stored kx, kz are fp64; alpha is formed from them exactly as the kernels do
        real alpha = (real)kx[n] * (real)kx[n] + (real)kz[m] * (real)kz[m];
        Mat Del(NN), DelDel(NN), LU, T, Delinv;
        for (size_t i = 0; i < NN; ++i) {
            Del[i] = D2[i];
            DelDel[i] = D4c[i] - 2.0L * alpha * D2[i];
        }
        for (int i = 0; i < Ni; ++i) {
            Del[(size_t)i * Ni + i] -= alpha;
            DelDel[(size_t)i * Ni + i] += alpha * alpha;
        }
        LU = Del;
        std::vector<int> piv;
        if (!lu_factor(LU, piv, Ni)) { fail |= 1; continue; }
        T = DelDel;
        lu_solve(LU, piv, T, Ni);                       // T = Delta^-1 Delta Delta (Eq. 12)
        Delinv.assign(NN, 0.0L);
        for (int i = 0; i < Ni; ++i) Delinv[(size_t)i * Ni + i] = 1.0L;
        lu_solve(LU, piv, Delinv, Ni);                  // IDELv (Listing 1)
        for (int hi = 0; hi < 2; ++hi) {
            real h = hi == 0 ? 0.5L : 1.0L;
            real g = h * dt / (2.0L * Re);
            Mat A(NN), Sm(NN), Ainv, AD, Sinv;
            for (size_t i = 0; i < NN; ++i) { A[i] = -g * T[i]; Sm[i] = -g * Del[i]; }
            for (int i = 0; i < Ni; ++i) { A[(size_t)i * Ni + i] += 1.0L; Sm[(size_t)i * Ni + i] += 1.0L; }
            if (!invert(A, Ainv, Ni) || !invert(Sm, Sinv, Ni)) { fail |= 1; continue; }
            matmul(Ainv, Delinv, AD, Ni);
            double* out = &mats[(((size_t)hi * nA + a) * 6) * BB];
            fold_block(Ainv, Ni, Kp, +1, Kh, out);
            fold_block(Ainv, Ni, Kp, -1, Kho, out + BB);
            fold_block(AD, Ni, Kp, +1, Kh, out + 2 * BB);
            fold_block(AD, Ni, Kp, -1, Kho, out + 3 * BB);
            fold_block(Sinv, Ni, Kp, +1, Kh, out + 4 * BB);
            fold_block(Sinv, Ni, Kp, -1, Kho, out + 5 * BB);
        }
        } catch (const std::bad_alloc&) {
            nomem |= 1;
        }
    }
    if (nomem) return DNS_ENOMEM;
    if (fail) return DNS_EINVAL;
    // ---- mean-flow operators (Eq. 14-15; boundary columns moved to the rhs)
    std::vector<double> S0inv(2 * NN), bc(2 * Ni), Ugam(2 * Ni);
    for (int hi = 0; hi < 2; ++hi) {
        real h = hi == 0 ? 0.5L : 1.0L;
        real g = h * dt / (2.0L * Re);
        Mat S0m(NN), inv;
        for (int i = 0; i < Ni; ++i)
            for (int j = 0; j < Ni; ++j)
                S0m[(size_t)i * Ni + j] = (i == j ? 1.0L : 0.0L) - g * D2F[(size_t)(i + 1) * Ny + (j + 1)];
        if (!invert(S0m, inv, Ni)) return DNS_EINVAL;
        real wug = 0.0L;
        for (int i = 0; i < Ni; ++i) {
            real s = 0.0L;
            for (int j = 0; j < Ni; ++j) {
                S0inv[(size_t)hi * NN + (size_t)i * Ni + j] = (double)inv[(size_t)i * Ni + j];
                s += inv[(size_t)i * Ni + j];
            }
            Ugam[(size_t)hi * Ni + i] = (double)(s * h * dt);
            wug += (real)w[i + 1] * (real)Ugam[(size_t)hi * Ni + i];
            real lo = -g * D2F[(size_t)(i + 1) * Ny + 0], hi_ = -g * D2F[(size_t)(i + 1) * Ny + N];
            bc[(size_t)hi * Ni + i] = (double)(lo * (-(real)d.Uw) + hi_ * (real)d.Uw);
        }
        d.wUg[hi] = (double)(0.5L * wug);
    }
    // ---- upload
    std::vector<double> Dfull_d((size_t)Ny * Ny), Dfrag_d(2 * BB, 0.0);
    for (size_t i = 0; i < Dfull_d.size(); ++i) Dfull_d[i] = (double)D[i];
    fold_block(Dii, Ni, Kp, -1, Kh, Dfrag_d.data());          // dd -> s
    fold_block(Dii, Ni, Kp, +1, Kho, Dfrag_d.data() + BB);    // s -> dd
    cudaError_t err = cudaSuccess;
    d.kx = upload(p, kx, &err);
    d.kz = upload(p, kz, &err);
    d.w = upload(p, w, &err);
    d.Dfull = upload(p, Dfull_d, &err);
    d.Dfrag = upload(p, Dfrag_d, &err);
    d.matsP = upload(p, mats, &err);
    d.S0inv = upload(p, S0inv, &err);
    d.bc = upload(p, bc, &err);
    d.Ugam = upload(p, Ugam, &err);
    d.twx = upload(p, twiddles(d.Mx), &err);
    d.twz = upload(p, twiddles(d.Mz), &err);
    if (d.lin) d.nlist = upload(p, p->nlist_host, &err);
    if (err == cudaErrorMemoryAllocation) return DNS_ENOMEM;
    return err == cudaSuccess ? DNS_OK : DNS_ECUDA;
}
