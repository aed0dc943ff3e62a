// Internal declarations shared by the translation units of libdns_b200 (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstddef>
#include <mutex>
#include <vector>

#include "../../include/dns.h"
#include "../../include/dns_debug.h"

// Everything a kernel needs, passed by value.  Spectral arrays are [Ny][nkx][nkz][E] complex (member index
// fastest: the paper's vectorised-ensemble axis, is the coalescing axis); mixed (kx, z) arrays
// are [Ny][Mz][ntl][nkx][2^etl] complex (member tiles, so that one (line, tile) block of a field is contiguous:
// one TMA bulk copy in the line kernel); mean-flow arrays are [Ny][E] real.
struct DnsDev {
    int Nx, Ny, Nz, E, Mx, Mz, nkx, nkz, nzh, P, Ni, flow;
    int form;              // DNS_FORM_CONVECTIVE (u . grad u_i) or DNS_FORM_ROTATIONAL (omega x u, row f1)
    int coupling;          // DNS_COUPLING_NONE or DNS_COUPLING_STREAMWISE_MEAN (row f2)
    double invEtot;        // 1 / (members of the whole ensemble, over all ranks) for the coupled mean
    // linearised forward / adjoint ensemble (row f3): every member has ONE streamwise mode, so the
    // spectral arrays are [Ny][nkz][E] (nkx = 1, P = nkz) while the operator tables keep all nkxm = Nx/2 modes
    int nkxm;              // streamwise modes in the kx and matrix tables (= nkx for a DNS plan)
    int lin, Eg, nmodes;   // lin = 1: E = nmodes * Eg members, member e has streamwise mode nlist[e / Eg]
    const int* nlist;      // [nmodes] (device)
    double* base;          // [9][Ny][Mz] U V W Uy Vy Wy Uz Vz Wz of the frozen streamwise-mean base flow (physical z)
    double* lin_scr;       // [E] energies, [E] gains, [Ny][E] partial sums
    int etl, ntl;          // mixed arrays are tile-major: member tile of 2^etl lanes, ntl = ceil(E / 2^etl) tiles
    double dt, Re, Uw, invMxMz;
    // plan-owned constant tables
    const double* kx;      // [nkx]
    const double* kz;      // [nkz] (FFT order)
    const double* w;       // [Ny] Clenshaw-Curtis weights
    const double* Dfull;   // [Ny][Ny]
    // reflection-parity blocks in DMMA fragment order (plan.cu: fold_block), Kp = 8 ceil(ceil(Ni/2)/8):
    const double* Dfrag;   // [2 (dd->s, s->dd)][Kp*Kp] interior block of D
    const double* matsP;   // [2 (h=1/2,1)][nkx*nzh][6 (Ainv s,dd; Ainv*Delinv s,dd; Sinv s,dd)][Kp*Kp]
    int Kp;
    const double* S0inv;   // [2][Ni*Ni]
    const double* bc;      // [2][Ni]   S0m[int,0]*U_lo + S0m[int,Ny-1]*U_hi
    const double* Ugam;    // [2][Ni]   S0inv * (h dt 1)
    double wUg[2];         // (1/2) w^T Ugam
    const double2* twx;    // [Mx] exp(-2 pi i k/Mx)
    const double2* twz;    // [Mz]
    // workspace
    double2 *vt, *et;      // state at time t
    double2* vs;           // v of the current stage (transform input)
    double2* es;           // eta of the current stage (rotational form only: omega_y is a transform input)
    double2 *uh, *wh;      // u, w of the current stage
    double2 *duh, *dwh;    // convective: du/dy, dw/dy ; rotational: omega_z = i kx v - du/dy, omega_x = dw/dy - i kz v
    double2* Nh;           // 3 fields: (u.grad)u, (u.grad)v, (u.grad)w in spectral space
    double2 *F0, *G0;      // history of the nonlinear terms: N0 after stage 0, N0 + 4 N1 after stage 1
    double2* I8;           // mixed-space inputs of the line kernel: u v w Du Dw uz vz wz (convective, 8 fields)
                           // or u v w omega_x omega_y omega_z (rotational, 6 fields)
    double2* I3;           // 3 mixed-space fields: Nu Nv Nw
    double2* uvpart;       // [Ny][Mz][E] (sum_x u v, sum_x w v) per z line; rotational: (sum_x H_x, sum_x H_z)
    double2* ens;          // coupled ensemble (row f2): [3][Ny][nkz] sums over the members of the kx = 0 plane of the
                           // nonlinear vector, then [Ny][Mz] sums of uvpart -- one contiguous exchange buffer
    double2* uvc0;         // [Ny][E] history of the plane means (as F0, G0)
    double *Ut, *Wt, *Us, *Ws;      // mean profiles at t and at the current stage
    double *gamma, *Qstar; // [E]
    double* diag;          // [E][6] + scratch [Ny][E]
    double* stat;          // [DNS_NSTAT][Ny][E] running sums of the one-point statistics
    double2* stage_io;     // staging for ABI-layout copies: 2 spectral fields
    size_t S;              // Ny*P*E
    size_t Isz;            // Ny*Mz*ntl*nkx*2^etl
};

// offset of element (plane j, line q, mode n, member e) inside one mixed field
__host__ __device__ inline size_t dns_mix_off(const DnsDev& d, int j, int q, int n, int e) {
    return ((((((size_t)j * d.Mz + q) * d.ntl + (e >> d.etl)) * d.nkx + n) << d.etl)) + (e & ((1 << d.etl) - 1));
}

struct dns_plan {
    DnsDev d{};
    double Lx = 0, Lz = 0;
    int R1x = 0, R2x = 0, R1z = 0, R2z = 0;   // four-step factorisations of Mx, Mz
    int ETy = 0, NTy = 0;                      // member tile of the per-pair kernel, n-tiles per warp
    int ETf = 0;                               // member tile of the transform kernels
    int line_grid = 0, line_grid_form = 0;     // persistent grid of the line kernel (set at first launch, per form)
    int line_tps = 0;                          // lanes per slot of the line kernel (4, 8 or 16)
    alignas(64) unsigned char tmaps[3][128];   // CUtensorMap of Nh, vt, et (encoded at dns_plan_bind)
    cudaStream_t side = nullptr;               // the mean-flow kernel runs here, under the z-forward and per-pair kernels
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    std::vector<void*> owned;                  // plan-owned device allocations
    std::vector<int> nlist_host;               // linearised ensemble: streamwise mode of every kx group
    bool has_base = false;
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    cudaStream_t stream = nullptr;
    bool bound = false, has_state = false;
    // coupled ensemble across ranks: sums dev_buf[0..count) over all ranks in place, ordered on the stream (include/dns.h)
    dns_exchange_fn exchange = nullptr;
    void* exchange_ctx = nullptr;
    // one time step (15 launches, fork/join with the side stream) captured once into a CUDA graph and replayed:
    // small ensembles are launch-bound.  graph_state: 0 not tried, 1 ready, -1 unavailable (direct launches)
    cudaStream_t capture_stream = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    int graph_state = 0;
    // linearised ensemble: one graph per direction (0 forward, 1 adjoint) of the 12 launches of a step, same states
    cudaGraph_t lin_graph[2] = {nullptr, nullptr};
    cudaGraphExec_t lin_graph_exec[2] = {nullptr, nullptr};
    int lin_graph_state[2] = {0, 0};
    int sticky = DNS_OK;
    long long nsteps_done = 0;
    long long nstat = 0;                       // samples in d.stat
    cudaEvent_t ev[2 * 16] = {};
    bool ev_init = false;
};

int dns_option(const char* name);            // test / tuning options (include/dns_debug.h); -1 = default
// Programmatic dependent launch between the kernels of a stage (option "pdl" = 1; OFF by default): every stage kernel lets
// its successor start launching at once (DNS_PDL_TRIGGER at its top) and waits for its predecessor to complete and flush
// (DNS_PDL_WAIT) before it touches anything a kernel wrote; every CTA of every such kernel executes the wait, so completion
// stays transitive along the chain.  Measured slower on every configuration (config 1: 59.4 -> 66.4 us per step, config 4:
// 12.02 -> 12.62 ms): the early CTAs of the successor take shared memory and registers from the running kernel, and the
// small configurations are bound by the latency of one CTA's dependent chain, not by launch gaps.  Without the launch
// attribute both instructions are no-ops.
#if defined(__CUDACC__)
#define DNS_PDL_TRIGGER() asm volatile("griddepcontrol.launch_dependents;" ::: "memory")
#define DNS_PDL_WAIT() asm volatile("griddepcontrol.wait;" ::: "memory")
template <class... KArgs, class... Args>
inline cudaError_t dns_launch(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = dns_option("pdl") == 1 ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
#endif

// Dynamic shared memory above 48 KB has to be granted per kernel with cudaFuncSetAttribute.  The grant is a property of the
// kernel ON ONE DEVICE, so the "already granted" size is remembered per device (a plan created on a second GPU of the same
// process must set it again there), and plans driven from several host threads may reach the same kernel at once: the
// check-and-set is under a mutex and the granted size only grows, so a smaller request can never undo a larger grant that
// another thread's launch relies on.  One DnsSmemGrant per kernel instantiation (a function-local static at the launch site;
// static storage = all zero).
constexpr int DNS_MAX_DEVICES = 64;
struct DnsSmemGrant {
    std::atomic<size_t> have[DNS_MAX_DEVICES];
    std::mutex m;
};
template <class K> inline void dns_grant_smem(K kern, size_t smem, DnsSmemGrant& g, size_t granted_at_load, bool carveout) {
    int dev = -1;
    const bool known = cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < DNS_MAX_DEVICES;
    if (known) {
        const size_t have = g.have[dev].load(std::memory_order_acquire);
        if ((have ? have : granted_at_load) >= smem) return;
    }
    std::lock_guard<std::mutex> lock(g.m);
    if (known) {
        const size_t have = g.have[dev].load(std::memory_order_relaxed);
        if ((have ? have : granted_at_load) >= smem) return;
    }
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (carveout) cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (known) g.have[dev].store(smem, std::memory_order_release);
}

// host precompute (plan.cu)
int dns_host_precompute(dns_plan* p);
bool dns_factor_len(int M, int* R1, int* R2);
int dns_line_tps(int Mx, int E);

// kernel launchers (kernels_*.cu); stage = 0,1,2
void launch_zinv(dns_plan* p, const double2* vin, const double2* ein);
void launch_ens(dns_plan* p, int phase);     // phase 0: sums -> d.ens ; 1: d.ens / Etot -> members ; 2: both
size_t dns_ens_count(const DnsDev& d);       // doubles in d.ens
void launch_line(dns_plan* p);
void launch_zfwd(dns_plan* p);
void launch_ypair(dns_plan* p, int stage, int derive_only);
size_t dns_ypair_smem(int Ni, int Ny, int ET);
int dns_ypair_encode_maps(dns_plan* p);
void launch_mean(dns_plan* p, int stage, int derive_only, cudaStream_t stream);
void launch_abi_to_internal(dns_plan* p, const double2* src_abi, double2* dst, int accumulate);
void launch_internal_to_abi(dns_plan* p, const double2* src, double2* dst_abi);
void launch_mean_in(dns_plan* p, const double* U_abi, const double* W_abi);
void launch_mean_out(dns_plan* p, double* U_abi, double* W_abi);
void launch_normalise_state(dns_plan* p);
void launch_diag(dns_plan* p, double t);
void launch_stats(dns_plan* p);
// linearised ensemble (kernels_lin.cu)
void launch_diag_energy_part(dns_plan* p, double* part);      // part[Ny][E]: weighted per-plane energy sums
void launch_lin_products(dns_plan* p, int adjoint);
void launch_lin_normalise(dns_plan* p);
void launch_lin_energy(dns_plan* p, double* out_dev);
void launch_lin_gs(dns_plan* p);
void launch_lin_base(dns_plan* lin, const dns_plan* dns, int member, cudaStream_t stream);
void dns_lin_drop_graphs(dns_plan* p);                       // api_lin.cu: the graphs hold workspace pointers and tensor maps
int dns_create_common(dns_plan** out, int Nx, int Ny, int Nz, int E, double Re, double Lx, double Lz, double dt, int flow,
                      int nmodes, const int* n_list, int Eg);
