// C ABI of libdns_b200 (include/dns.h): argument checks, workspace carving, and the launch sequence of one
// CN/RK3 step: three stages, each = z-inverse FFT -> fused x-line kernel -> z-forward FFT ->
// per-pair contractions -> mean flow.  Every step of the path runs in this library's kernels.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "dns_internal.h"

namespace {

// test / tuning options of include/dns_debug.h (process-wide; -1 = default)
struct Option { const char* name; int value; };
Option g_options[] = {{"graph", -1}, {"zreg", -1}, {"etf", -1}, {"ety", -1}, {"nty", -1}, {"line_tps", -1}, {"line_alt", -1}, {"line_ring", -1}, {"line_pair", -1}, {"pdl", -1}, {"zinv_tp", -1}};

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

int pow2ceil(int x) { int p = 1; while (p < x) p <<= 1; return p; }

bool is_23_smooth(int M) {
    if (M < 1) return false;
    while (M % 2 == 0) M /= 2;
    while (M % 3 == 0) M /= 3;
    return M == 1;
}

struct Carve {
    char* base;
    size_t off = 0;
    template <class T> T* take(size_t n) {
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += align256(n * sizeof(T));
        return p;
    }
};

// lays the workspace out; with base == nullptr only measures
size_t carve_workspace(dns_plan* p, void* base) {
    DnsDev& d = p->d;
    Carve c{static_cast<char*>(base)};
    const size_t S = d.S, I = d.Isz, NE = (size_t)d.Ny * d.E;
    d.vt = c.take<double2>(S);  d.et = c.take<double2>(S);  d.vs = c.take<double2>(S);  d.es = c.take<double2>(S);
    d.uh = c.take<double2>(S);  d.wh = c.take<double2>(S);  d.duh = c.take<double2>(S);  d.dwh = c.take<double2>(S);
    d.Nh = c.take<double2>(3 * S);
    d.F0 = c.take<double2>(S);  d.G0 = c.take<double2>(S);
    d.I8 = c.take<double2>(8 * I);
    d.I3 = c.take<double2>(3 * I);
    d.uvpart = c.take<double2>((size_t)d.Ny * d.Mz * d.E);
    d.uvc0 = c.take<double2>(NE);
    d.ens = c.take<double2>(dns_ens_count(d) / 2);
    d.base = c.take<double>(d.lin ? (size_t)9 * d.Ny * d.Mz : 1);
    d.lin_scr = c.take<double>(d.lin ? (size_t)2 * d.E + (size_t)d.Ny * d.E : 1);
    d.Ut = c.take<double>(NE);  d.Wt = c.take<double>(NE);  d.Us = c.take<double>(NE);  d.Ws = c.take<double>(NE);
    d.gamma = c.take<double>(d.E);  d.Qstar = c.take<double>(d.E);
    d.diag = c.take<double>((size_t)d.E * 6 + NE);
    d.stat = c.take<double>((size_t)DNS_NSTAT * NE);
    d.stage_io = c.take<double2>(2 * S + 2 * NE);
    return c.off;
}

int cuda_status(dns_plan* p, cudaError_t e) {
    if (e == cudaSuccess) return DNS_OK;
    p->sticky = (e == cudaErrorMemoryAllocation) ? DNS_ENOMEM : DNS_ECUDA;
    return p->sticky;
}

bool is_device_ptr(const void* q) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, q) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

int run_stage(dns_plan* p, int s, cudaEvent_t* ev) {
    // ev (optional): 5 events bracketing the 4 kernel classes (the mean flow rides beside the per-pair launch)
    const double2* vin = s == 0 ? p->d.vt : p->d.vs;
    const double2* ein = s == 0 ? p->d.et : p->d.es;
    const bool coupled = p->d.coupling == DNS_COUPLING_STREAMWISE_MEAN;
    if (ev) cudaEventRecord(ev[0], p->stream);
    launch_zinv(p, vin, ein);
    if (ev) cudaEventRecord(ev[1], p->stream);
    launch_line(p);
    if (ev) cudaEventRecord(ev[2], p->stream);
    // the mean flow (row a10) needs only the plane sums of the line kernel: fork it onto the side stream, join at the end.
    // Coupled ensemble (row f2): it must wait for the ensemble means, which follow the z-forward transform.
    if (!coupled) {
        cudaEventRecord(p->ev_fork, p->stream);
        cudaStreamWaitEvent(p->side, p->ev_fork, 0);
        launch_mean(p, s, 0, p->side);
        cudaEventRecord(p->ev_join, p->side);
    }
    launch_zfwd(p);
    if (ev) cudaEventRecord(ev[3], p->stream);
    if (coupled) {
        if (p->exchange) {
            launch_ens(p, 0);
            if (p->exchange(p->exchange_ctx, reinterpret_cast<double*>(p->d.ens), dns_ens_count(p->d), p->stream) != 0) return DNS_ECUDA;
            launch_ens(p, 1);
        } else {
            launch_ens(p, 2);
        }
        cudaEventRecord(p->ev_fork, p->stream);
        cudaStreamWaitEvent(p->side, p->ev_fork, 0);
        launch_mean(p, s, 0, p->side);
        cudaEventRecord(p->ev_join, p->side);
    }
    launch_ypair(p, s, 0);
    cudaStreamWaitEvent(p->stream, p->ev_join, 0);
    if (ev) cudaEventRecord(ev[4], p->stream);
    return DNS_OK;
}

// Captures one time step into a CUDA graph (on an internal stream: the plan's stream may be the legacy default stream,
// which cannot be captured).  On any failure the plan falls back to direct launches for good.
void build_step_graph(dns_plan* p) {
    p->graph_state = -1;
    if (dns_option("graph") == 0 || p->exchange) return;
    if (cudaPeekAtLastError() != cudaSuccess) return;     // a pending error is reported by the caller, not cleared here
    if (!p->capture_stream && cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return; }
    cudaStream_t user = p->stream;
    if (cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return; }
    p->stream = p->capture_stream;
    for (int s = 0; s < 3; ++s) run_stage(p, s, nullptr);
    p->stream = user;
    cudaGraph_t g = nullptr;
    const cudaError_t e1 = cudaStreamEndCapture(p->capture_stream, &g);
    if (e1 != cudaSuccess || !g) { cudaGetLastError(); return; }
    cudaGraphExec_t ge = nullptr;
    if (cudaGraphInstantiate(&ge, g, 0) != cudaSuccess || !ge) { cudaGetLastError(); cudaGraphDestroy(g); return; }
    p->graph = g;
    p->graph_exec = ge;
    p->graph_state = 1;
}

void drop_step_graph(dns_plan* p) {
    dns_lin_drop_graphs(p);
    if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
    if (p->graph) cudaGraphDestroy(p->graph);
    p->graph_exec = nullptr;
    p->graph = nullptr;
    p->graph_state = 0;
}

}  // namespace

extern "C" {

const char* dns_strerror(int s) {
    switch (s) {
        case DNS_OK: return "ok";
        case DNS_EINVAL: return "invalid argument";
        case DNS_ENOMEM: return "out of memory";
        case DNS_ECUDA: return "CUDA error or no CUDA device";
        case DNS_ENONFINITE: return "non-finite energy";
        case DNS_ESTATE: return "call out of order (workspace not bound or state not set)";
        case DNS_ELIMIT: return "problem exceeds the fixed capacity of the allocation-free entry point (Ny * E > 65536)";
        default: return "unknown status";
    }
}

}  // extern "C"

// dns_plan_create and dns_lin_plan_create: nmodes = 0 for a DNS plan; otherwise E = nmodes * Eg single-kx members
int dns_create_common(dns_plan** out, int Nx, int Ny, int Nz, int E, double Re, double Lx, double Lz, double dt, int flow,
                      int nmodes, const int* n_list, int Eg) {
    if (!out) return DNS_EINVAL;
    *out = nullptr;
    if (Nx < 2 || Nz < 4 || (Nx & 1) || (Nz & 1)) return DNS_EINVAL;
    const int Mx = 3 * Nx / 2, Mz = 3 * Nz / 2;
    int r1, r2;
    if (Mx < 16 || Mx > 128 || Mz < 16 || Mz > 128 || !is_23_smooth(Mx) || !is_23_smooth(Mz)) return DNS_EINVAL;
    if (!dns_factor_len(Mx, &r1, &r2) || !dns_factor_len(Mz, &r1, &r2)) return DNS_EINVAL;
    if (Ny < 5 || Ny > 257 || E < 1) return DNS_EINVAL;
    if (!(Re > 0.0) || !(Lx > 0.0) || !(Lz > 0.0) || !(dt > 0.0)) return DNS_EINVAL;
    if (!std::isfinite(Re) || !std::isfinite(Lx) || !std::isfinite(Lz) || !std::isfinite(dt)) return DNS_EINVAL;
    if (flow != DNS_COUETTE && flow != DNS_POISEUILLE_CMF) return DNS_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return DNS_ECUDA; }
    dns_plan* p = new (std::nothrow) dns_plan();
    if (!p) return DNS_ENOMEM;
    DnsDev& d = p->d;
    d.Nx = Nx; d.Ny = Ny; d.Nz = Nz; d.E = E; d.Mx = Mx; d.Mz = Mz;
    d.nkxm = Nx / 2; d.lin = nmodes > 0; d.nmodes = nmodes; d.Eg = Eg;
    d.nkx = d.lin ? 1 : Nx / 2; d.nkz = Nz - 1; d.nzh = Nz / 2; d.P = d.nkx * d.nkz; d.Ni = Ny - 2; d.flow = flow;
    if (d.lin) {
        for (int g = 0; g < nmodes; ++g)
            if (n_list[g] < 1 || n_list[g] >= d.nkxm) { delete p; return DNS_EINVAL; }
        p->nlist_host.assign(n_list, n_list + nmodes);
    }
    d.dt = dt; d.Re = Re; d.Uw = flow == DNS_COUETTE ? 1.0 : 0.0;
    d.invMxMz = d.lin ? 1.0 / Mz : 1.0 / ((double)Mx * Mz);       // single-kx members: x is analytic, only z is transformed
    d.form = DNS_FORM_CONVECTIVE; d.coupling = DNS_COUPLING_NONE; d.invEtot = 1.0 / E;
    d.S = (size_t)Ny * d.P * E;
    {
        const int tps = dns_line_tps(d.lin ? Mz : Mx, E);   // lanes per slot of the line kernel = largest member tile
        p->line_tps = tps;
        int et = 1, lg = 0;
        while (et < tps && et < E) { et <<= 1; ++lg; }
        d.etl = lg;
        d.ntl = (E + et - 1) / et;
        d.Isz = ((size_t)Ny * Mz * d.ntl * d.nkx) << lg;
    }
    p->Lx = Lx; p->Lz = Lz;
    // member tiles
    p->ETf = pow2ceil(E) < 32 ? pow2ceil(E) : 32;
    { const int v = dns_option("etf"); if ((v == 4 || v == 8 || v == 16 || v == 32) && v <= pow2ceil(E)) p->ETf = v; }
    d.Kp = (((d.Ni + 1) / 2 + 7) / 8) * 8;
    const int Etile = d.lin ? Eg : E;                    // a member tile of the per-pair kernel lies inside one kx group
    int ETy = pow2ceil(Etile) < 16 ? pow2ceil(Etile) : 16;
    if (ETy < 4) ETy = 4;
    while (ETy > 4 && dns_ypair_smem(d.Ni, Ny, ETy) > 75 * 1024) ETy >>= 1;
    { const int v = dns_option("ety"); if (v == 4 || v == 8 || v == 16) ETy = v; }
    if (dns_ypair_smem(d.Ni, Ny, ETy) > 227 * 1024) { delete p; return DNS_EINVAL; }
    p->ETy = ETy;
    p->NTy = ETy >= 8 ? 2 : 1;
    { const int v = dns_option("nty"); if ((v == 1 || v == 2 || v == 4) && 4 * v <= ETy) p->NTy = v; }
    while (32 * (d.Kp / 8) * (ETy / (4 * p->NTy)) > 1024) p->NTy *= 2;
    if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        dns_plan_destroy(p);
        return DNS_ECUDA;
    }
    int st = DNS_OK;
    try {
        st = dns_host_precompute(p);
    } catch (const std::bad_alloc&) {
        st = DNS_ENOMEM;
    }
    if (st != DNS_OK) { dns_plan_destroy(p); return st; }
    p->workspace_bytes = carve_workspace(p, nullptr);
    *out = p;
    return DNS_OK;
}

extern "C" {

int dns_plan_create(dns_plan** out, int Nx, int Ny, int Nz, int E, double Re, double Lx, double Lz, double dt,
                    int flow) {
    return dns_create_common(out, Nx, Ny, Nz, E, Re, Lx, Lz, dt, flow, 0, nullptr, 0);
}

size_t dns_plan_workspace_bytes(const dns_plan* p) { return p ? p->workspace_bytes : 0; }

int dns_plan_bind(dns_plan* p, void* ws, size_t bytes, void* stream) {
    if (!p || !ws) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (bytes < p->workspace_bytes || (reinterpret_cast<size_t>(ws) & 255)) return DNS_EINVAL;
    if (!is_device_ptr(ws)) return DNS_EINVAL;
    p->workspace = ws;
    p->stream = static_cast<cudaStream_t>(stream);
    carve_workspace(p, ws);
    drop_step_graph(p);                                  // the graph holds the old workspace pointers and tensor maps
    const int st = dns_ypair_encode_maps(p);
    if (st != DNS_OK) { p->sticky = st; return st; }
    p->bound = true;
    p->has_state = false;
    p->has_base = false;
    p->nstat = 0;
    return cuda_status(p, cudaMemsetAsync(ws, 0, p->workspace_bytes, p->stream));
}

// copies up to four ABI arrays into the staging area; *all_dev = every given pointer is a device pointer
static cudaError_t stage_in(dns_plan* p, const double* vhat, const double* etahat, const double* U00, const double* W00,
                            bool* all_dev) {
    DnsDev& d = p->d;
    const size_t S = d.S, NE = (size_t)d.Ny * d.E;
    double2* sv = d.stage_io;
    double2* se = sv + S;
    double* sU = reinterpret_cast<double*>(se + S);
    double* sW = sU + NE;
    cudaError_t e = cudaSuccess;
    *all_dev = true;
    auto in = [&](void* dst, const void* src, size_t bytes) {
        if (!src || e != cudaSuccess) return;
        const bool dev = is_device_ptr(src);
        if (!dev) *all_dev = false;
        e = cudaMemcpyAsync(dst, src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    };
    in(sv, vhat, S * sizeof(double2));
    in(se, etahat, S * sizeof(double2));
    in(sU, U00, NE * sizeof(double));
    in(sW, W00, NE * sizeof(double));
    return e;
}

int dns_set_state(dns_plan* p, const double* vhat, const double* etahat, const double* U00, const double* W00) {
    if (!p || !vhat || !etahat || !U00 || !W00) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound) return DNS_ESTATE;
    DnsDev& d = p->d;
    const size_t S = d.S, NE = (size_t)d.Ny * d.E;
    double2* sv = d.stage_io;
    double2* se = sv + S;
    double* sU = reinterpret_cast<double*>(se + S);
    double* sW = sU + NE;
    bool all_dev = true;
    cudaError_t e = stage_in(p, vhat, etahat, U00, W00, &all_dev);
    if (e != cudaSuccess) return cuda_status(p, e);
    launch_abi_to_internal(p, sv, d.vt, 0);
    launch_abi_to_internal(p, se, d.et, 0);
    launch_normalise_state(p);
    launch_mean_in(p, sU, sW);
    launch_ypair(p, 0, 1);          // derive u, w, du/dy, dw/dy (or omega_x, omega_z) of the initial state (Eq. 17-18)
    launch_mean(p, 0, 1, p->stream);   // and their (0,0) column
    p->has_state = true;
    p->nsteps_done = 0;
    e = cudaGetLastError();
    // any host source: its copy may still be in flight (pinned memory), so the call only returns once it has landed
    if (e == cudaSuccess && !all_dev) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_add_increment(dns_plan* p, const double* dv, const double* deta) {
    if (!p || !dv || !deta) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    DnsDev& d = p->d;
    double2* sv = d.stage_io;
    double2* se = sv + d.S;
    bool all_dev = true;
    cudaError_t e = stage_in(p, dv, deta, nullptr, nullptr, &all_dev);
    if (e != cudaSuccess) return cuda_status(p, e);
    launch_abi_to_internal(p, sv, d.vt, 1);            // accumulate
    launch_abi_to_internal(p, se, d.et, 1);
    launch_normalise_state(p);
    launch_ypair(p, 0, 1);
    launch_mean(p, 0, 1, p->stream);
    e = cudaGetLastError();
    if (e == cudaSuccess && !all_dev) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_plan_set_form(dns_plan* p, int form) {
    if (!p || p->d.lin || (form != DNS_FORM_CONVECTIVE && form != DNS_FORM_ROTATIONAL)) return DNS_EINVAL;
    if (p->has_state) return DNS_ESTATE;
    if (form != p->d.form) drop_step_graph(p);
    p->d.form = form;
    return DNS_OK;
}

int dns_plan_set_coupling(dns_plan* p, int mode, long long E_total) {
    if (!p || p->d.lin || (mode != DNS_COUPLING_NONE && mode != DNS_COUPLING_STREAMWISE_MEAN)) return DNS_EINVAL;
    if (mode == DNS_COUPLING_STREAMWISE_MEAN && E_total < p->d.E) return DNS_EINVAL;
    if (p->has_state) return DNS_ESTATE;
    drop_step_graph(p);
    p->d.coupling = mode;
    p->d.invEtot = 1.0 / (double)(mode == DNS_COUPLING_NONE ? p->d.E : E_total);
    return DNS_OK;
}

int dns_plan_set_exchange(dns_plan* p, dns_exchange_fn fn, void* ctx) {
    if (!p) return DNS_EINVAL;
    drop_step_graph(p);
    p->exchange = fn;
    p->exchange_ctx = ctx;
    return DNS_OK;
}

int dns_step(dns_plan* p, int nsteps) {
    if (!p || nsteps < 0) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    if (p->graph_state == 0 && nsteps > 0) build_step_graph(p);
    for (int it = 0; it < nsteps; ++it) {
        if (p->graph_state == 1) {
            if (cudaGraphLaunch(p->graph_exec, p->stream) != cudaSuccess) return cuda_status(p, cudaGetLastError());
        } else {
            for (int s = 0; s < 3; ++s)
                if (run_stage(p, s, nullptr) != DNS_OK) { p->sticky = DNS_ECUDA; return DNS_ECUDA; }
        }
        ++p->nsteps_done;
    }
    return cuda_status(p, cudaGetLastError());
}

int dns_step_profile(dns_plan* p, int nsteps, double* ms) {
    if (!p || nsteps < 0 || !ms) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    if (!p->ev_init) {
        for (auto& e : p->ev)
            if (cudaEventCreate(&e) != cudaSuccess) return cuda_status(p, cudaGetLastError());
        p->ev_init = true;
    }
    for (int it = 0; it < nsteps; ++it) {
        for (int s = 0; s < 3; ++s)
            if (run_stage(p, s, p->ev + 5 * s) != DNS_OK) { p->sticky = DNS_ECUDA; return DNS_ECUDA; }
        cudaError_t e = cudaStreamSynchronize(p->stream);
        if (e != cudaSuccess) return cuda_status(p, e);
        for (int s = 0; s < 3; ++s)
            for (int c = 0; c < DNS_NCLASS; ++c) {
                float t = 0.f;
                cudaEventElapsedTime(&t, p->ev[5 * s + c], p->ev[5 * s + c + 1]);
                ms[c] += t;
            }
        ++p->nsteps_done;
    }
    return cuda_status(p, cudaGetLastError());
}

int dns_get_state(dns_plan* p, double* vhat, double* etahat, double* U00, double* W00) {
    if (!p) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    DnsDev& d = p->d;
    const size_t S = d.S, NE = (size_t)d.Ny * d.E;
    double2* sv = d.stage_io;
    double2* se = sv + S;
    double* sU = reinterpret_cast<double*>(se + S);
    double* sW = sU + NE;
    cudaError_t e = cudaSuccess;
    auto out = [&](void* dst, const void* src, size_t bytes) {
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(dst, src, bytes, is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, p->stream);
    };
    if (vhat) { launch_internal_to_abi(p, d.vt, sv); out(vhat, sv, S * sizeof(double2)); }
    if (etahat) { launch_internal_to_abi(p, d.et, se); out(etahat, se, S * sizeof(double2)); }
    if (U00 || W00) {
        launch_mean_out(p, U00 ? sU : nullptr, W00 ? sW : nullptr);
        if (U00) out(U00, sU, NE * sizeof(double));
        if (W00) out(W00, sW, NE * sizeof(double));
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_diagnostics(dns_plan* p, double* out) {
    if (!p || !out) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    DnsDev& d = p->d;
    std::vector<double> h;
    try { h.resize((size_t)d.E * 6); } catch (...) { return DNS_ENOMEM; }      // nothing may throw across the ABI
    launch_diag(p, (double)p->nsteps_done * d.dt);
    cudaError_t e = cudaMemcpyAsync(h.data(), d.diag, h.size() * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e == cudaSuccess)
        e = cudaMemcpy(out, h.data(), h.size() * sizeof(double), is_device_ptr(out) ? cudaMemcpyHostToDevice : cudaMemcpyHostToHost);
    if (e != cudaSuccess) return cuda_status(p, e);
    for (int i = 0; i < d.E; ++i)
        if (!std::isfinite(h[(size_t)i * 6])) return DNS_ENONFINITE;
    return DNS_OK;
}

int dns_stats_reset(dns_plan* p) {
    if (!p) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound) return DNS_ESTATE;
    p->nstat = 0;
    return cuda_status(p, cudaMemsetAsync(p->d.stat, 0, (size_t)DNS_NSTAT * p->d.Ny * p->d.E * sizeof(double), p->stream));
}

int dns_stats_accumulate(dns_plan* p) {
    if (!p) return DNS_EINVAL;
    if (p->d.lin) return DNS_EINVAL;                      // a linearised-ensemble plan: use dns_lin_*
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    launch_stats(p);
    ++p->nstat;
    return cuda_status(p, cudaGetLastError());
}

int dns_stats_get(dns_plan* p, double* out, long long* nsamples) {
    if (!p || !out) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound) return DNS_ESTATE;
    const DnsDev& d = p->d;
    const size_t NE = (size_t)d.Ny * d.E;
    std::vector<double> h, t;
    try { h.resize((size_t)DNS_NSTAT * NE); t.assign((size_t)DNS_NSTAT * NE, 0.0); } catch (...) { return DNS_ENOMEM; }
    cudaError_t e = cudaMemcpyAsync(h.data(), d.stat, h.size() * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return cuda_status(p, e);
    if (p->nstat > 0) {
        const double inv = 1.0 / (double)p->nstat;
        for (int k = 0; k < DNS_NSTAT; ++k)
            for (int j = 0; j < d.Ny; ++j)
                for (int m = 0; m < d.E; ++m) t[((size_t)m * d.Ny + j) * DNS_NSTAT + k] = h[(size_t)k * NE + (size_t)j * d.E + m] * inv;
    }
    e = cudaMemcpy(out, t.data(), t.size() * sizeof(double), is_device_ptr(out) ? cudaMemcpyHostToDevice : cudaMemcpyHostToHost);
    if (nsamples) *nsamples = p->nstat;
    return cuda_status(p, e);
}

int dns_debug_fetch(dns_plan* p, int which, void* dst, size_t nbytes) {
    if (!p || !dst) return DNS_EINVAL;
    if (!p->bound) return DNS_ESTATE;
    const DnsDev& d = p->d;
    const size_t S = d.S * sizeof(double2), NE = (size_t)d.Ny * d.E * sizeof(double);
    const void* src = nullptr;
    size_t sz = S;
    switch (which) {
        case 0: src = d.uh; break;
        case 1: src = d.wh; break;
        case 2: src = d.duh; break;
        case 3: src = d.dwh; break;
        case 4: src = d.Nh; sz = 3 * S; break;
        case 5: src = d.F0; break;
        case 6: src = d.G0; break;
        case 7: src = d.vs; break;
        case 8: src = d.Us; sz = NE; break;
        case 9: src = d.Ws; sz = NE; break;
        case 10: src = d.es; break;
        default: return DNS_EINVAL;
    }
    if (nbytes != sz) return DNS_EINVAL;
    cudaError_t e = cudaStreamSynchronize(p->stream);
    if (e == cudaSuccess) e = cudaMemcpy(dst, src, sz, cudaMemcpyDeviceToHost);
    return cuda_status(p, e);
}

int dns_debug_stage(dns_plan* p, int stage) {
    if (!p || stage < 0 || stage > 2) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    if (run_stage(p, stage, nullptr) != DNS_OK) { p->sticky = DNS_ECUDA; return DNS_ECUDA; }
    if (stage == 2) ++p->nsteps_done;
    return cuda_status(p, cudaGetLastError());
}

int dns_launches_per_step(const dns_plan* p) {
    if (!p) return 0;
    const int ens = p->d.coupling == DNS_COUPLING_STREAMWISE_MEAN ? (p->exchange ? 2 : 1) : 0;
    return 3 * (5 + ens);
}

int dns_debug_set_option(const char* name, int value) {
    if (!name) return DNS_EINVAL;
    for (auto& o : g_options)
        if (strcmp(o.name, name) == 0) { o.value = value < 0 ? -1 : value; return DNS_OK; }
    return DNS_EINVAL;
}

int dns_plan_destroy(dns_plan* p) {
    if (!p) return DNS_OK;
    for (void* q : p->owned) cudaFree(q);
    drop_step_graph(p);
    if (p->capture_stream) cudaStreamDestroy(p->capture_stream);
    if (p->side) cudaStreamDestroy(p->side);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->ev_init)
        for (auto& e : p->ev) cudaEventDestroy(e);
    delete p;
    return DNS_OK;
}

}  // extern "C"

int dns_option(const char* name) {
    for (auto& o : g_options)
        if (strcmp(o.name, name) == 0) return o.value;
    return -1;
}
