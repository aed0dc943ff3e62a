// C ABI of libdns_b200 (include/dns.h): argument checks, workspace carving, and the launch sequence of one
// CN/RK3 step: three stages, each = z-inverse FFT -> fused x-line kernel -> z-forward FFT ->
// per-pair contractions -> mean flow.  Every step of the path runs in this library's kernels.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <new>

#include "dns_internal.h"

namespace {

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
    d.vt = c.take<double2>(S);  d.et = c.take<double2>(S);  d.vs = c.take<double2>(S);
    d.uh = c.take<double2>(S);  d.wh = c.take<double2>(S);  d.duh = c.take<double2>(S);  d.dwh = c.take<double2>(S);
    d.Nh = c.take<double2>(3 * S);
    d.F0 = c.take<double2>(S);  d.G0 = c.take<double2>(S);
    d.I8 = c.take<double2>(8 * I);
    d.I3 = c.take<double2>(3 * I);
    d.uvpart = c.take<double2>((size_t)d.Ny * d.Mz * d.E);
    d.uvc0 = c.take<double2>(NE);
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

void run_stage(dns_plan* p, int s, cudaEvent_t* ev) {
    // ev (optional): 5 events bracketing the 4 kernel launches (the mean flow rides inside the per-pair launch)
    const double2* vin = s == 0 ? p->d.vt : p->d.vs;
    if (ev) cudaEventRecord(ev[0], p->stream);
    launch_zinv(p, vin);
    if (ev) cudaEventRecord(ev[1], p->stream);
    launch_line(p);
    // the mean flow (row a10) needs only the plane sums of the line kernel: fork it onto the side stream, join at the end
    cudaEventRecord(p->ev_fork, p->stream);
    cudaStreamWaitEvent(p->side, p->ev_fork, 0);
    launch_mean(p, s, 0, p->side);
    cudaEventRecord(p->ev_join, p->side);
    if (ev) cudaEventRecord(ev[2], p->stream);
    launch_zfwd(p);
    if (ev) cudaEventRecord(ev[3], p->stream);
    launch_ypair(p, s, 0);
    cudaStreamWaitEvent(p->stream, p->ev_join, 0);
    if (ev) cudaEventRecord(ev[4], p->stream);
}

// Captures one time step into a CUDA graph (on an internal stream: the plan's stream may be the legacy default stream,
// which cannot be captured).  On any failure the plan falls back to direct launches for good.
void build_step_graph(dns_plan* p) {
    p->graph_state = -1;
    if (getenv("DNS_GRAPH") && atoi(getenv("DNS_GRAPH")) == 0) return;
    if (cudaGetLastError() != cudaSuccess) return;
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
        default: return "unknown status";
    }
}

int dns_plan_create(dns_plan** out, int Nx, int Ny, int Nz, int E, double Re, double Lx, double Lz, double dt,
                    int flow) {
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
    d.nkx = Nx / 2; d.nkz = Nz - 1; d.nzh = Nz / 2; d.P = d.nkx * d.nkz; d.Ni = Ny - 2; d.flow = flow;
    d.dt = dt; d.Re = Re; d.Uw = flow == DNS_COUETTE ? 1.0 : 0.0; d.invMxMz = 1.0 / ((double)Mx * Mz);
    d.S = (size_t)Ny * d.P * E;
    {
        const int tps = dns_line_tps(Mx, E);             // lanes per slot of the line kernel = largest member tile
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
    if (const char* s = getenv("DNS_ETF")) { int v = atoi(s); if ((v == 4 || v == 8 || v == 16 || v == 32) && v <= pow2ceil(E)) p->ETf = v; }
    d.Kp = (((d.Ni + 1) / 2 + 7) / 8) * 8;
    int ETy = pow2ceil(E) < 16 ? pow2ceil(E) : 16;
    if (ETy < 4) ETy = 4;
    while (ETy > 4 && dns_ypair_smem(d.Ni, Ny, ETy) > 75 * 1024) ETy >>= 1;
    if (const char* s = getenv("DNS_ETY")) { int v = atoi(s); if (v == 4 || v == 8 || v == 16) ETy = v; }
    if (dns_ypair_smem(d.Ni, Ny, ETy) > 227 * 1024) { delete p; return DNS_EINVAL; }
    p->ETy = ETy;
    p->NTy = ETy >= 8 ? 2 : 1;
    if (const char* s = getenv("DNS_NTY")) { int v = atoi(s); if ((v == 1 || v == 2 || v == 4) && 4 * v <= ETy) p->NTy = v; }
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
    p->nstat = 0;
    return cuda_status(p, cudaMemsetAsync(ws, 0, p->workspace_bytes, p->stream));
}

int dns_set_state(dns_plan* p, const double* vhat, const double* etahat, const double* U00, const double* W00) {
    if (!p || !vhat || !etahat || !U00 || !W00) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound) return DNS_ESTATE;
    DnsDev& d = p->d;
    const size_t S = d.S, NE = (size_t)d.Ny * d.E;
    double2* sv = d.stage_io;
    double2* se = sv + S;
    double* sU = reinterpret_cast<double*>(se + S);
    double* sW = sU + NE;
    const bool dev = is_device_ptr(vhat);
    const cudaMemcpyKind kind = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    cudaError_t e = cudaMemcpyAsync(sv, vhat, S * sizeof(double2), kind, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(se, etahat, S * sizeof(double2), is_device_ptr(etahat) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(sU, U00, NE * sizeof(double), is_device_ptr(U00) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(sW, W00, NE * sizeof(double), is_device_ptr(W00) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    if (e != cudaSuccess) return cuda_status(p, e);
    launch_abi_to_internal(p, sv, d.vt);
    launch_abi_to_internal(p, se, d.et);
    launch_normalise_state(p);
    launch_mean_in(p, sU, sW);
    launch_ypair(p, 0, 1);          // derive u, w, du/dy, dw/dy of the initial state (Eq. 17-18)
    launch_mean(p, 0, 1, p->stream);   // and their (0,0) column
    p->has_state = true;
    p->nsteps_done = 0;
    e = cudaGetLastError();
    if (e == cudaSuccess && !dev) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_step(dns_plan* p, int nsteps) {
    if (!p || nsteps < 0) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    if (p->graph_state == 0 && nsteps > 0) build_step_graph(p);
    for (int it = 0; it < nsteps; ++it) {
        if (p->graph_state == 1) {
            if (cudaGraphLaunch(p->graph_exec, p->stream) != cudaSuccess) return cuda_status(p, cudaGetLastError());
        } else {
            for (int s = 0; s < 3; ++s) run_stage(p, s, nullptr);
        }
        ++p->nsteps_done;
    }
    return cuda_status(p, cudaGetLastError());
}

int dns_step_profile(dns_plan* p, int nsteps, double* ms) {
    if (!p || nsteps < 0 || !ms) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    if (!p->ev_init) {
        for (auto& e : p->ev)
            if (cudaEventCreate(&e) != cudaSuccess) return cuda_status(p, cudaGetLastError());
        p->ev_init = true;
    }
    for (int it = 0; it < nsteps; ++it) {
        for (int s = 0; s < 3; ++s) run_stage(p, s, p->ev + 5 * s);
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
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    DnsDev& d = p->d;
    launch_diag(p, (double)p->nsteps_done * d.dt);
    std::vector<double> h((size_t)d.E * 6);
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
    std::vector<double> h((size_t)DNS_NSTAT * NE), t((size_t)DNS_NSTAT * NE, 0.0);
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
    run_stage(p, stage, nullptr);
    if (stage == 2) ++p->nsteps_done;
    return cuda_status(p, cudaGetLastError());
}

int dns_launches_per_step(const dns_plan* p) { return p ? 3 * 5 : 0; }

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
