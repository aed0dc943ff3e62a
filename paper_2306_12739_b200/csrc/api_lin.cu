// C ABI of the linearised forward / adjoint ensemble (include/dns.h, dns_lin_*; PAPER.md:296-317,
// Appendix B).  A linear plan is a dns_plan whose spectral arrays hold one streamwise mode per member; workspace, binding
// and destruction go through dns_plan_workspace_bytes / dns_plan_bind / dns_plan_destroy.
#include <cmath>
#include <vector>

#include "dns_internal.h"

namespace {

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
bool all_finite(const double* x, int n) {
    for (int i = 0; i < n; ++i)
        if (!std::isfinite(x[i])) return false;
    return true;
}
int check(dns_plan* p, bool need_state) {
    if (!p) return DNS_EINVAL;
    if (!p->d.lin) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound) return DNS_ESTATE;
    if (need_state && (!p->has_state || !p->has_base)) return DNS_ESTATE;
    return DNS_OK;
}

// one CN/RK3 stage of Eq. 12-13 with the linear vector in place of u.grad u
void lin_stage(dns_plan* p, int s, int adjoint) {
    launch_zinv(p, s == 0 ? p->d.vt : p->d.vs, nullptr);     // u v w du/dy dw/dy -> 8 mixed fields (i kz on load)
    launch_lin_products(p, adjoint);
    launch_zfwd(p);
    launch_ypair(p, s, 0);
}

// One linear step (3 stages x 4 launches) captured into a CUDA graph per direction, as dns_step does for the DNS step: at
// the paper's size (45 disturbances) every kernel of the step lasts a few microseconds and the step is bound by
// launch overhead.  Captured on the plan's internal stream; any failure leaves the direction on direct launches for good.
void build_lin_graph(dns_plan* p, int adjoint) {
    p->lin_graph_state[adjoint] = -1;
    if (dns_option("graph") == 0) return;
    if (cudaPeekAtLastError() != cudaSuccess) return;
    if (!p->capture_stream && cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return; }
    cudaStream_t user = p->stream;
    if (cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return; }
    p->stream = p->capture_stream;
    for (int s = 0; s < 3; ++s) lin_stage(p, s, adjoint);
    p->stream = user;
    cudaGraph_t g = nullptr;
    if (cudaStreamEndCapture(p->capture_stream, &g) != cudaSuccess || !g) { cudaGetLastError(); return; }
    cudaGraphExec_t ge = nullptr;
    if (cudaGraphInstantiate(&ge, g, 0) != cudaSuccess || !ge) { cudaGetLastError(); cudaGraphDestroy(g); return; }
    p->lin_graph[adjoint] = g;
    p->lin_graph_exec[adjoint] = ge;
    p->lin_graph_state[adjoint] = 1;
}

}  // namespace

void dns_lin_drop_graphs(dns_plan* p) {
    for (int a = 0; a < 2; ++a) {
        if (p->lin_graph_exec[a]) cudaGraphExecDestroy(p->lin_graph_exec[a]);
        if (p->lin_graph[a]) cudaGraphDestroy(p->lin_graph[a]);
        p->lin_graph_exec[a] = nullptr;
        p->lin_graph[a] = nullptr;
        p->lin_graph_state[a] = 0;
    }
}

extern "C" {

int dns_lin_plan_create(dns_plan** out, int Nx, int Ny, int Nz, int nmodes, const int* n_list, int Eg, double Re, double Lx,
                        double Lz, double dt_lin) {
    if (!out) return DNS_EINVAL;
    *out = nullptr;
    if (nmodes < 1 || !n_list || Eg < 1 || (long long)nmodes * Eg > (1 << 20)) return DNS_EINVAL;
    return dns_create_common(out, Nx, Ny, Nz, nmodes * Eg, Re, Lx, Lz, dt_lin, DNS_COUETTE, nmodes, n_list, Eg);
}

int dns_lin_set_base(dns_plan* lin, dns_plan* dns, int member) {
    const int st = check(lin, false);
    if (st != DNS_OK) return st;
    if (!dns || dns->d.lin || member < 0 || member >= dns->d.E) return DNS_EINVAL;
    if (dns->d.Ny != lin->d.Ny || dns->d.Nz != lin->d.Nz || dns->d.Nx != lin->d.Nx || dns->Lz != lin->Lz || dns->Lx != lin->Lx)
        return DNS_EINVAL;
    if (dns->d.form != DNS_FORM_CONVECTIVE) return DNS_EINVAL;        // the mixed arrays must hold du/dy, dw/dy
    if (dns->sticky != DNS_OK) return dns->sticky;
    if (!dns->bound || !dns->has_state) return DNS_ESTATE;
    // linear steps still in flight on the linear plan's stream read the base flow that is about to be rewritten
    const cudaError_t e0 = cudaStreamSynchronize(lin->stream);
    if (e0 != cudaSuccess) return cuda_status(lin, e0);
    // the DNS plan's transform inputs (u, w, du/dy, dw/dy of its current state) -> mixed (kx, z) arrays; their kx = 0
    // column is the streamwise-mean flow in physical z.  I8 is scratch of the DNS plan, rewritten by its next stage.
    launch_zinv(dns, dns->d.vt, dns->d.et);
    launch_lin_base(lin, dns, member, dns->stream);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(dns->stream);    // the linear plan may work on another stream
    if (e != cudaSuccess) return cuda_status(lin, e);
    lin->has_base = true;
    return DNS_OK;
}

int dns_lin_set_state(dns_plan* p, const double* vhat, const double* etahat) {
    const int st = check(p, false);
    if (st != DNS_OK) return st;
    if (!vhat || !etahat) return DNS_EINVAL;
    DnsDev& d = p->d;
    double2* sv = d.stage_io;
    double2* se = sv + d.S;
    const bool dv = is_device_ptr(vhat), de = is_device_ptr(etahat);
    cudaError_t e = cudaMemcpyAsync(sv, vhat, d.S * sizeof(double2), dv ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(se, etahat, d.S * sizeof(double2), de ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream);
    if (e != cudaSuccess) return cuda_status(p, e);
    launch_abi_to_internal(p, sv, d.vt, 0);
    launch_abi_to_internal(p, se, d.et, 0);
    launch_lin_normalise(p);
    launch_ypair(p, 0, 1);                                   // u, w, du/dy, dw/dy of the state (Eq. 17-18)
    p->has_state = true;
    e = cudaGetLastError();
    if (e == cudaSuccess && !(dv && de)) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_lin_get_state(dns_plan* p, double* vhat, double* etahat) {
    const int st = check(p, false);
    if (st != DNS_OK) return st;
    if (!p->has_state) return DNS_ESTATE;
    DnsDev& d = p->d;
    double2* sv = d.stage_io;
    double2* se = sv + d.S;
    cudaError_t e = cudaSuccess;
    if (vhat) {
        launch_internal_to_abi(p, d.vt, sv);
        e = cudaMemcpyAsync(vhat, sv, d.S * sizeof(double2), is_device_ptr(vhat) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, p->stream);
    }
    if (etahat && e == cudaSuccess) {
        launch_internal_to_abi(p, d.et, se);
        e = cudaMemcpyAsync(etahat, se, d.S * sizeof(double2), is_device_ptr(etahat) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, p->stream);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    return cuda_status(p, e);
}

int dns_lin_step(dns_plan* p, int nsteps, int adjoint) {
    const int st = check(p, true);
    if (st != DNS_OK) return st;
    if (nsteps < 0 || (adjoint != 0 && adjoint != 1)) return DNS_EINVAL;
    if (p->lin_graph_state[adjoint] == 0 && nsteps > 0) build_lin_graph(p, adjoint);
    for (int it = 0; it < nsteps; ++it) {
        if (p->lin_graph_state[adjoint] == 1) {
            if (cudaGraphLaunch(p->lin_graph_exec[adjoint], p->stream) != cudaSuccess) return cuda_status(p, cudaGetLastError());
        } else {
            for (int s = 0; s < 3; ++s) lin_stage(p, s, adjoint);
        }
    }
    return cuda_status(p, cudaGetLastError());
}

int dns_lin_energy(dns_plan* p, double* out) {
    const int st = check(p, false);
    if (st != DNS_OK) return st;
    if (!out) return DNS_EINVAL;
    if (!p->has_state) return DNS_ESTATE;
    launch_lin_energy(p, p->d.lin_scr);
    const bool dev = is_device_ptr(out);
    cudaError_t e = cudaMemcpyAsync(out, p->d.lin_scr, p->d.E * sizeof(double),
                                    dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return cuda_status(p, e);
    return (!dev && !all_finite(out, p->d.E)) ? DNS_ENONFINITE : DNS_OK;
}

int dns_lin_orthonormalise(dns_plan* p) {
    const int st = check(p, false);
    if (st != DNS_OK) return st;
    if (!p->has_state) return DNS_ESTATE;
    launch_lin_gs(p);
    launch_ypair(p, 0, 1);                                   // refresh the transform inputs of the new vectors
    return cuda_status(p, cudaGetLastError());
}

int dns_lin_optimals(dns_plan* p, int nsteps, int niter, double* gains) {
    int st = check(p, true);
    if (st != DNS_OK) return st;
    if (nsteps < 1 || niter < 1 || !gains) return DNS_EINVAL;
    if ((st = dns_lin_orthonormalise(p)) != DNS_OK) return st;
    double* g = p->d.lin_scr + p->d.E;
    for (int it = 0; it < niter; ++it) {
        if ((st = dns_lin_step(p, nsteps, 0)) != DNS_OK) return st;
        launch_lin_energy(p, g);                             // the initial energies are 1: E(T_opt) is the gain (B.1)
        if ((st = dns_lin_step(p, nsteps, 1)) != DNS_OK) return st;
        if ((st = dns_lin_orthonormalise(p)) != DNS_OK) return st;
    }
    const bool dev = is_device_ptr(gains);
    cudaError_t e = cudaMemcpyAsync(gains, g, p->d.E * sizeof(double),
                                    dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return cuda_status(p, e);
    return (!dev && !all_finite(gains, p->d.E)) ? DNS_ENONFINITE : DNS_OK;
}

int dns_lin_launches_per_step(const dns_plan* p) { return (p && p->d.lin) ? 3 * 4 : 0; }

}  // extern "C"
