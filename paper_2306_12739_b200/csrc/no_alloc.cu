// dns_energy_noalloc (include/dns.h): the per-member kinetic energy of Eq. B.1 for callers that must not
// allocate.  It is the energy kernel pair of dns_diagnostics / dns_lin_energy (kernels_y.cu: k_diag_energy + the row sum)
// restated here with one difference: the [Ny][E] table of per-plane partial sums that sits between the two kernels does
// not live in anyone's allocation.  It lives in g_energy_scratch below, a fixed array that is part of the library image
// and therefore exists on every GPU that loads the library, from load to process exit, whether or not this call is used.
//
// Rules of that array, for whoever edits this file:
//   * In HOST code the name g_energy_scratch is only a handle for the runtime, not a device address.  Handing it to a
//     kernel would make the kernel fault, or, on a machine where the GPU can reach host memory, quietly read and write
//     the wrong bytes.  The device address is looked up with cudaGetSymbolAddress, once per device, with that device
//     current, and the kernels are given the looked-up pointer.
//   * All calls on one GPU share it and it is never cleared: it still holds the previous call's partial sums.  That is
//     harmless because k_energy_planes writes every element (j < Ny, e < E) that k_energy_members of the same call reads,
//     so nothing needs to start at zero.  Two calls whose kernels overlap on the GPU (different streams) race on it.
//   * Nothing in this file may allocate, on the host or on the device: no cudaMalloc / cudaFree, no std::vector, no
//     library routine that allocates behind the scenes.
#include <mutex>

#include "dns_internal.h"

namespace {

static __device__ __align__(256) double g_energy_scratch[DNS_NOALLOC_MAX_DOUBLES];      // 512 KiB per GPU

constexpr int kMaxDevices = 64;
std::mutex g_lookup_mutex;
double* g_scratch_addr[kMaxDevices] = {};       // device address of g_energy_scratch on device i, nullptr = not looked up

// Set-up, once per device: the address of the array ON THE CURRENT DEVICE.  The first lookup also makes the runtime load
// this module onto that device, which is why the first call should not happen inside a stream capture.
cudaError_t scratch_address(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_lookup_mutex);
    if (!g_scratch_addr[dev]) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_energy_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

__device__ __forceinline__ int member_block(int E) { int b = 1; while (b < E && b < 256) b <<= 1; return b; }

// part[j][e] = (1/4) w_j sum_p c_p (|u|^2 + |v|^2 + |w|^2) over the retained modes p of plane j = blockIdx.x; c_p = 2 for a
// stored mode that stands for +-kx, 1 on the kx = 0 plane of a DNS plan (both signs of kz are stored there).  Same thread
// mapping and the same order of additions as k_diag_energy: 256 threads = EB member lanes x (256 / EB) mode slots, slot
// sums added in ascending slot order, so the result does not depend on scheduling and equals the existing path's.
__global__ void __launch_bounds__(256) k_energy_planes(DnsDev d, double* __restrict__ part) {
    __shared__ double sm[256];
    const int j = blockIdx.x, EB = member_block(d.E);
    const int el = threadIdx.x % EB, slot = threadIdx.x / EB, nslot = blockDim.x / EB;
    for (int e0 = 0; e0 < d.E; e0 += EB) {
        const int e = e0 + el;
        double acc = 0.0;
        if (e < d.E)
            for (int p = slot; p < d.P; p += nslot) {
                const size_t gi = ((size_t)j * d.P + p) * d.E + e;
                const double2 u = d.uh[gi], v = d.vt[gi], w = d.wh[gi];
                const double cn = (!d.lin && (p / d.nkz) == 0) ? 1.0 : 2.0;
                acc += cn * (u.x * u.x + u.y * u.y + v.x * v.x + v.y * v.y + w.x * w.x + w.y * w.y);
            }
        sm[slot * EB + el] = acc;
        __syncthreads();
        if (slot == 0 && e < d.E) {
            double t = 0.0;
            for (int q = 0; q < nslot; ++q) t += sm[q * EB + el];
            part[(size_t)j * d.E + e] = 0.25 * d.w[j] * t;
        }
        __syncthreads();
    }
}

// energy[e] = sum_j part[j][e], ascending j
__global__ void k_energy_members(int Ny, int E, const double* __restrict__ part, double* __restrict__ energy) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= E) return;
    double s = 0.0;
    for (int j = 0; j < Ny; ++j) s += part[(size_t)j * E + e];
    energy[e] = s;
}

}  // namespace

extern "C" int dns_energy_noalloc(dns_plan* p, double* energy_dev) {
    if (!p || !energy_dev) return DNS_EINVAL;
    if (p->sticky != DNS_OK) return p->sticky;
    if (!p->bound || !p->has_state) return DNS_ESTATE;
    const DnsDev& d = p->d;
    if ((size_t)d.Ny * (size_t)d.E > (size_t)DNS_NOALLOC_MAX_DOUBLES) return DNS_ELIMIT;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, energy_dev) != cudaSuccess) { cudaGetLastError(); return DNS_EINVAL; }
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) return DNS_EINVAL;
    double* part = nullptr;
    if (scratch_address(&part) != cudaSuccess) { cudaGetLastError(); return DNS_ECUDA; }
    k_energy_planes<<<d.Ny, 256, 0, p->stream>>>(d, part);
    k_energy_members<<<(d.E + 127) / 128, 128, 0, p->stream>>>(d.Ny, d.E, part, energy_dev);
    return cudaGetLastError() == cudaSuccess ? DNS_OK : DNS_ECUDA;
}
