/* dns.h -- C ABI of libdns_b200: the vectorised ensemble time step of arXiv 2306.12739
 * ("A vectorized Navier-Stokes ensemble DNS code for plane parallel flows") on one NVIDIA B200 (sm_100a).
 *
 * The library advances E independent realisations of 3-D incompressible plane Couette / constant-mass-flux
 * Poiseuille flow at once.  State = wall-normal velocity v and wall-normal vorticity eta (PAPER.md:68,
 * Eq. 4-5 :72-74) in Fourier space in x,z and on Ny Chebyshev-Gauss-Lobatto points in y, plus the mean
 * profiles U00(y), W00(y) (Eq. 6-7 :76-78).  Time stepping is the combined Crank-Nicolson / 3rd-order
 * Runge-Kutta scheme (Eq. 11); next-stage fields come from precomputed per-(kx,kz) matrix
 * inverses (Eq. 12-15 :153-163, Listings 3-5) applied to all members at once.
 *
 * Every entry point returns an int status (DNS_OK = 0, negative on error); nothing throws or aborts across
 * the ABI.  No torch / C++ types appear in the signatures.  All compute runs in the library's CUDA kernels;
 * there is no CPU fallback: without a CUDA device every call that needs one returns DNS_ECUDA.
 *
 * Array layouts at the ABI (C order, last index fastest):
 *   vhat, etahat : [E][nkx][nkz][Ny] complex128 as interleaved (re, im) doubles
 *                  nkx = Nx/2, streamwise mode n = 0 .. Nx/2-1            (kx = 2 pi n / Lx)
 *                  nkz = Nz-1, spanwise mode m in FFT order 0,1,..,Nz/2-1, -(Nz/2-1),..,-1
 *                                                                       (kz = 2 pi m / Lz; `mrange`)
 *                  y_j = -cos(pi j/(Ny-1)), j = 0..Ny-1, ascending from the lower wall
 *   U00, W00     : [E][Ny] float64
 * Fourier convention: f(x,z) = sum_{n,m} fhat(n,m) exp(+i(kx x + kz z)); coefficients are amplitudes; only
 * n >= 0 is stored, fhat(-n,-m) = conj fhat(n,m).  The Nyquist modes n = Nx/2, m = -Nz/2 are not stored and
 * are identically zero (3/2-rule dealiasing on an Mx = 3Nx/2, Mz = 3Nz/2 grid).
 * Pointers passed to set/get/diagnostics may be HOST or DEVICE pointers (detected with
 * cudaPointerGetAttributes); the caller owns them and the library keeps no reference after the call returns.
 */
#ifndef DNS_B200_H
#define DNS_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dns_plan dns_plan; /* opaque, owned by the library */

enum { DNS_COUETTE = 0, DNS_POISEUILLE_CMF = 1 }; /* flow */

enum {
    DNS_OK = 0,
    DNS_EINVAL = -1,     /* bad argument (see each call) */
    DNS_ENOMEM = -2,     /* host or device allocation failed */
    DNS_ECUDA = -3,      /* CUDA runtime error or no device; sticky on the plan */
    DNS_ENONFINITE = -4, /* a member's energy is not finite (dns_diagnostics) */
    DNS_ESTATE = -5,     /* call out of order (no workspace bound, no state set) */
    DNS_ELIMIT = -6      /* the problem is larger than the fixed capacity of dns_energy_noalloc */
};

/* kernel classes reported by dns_step_profile (north_star subsystems (1)-(4)) */
enum {
    DNS_CLASS_FFT_Z_INV = 0, /* a4, z direction: zero-pad + i kz + complex inverse FFT            */
    DNS_CLASS_LINE = 1,      /* a4 x direction + a5 products + a6 x direction, fused per (y,z) line */
    DNS_CLASS_FFT_Z_FWD = 2, /* a6, z direction: forward FFT + truncation + 1/(Mx Mz)              */
    DNS_CLASS_YPAIR = 3,     /* a7,a8,a9,a1,a2,a3: per-(kx,kz) DMMA contractions + stage algebra;
                                a10 (mean flow, wall lift, mass-flux gamma) is a small kernel on an internal side stream
                                that runs under classes 2 and 3 and is joined before this class's closing event */
    DNS_NCLASS = 4
};

/* dns_plan_create -- precompute everything that is constant for a fixed dt: Chebyshev D,
 * D2 = D*D, the clamped fourth derivative, and for every distinct
 * alpha = kx^2+kz^2 and h in {1/2, 1} the inverses of Eq. 12-13 (Listing 3) and of the
 * mean-flow operator of Eq. 14-15; uploads them to the current CUDA device.
 *   Nx, Nz : un-padded Fourier grid, even; Mx = 3Nx/2 and Mz = 3Nz/2 must be 2^a 3^b within 16..128
 *   Ny     : Chebyshev-Gauss-Lobatto points including both walls, 5 <= Ny <= 257
 *   E      : ensemble members (PAPER.md:131 `Fn`), >= 1
 *   Re     : 1/nu in the units of the state; Lx, Lz periodic lengths (y in [-1,1]); dt fixed step
 *   flow   : DNS_COUETTE (walls at +-1 move with U = +-1, gamma = 0) or DNS_POISEUILLE_CMF (walls at rest,
 *            gamma(t) solved every stage so that the bulk flux (1/2) int U00 dy keeps the value it had in
 *            dns_set_state)
 * Errors: DNS_EINVAL (null out, bad sizes, non-positive Re/Lx/Lz/dt, unknown flow), DNS_ENOMEM, DNS_ECUDA.
 * On success *out owns host and device memory until dns_plan_destroy. */
int dns_plan_create(dns_plan** out, int Nx, int Ny, int Nz, int E, double Re, double Lx, double Lz, double dt,
                    int flow);

/* dns_plan_set_form -- form of the nonlinear term.  DNS_FORM_CONVECTIVE (default) is the
 * paper's u . grad u_i.  DNS_FORM_ROTATIONAL forms H = omega x u instead, omega = curl u:
 * (u . grad)u = omega x u + grad(|u|^2/2) and Eq. 4-5 are what is left of the momentum equation once
 * gradients are eliminated (:68), so F and G keep their form with H in place of u . grad u; the mean-flow sources of
 * Eq. 6-7 become the plane means of H_x and H_z.  6 instead of 11 physical fields are transformed per stage.  The two
 * forms agree to round-off wherever the wall-normal products are resolved and differ at y-truncation level otherwise.
 * Call before dns_set_state.  Errors: DNS_EINVAL (null, unknown form), DNS_ESTATE (a state is already set). */
enum { DNS_FORM_CONVECTIVE = 0, DNS_FORM_ROTATIONAL = 1 };
int dns_plan_set_form(dns_plan* plan, int form);

/* dns_plan_set_coupling -- ensemble-coupled streamwise-mean flow ("Each
 * ensemble member shares a common streamwise mean flow, which is updated at every time-step by the perturbation
 * Reynolds stresses averaged over the ensemble members").  With DNS_COUPLING_STREAMWISE_MEAN every stage replaces the
 * kx = 0 part of the nonlinear vector (all that forces the streamwise-mean flow) and the mean-flow sources of Eq. 6-7
 * by their average over ALL members, summed in a fixed order; kx != 0 is untouched.  Members whose kx = 0 components
 * and U00, W00 are equal in dns_set_state keep them equal.  E_total = members of the whole ensemble: plan E on one
 * GPU; with members sharded over ranks the sum of the ranks' E, and dns_plan_set_exchange must be given.
 * Call before dns_set_state.  Errors: DNS_EINVAL (null, unknown mode, E_total < E), DNS_ESTATE. */
enum { DNS_COUPLING_NONE = 0, DNS_COUPLING_STREAMWISE_MEAN = 1 };
int dns_plan_set_coupling(dns_plan* plan, int mode, long long E_total);

/* dns_plan_set_exchange -- the one exchange step of the path (coupled ensembles sharded over GPUs): fn must replace
 * dev_buf[0..count) (doubles, DEVICE memory inside the bound workspace) by its element-wise sum over all ranks, ordered
 * after the work already enqueued on cuda_stream and before anything enqueued later (e.g. an NCCL all-reduce on that
 * stream), and return 0 on success.  It is called once per stage (3 times per step) from dns_step; count is
 * (3 Ny (Nz-1) + Ny 3Nz/2) * 2.  With an exchange set dns_step launches directly (a host call cannot be replayed from a
 * CUDA graph).  fn = NULL removes it.  ctx is passed back verbatim and never dereferenced by the library. */
typedef int (*dns_exchange_fn)(void* ctx, double* dev_buf, size_t count, void* cuda_stream);
int dns_plan_set_exchange(dns_plan* plan, dns_exchange_fn fn, void* ctx);

/* dns_add_increment -- state += (dvhat, detahat) between two steps (layout of dns_set_state; host or device): how a
 * caller applies one realisation of a stochastic forcing (the realisations are the caller's).  The
 * result is normalised as in dns_set_state (wall rows, (0,0) column, Hermitian kx = 0 plane) and the transform inputs
 * are re-derived; time, step count and the Poiseuille target flux are kept.  Errors: DNS_EINVAL, DNS_ESTATE, DNS_ECUDA. */
int dns_add_increment(dns_plan* plan, const double* dvhat, const double* detahat);

/* Bytes of DEVICE workspace the caller must provide to dns_plan_bind (state, stage buffers, transform
 * intermediates).  0 if plan is null. */
size_t dns_plan_workspace_bytes(const dns_plan* plan);

/* dns_plan_bind -- hand the plan a device buffer (256-byte aligned, >= dns_plan_workspace_bytes) and the CUDA
 * stream (cudaStream_t as void*, NULL = default stream) every later call works on.  The buffer stays owned by
 * the caller and must outlive the plan or the next bind; it is zero-filled here.
 * Errors: DNS_EINVAL (null plan/buffer, too small, misaligned), DNS_ECUDA. */
int dns_plan_bind(dns_plan* plan, void* dev_workspace, size_t bytes, void* cuda_stream);

/* dns_set_state -- load the state at time t = 0 (ABI layout above; host or device pointers).  Input is
 * normalised: wall rows of vhat, etahat and their (0,0) column are set to 0 (PAPER.md:82 Eq. 8, :87); wall rows
 * of U00 to -+1 (Couette) or 0, of W00 to 0 (Eq. 9 :85); on the n = 0 plane entries with m < 0 are replaced by
 * the conjugates of m > 0.  The Poiseuille target flux of member e is the Clenshaw-Curtis bulk mean of U00[e].
 * Also derives u, w, dU/dy ... needed by the first nonlinear evaluation (Eq. 17-18 :214-216).  Asynchronous
 * for device pointers; for host pointers the copies are enqueued on the plan's stream and synchronised.
 * Errors: DNS_EINVAL (null), DNS_ESTATE (no workspace), DNS_ECUDA. */
int dns_set_state(dns_plan* plan, const double* vhat, const double* etahat, const double* U00,
                  const double* W00);

/* dns_step -- enqueue nsteps full CN/RK3 time steps (3 stages each) on the plan's stream
 * and return without synchronising.  The launches of a step (dns_launches_per_step: 15, 18 with the coupled ensemble, 21 with
 * an exchange) are captured once into a CUDA graph (on an internal
 * stream, at the first call after dns_plan_bind) and replayed per step; a failed capture (or the test option "graph" = 0 of include/dns_debug.h) falls back to
 * direct launches with identical results.  Errors: DNS_EINVAL (nsteps < 0), DNS_ESTATE (no state), DNS_ECUDA. */
int dns_step(dns_plan* plan, int nsteps);

/* dns_step_profile -- as dns_step, but brackets every kernel class with CUDA events on the plan's stream,
 * synchronises, and adds the elapsed milliseconds per class to ms_by_class[DNS_NCLASS] (host array). */
int dns_step_profile(dns_plan* plan, int nsteps, double* ms_by_class);

/* dns_get_state -- copy the current state out (same layout as dns_set_state; any pointer may be NULL to skip
 * that array); synchronises the stream.  Errors: DNS_ESTATE, DNS_ECUDA. */
int dns_get_state(dns_plan* plan, double* vhat, double* etahat, double* U00, double* W00);

/* dns_diagnostics -- out[E][6] (host or device): [0] kinetic energy 1/(2V) int |u|^2 dV,
 * [1] dU00/dy at the lower wall, [2] at the upper wall (tau_w = (1/Re) dU00/dy), [3] bulk flux
 * (1/2) int U00 dy, [4] gamma used in the last stage, [5] time t.  Synchronises.
 * Returns DNS_ENONFINITE if any member's energy is not finite (rows are still filled). */
int dns_diagnostics(dns_plan* plan, double* out);

/* One-point statistics: running sums, per member and wall-normal point, of
 * U (plane-mean streamwise velocity), <u'u'>, <v'v'>, <w'w'>, <u'v'> (primes = deviations from the (x,z) plane mean),
 * evaluated from the spectral state by Parseval over the retained modes.
 *   dns_stats_reset      -- zero the sums and the sample count (also done by dns_plan_bind)
 *   dns_stats_accumulate -- enqueue: add the statistics of the current state as one sample
 *   dns_stats_get        -- out[E][Ny][5] (host or device) = sums / samples; *nsamples (may be NULL) = sample count;
 *                           synchronises.  With no sample yet out is zero-filled.
 * Errors: DNS_EINVAL (null), DNS_ESTATE (no workspace / no state), DNS_ECUDA. */
enum { DNS_NSTAT = 5 };
int dns_stats_reset(dns_plan* plan);
int dns_stats_accumulate(dns_plan* plan);
int dns_stats_get(dns_plan* plan, double* out, long long* nsamples);

/* ---- Linearised forward / adjoint ensemble (section 4.1.1, Appendix B :390-417) ----
 * E = nmodes * Eg disturbance vectors advanced at once.  Vector e = g Eg + i has the single streamwise wavenumber
 * kx = 2 pi n_list[g] / Lx ("we may specify the streamwise wavenumber of each disturbance") and no mean flow, so only
 * Eq. 12-13 are solved, with the precomputed single-kx operators of that vector, which also serve the adjoint.
 * The base flow (U, V, W)(y, z) is the frozen streamwise-mean (kx = 0) part of a DNS state (Fig. 7(a)).
 *   forward (Eq. B.2):  d u'/dt     = -[(U.grad)u' + (u'.grad)U] - grad p' + (1/Re) Lap u'
 *   adjoint (Eq. B.5):  d lam/d tau = +[(U.grad)lam + U_i grad lam_i] - grad b + (1/Re) Lap lam,  tau = T - t (reversed time)
 * stepped with the CN/RK3 scheme of PAPER.md:120-126 at dt_lin = t_f dt (time-step factor t_f, :315).  Energy inner product
 * (Eq. B.1) <a,b> = 1/(2V) int conj(a).b dV.  Layout: vhat, etahat [E][nkz][Ny] complex128 (m in FFT order, y ascending).
 *
 * dns_lin_plan_create  -- as dns_plan_create (same grid limits); n_list[nmodes] with 1 <= n < Nx/2; Eg members per mode;
 *                         dt_lin the step of the linear problem.  Workspace, binding and destruction:
 *                         dns_plan_workspace_bytes, dns_plan_bind, dns_plan_destroy.  Errors: DNS_EINVAL, DNS_ENOMEM, DNS_ECUDA.
 * dns_lin_set_base     -- base flow := streamwise-mean flow of member `member` of the CURRENT state of a DNS plan with the
 *                         same grid and box, in the convective form (its transform scratch is overwritten; synchronises that
 *                         plan's stream).  Errors: DNS_EINVAL (mismatch, rotational form, bad member), DNS_ESTATE, DNS_ECUDA.
 * dns_lin_set_state / dns_lin_get_state -- host or device pointers; wall rows are set to 0; get synchronises.
 * dns_lin_step         -- enqueue nsteps steps of the forward (adjoint = 0) or adjoint (adjoint = 1) equations.  As in
 *                         dns_step the 12 launches of a step are captured once per direction into a CUDA graph and replayed
 *                         (identical results; direct launches if the capture fails or with the test option "graph" = 0).
 * dns_lin_energy       -- out[E] = <q_e, q_e> (host or device); synchronises.  DNS_ENONFINITE if out is a host pointer and
 *                         an energy is not finite (out is still filled; a device out is not inspected).
 * dns_lin_orthonormalise -- modified Gram-Schmidt in member order within every kx group, energy inner product (:417).
 *                         A member whose energy is exactly zero (or not finite) when its turn comes, e.g. a zero vector, is
 *                         set to zero rather than divided by zero; its energy and gain then read 0 and the other members of
 *                         its group are unaffected.
 * dns_lin_optimals     -- the power iteration of :417: orthonormalise; niter times { nsteps forward, record the gains
 *                         E(T_opt)/E(0), nsteps adjoint from the forward final state, orthonormalise }; gains[E] (host or
 *                         device) are those of the last forward leg.  T_opt = nsteps dt_lin.  Synchronises.
 *                         DNS_ENONFINITE as for dns_lin_energy.
 * All: DNS_EINVAL for a non-linear plan or bad arguments, DNS_ESTATE before bind / set_base / set_state, DNS_ECUDA. */
int dns_lin_plan_create(dns_plan** out, int Nx, int Ny, int Nz, int nmodes, const int* n_list, int Eg, double Re, double Lx,
                        double Lz, double dt_lin);
int dns_lin_set_base(dns_plan* lin, dns_plan* dns, int member);
int dns_lin_set_state(dns_plan* lin, const double* vhat, const double* etahat);
int dns_lin_get_state(dns_plan* lin, double* vhat, double* etahat);
int dns_lin_step(dns_plan* lin, int nsteps, int adjoint);
int dns_lin_energy(dns_plan* lin, double* out);
int dns_lin_orthonormalise(dns_plan* lin);
int dns_lin_optimals(dns_plan* lin, int nsteps, int niter, double* gains);
int dns_lin_launches_per_step(const dns_plan* lin);

/* dns_energy_noalloc -- energy_dev[E] = kinetic energy 1/(2V) int |u|^2 dV (Eq. B.1) of every member of
 * the plan's current state: the number dns_diagnostics reports in column 0 (DNS plan) and dns_lin_energy reports
 * (linearised plan), computed in the same order of operations.
 *
 * Who it is for.  The other two calls stage their result through memory carved from the workspace or through a host
 * vector.  Some callers may not create memory at the point where they want an energy: a monitor that runs inside a
 * time loop whose every device byte was handed out up front (a pool or caching allocator owns the GPU, or the job runs
 * under a fixed memory budget on a shared or partitioned GPU, so a fresh device allocation can fail long into a run);
 * code on a latency-critical path, where a device allocation or free stalls the whole GPU until earlier work has
 * drained; and host code that is simply not allowed to call the CUDA allocator (plug-ins, callbacks).  This call
 * allocates nothing, neither on the host nor on the device, and frees nothing.  The table of per-plane partial sums it
 * needs between its two kernels is a fixed 512 KiB array inside the library image; every GPU that loads the library
 * holds those 512 KiB until the process exits, used or not.
 *
 * Limit.  Ny * E <= DNS_NOALLOC_MAX_DOUBLES (65536; e.g. Ny = 65 with up to 1008 members).  A larger plan is refused with
 * DNS_ELIMIT and nothing is launched: use dns_diagnostics / dns_lin_energy there.
 *
 * Arguments.  plan: bound and with a state (DNS or linearised); its device must be the current one.  energy_dev: DEVICE
 * pointer to E doubles owned by the caller (a host pointer is refused with DNS_EINVAL: copying to pageable host memory
 * would need a staging buffer).  Two kernels are enqueued on the plan's stream; the call does not synchronise, so read
 * energy_dev in stream order.
 *
 * First call on a device.  It looks up where the fixed array lives on that device (once per device, remembered
 * afterwards), which can also make the CUDA runtime load the library's code onto the device.  Make that first call
 * during set-up, outside any stream capture.
 *
 * Sharing.  All plans and all calls on one GPU use the same array, and it keeps whatever the last call left in it.
 * Every entry a call reads it has written itself first, so stale contents never reach a result.  But two calls whose
 * kernels can run at the same time on one GPU (plans bound to different streams, or several host threads) overwrite
 * each other's partial sums: order such calls yourself (one stream, or an event between them).
 * Errors: DNS_EINVAL (null, host pointer), DNS_ESTATE (no workspace / no state), DNS_ELIMIT, DNS_ECUDA. */
#define DNS_NOALLOC_MAX_DOUBLES 65536
int dns_energy_noalloc(dns_plan* plan, double* energy_dev);

/* Number of kernel launches one dns_step(1) enqueues (for bench.py's gpu_launches). */
int dns_launches_per_step(const dns_plan* plan);

/* Frees plan-owned host and device memory (not the bound workspace).  Null is accepted. */
int dns_plan_destroy(dns_plan* plan);

/* Static string for a status code. */
const char* dns_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* DNS_B200_H */
