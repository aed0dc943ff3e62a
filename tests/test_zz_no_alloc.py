"""dns_energy_noalloc (include/dns.h) against the calls that were there before it.

Why the entry point exists: dns_diagnostics and dns_lin_energy pass their result through staging memory (a host vector, a
slice of the workspace).  A caller that has given every device byte to a pool up front, that runs under a fixed memory
budget, that sits on a latency-critical path where a device allocation would stall the GPU, or that is simply not allowed
to call the CUDA allocator, needs an energy read-out that creates no memory at all.  dns_energy_noalloc keeps the one
table it needs between its two kernels in a fixed 512 KiB array inside the library, which limits it to
Ny * E <= DNS_NOALLOC_MAX_DOUBLES, and which every call on a GPU shares.

What is checked: the energies equal the existing paths' within the tolerance the other energy tests use (1e-12 relative,
tests/test_gpu_linear.py), on calls made back to back, so that the second and third call find the previous call's partial
sums still in the shared array -- laid out for another Ny and E -- and must not be affected by them; and the limit and
the argument checks.  The output tensors are created before the call under test: the call itself must not need any.

This file is named to be collected last (pytest -x stops at the first failure), and it passes alone in a fresh process
(the first call then does the per-device set-up) as well as after the other GPU tests."""
import numpy as np
import pytest

from paper_2306_12739_b200 import binding, inputs

pytestmark = pytest.mark.gpu

PI = np.pi
TOL = 1e-12          # relative, as in tests/test_gpu_linear.py for energies


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def test_noalloc_energy_equals_existing_paths_on_calls_in_a_row():
    import torch

    # a DNS plan (Ny * E = 33 * 5) and a linearised plan with another Ny and E (25 * 15), both with a few steps behind them
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 33, 16, 5, 0.02, 1, 0.3, 0, box=3)
    st = inputs.make_state(cfg)
    dns = binding.Plan(*inputs.plan_args(cfg))
    dns.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    dns.step(2)

    cl = inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 25, 16, 2, 0.02, 1, 0.3, 0, box=3)
    sl = inputs.make_state(cl)
    base = binding.Plan(*inputs.plan_args(cl))
    base.set_state(sl["vhat"], sl["etahat"], sl["U00"], sl["W00"])
    n_list, Eg = [1, 2, 3], 5
    lin = binding.LinPlan(cl.Nx, cl.Ny, cl.Nz, n_list, Eg, cl.Re, cl.Lx, cl.Lz, 5 * cl.dt)
    lin.set_base(base, 1)
    pert = inputs.make_state(inputs.Config(**{**cl.__dict__, "E": lin.E}), range(20, 20 + lin.E))
    lin.set_state(np.stack([pert["vhat"][e, n_list[e // Eg]] for e in range(lin.E)]),
                  np.stack([pert["etahat"][e, n_list[e // Eg]] for e in range(lin.E)]))
    lin.step(1, False)

    # reference values from the calls that existed before, and the outputs of the new call, all made BEFORE it runs
    want_dns = dns.diagnostics()[:, 0].copy()
    want_lin = lin.energy().copy()
    out1 = torch.full((cfg.E,), float("nan"), dtype=torch.float64, device="cuda")
    out2 = torch.full((lin.E,), float("nan"), dtype=torch.float64, device="cuda")
    out3 = torch.full((cfg.E,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()

    dns.energy_noalloc(out1)          # first call (in a fresh process: also the per-device set-up)
    lin.energy_noalloc(out2)          # second call, same stream: the array still holds the [33][5] table of the first
    dns.energy_noalloc(out3)          # third call: now it holds the [25][15] table of the second
    torch.cuda.synchronize()
    got1, got2, got3 = out1.cpu().numpy(), out2.cpu().numpy(), out3.cpu().numpy()
    assert np.isfinite(got1).all() and np.isfinite(got2).all() and (want_dns > 0).all() and (want_lin > 0).all()
    assert rel(got1, want_dns) < TOL, rel(got1, want_dns)
    assert rel(got2, want_lin) < TOL, rel(got2, want_lin)
    assert rel(got3, want_dns) < TOL, rel(got3, want_dns)
    assert np.array_equal(got1, got3)                     # same state, same order of additions: identical bits

    # the state moves on; two more calls in a row follow it
    dns.step(1)
    lin.step(1, True)
    want_dns, want_lin = dns.diagnostics()[:, 0].copy(), lin.energy().copy()
    dns.energy_noalloc(out1)
    lin.energy_noalloc(out2)
    torch.cuda.synchronize()
    assert rel(out1.cpu().numpy(), want_dns) < TOL
    assert rel(out2.cpu().numpy(), want_lin) < TOL
    assert not np.array_equal(out1.cpu().numpy(), got1)
    for p in (lin, base, dns):
        p.close()


def test_noalloc_energy_at_the_headline_shape():
    """BASELINE config 4's Ny and E (65 x 256 = 16640 table entries, several member blocks per plane) on a small x-z grid."""
    import torch

    cfg = inputs.Config(4, inputs.POISEUILLE_CMF, 3250.0, 1.75 * PI, 1.2 * PI, 16, 65, 16, 256, 0.008, 1, 0.3, 0, box=3)
    st = inputs.make_state(cfg)
    p = binding.Plan(*inputs.plan_args(cfg))
    p.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    p.step(1)
    want = p.diagnostics()[:, 0].copy()
    out = torch.zeros(cfg.E, dtype=torch.float64, device="cuda")
    for _ in range(2):
        out.fill_(float("nan"))
        p.energy_noalloc(out)
        torch.cuda.synchronize()
        assert rel(out.cpu().numpy(), want) < TOL
    p.close()


def test_noalloc_energy_refuses_what_it_cannot_do():
    import torch

    # no state yet
    p = binding.Plan(16, 17, 16, 2, 400.0, 5.0, 3.0, 0.02, binding.DNS_COUETTE)
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    assert binding.dns_energy_noalloc(p.h, out) == binding.DNS_ESTATE
    z = np.zeros(p.shape, np.complex128)
    p.set_state(z, z, np.zeros((2, 17)), np.zeros((2, 17)))
    assert binding.dns_energy_noalloc(p.h, None) == binding.DNS_EINVAL
    assert binding.dns_energy_noalloc(p.h, np.zeros(2)) == binding.DNS_EINVAL          # host memory
    assert binding.dns_energy_noalloc(None, out) == binding.DNS_EINVAL
    p.close()

    # one table entry too many for the fixed array: 17 * 3856 = 65552 > 65536
    E = 3856
    assert 17 * E > binding.DNS_NOALLOC_MAX_DOUBLES >= 17 * (E - 1)
    big = binding.Plan(12, 17, 12, E, 400.0, 5.0, 3.0, 0.02, binding.DNS_COUETTE)
    z = np.zeros(big.shape, np.complex128)
    big.set_state(z, z, np.zeros((E, 17)), np.zeros((E, 17)))
    out = torch.full((E,), -1.0, dtype=torch.float64, device="cuda")
    assert binding.dns_energy_noalloc(big.h, out) == binding.DNS_ELIMIT
    with pytest.raises(binding.DnsError, match="fixed capacity"):
        big.energy_noalloc(out)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == -1.0).all()              # nothing was launched
    assert np.isfinite(big.diagnostics()[:, 0]).all()     # the plan is still usable through the allocating path
    big.close()

    # the largest table that fits: 17 * 3855 = 65535 entries
    ok = binding.Plan(12, 17, 12, E - 1, 400.0, 5.0, 3.0, 0.02, binding.DNS_COUETTE)
    z = np.zeros(ok.shape, np.complex128)
    ok.set_state(z, z, np.zeros((E - 1, 17)), np.zeros((E - 1, 17)))
    out = torch.full((E - 1,), -1.0, dtype=torch.float64, device="cuda")
    ok.energy_noalloc(out)
    torch.cuda.synchronize()
    want = ok.diagnostics()[:, 0]
    assert np.abs(out.cpu().numpy() - want).max() <= TOL * max(np.abs(want).max(), 1.0)
    ok.close()
