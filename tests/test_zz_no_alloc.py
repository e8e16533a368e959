"""wslda_gradient_densities_static: the allocation-free entry point (scratch in a file-scope device array) against the
existing context path (wslda_densities with TAU | J -> gdens.cuh with the caller's workspace), on two calls in a row.
Collected last on purpose (the run uses -x)."""
import ctypes as C

import numpy as np
import pytest

import paper_2602_08982_b200 as ws
import workloads as wl

TOL_D = 1e-11               # the density tolerance of tests/test_gpu_parity.py (north_star)
FIELDS_TAU = ("tau_a", "tau_b")
FIELDS_J = ("ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z")


def relerr(x, ref):
    d = np.max(np.abs(ref))
    return float(np.max(np.abs(x - ref)) / (d if d > 0 else 1.0))


def _existing_path(shape, dx, psi, wa, wb):
    """tau and j through a context: [2][M] and [2][3][M] as numpy arrays."""
    import torch
    n = psi.shape[0]
    g = ws.Context(3, shape, dx, n, func_id=0, kin_form=0)
    g.set_mu(0.0, 0.0)
    g.set_weights(wa, wb)
    g.densities(psi, which=ws.D_TAU | ws.D_J)
    tau = torch.stack([g.get_field(f) for f in FIELDS_TAU]).cpu().numpy().reshape(2, -1)
    j = torch.stack([g.get_field(f) for f in FIELDS_J]).cpu().numpy().reshape(2, 3, -1)
    torch.cuda.synchronize()
    return tau, j


def _case(seed, n, side, dx):
    import torch
    shape = (side,) * 3
    psi = torch.from_numpy(np.ascontiguousarray(wl.random_spinors(seed, n, shape))).cuda()
    wa, wb = wl.uniform01(seed + 1, 0, n), wl.uniform01(seed + 2, 0, n)
    wa[n // 2] = 0.0                                          # a spinor one spin skips
    return shape, dx, psi, wa, wb


@pytest.mark.gpu
@pytest.mark.parametrize("side,n1,n2", [(32, 21, 5), (64, 3, 2)])
def test_static_scratch_entry_point_matches_the_context_path_twice(side, n1, n2):
    import torch
    M = side ** 3
    assert ws.lib().wslda_static_scratch_bytes() == 24 << 20
    tau = torch.empty(2, M, dtype=torch.float64, device="cuda")
    j = torch.empty(2, 3, M, dtype=torch.float64, device="cuda")
    # second call: fewer spinors (fewer groups at 32^3), other spacings -- what the first call left in the scratch must not leak
    for k, (seed, n, dx) in enumerate([(7100, n1, (1.0, 0.9, 1.1)), (7200, n2, (0.8, 1.0, 1.25))]):
        shape, dx, psi, wa, wb = _case(seed + side, n, side, dx)
        ref_tau, ref_j = _existing_path(shape, dx, psi, wa, wb)
        cwa, cwb = torch.from_numpy(wa).cuda(), torch.from_numpy(wb).cuda()
        tau.fill_(float("nan")); j.fill_(float("nan"))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        ws.gradient_densities_static(psi, cwa, cwb, dx, tau, j)
        torch.cuda.synchronize()
        if k == 1:                                            # warm call: the device's free memory has not moved
            assert torch.cuda.mem_get_info()[0] == free0
        got_tau, got_j = tau.cpu().numpy(), j.cpu().numpy()
        assert np.isfinite(got_tau).all() and np.isfinite(got_j).all()
        assert np.abs(ref_tau).max() > 0 and np.abs(ref_j).max() > 0
        for s in range(2):
            assert relerr(got_tau[s], ref_tau[s]) < TOL_D, (k, "tau", s)
            for d in range(3):
                assert relerr(got_j[s, d], ref_j[s, d]) < TOL_D, (k, "j", s, d)
    # tau alone / j alone, on a side stream, same bits as the call that produced both
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        t2 = torch.full_like(tau, float("nan")); j2 = torch.full_like(j, float("nan"))
        ws.gradient_densities_static(psi, cwa, cwb, dx, t2, None)
        ws.gradient_densities_static(psi, cwa, cwb, dx, None, j2)
    st.synchronize()
    assert torch.equal(t2, tau) and torch.equal(j2, j)


def test_static_entry_point_rejects_sizes_beyond_the_maximum():
    """Host-side argument checks come before any CUDA call: they run without a GPU."""
    L = ws.lib()
    dx = (C.c_double * 3)(1.0, 1.0, 1.0)
    p = C.c_void_p(256)                                       # never dereferenced: every call below is refused

    def call(n_wf, side, psi=p, tau=p):
        rc = L.wslda_gradient_densities_static(psi, p, p, n_wf, side, dx, tau, None, None)
        return rc, L.wslda_last_error(None).decode()

    rc, msg = call(4, 128)
    assert rc == 1 and "beyond the maximum of 64" in msg
    rc, msg = call(4, 48)
    assert rc == 1 and "32 or 64" in msg
    rc, msg = call(ws.STATIC_MAX_SPINORS + 1, 32)
    assert rc == 1 and "65536" in msg
    rc, msg = call(0, 32)
    assert rc == 1
    rc, msg = call(4, 32, psi=None)
    assert rc == 1 and "null" in msg
    rc, msg = call(4, 32, tau=None)
    assert rc == 1 and "null" in msg
    bad = (C.c_double * 3)(1.0, 0.0, 1.0)
    assert L.wslda_gradient_densities_static(p, p, p, 4, 32, bad, p, None, None) == 1
