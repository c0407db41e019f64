"""chem_integrate_noalloc (include/chem.h) against the allocating path chem_integrate_ex (-m gpu).

Who needs the entry point under test: a host program that cannot ask CUDA for device memory while it runs -- it gave the
whole card to its own arena at start-up, or it lives under a fixed memory budget, or it sits in a loop where an allocator
call (driver lock, possible device synchronisation) is not acceptable.  For such callers the library keeps the scratch of
the integration kernels (work-queue head, start order) in a fixed 4 MiB array inside libchem.so.  That array is shared by
all calls and keeps the last call's contents, so the property worth testing is that a call is right when it FOLLOWS another
one: every case below makes at least two calls in a row without synchronising in between, with different batch sizes, and
compares each with chem_integrate_ex on the same kernel id.  The two run the same kernels, so the comparison is bit for
bit; the north_star tolerance the parity tests use (|dy| <= 1e-9 + 1e-6 |y|) is asserted as well.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this add-on must not hide
the parity tests.  Nothing here depends on what ran before it in the process (the fixtures are this file's own).
"""
import numpy as np
import pytest

from paper_1607_03884_b200 import synth

pytestmark = pytest.mark.gpu

P = synth.P_ATM
RTOL, ATOL = synth.RTOL, synth.ATOL


@pytest.fixture(scope="module")
def env(mech_h2co, mech_gri):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1607_03884_b200 import binding
    return {"torch": torch, "binding": binding, "desc": {"h2co": mech_h2co, "gri": mech_gri},
            "mech": {"h2co": binding.chem_mech_load(mech_h2co), "gri": binding.chem_mech_load(mech_gri)}}


def _batch(env, kind, n, seed, dist="ignition"):
    return env["torch"].from_numpy(synth.make_states(env["desc"][kind], n, dist, seed)).cuda()


def _reference(env, kind, y0, t_end, kernel):
    """the existing (allocating) path on the same kernel id"""
    b = env["binding"]
    y, st = b.chem_integrate_ex(env["mech"][kind], P, t_end, RTOL, ATOL, y0, kernel=kernel)
    assert b.chem_last_kernel(env["mech"][kind]) == kernel
    return y, st


def _fresh_outputs(env, y0):
    """caller-owned outputs, poisoned so that a state the kernel never wrote is seen"""
    torch = env["torch"]
    y = torch.full_like(y0, float("nan"))
    st = torch.full((y0.shape[0], 48), 0xEE, dtype=torch.uint8, device=y0.device)
    return y, st


def _assert_same(env, got, ref):
    torch = env["torch"]
    (y, st), (y_ref, st_ref) = got, ref
    assert not torch.isnan(y).any(), "a state was not written"
    yn, rn = y.cpu().numpy(), y_ref.cpu().numpy()
    assert np.all(np.abs(yn - rn) <= 1e-9 + 1e-6 * np.abs(rn))          # the tolerance of the parity tests
    assert torch.equal(y, y_ref)                                         # and in fact the same bits
    a, b = env["binding"].stats_to_numpy(st), env["binding"].stats_to_numpy(st_ref)
    for f in ("status", "nstep", "naccpt", "nrejct", "nfcn", "njac", "ndec", "nsol", "nnewt_fail", "h_last"):
        assert np.array_equal(a[f], b[f]), f


@pytest.mark.parametrize("kind,kernel,n1,n2,t_end", [("h2co", 2, 3001, 1777, 1e-5), ("h2co", 1, 1500, 700, 1e-5),
                                                    ("gri", 1, 67, 40, 1e-6)])
def test_noalloc_matches_allocating_path_on_calls_in_a_row(kind, kernel, n1, n2, t_end, env):
    """Three calls back to back on one stream, no synchronisation between them: a plain one, a shorter one that also asks
    for cost ordering (stale queue head far past its n, stale order entries behind its own), and the first again."""
    b, torch = env["binding"], env["torch"]
    m = env["mech"][kind]
    ya, yb = _batch(env, kind, n1, 301), _batch(env, kind, n2, 302, "uniform")
    ref_a, ref_b = _reference(env, kind, ya, t_end, kernel), _reference(env, kind, yb, t_end, kernel)
    cost = torch.from_numpy(b.stats_to_numpy(ref_b[1])["nstep"].copy()).cuda()
    out1, out2, out3 = _fresh_outputs(env, ya), _fresh_outputs(env, yb), _fresh_outputs(env, ya)
    torch.cuda.synchronize()
    launches = b.chem_launch_count()
    b.chem_integrate_noalloc(m, P, t_end, RTOL, ATOL, ya, out1[0], out1[1], kernel=kernel)
    assert b.chem_last_kernel(m) == kernel
    b.chem_integrate_noalloc(m, P, t_end, RTOL, ATOL, yb, out2[0], out2[1], kernel=kernel, reorder=1, cost_hint=cost)
    b.chem_integrate_noalloc(m, P, t_end, RTOL, ATOL, ya, out3[0], out3[1], kernel=kernel)
    assert b.chem_launch_count() - launches == 1 + 4 + 1        # the ordered call adds three small kernels
    torch.cuda.synchronize()
    _assert_same(env, out1, ref_a)
    _assert_same(env, out2, ref_b)
    _assert_same(env, out3, ref_a)


def test_noalloc_auto_kernel_options_and_in_place(env):
    """kernel = 0 takes the warp-per-state kernel for the small mechanism and the group kernel for the large one; per-state
    pressure and the other options pass through; y_out may be y_in; stats may be omitted"""
    b, torch = env["binding"], env["torch"]
    y0 = _batch(env, "h2co", 999, 303)
    Ps = torch.from_numpy(P * (0.5 + np.random.default_rng(5).random(999))).cuda()
    y_ref, _ = b.chem_integrate_ex(env["mech"]["h2co"], P, 1e-5, RTOL, ATOL, y0, kernel=2, P_per_state=Ps, newton_max=5)
    y = y0.clone()
    for _ in range(2):                       # second pass integrates the first pass's result: only the first is compared
        got, st = b.chem_integrate_noalloc(env["mech"]["h2co"], P, 1e-5, RTOL, ATOL, y, y, P_per_state=Ps, newton_max=5)
        assert st is None and b.chem_last_kernel(env["mech"]["h2co"]) == 2
        if _ == 0:
            assert torch.equal(got, y_ref)
    yg = _batch(env, "gri", 33, 304)
    out = _fresh_outputs(env, yg)
    b.chem_integrate_noalloc(env["mech"]["gri"], P, 1e-6, RTOL, ATOL, yg, out[0], out[1])
    assert b.chem_last_kernel(env["mech"]["gri"]) == 1
    _assert_same(env, out, _reference(env, "gri", yg, 1e-6, 1))
    empty = torch.empty((0, 13), dtype=torch.float64, device="cuda")
    b.chem_integrate_noalloc(env["mech"]["h2co"], P, 1e-6, RTOL, ATOL, empty, empty.clone())


def test_noalloc_rejects_what_the_fixed_array_cannot_hold(env):
    """more states than the array has order slots, and the thread-per-state kernel (277 MB workspace): a clear error and no
    launch; the next valid call is unaffected; exactly the maximum is accepted"""
    b, torch = env["binding"], env["torch"]
    m = env["mech"]["h2co"]
    n_max = b.NOALLOC_MAX_STATES
    small = _batch(env, "h2co", 64, 305, "uniform")
    big = small.repeat((n_max + 1 + 63) // 64, 1)[: n_max + 1].contiguous()
    out = torch.full_like(big, float("nan"))
    launches = b.chem_launch_count()
    with pytest.raises(b.ChemError, match="CHEM_NOALLOC_MAX_STATES"):
        b.chem_integrate_noalloc(m, P, 1e-6, RTOL, ATOL, big, out)
    with pytest.raises(b.ChemError, match="thread-per-state"):
        b.chem_integrate_noalloc(m, P, 1e-6, RTOL, ATOL, small, out[:64], kernel=3)
    assert b.chem_launch_count() == launches
    torch.cuda.synchronize()
    assert torch.isnan(out).all()
    # exactly the maximum, with ordering (every order slot in use): all states written, copies of one state agree
    cost = (torch.arange(n_max, device="cuda", dtype=torch.int32) * 7) % 1500       # classes 0..1023 and the clamp above
    b.chem_integrate_noalloc(m, P, 1e-6, RTOL, ATOL, big[:n_max], out[:n_max], reorder=1, cost_hint=cost)
    torch.cuda.synchronize()
    ref, _ = b.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, small, kernel=2)
    assert not torch.isnan(out[:n_max]).any()
    assert torch.equal(out[:n_max].view(-1, 64, 13), ref.unsqueeze(0).expand(n_max // 64, 64, 13))
