"""Parity of the CUDA path against the CPU oracle, element by element, through the C ABI (-m gpu)."""
import numpy as np
import pytest

from paper_1607_03884_b200 import synth

pytestmark = pytest.mark.gpu

P = synth.P_ATM
RTOL, ATOL = synth.RTOL, synth.ATOL


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def gpu_mechs(torch_cuda, mech_h2co, mech_gri):
    from paper_1607_03884_b200 import binding
    return {"h2co": binding.chem_mech_load(mech_h2co), "gri": binding.chem_mech_load(mech_gri)}


@pytest.fixture(scope="module")
def orc_mechs(mech_h2co, mech_gri):
    from oracle import oracle as orc
    return {"h2co": orc.Mechanism(mech_h2co), "gri": orc.Mechanism(mech_gri)}


def descs(request):
    return {"h2co": request.getfixturevalue("mech_h2co"), "gri": request.getfixturevalue("mech_gri")}


@pytest.mark.parametrize("kind,n", [("h2co", 203), ("gri", 67)])
def test_rhs_matches_oracle(kind, n, torch_cuda, gpu_mechs, orc_mechs, request):
    """1e-10 x the per-state magnitude of the species source terms (1e-11 x the batch maximum); the
    temperature equation against |f_T| + 1e5 x that magnitude"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y = np.concatenate([synth.make_states(mech, n // 2, "uniform", 11), synth.make_states(mech, n - n // 2, "ignition", 12)])
    f = binding.chem_rhs(gpu_mechs[kind], P, torch.from_numpy(y).cuda()).cpu().numpy()
    ref = orc_mechs[kind].rhs(P, y)
    # scale: rates of individual reactions can cancel; use the per-state magnitude of the species source terms
    scale = np.abs(ref[:, 1:]).max(axis=1, keepdims=True) + 1e-300
    assert np.abs(f[:, 1:] - ref[:, 1:]).max() <= 1e-11 * scale.max()
    assert np.all(np.abs(f[:, 1:] - ref[:, 1:]) <= 1e-10 * scale)
    tscale = np.abs(ref[:, :1]) + scale * 1e5
    assert np.all(np.abs(f[:, :1] - ref[:, :1]) <= 1e-10 * tscale)


@pytest.mark.parametrize("kind,n", [("h2co", 101), ("gri", 37)])
def test_jacobian_matches_oracle(kind, n, torch_cuda, gpu_mechs, orc_mechs, request):
    """1e-9 x the column maximum of J (the two sides use different but equivalent formulations)"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y = np.concatenate([synth.make_states(mech, n // 2, "uniform", 21), synth.make_states(mech, n - n // 2, "ignition", 22)])
    J = binding.chem_jacobian(gpu_mechs[kind], P, torch.from_numpy(y).cuda()).cpu().numpy()
    ref = orc_mechs[kind].jacobian(P, y)
    col = np.abs(ref).max(axis=1, keepdims=True) + 1e-300
    assert np.all(np.abs(J - ref) <= 1e-9 * col)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [1, 2, 5, 13, 16, 17, 32, 33, 53, 64, 70])    # n <= 16: warp path routines; <= 64: lu2_pair + solves of the group kernels; above: generic LU
def test_lu_solve_matches_oracle(n, cplx, torch_cuda):
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    rng = np.random.default_rng(n + 100 * cplx)
    batch = 37
    A = rng.standard_normal((batch, n, n)) + (1j * rng.standard_normal((batch, n, n)) if cplx else 0)
    b = rng.standard_normal((batch, n)) + (1j * rng.standard_normal((batch, n)) if cplx else 0)
    A[-1] = 0.0                                      # singular system: info != 0
    x, info = binding.chem_lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
    x, info = x.cpu().numpy(), info.cpu().numpy()
    assert info[-1] != 0 and np.all(info[:-1] == 0)
    for s in range(batch - 1):
        if cplx:
            LU, ip, ier = orc.lu_complex(A[s])
            ref = orc.lu_solve_complex(LU, ip, b[s])
        else:
            LU, ip, ier = orc.lu_real(A[s])
            ref = orc.lu_solve_real(LU, ip, b[s])
        assert np.allclose(x[s], ref, rtol=1e-9, atol=1e-11 * np.abs(ref).max())


@pytest.mark.parametrize("n", [13, 16, 40, 53])
def test_lu_solve_stiff_newton_matrices(n, torch_cuda):
    """Matrices of the shape the integrator factors, gamma/h I - J and (alpha + i beta)/h I - J with a stiff J
    (eigenvalues spread over 12 decades): the residual of the device solve must be at the level of a backward-stable
    solve of a system with this condition number (the warp path applies an explicit inverse)."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    rng = np.random.default_rng(7 + n)
    batch = 24
    for cplx in (False, True):
        A = np.empty((batch, n, n), dtype=complex if cplx else float)
        conds = []
        for s in range(batch):
            V = rng.standard_normal((n, n))
            lam = -10.0 ** rng.uniform(-2, 10, n)
            J = V @ np.diag(lam) @ np.linalg.inv(V)
            fac = (3.6378 + (0.0 if not cplx else 3.0j)) / 10.0 ** rng.uniform(-8, -4)
            A[s] = fac * np.eye(n) - J
            conds.append(np.linalg.cond(A[s]))
        b = rng.standard_normal((batch, n)) + (1j * rng.standard_normal((batch, n)) if cplx else 0)
        x, info = binding.chem_lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x, info = x.cpu().numpy(), info.cpu().numpy()
        assert np.all(info == 0)
        for s in range(batch):
            ref = np.linalg.solve(A[s], b[s])
            err = np.abs(x[s] - ref).max() / np.abs(ref).max()
            assert err <= 1e-13 * conds[s] + 1e-12, (n, cplx, s, err, conds[s])


def compare_integration(y_gpu, st_gpu, y_ref, st_ref):
    """north_star bar: |dy| <= 1e-9 + 1e-6 |y_oracle| per component; accepted-step counts identical on >= 99 %"""
    assert np.all(st_gpu["status"] == st_ref["status"])
    same = (st_gpu["naccpt"] == st_ref["naccpt"])
    assert same.mean() >= 0.99, same.mean()
    tol = 1e-9 + 1e-6 * np.abs(y_ref)
    bad = np.abs(y_gpu - y_ref) > tol
    assert not bad.any(), (np.argwhere(bad)[:5], np.abs(y_gpu - y_ref).max())


CASES = [("h2co", "uniform", 1e-6, 4096), ("h2co", "ignition", 1e-4, 1037), ("gri", "uniform", 1e-6, 301),
         ("gri", "ignition", 1e-4, 157)]


@pytest.mark.parametrize("kind,dist,t_end,n", CASES)
def test_integrate_matches_oracle(kind, dist, t_end, n, torch_cuda, gpu_mechs, orc_mechs, request):
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y0 = synth.make_states(mech, n, dist, synth.STATE_SEED)
    y_ref, st_ref, _ = orc_mechs[kind].integrate(y0, P, t_end, RTOL, ATOL)
    # kernel 1 = shared-memory groups, 2 = warp per state, 3 = thread per state (2, 3: h2co only), 0 = auto
    for kernel in ((1, 2, 3, 0) if kind == "h2co" else (1, 0)):
        y_dev, st = binding.chem_integrate_ex(gpu_mechs[kind], P, t_end, RTOL, ATOL, torch.from_numpy(y0).cuda(),
                                              kernel=kernel)
        torch.cuda.synchronize()
        compare_integration(y_dev.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)
    # the plain entry point and the host-buffer entry point give the same bits
    y2 = binding.chem_integrate(gpu_mechs[kind], P, t_end, RTOL, ATOL, torch.from_numpy(y0).cuda())
    assert torch.equal(y2, y_dev)
    y3 = binding.chem_integrate_host(gpu_mechs[kind], P, t_end, RTOL, ATOL, y0)
    assert np.array_equal(y3, y_dev.cpu().numpy())


def test_edge_cases(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    m = gpu_mechs["h2co"]
    empty = torch.empty((0, 13), dtype=torch.float64, device="cuda")
    assert binding.chem_integrate(m, P, 1e-6, RTOL, ATOL, empty).shape == (0, 13)
    y0 = synth.make_states(mech_h2co, 5, "uniform", 1)
    y0[2, 3] = np.nan
    y, st = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, torch.from_numpy(y0).cuda())
    st = binding.stats_to_numpy(st)
    assert st["status"][2] == -4 and np.all(st["status"][[0, 1, 3, 4]] == 0)      # one bad state does not affect others
    y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0, P, 1e-6, RTOL, ATOL)
    assert st_ref["status"][2] == -4
    ok = [0, 1, 3, 4]
    assert np.all(np.abs(y.cpu().numpy()[ok] - y_ref[ok]) <= 1e-9 + 1e-6 * np.abs(y_ref[ok]))
    # max_steps limit reported as -1 on both sides
    y0 = synth.make_states(mech_h2co, 64, "ignition", 2)
    _, st = binding.chem_integrate_ex(m, P, 1e-4, RTOL, ATOL, torch.from_numpy(y0).cuda(), max_steps=3)
    _, st_ref, _ = orc_mechs["h2co"].integrate(y0, P, 1e-4, RTOL, ATOL, max_steps=3)
    assert np.array_equal(binding.stats_to_numpy(st)["status"], st_ref["status"])
    with pytest.raises(binding.ChemError):
        binding.chem_integrate(m, P, -1.0, RTOL, ATOL, torch.from_numpy(y0).cuda())


def test_full_size_config1_sampled_against_oracle(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    """BASELINE.json configs[1] at full size (1,048,576 states) in the launch configuration bench.py times (plain
    chem_integrate, auto kernel): a random sample of states is recomputed by the oracle one by one; properties that
    hold at any size are checked on ALL states."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    y0 = synth.make_states(mech_h2co, cfg["n_states"], cfg["dist"], synth.STATE_SEED)
    y_dev = torch.from_numpy(y0).cuda()
    y1 = binding.chem_integrate(gpu_mechs["h2co"], P, cfg["t_end"], RTOL, ATOL, y_dev).cpu().numpy()
    assert binding.chem_last_kernel(gpu_mechs["h2co"]) == 3     # the headline runs on the thread-per-state kernel
    assert np.all(np.isfinite(y1))
    # all states: element mass fractions are linear invariants of the method; mass fractions stay in [-atol-ish, 1]
    W = mech_h2co["mol_weight"]
    comp = mech_h2co["elem_comp"].astype(np.float64)

    def elem(y):
        Y = np.concatenate([y[:, 1:], 1.0 - y[:, 1:].sum(axis=1, keepdims=True)], axis=1)
        return (Y / W) @ comp
    assert np.abs(elem(y1) - elem(y0)).max() < 1e-12
    assert y1[:, 1:].min() > -1e-7 and y1[:, 1:].max() < 1.0 + 1e-9
    assert np.all(y1[:, 0] > 500.0) and np.all(y1[:, 0] < 4000.0)
    # sample: 2048 random states + the ragged tail of the last CTA
    rng = np.random.default_rng(123)
    idx = np.unique(np.concatenate([rng.choice(cfg["n_states"], 2048, replace=False), np.arange(cfg["n_states"] - 9, cfg["n_states"])]))
    y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0[idx], P, cfg["t_end"], RTOL, ATOL)
    assert np.all(st_ref["status"] == 0)
    assert np.all(np.abs(y1[idx] - y_ref) <= 1e-9 + 1e-6 * np.abs(y_ref))
    # statistics of the same launch configuration with the counters on
    _, st = binding.chem_integrate_ex(gpu_mechs["h2co"], P, cfg["t_end"], RTOL, ATOL, y_dev)
    st = binding.stats_to_numpy(st)
    assert np.all(st["status"] == 0)
    assert (st["naccpt"][idx] == st_ref["naccpt"]).mean() >= 0.99
    assert (st["nstep"][idx] == st_ref["nstep"]).mean() >= 0.99


@pytest.mark.parametrize("ci,n_sample", [(2, 1024), (3, 128), (4, 96)])
def test_full_size_other_configs_sampled_against_oracle(ci, n_sample, torch_cuda, gpu_mechs, orc_mechs, request):
    """BASELINE.json configs[2..4] at FULL size through the plain entry point; a random sample (plus the ragged tail) is
    recomputed by the oracle one by one; element conservation is checked on every state"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    cfg = synth.CONFIGS[ci]
    mech = descs(request)[cfg["kind"]]
    y0 = synth.make_states(mech, cfg["n_states"], cfg["dist"], synth.STATE_SEED)
    y1 = binding.chem_integrate(gpu_mechs[cfg["kind"]], P, cfg["t_end"], RTOL, ATOL, torch.from_numpy(y0).cuda()).cpu().numpy()
    assert np.all(np.isfinite(y1))
    W, comp = mech["mol_weight"], mech["elem_comp"].astype(np.float64)

    def elem(y):
        Y = np.concatenate([y[:, 1:], 1.0 - y[:, 1:].sum(axis=1, keepdims=True)], axis=1)
        return (Y / W) @ comp
    assert np.abs(elem(y1) - elem(y0)).max() < 1e-11
    rng = np.random.default_rng(1000 + ci)
    idx = np.unique(np.concatenate([rng.choice(cfg["n_states"], n_sample, replace=False),
                                    np.arange(cfg["n_states"] - 5, cfg["n_states"])]))
    y_ref, st_ref, _ = orc_mechs[cfg["kind"]].integrate(y0[idx], P, cfg["t_end"], RTOL, ATOL)
    assert np.all(st_ref["status"] == 0)
    assert np.all(np.abs(y1[idx] - y_ref) <= 1e-9 + 1e-6 * np.abs(y_ref))
    # step counts of the sampled states (the same states through chem_integrate_ex; results do not depend on the batch)
    y_s, st = binding.chem_integrate_ex(gpu_mechs[cfg["kind"]], P, cfg["t_end"], RTOL, ATOL, torch.from_numpy(y0[idx].copy()).cuda(),
                                        kernel=binding.chem_last_kernel(gpu_mechs[cfg["kind"]]))   # the kernel auto chose for the full batch
    st = binding.stats_to_numpy(st)
    assert np.array_equal(y_s.cpu().numpy(), y1[idx])
    assert np.all(st["status"] == 0)
    assert (st["naccpt"] == st_ref["naccpt"]).mean() >= 0.99
    assert (st["nstep"] == st_ref["nstep"]).mean() >= 0.99


@pytest.mark.parametrize("kind,n", [("h2co", 5000), ("gri", 300)])
def test_cost_ordering_does_not_change_results(kind, n, torch_cuda, gpu_mechs, request):
    """chem_opts.reorder only changes WHEN a state is started: results are bit-identical"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y0 = torch.from_numpy(synth.make_states(mech, n, "ignition", 77)).cuda()
    y_a, st_a = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, y0)
    nstep = torch.from_numpy(binding.stats_to_numpy(st_a)["nstep"].copy()).cuda()
    y_b, st_b = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, y0, reorder=1, cost_hint=nstep)
    torch.cuda.synchronize()
    assert torch.equal(y_a, y_b)
    assert np.array_equal(binding.stats_to_numpy(st_a), binding.stats_to_numpy(st_b))


@pytest.mark.parametrize("kind,n", [("h2co", 20011), ("gri", 601)])
def test_results_are_reproducible_and_independent_of_the_batch(kind, n, torch_cuda, gpu_mechs, request):
    """Work-queue scheduling, the butterfly sums and the gather schedule are deterministic: the same state gives the same
    bits whatever else is in the batch, in every launch, through the device and the host entry point."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y0 = synth.make_states(mech, n, "ignition", 91)
    y_a, st_a = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, torch.from_numpy(y0).cuda())
    y_b, st_b = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, torch.from_numpy(y0).cuda())
    assert torch.equal(y_a, y_b)
    assert np.array_equal(binding.stats_to_numpy(st_a), binding.stats_to_numpy(st_b))
    perm = np.random.default_rng(5).permutation(n)[: n // 3]            # a shuffled third of the batch
    y_c, _ = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, torch.from_numpy(y0[perm].copy()).cuda())
    assert np.array_equal(y_c.cpu().numpy(), y_a.cpu().numpy()[perm])
    y_h = binding.chem_integrate_host(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, y0)
    assert np.array_equal(y_h, y_a.cpu().numpy())


@pytest.mark.parametrize("kind,n,kernels", [("h2co", 1500, (1, 2, 3)), ("gri", 300, (0,))])
def test_finite_difference_jacobian_matches_oracle(kind, n, kernels, torch_cuda, gpu_mechs, orc_mechs, request):
    """PAPER.md L82 / Sec. 3.4: the CVODE-style FD Jacobian variant (R13) against the oracle's"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y0 = synth.make_states(mech, n, "ignition", 31)
    y_ref, st_ref, _ = orc_mechs[kind].integrate(y0, P, 1e-5, RTOL, ATOL, fd_jacobian=1)
    for kernel in kernels:
        y, st = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-5, RTOL, ATOL, torch.from_numpy(y0).cuda(), kernel=kernel,
                                          fd_jacobian=1)
        torch.cuda.synchronize()
        st = binding.stats_to_numpy(st)
        y = y.cpu().numpy()
        # The difference quotient carries ~1e-8 relative rounding noise that differs between the two sides; a Newton
        # iteration more or less moves the result by the Newton tolerance.  Bar for this variant: identical status,
        # accepted-step counts identical on >= 97 %, the north_star tolerance on >= 97 % of the states, and every
        # state within 100 units of the paper's error metric (Eq. 1) of the oracle.
        assert np.all(st["status"] == st_ref["status"])
        assert (st["naccpt"] == st_ref["naccpt"]).mean() >= 0.97
        ok = np.all(np.abs(y - y_ref) <= 1e-9 + 1e-6 * np.abs(y_ref), axis=1)
        assert ok.mean() >= 0.97, ok.mean()
        from oracle import oracle as orc
        Emax, _ = orc.error_metric(y, y_ref, RTOL, ATOL)
        assert Emax < 100.0, Emax
        assert (st["nfcn"] == st_ref["nfcn"]).mean() >= 0.85
        assert (st["njac"] == st_ref["njac"]).mean() >= 0.97


@pytest.mark.parametrize("kind,n,kernels", [("h2co", 600, (1, 2, 3)), ("gri", 60, (0,))])
def test_fixed_step_mode_matches_oracle(kind, n, kernels, torch_cuda, gpu_mechs, orc_mechs, request):
    """solver-verification mode of PAPER.md L106-L128: a given number of equal internal steps, no error control"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = descs(request)[kind]
    y0 = synth.make_states(mech, n, "uniform", 41)
    for steps in (1, 4, 16):
        y_ref, st_ref, _ = orc_mechs[kind].integrate(y0, P, 1e-6, RTOL, ATOL, fixed_steps=steps)
        for kernel in kernels:
            y, st = binding.chem_integrate_ex(gpu_mechs[kind], P, 1e-6, RTOL, ATOL, torch.from_numpy(y0).cuda(),
                                              kernel=kernel, fixed_steps=steps)
            st = binding.stats_to_numpy(st)
            # one giant step may blow up: such a state ends with status -5 on both sides (R14)
            assert np.array_equal(st["status"], st_ref["status"]) and np.all(np.isin(st_ref["status"], (0, -5)))
            ok0 = st_ref["status"] == 0
            assert ok0.mean() > 0.9
            assert np.array_equal(st["naccpt"], st_ref["naccpt"]) and np.all(st["naccpt"][ok0] == steps)
            y = y.cpu().numpy()
            assert np.all(np.isfinite(y[ok0]))
            ok = np.all(np.abs(y[ok0] - y_ref[ok0]) <= 1e-9 + 1e-6 * np.abs(y_ref[ok0]), axis=1)
            assert ok.all(), (steps, kernel, ok.mean())


def test_fixed_step_convergence_like_fig2(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    """Fig. 2 of the paper on synthetic states: |E| (Eq. 2) against a tight-tolerance truth falls steeply with the
    number of internal steps (about four orders of magnitude from 1 to 10 steps for Radau IIA)"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    y0 = synth.make_states(mech_h2co, 1000, "uniform", 43)
    truth, st_t, _ = orc_mechs["h2co"].integrate(y0, P, 1e-6, 1e-12, 1e-18)
    assert np.all(st_t["status"] == 0)
    E = []
    for steps in (1, 10, 100):
        y, _ = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-6, RTOL, ATOL, torch.from_numpy(y0).cuda(), fixed_steps=steps)
        y = y.cpu().numpy()
        fin = np.all(np.isfinite(y), axis=1)
        Emax, Ei = orc.error_metric(y[fin], truth[fin], RTOL, ATOL)
        E.append(Emax)
    # oracle values on these states: |E| = 3.7e4, 0.46, 0.22 for 1, 10, 100 steps (then the Newton tolerance floor)
    assert E[1] < 1e-3 * E[0] and E[2] < 10.0 * E[1] and E[2] < 1.0, E


def _tiny(rxn_type, **kw):
    from tests.test_oracle_chem import tiny_mech
    nasa = np.array([[3.5, 1e-3, 0, 0, 0, 2000.0, 4.0], [4.0, 5e-4, 1e-7, 0, 0, -3000.0, 6.0],
                     [4.5, 2e-3, -2e-7, 0, 0, -9000.0, 5.0], [2.5, 0, 0, 0, 0, 0.0, 5.0]])
    return tiny_mech(rxn_type=rxn_type, A=1.0e9, b=0.7, Ea=8000.0, low=(3.0e13, -0.5, 3000.0),
                     troe=(0.6, 150.0, 1800.0, 4000.0), eff=((0, 3.0), (2, 0.4)), reac=((0, 1), (1, 1)), prod=((2, 1),),
                     W=(10.0, 18.0, 28.0, 40.0), nasa=nasa, **kw)


@pytest.mark.parametrize("rxn_type", [0, 1, 2, 3])
def test_tiny_mechanisms_every_reaction_type(rxn_type, torch_cuda):
    """degenerate sizes (4 species, 1 reaction) and the Lindemann type, which the synthetic mechanisms do not contain:
    source term, Jacobian and integration through both kernels against the oracle"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = _tiny(rxn_type)
    gm, om = binding.chem_mech_load(mech), orc.Mechanism(mech)
    rng = np.random.default_rng(rxn_type)
    n = 70
    Y = rng.uniform(0.05, 0.4, (n, 4))
    Y /= Y.sum(axis=1, keepdims=True)
    y0 = np.concatenate([rng.uniform(900.0, 1900.0, (n, 1)), Y[:, :3]], axis=1)
    yd = torch.from_numpy(y0).cuda()
    f, f_ref = binding.chem_rhs(gm, P, yd).cpu().numpy(), om.rhs(P, y0)
    assert np.all(np.abs(f - f_ref) <= 1e-10 * np.abs(f_ref).max(axis=1, keepdims=True) + 1e-300)
    J, J_ref = binding.chem_jacobian(gm, P, yd).cpu().numpy(), om.jacobian(P, y0)
    assert np.all(np.abs(J - J_ref) <= 1e-9 * np.abs(J_ref).max(axis=1, keepdims=True) + 1e-300)
    y_ref, st_ref, _ = om.integrate(y0, P, 1e-3, RTOL, ATOL)
    for kernel in (1, 2, 3):
        y, st = binding.chem_integrate_ex(gm, P, 1e-3, RTOL, ATOL, yd, kernel=kernel)
        compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)


def test_mechanism_outside_the_fast_paths(torch_cuda, orc_mechs, mech_h2co):
    """species with different NASA switch temperatures: neither the warp path nor the exp-job source term applies, the
    reaction-by-reaction group kernel must give the same answers"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = dict(mech_h2co)
    mech["nasa_tmid"] = mech_h2co["nasa_tmid"].copy()
    mech["nasa_tmid"][3] = 1200.0
    gm, om = binding.chem_mech_load(mech), orc.Mechanism(mech)
    y0 = synth.make_states(mech_h2co, 700, "ignition", 51)
    with pytest.raises(binding.ChemError):
        binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, torch.from_numpy(y0).cuda(), kernel=2)
    y_ref, st_ref, _ = om.integrate(y0, P, 1e-5, RTOL, ATOL)
    y, st = binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, torch.from_numpy(y0).cuda())
    compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)


def test_single_state_and_per_state_pressure(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    y0 = synth.make_states(mech_h2co, 33, "uniform", 61)
    y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0[:1], P, 1e-6, RTOL, ATOL)
    y, st = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-6, RTOL, ATOL, torch.from_numpy(y0[:1]).cuda())
    compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)
    # per-state pressure: each state at its own P equals separate calls at that P
    Ps = np.linspace(0.5, 5.0, 33) * P
    y, _ = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-6, RTOL, ATOL, torch.from_numpy(y0).cuda(),
                                     P_per_state=torch.from_numpy(Ps).cuda())
    y = y.cpu().numpy()
    for s in (0, 16, 32):
        yr, _, _ = orc_mechs["h2co"].integrate(y0[s:s + 1], float(Ps[s]), 1e-6, RTOL, ATOL)
        assert np.all(np.abs(y[s] - yr[0]) <= 1e-9 + 1e-6 * np.abs(yr[0]))


def test_concurrent_launches_on_two_streams(torch_cuda, gpu_mechs, mech_h2co):
    """include/chem.h: calls on different streams may run concurrently with the same chem_mech (every launch has its own
    work-queue head and scratch).  Two different batches on two streams, interleaved several times, must give the bits
    of sequential runs -- for every kernel."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    m = gpu_mechs["h2co"]
    ya = torch.from_numpy(synth.make_states(mech_h2co, 30011, "ignition", 101)).cuda()
    yb = torch.from_numpy(synth.make_states(mech_h2co, 17003, "uniform", 102)).cuda()
    for kernel in (1, 2, 3):
        ref_a, sa = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, ya, kernel=kernel)
        ref_b, sb = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, yb, kernel=kernel)
        torch.cuda.synchronize()
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        outs = []
        for rep in range(4):
            oa, ta = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, ya, kernel=kernel, stream=s1)
            ob, tb = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, yb, kernel=kernel, stream=s2)
            outs.append((oa, ta, ob, tb))
        torch.cuda.synchronize()
        for oa, ta, ob, tb in outs:
            assert torch.equal(oa, ref_a) and torch.equal(ob, ref_b), kernel
            assert torch.equal(ta, sa) and torch.equal(tb, sb), kernel


def test_divergence_measure_matches_oracle_definition(torch_cuda, gpu_mechs, mech_h2co):
    """PAPER.md Eq. 3 (L190): the product-side D (paper_1607_03884_b200/diagnostics.py, reported by bench.py) against the
    oracle's routine on the SAME per-state step counters taken from the GPU run; Eq. 1-2 likewise"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding, diagnostics
    torch = torch_cuda
    y0 = synth.make_states(mech_h2co, 4099, "ignition", 111)           # ragged: 128 complete warps + 3 states
    y, st = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-4, RTOL, ATOL, torch.from_numpy(y0).cuda())
    st = binding.stats_to_numpy(st)
    D = diagnostics.divergence(st["nstep"])
    D_ref = orc.divergence(st["nstep"])
    assert D.shape == D_ref.shape == (128,)
    assert np.array_equal(D, D_ref)
    assert 0.0 <= D.min() and D.max() < 1.0 and D.mean() > 0.1            # dt = 1e-4: visibly divergent step counts
    summ = diagnostics.divergence_summary(st["nstep"])
    assert summ["warps"] == 128 and abs(sum(summ["hist"]) - 1.0) < 1e-3
    y = y.cpu().numpy()
    Emax, E = diagnostics.error_metric(y, y0, RTOL, ATOL)
    Emax_ref, E_ref = orc.error_metric(y, y0, RTOL, ATOL)
    assert np.allclose(E, E_ref, rtol=1e-13, atol=0.0) and np.isclose(Emax, Emax_ref, rtol=1e-13)


def _backward_error(A, x, b):
    """componentwise backward error of x for A x = b (Oettli-Prager): max_i |A x - b|_i / (|A| |x| + |b|)_i"""
    return (np.abs(A @ x - b) / (np.abs(A) @ np.abs(x) + np.abs(b))).max()


@pytest.mark.parametrize("ci", [1, 2])
def test_linear_algebra_on_the_matrices_the_integrator_forms(ci, torch_cuda, gpu_mechs, mech_h2co):
    """the device solve (n = 13: the warp path's pivoted Gauss-Jordan inverse) on the
    WORST-conditioned matrices the integrator actually forms: E1 = gamma/h I - J and E2 = (alpha + i beta)/h I - J rebuilt
    from chem_jacobian at the states of the config with h = h_last of their integration, ranked by condition number.
    The bar is a componentwise BACKWARD error in units of u (DESIGN.md 8 states the measured worst case)."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    cfg = synth.CONFIGS[ci]
    m = gpu_mechs["h2co"]
    y0 = synth.make_states(mech_h2co, 8192, cfg["dist"], synth.STATE_SEED)
    yd = torch.from_numpy(y0).cuda()
    y1, st = binding.chem_integrate_ex(m, P, cfg["t_end"], RTOL, ATOL, yd)
    h = binding.stats_to_numpy(st)["h_last"]
    J = np.concatenate([binding.chem_jacobian(m, P, yd).cpu().numpy(), binding.chem_jacobian(m, P, y1).cpu().numpy()])
    h = np.concatenate([h, h])
    U1, AL, BE = 3.637834252744495732, 2.681082873627752134, 3.050430199247410569
    eye = np.eye(13)
    E1 = (U1 / h)[:, None, None] * eye - J
    E2 = ((AL + 1j * BE) / h)[:, None, None] * eye - J
    cond = np.linalg.cond(E1)
    worst = np.argsort(cond)[-256:]
    rng = np.random.default_rng(5 + ci)
    u = 2.0 ** -53
    worst_eta = 0.0
    for A in (E1[worst], E2[worst]):
        b = rng.standard_normal((256, 13)) + (1j * rng.standard_normal((256, 13)) if np.iscomplexobj(A) else 0)
        x, info = binding.chem_lu_solve(torch.from_numpy(np.ascontiguousarray(A)).cuda(), torch.from_numpy(b).cuda())
        x, info = x.cpu().numpy(), info.cpu().numpy()
        assert np.all(info == 0)
        eta = max(_backward_error(A[s], x[s], b[s]) for s in range(256))
        eta_ref = max(_backward_error(A[s], np.linalg.solve(A[s], b[s]), b[s]) for s in range(256))
        worst_eta = max(worst_eta, eta)
        print(f"config {ci} {'complex' if np.iscomplexobj(A) else 'real'}: cond up to {cond[worst].max():.2e}, "
              f"backward error device {eta / u:.3g} u, LAPACK {eta_ref / u:.3g} u")
    assert worst_eta <= 1024 * u, worst_eta / u        # measured: 211 u (LAPACK on the same matrices: 61 u)


def test_small_mechanism_kernels_at_their_size_limit(torch_cuda):
    """16 species / 28 reactions (synth kind "lim16"): the largest shape the warp-per-state and thread-per-state kernels
    are compiled for; the thread-per-state kernel runs its compile-time-N instantiation <16, 4> here, and the
    warp-per-state kernel must decline (its CTA does not fit in shared memory) instead of failing in auto"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = synth.make_mechanism("lim16", 7)
    gm, om = binding.chem_mech_load(mech), orc.Mechanism(mech)
    y0 = synth.make_states(mech, 1500, "ignition", 3)
    yd = torch.from_numpy(y0).cuda()
    f, f_ref = binding.chem_rhs(gm, P, yd).cpu().numpy(), om.rhs(P, y0)
    scale = np.abs(f_ref[:, 1:]).max(axis=1, keepdims=True) + 1e-300
    assert np.all(np.abs(f[:, 1:] - f_ref[:, 1:]) <= 1e-10 * scale)
    y_ref, st_ref, _ = om.integrate(y0, P, 1e-5, RTOL, ATOL)
    with pytest.raises(binding.ChemError):      # one 640-thread CTA of the warp-per-state kernel does not fit at N = 16
        binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, yd, kernel=2)
    for kernel in (1, 3, 0):
        y, st = binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, yd, kernel=kernel)
        compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)
    assert binding.chem_last_kernel(gm) == 1    # auto: small batch, no warp kernel -> group kernel


def test_newton_iterates_with_nonpositive_temperature(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    """a huge first step (h0 = t_end = 1e-2 s on ignition states) drives Newton iterates to T <= 0; log T is
    then NaN on every path (libm in the oracle and the generic source term, an explicit guard around the compact log in
    the stage-batched ones), the step is rejected (R11) and every kernel takes the oracle's step sequence."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    y0 = synth.make_states(mech_h2co, 2000, "ignition", 121)
    y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0, P, 1e-2, RTOL, ATOL)
    assert st_ref["nnewt_fail"].sum() > 500                 # the case does exercise failed Newton iterations
    for kernel in (1, 2, 3):
        y, st = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-2, RTOL, ATOL, torch.from_numpy(y0).cuda(), kernel=kernel)
        compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)


def test_fixed_step_that_cannot_be_taken_ends_the_state(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    """DESIGN.md R14: in fixed-step mode a step whose Newton iterate or error estimate is not finite (or whose
    matrix is singular) ends the state with status -5 instead of silently halving the step; one giant step of 1e-2 s on
    ignition states does that to about a third of them, identically in the oracle and in every kernel"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    y0 = synth.make_states(mech_h2co, 600, "ignition", 131)
    for steps in (1, 2):
        y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0, P, 1e-2, RTOL, ATOL, fixed_steps=steps)
        assert (st_ref["status"] == -5).sum() > 100 and (st_ref["status"] == 0).sum() > 100
        for kernel in (1, 2, 3):
            y, st = binding.chem_integrate_ex(gpu_mechs["h2co"], P, 1e-2, RTOL, ATOL, torch.from_numpy(y0).cuda(),
                                              kernel=kernel, fixed_steps=steps)
            st = binding.stats_to_numpy(st)
            # whether a wildly diverging iterate of such a step overflows within 7 iterations is marginal between two
            # implementations of the arithmetic: statuses must agree on >= 97 % of the states, results where both finish
            same = st["status"] == st_ref["status"]
            print(f"fixed_steps={steps} kernel={kernel}: status agreement {same.mean():.4f}")
            assert np.all(np.isin(st["status"], (0, -5))) and same.mean() >= 0.97, (steps, kernel, same.mean())
            ok0 = (st_ref["status"] == 0) & (st["status"] == 0)
            assert np.all(st["naccpt"][ok0] == steps) and np.all(st_ref["naccpt"][ok0] == steps)
            y = y.cpu().numpy()
            good = np.all(np.abs(y[ok0] - y_ref[ok0]) <= 1e-9 + 1e-6 * np.abs(y_ref[ok0]), axis=1)
            assert good.mean() >= 0.97, (steps, kernel, good.mean())


@pytest.mark.parametrize("n", [1, 2, 5, 8, 9, 10, 11, 12, 13, 14, 15, 16])
def test_thread_per_state_linear_algebra_matches_lapack(n, torch_cuda, gpu_mechs, mech_h2co):
    """PAPER.md L86 (LU factorisation): the thread-per-state kernel's LU + triangular solves -- lu_pair_t<n> / solve3_t<n>
    for every 8 <= n <= 16, the runtime-N forms below that: the hook dispatches through the same table as the integration
    kernel -- on E1 = fac1 I - J and E2 = (alphn + i betan) I - J against numpy / LAPACK: random matrices with heavy
    pivoting, stiff matrices of the integrator's shape (n = 13: the Jacobians of config 2 states), and a matrix without
    a pivot (info)."""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    rng = np.random.default_rng(300 + n)
    batch = 301                                              # several warps and a ragged tail
    J = rng.standard_normal((batch, n, n))
    fac1, alphn, betan = 3.6378e0, 2.6811e0, 3.0504e0        # h = 1: the shift does not dominate, pivots move
    if n == 13:
        y0 = synth.make_states(mech_h2co, 150, "ignition", 5)
        J[:150] = binding.chem_jacobian(gpu_mechs["h2co"], P, torch.from_numpy(y0).cuda()).cpu().numpy() * 1e-5   # h = 1e-5 s
    J[-1] = 0.0
    J[-1, 0, 0] = fac1                                       # fac1 I - J has a zero first column: no pivot
    b = rng.standard_normal((batch, 3, n))
    x, info = binding.chem_tps_radau_solve(torch.from_numpy(J).cuda(), fac1, alphn, betan, torch.from_numpy(b).cuda())
    x, info = x.cpu().numpy(), info.cpu().numpy()
    if n > 1:
        assert info[-1] != 0
    assert np.all(info[:-1] == 0)
    eye = np.eye(n)
    u = 2.0 ** -53
    worst, worst_ref = 0.0, 0.0
    for s in range(batch - 1):
        E1 = fac1 * eye - J[s]
        E2 = (alphn + 1j * betan) * eye - J[s]
        for A, rhs, sol in ((E1, b[s, 0], x[s, 0]), (E2, b[s, 1] + 1j * b[s, 2], x[s, 1] + 1j * x[s, 2])):
            ref = np.linalg.solve(A, rhs)
            cond = np.linalg.cond(A)
            assert np.abs(sol - ref).max() <= 1e-13 * cond * np.abs(ref).max() + 1e-300, (n, s, cond)
            worst = max(worst, _backward_error(A, sol, rhs) / u)
            worst_ref = max(worst_ref, _backward_error(A, ref, rhs) / u)
    print(f"n = {n}: componentwise backward error device {worst:.3g} u, LAPACK {worst_ref:.3g} u")
    assert worst <= 8.0 * worst_ref + 64.0, (worst, worst_ref)   # that of a pivoted LU solve on the same (badly scaled) matrices


def test_other_small_mechanism_sizes(torch_cuda):
    """a 9-species / 20-reaction hydrogen-oxygen sized shape (synth kind "h2_9"): the thread-per-state kernel has a
    compile-time-N instantiation for every 8 <= N <= 16 (13 is the one the BASELINE.json configs exercise); this is N = 9,
    and the warp-per-state and group kernels at a size other than the benchmark's"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = synth.make_mechanism("h2_9", 1)
    gm, om = binding.chem_mech_load(mech), orc.Mechanism(mech)
    y0 = synth.make_states(mech, 3000, "ignition", 3)
    yd = torch.from_numpy(y0).cuda()
    y_ref, st_ref, _ = om.integrate(y0, P, 1e-5, RTOL, ATOL)
    assert np.all(st_ref["status"] == 0)
    for kernel in (1, 2, 3):
        y, st = binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, yd, kernel=kernel)
        compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)


@pytest.mark.parametrize("n_sp", [8, 10, 11, 12, 14, 15])
def test_every_compile_time_size_of_the_thread_per_state_kernel(n_sp, torch_cuda):
    """integrate_tps_kernel<N, 4> for the N that no other test reaches (synth kinds "sz<N>"; 9, 13 and 16 run elsewhere):
    integration parity against the oracle, beside the group kernel on the same states"""
    from oracle import oracle as orc
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    mech = synth.make_mechanism(f"sz{n_sp}", 1)
    assert mech["n_species"] == n_sp
    gm, om = binding.chem_mech_load(mech), orc.Mechanism(mech)
    y0 = synth.make_states(mech, 1300, "ignition", 3)
    yd = torch.from_numpy(y0).cuda()
    y_ref, st_ref, _ = om.integrate(y0, P, 1e-5, RTOL, ATOL)
    assert np.all(st_ref["status"] == 0)
    for kernel in (3, 1):
        y, st = binding.chem_integrate_ex(gm, P, 1e-5, RTOL, ATOL, yd, kernel=kernel)
        assert binding.chem_last_kernel(gm) == kernel
        compare_integration(y.cpu().numpy(), binding.stats_to_numpy(st), y_ref, st_ref)


def test_host_entry_point_picks_one_kernel_for_the_whole_batch(torch_cuda, gpu_mechs, mech_h2co):
    """with kernel = 0 the choice depends on the batch size; the pageable path of chem_integrate_host splits
    the batch in two chunks and must still run the kernel the whole batch selects (400,000 states: thread per state; a
    200,000-state chunk alone would select warp per state), so that pinned and pageable buffers give the same bits"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    m = gpu_mechs["h2co"]
    y0 = synth.make_states(mech_h2co, 400_000, "uniform", 77)
    y_dev = binding.chem_integrate(m, P, 1e-6, RTOL, ATOL, torch.from_numpy(y0).cuda()).cpu().numpy()
    assert binding.chem_last_kernel(m) == 3
    y_pageable = binding.chem_integrate_host(m, P, 1e-6, RTOL, ATOL, y0)
    assert binding.chem_last_kernel(m) == 3
    pin_in = torch.from_numpy(y0).pin_memory()
    pin_out = torch.empty(pin_in.shape, dtype=torch.float64, pin_memory=True)
    binding.chem_integrate_host(m, P, 1e-6, RTOL, ATOL, pin_in.numpy(), pin_out.numpy())
    assert binding.chem_last_kernel(m) == 3
    assert np.array_equal(y_pageable, y_dev) and np.array_equal(pin_out.numpy(), y_dev)
    binding.chem_scratch_trim()                     # the pool gives its blocks back and the next launch still works
    y_again = binding.chem_integrate(m, P, 1e-6, RTOL, ATOL, torch.from_numpy(y0[:5000]).cuda(), ).cpu().numpy()
    assert y_again.shape == (5000, 13) and np.all(np.isfinite(y_again))


def test_library_stiffness_ordering_changes_no_bit(torch_cuda, gpu_mechs, mech_h2co, mech_gri):
    """chem_opts.reorder = 2 (the library's own estimate t_end ||f(y0) / scal||_rms) and the auto mode that
    switches it on for large thread-per-state launches only change the order in which states start: y and every counter
    are bit-identical to reorder = -1 (off) on all three kernels; the estimate needs a small mechanism"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    m = gpu_mechs["h2co"]
    y0 = synth.make_states(mech_h2co, 30011, "ignition", 93)
    y0[7, 2] = np.nan                                                     # a non-finite state gets key 0 and status -4
    yd = torch.from_numpy(y0).cuda()
    for kernel in (1, 2, 3):
        y_off, st_off = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, yd, kernel=kernel, reorder=-1)
        l0 = binding.chem_launch_count()
        y_est, st_est = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, yd, kernel=kernel, reorder=2)
        assert binding.chem_launch_count() - l0 > 2                       # estimate + sort + integration
        assert torch.equal(torch.nan_to_num(y_off, nan=-1.0), torch.nan_to_num(y_est, nan=-1.0)) and torch.equal(st_off, st_est)
        assert binding.stats_to_numpy(st_est)["status"][7] == -4
    big = torch.from_numpy(synth.make_states(mech_h2co, 320_000, "uniform", 94)).cuda()      # >= 8 x 37,888: auto orders
    y_off, st_off = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, big, reorder=-1)
    l0 = binding.chem_launch_count()
    y_auto, st_auto = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, big)
    assert binding.chem_last_kernel(m) == 3 and binding.chem_launch_count() - l0 > 2
    assert torch.equal(y_off, y_auto) and torch.equal(st_off, st_auto)
    yg = torch.from_numpy(synth.make_states(mech_gri, 16, "uniform", 95)).cuda()
    with pytest.raises(binding.ChemError, match="small mechanism"):
        binding.chem_integrate_ex(gpu_mechs["gri"], P, 1e-6, RTOL, ATOL, yg, reorder=2)
    with pytest.raises(binding.ChemError, match="reorder"):
        binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, yd, reorder=3)


def test_thread_per_state_kernel_options_and_reproducibility(torch_cuda, gpu_mechs, orc_mechs, mech_h2co):
    """the thread-per-state kernel (what auto takes for the full-size h2co configs) with the options and properties the
    other kernels are tested for: per-state pressure, cost ordering (bit-identical results), bit-reproducible results that
    do not depend on what else is in the batch or on how the lanes were refilled, exact zeros in the state"""
    from paper_1607_03884_b200 import binding
    torch = torch_cuda
    m = gpu_mechs["h2co"]
    y0 = synth.make_states(mech_h2co, 20011, "ignition", 91)
    y0[::97, 3] = 0.0                                                     # some exact zeros among the mass fractions
    yd = torch.from_numpy(y0).cuda()
    y_a, st_a = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, yd, kernel=3)
    y_b, st_b = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, yd, kernel=3)
    assert torch.equal(y_a, y_b) and torch.equal(st_a, st_b)
    sa = binding.stats_to_numpy(st_a)
    assert np.all(sa["status"] == 0)
    # a shuffled third of the batch: other neighbours in the warp, other refill pattern, same bits
    perm = np.random.default_rng(5).permutation(20011)[:6667]
    y_c, st_c = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, torch.from_numpy(y0[perm].copy()).cuda(), kernel=3)
    assert np.array_equal(y_c.cpu().numpy(), y_a.cpu().numpy()[perm])
    assert np.array_equal(binding.stats_to_numpy(st_c), sa[perm])
    # cost ordering only changes when a state starts
    nstep = torch.from_numpy(sa["nstep"].copy()).cuda()
    y_d, st_d = binding.chem_integrate_ex(m, P, 1e-5, RTOL, ATOL, yd, kernel=3, reorder=1, cost_hint=nstep)
    assert torch.equal(y_a, y_d) and torch.equal(st_a, st_d)
    # against the oracle on a sample (including states with zeros), and per-state pressure
    idx = np.r_[np.arange(0, 20011, 97)[:60], np.arange(1, 400, 7)]
    y_ref, st_ref, _ = orc_mechs["h2co"].integrate(y0[idx], P, 1e-5, RTOL, ATOL)
    compare_integration(y_a.cpu().numpy()[idx], sa[idx], y_ref, st_ref)
    Ps = np.linspace(0.5, 5.0, 20011) * P
    y_p, _ = binding.chem_integrate_ex(m, P, 1e-6, RTOL, ATOL, yd, kernel=3, P_per_state=torch.from_numpy(Ps).cuda())
    y_p = y_p.cpu().numpy()
    for s in (0, 9999, 20010):
        yr, _, _ = orc_mechs["h2co"].integrate(y0[s:s + 1], float(Ps[s]), 1e-6, RTOL, ATOL)
        assert np.all(np.abs(y_p[s] - yr[0]) <= 1e-9 + 1e-6 * np.abs(yr[0]))
    # host entry point: pinned buffers are read and written through their device mapping, pageable ones are staged
    y_pin = torch.from_numpy(y0).pin_memory()
    o_pin = torch.empty(y_pin.shape, dtype=torch.float64, pin_memory=True)
    binding.chem_integrate_host(m, P, 1e-5, RTOL, ATOL, y_pin.numpy(), o_pin.numpy(), kernel=3)
    assert np.array_equal(o_pin.numpy(), y_a.cpu().numpy())
    y_h, st_h = binding.chem_integrate_host(m, P, 1e-5, RTOL, ATOL, y0, want_stats=True, kernel=3)
    assert np.array_equal(y_h, y_a.cpu().numpy()) and np.array_equal(st_h, sa)
