"""Pins of the oracle's thermochemistry, source term and analytical Jacobian.

Independent checks only: closed forms, limits, invariants, finite differences of a different
routine, a library integrator.  Nothing here comes from the CUDA path."""
import numpy as np
import pytest
import scipy.integrate

from oracle import oracle as orc
from paper_1607_03884_b200 import synth

R_ERG = 8.31446261815324e7
P_ATM = synth.P_ATM


def tiny_mech(rxn_type=0, A=1.0e10, b=0.0, Ea=0.0, low=(0.0, 0.0, 0.0), troe=(0, 0, 0, 0), eff=(),
              reac=((0, 1),), prod=((1, 1),), W=(10.0, 10.0, 28.0), nasa=None):
    """hand-made mechanism: species 0, 1 reactive, species 2 inert bath; one reaction"""
    ns = len(W)
    if nasa is None:
        nasa = np.tile(np.array([3.5, 0, 0, 0, 0, -1000.0, 4.0]), (ns, 1))
    return dict(n_species=ns, n_reactions=1, n_elements=1, elem_comp=np.ones((ns, 1), dtype=np.int32),
                mol_weight=np.array(W, dtype=float), nasa_lo=np.array(nasa, dtype=float),
                nasa_hi=np.array(nasa, dtype=float), nasa_tmid=np.full(ns, 1000.0),
                rxn_type=np.array([rxn_type], dtype=np.int32),
                reac_ptr=np.array([0, len(reac)], dtype=np.int32), reac_sp=np.array([r[0] for r in reac], dtype=np.int32),
                reac_nu=np.array([r[1] for r in reac], dtype=np.int32),
                prod_ptr=np.array([0, len(prod)], dtype=np.int32), prod_sp=np.array([p[0] for p in prod], dtype=np.int32),
                prod_nu=np.array([p[1] for p in prod], dtype=np.int32),
                arr_A=np.array([A]), arr_b=np.array([b]), arr_Ea=np.array([Ea]),
                low_A=np.array([low[0]]), low_b=np.array([low[1]]), low_Ea=np.array([low[2]]),
                troe=np.array([troe], dtype=float),
                eff_ptr=np.array([0, len(eff)], dtype=np.int32), eff_sp=np.array([e[0] for e in eff], dtype=np.int32),
                eff_val=np.array([e[1] for e in eff], dtype=float))


def well_scaled_state(mech, T, seed=0):
    rng = np.random.default_rng(seed)
    Y = rng.uniform(0.02, 0.1, mech["n_species"])
    Y /= Y.sum()
    return np.concatenate([[T], Y[:-1]])


# ---------------------------------------------------------------- thermo
@pytest.mark.parametrize("kind", ["h2co", "gri"])
def test_nasa_polynomials_are_consistent(kind, request):
    """h and s must be the integrals of cp (a wrong 1/2, 1/3 ... or a5/T term fails), and the two
    ranges join continuously at T_mid (generator acceptance: 'NASA continuity at T_mid')"""
    mech = request.getfixturevalue("mech_" + kind)
    M = orc.Mechanism(mech)
    for T in (450.0, 1700.0, 2900.0):
        d = 1e-3 * T
        cp, h, s = M.thermo(T)
        _, hp, sp = M.thermo(T + d)
        _, hm, sm = M.thermo(T - d)
        dH = (hp * (T + d) - hm * (T - d)) / (2 * d)          # d(H/R)/dT = cp/R
        assert np.allclose(dH, cp, rtol=2e-6)
        assert np.allclose((sp - sm) / (2 * d), cp / T, rtol=2e-6)
    lo = M.thermo(1000.0)                                      # T <= tmid -> low range
    hi = M.thermo(1000.0 * (1 + 1e-13))
    for a, b_ in zip(lo, hi):
        assert np.allclose(a, b_, rtol=1e-9)
    cp = np.array([M.thermo(T)[0] for T in np.linspace(300, 3000, 28)])
    assert cp.min() >= 2.5 - 1e-9 and cp.max() <= synth.KINDS[kind]["cp_max"] + 1e-9
    a = mech["nasa_lo"][0]
    T = 700.0
    cp0, h0, s0 = (x[0] for x in M.thermo(T))
    # hand evaluation of one species, written with Horner's rule (different form)
    assert np.isclose(cp0, a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4]))), rtol=1e-14)
    assert np.isclose(s0, a[0] * np.log(T) + T * (a[1] + T * (a[2] / 2 + T * (a[3] / 3 + T * a[4] / 4))) + a[6], rtol=1e-14)


def test_ideal_gas_density_and_concentrations(mech_h2co):
    """sum_k C_k = P/(R T) and rho = sum_k C_k W_k: pins Wbar, rho, R and the closure Y_N = 1 - sum Y"""
    M = orc.Mechanism(mech_h2co)
    y = well_scaled_state(mech_h2co, 1350.0)
    r = M.rates(2.5 * P_ATM, y)
    assert np.isclose(r["C"].sum(), 2.5 * P_ATM / (R_ERG * 1350.0), rtol=1e-13)
    assert np.isclose((r["C"] * mech_h2co["mol_weight"]).sum(), r["rho"], rtol=1e-13)
    Y = np.append(y[1:], 1 - y[1:].sum())
    assert np.allclose(r["C"] * mech_h2co["mol_weight"] / r["rho"], Y, rtol=1e-12)


# ---------------------------------------------------------------- rate constants
def test_arrhenius_units_and_form():
    """Ea is in cal/mol: Ea = 1000 K * R_cal gives exp(-1) at 1000 K; T^b factor"""
    m = tiny_mech(A=3.0e9, b=0.0, Ea=1000.0 * 1.98720425864083)
    kf = orc.Mechanism(m).rates(P_ATM, [1000.0, 0.3, 0.3])["kf"][0]
    assert np.isclose(kf, 3.0e9 * np.exp(-1.0), rtol=1e-13)
    m = tiny_mech(A=2.0, b=1.5, Ea=0.0)
    assert np.isclose(orc.Mechanism(m).rates(P_ATM, [900.0, 0.3, 0.3])["kf"][0], 2.0 * 900.0**1.5, rtol=1e-13)


def test_equilibrium_constant_pressure_factor():
    """A <=> 2B with identical thermo: Kc = (P_atm/(R T))^(+1) * exp(-(g_B*2 - g_A)); with s = h = const per
    species the exponent is hand-computable"""
    nasa = np.array([[3.5, 0, 0, 0, 0, -1000.0, 4.0], [3.5, 0, 0, 0, 0, 500.0, 6.0], [3.5, 0, 0, 0, 0, 0.0, 5.0]])
    m = tiny_mech(A=1.0e8, prod=((1, 2),), W=(20.0, 10.0, 28.0), nasa=nasa)
    T = 800.0
    r = orc.Mechanism(m).rates(P_ATM, [T, 0.2, 0.2])
    g = lambda a: a[0] * (1 - np.log(T)) + a[5] / T - a[6]            # h/RT - s/R for constant cp
    Kc = (P_ATM / (R_ERG * T)) * np.exp(-(2 * g(nasa[1]) - g(nasa[0])))
    assert np.isclose(r["kf"][0] / r["kr"][0], Kc, rtol=1e-12)
    # rate of progress: kf [A] - kr [B]^2
    assert np.isclose(r["q"][0], r["kf"][0] * r["C"][0] - r["kr"][0] * r["C"][1] ** 2, rtol=1e-12)
    assert np.allclose(r["wdot"], [-r["q"][0], 2 * r["q"][0], 0.0], rtol=1e-13)


@pytest.mark.parametrize("kind", ["h2co", "gri"])
def test_detailed_balance_at_constructed_equilibrium(kind, request):
    """element-potential construction: C_k = (P_atm/RT) exp(-g_k/RT + sum_e a_ke lambda_e) makes every
    element-balanced reaction satisfy Kc exactly, so every net rate of progress must vanish
    ('relaxation toward the equilibrium implied by the thermo data').  A wrong sign of dG, a missing
    (P_atm/RT)^dnu, or a stoichiometry slip leaves |q| ~ forward rate."""
    mech = request.getfixturevalue("mech_" + kind)
    M = orc.Mechanism(mech)
    rng = np.random.default_rng(3)
    T = 1600.0
    cp, h, s = M.thermo(T)
    lam = rng.uniform(-2.0, 0.0, mech["n_elements"])
    lnC = np.log(P_ATM / (R_ERG * T)) - (h - s) + mech["elem_comp"] @ lam
    C = np.exp(lnC)
    P = C.sum() * R_ERG * T
    Y = C * mech["mol_weight"]
    Y /= Y.sum()
    y = np.concatenate([[T], Y[:-1]])
    r = M.rates(P, y)
    assert np.allclose(r["C"], C, rtol=1e-10)
    # forward rates of progress for scale
    fwd = np.empty(mech["n_reactions"])
    for i in range(mech["n_reactions"]):
        p = slice(mech["reac_ptr"][i], mech["reac_ptr"][i + 1])
        fwd[i] = r["kf"][i] * np.prod(C[mech["reac_sp"][p]] ** mech["reac_nu"][p])
    ratio = np.empty(mech["n_reactions"])
    for i in range(mech["n_reactions"]):
        p = slice(mech["prod_ptr"][i], mech["prod_ptr"][i + 1])
        ratio[i] = r["kr"][i] * np.prod(C[mech["prod_sp"][p]] ** mech["prod_nu"][p]) / fwd[i]
    assert np.allclose(ratio, 1.0, rtol=1e-9)
    f = M.rhs(P, y)
    scale = np.abs(fwd).max() * mech["mol_weight"].max() / r["rho"]
    assert np.abs(f[1:]).max() < 1e-8 * scale


def test_three_body_and_falloff_limits():
    """[M] = sum alpha_k C_k; Lindemann: Pr >> 1 gives k_inf, Pr << 1 gives k_0 [M]; Troe with
    Fcent = 1 is Lindemann; Troe at log10 Pr + c = 0 gives F = Fcent"""
    T = 1200.0
    y = [T, 0.2, 0.3]
    base = orc.Mechanism(tiny_mech(A=1.0e7)).rates(P_ATM, y)
    Cs = base["C"]
    r3 = orc.Mechanism(tiny_mech(rxn_type=1, A=1.0e7, eff=((0, 2.5), (2, 0.5)))).rates(P_ATM, y)
    Mconc = 2.5 * Cs[0] + Cs[1] + 0.5 * Cs[2]
    assert np.isclose(r3["q"][0], Mconc * base["q"][0], rtol=1e-13)
    # Lindemann limits
    hi = orc.Mechanism(tiny_mech(rxn_type=2, A=1.0e7, low=(1.0e30, 0.0, 0.0))).rates(P_ATM, y)
    assert np.isclose(hi["q"][0], base["q"][0], rtol=1e-9)
    lo = orc.Mechanism(tiny_mech(rxn_type=2, A=1.0e7, low=(1.0e2, 0.0, 0.0))).rates(P_ATM, y)
    Msum = Cs.sum()
    Pr = 1.0e2 * Msum / 1.0e7
    assert np.isclose(lo["q"][0], base["q"][0] * Pr / (1 + Pr), rtol=1e-12)
    assert np.isclose(lo["q"][0] / base["q"][0], 1.0e2 * Msum / 1.0e7, rtol=1e-4)       # k_0 [M] / k_inf
    # Troe: Fcent -> 1 when T*** and T* are huge and T** is huge: (1-a) + a + 0
    tl = orc.Mechanism(tiny_mech(rxn_type=3, A=1.0e7, low=(1.0e12, 0.0, 0.0), troe=(0.6, 1e30, 1e30, 1e30))).rates(P_ATM, y)
    ll = orc.Mechanism(tiny_mech(rxn_type=2, A=1.0e7, low=(1.0e12, 0.0, 0.0))).rates(P_ATM, y)
    assert np.isclose(tl["q"][0], ll["q"][0], rtol=1e-12)
    # Troe centre: choose k_0 so that log10 Pr = -c = 0.4 + 0.67 log10 Fcent  =>  F = Fcent
    al, T3, T1, T2 = 0.7, 200.0, 1500.0, 5000.0
    Fc = (1 - al) * np.exp(-T / T3) + al * np.exp(-T / T1) + np.exp(-T2 / T)
    Pr = 10.0 ** (0.4 + 0.67 * np.log10(Fc))
    A0 = Pr * 1.0e7 / Msum
    tc = orc.Mechanism(tiny_mech(rxn_type=3, A=1.0e7, low=(A0, 0.0, 0.0), troe=(al, T3, T1, T2))).rates(P_ATM, y)
    assert np.isclose(tc["q"][0], base["q"][0] * Pr / (1 + Pr) * Fc, rtol=1e-11)
    # and away from the centre F lies strictly between Fcent and 1
    tf = orc.Mechanism(tiny_mech(rxn_type=3, A=1.0e7, low=(A0 * 100, 0.0, 0.0), troe=(al, T3, T1, T2))).rates(P_ATM, y)
    F = tf["q"][0] / (base["q"][0] * (100 * Pr) / (1 + 100 * Pr))
    assert Fc < F < 1.0


# ---------------------------------------------------------------- source term invariants
@pytest.mark.parametrize("kind", ["h2co", "gri"])
def test_mass_and_element_conservation_of_rates(kind, request):
    """sum_k W_k wdot_k = 0 and sum_k a_ke wdot_k = 0 (a stoichiometric sign slip breaks both)"""
    mech = request.getfixturevalue("mech_" + kind)
    M = orc.Mechanism(mech)
    for seed, T in ((1, 900.0), (2, 2100.0)):
        r = M.rates(P_ATM, well_scaled_state(mech, T, seed))
        w = r["wdot"]
        assert abs((mech["mol_weight"] * w).sum()) < 1e-12 * np.abs(mech["mol_weight"] * w).sum()
        el = mech["elem_comp"].T @ w
        assert np.all(np.abs(el) < 1e-12 * (np.abs(mech["elem_comp"]).T @ np.abs(w) + 1e-300))
        # wdot is S q with the CSR stoichiometry (scatter written independently here)
        S = np.zeros((mech["n_species"], mech["n_reactions"]))
        for i in range(mech["n_reactions"]):
            for p in range(mech["reac_ptr"][i], mech["reac_ptr"][i + 1]):
                S[mech["reac_sp"][p], i] -= mech["reac_nu"][p]
            for p in range(mech["prod_ptr"][i], mech["prod_ptr"][i + 1]):
                S[mech["prod_sp"][p], i] += mech["prod_nu"][p]
        assert np.allclose(S @ r["q"], w, rtol=1e-10, atol=1e-14 * np.abs(w).max())


@pytest.mark.parametrize("kind", ["h2co", "gri"])
def test_rhs_conserves_enthalpy_to_first_order(kind, request):
    """constant-pressure adiabatic reactor: d/dt sum_k Y_k h_k(T) = 0, i.e.
    cp Tdot + sum_k h_k Ydot_k = 0 with mass-specific h_k, cp (pins the temperature equation)"""
    mech = request.getfixturevalue("mech_" + kind)
    M = orc.Mechanism(mech)
    W = mech["mol_weight"]
    y = well_scaled_state(mech, 1400.0, 4)
    f = M.rhs(P_ATM, y)
    cp, h, s = M.thermo(1400.0)
    Y = np.append(y[1:], 1 - y[1:].sum())
    Ydot = np.append(f[1:], -f[1:].sum())
    cp_mass = (Y * cp * R_ERG / W).sum()
    h_mass = h * R_ERG * 1400.0 / W
    assert abs(cp_mass * f[0] + (h_mass * Ydot).sum()) < 1e-11 * np.abs(h_mass * Ydot).sum()


# ---------------------------------------------------------------- Jacobian
@pytest.mark.parametrize("kind,T", [("h2co", 800.0), ("h2co", 1500.0), ("gri", 900.0), ("gri", 2000.0)])
def test_jacobian_matches_finite_differences(kind, T, request):
    """analytical Jacobian vs central differences of the (separately pinned) source term; every reaction
    type is present in both mechanisms, both NASA ranges are visited.  A dropped term in any of
    d/dT (Arrhenius, Kc, Troe, [M], rho) or d/dY (rho, Wbar, closure species) shows at 1e-2..1; FD noise is 1e-7."""
    mech = request.getfixturevalue("mech_" + kind)
    M = orc.Mechanism(mech)
    y = well_scaled_state(mech, T, 7)
    N = mech["n_species"]
    J = M.jacobian(P_ATM, y)
    Jfd = np.empty((N, N))
    for j in range(N):
        d = 2e-5 * y[j]
        yp, ym = y.copy(), y.copy()
        yp[j] += d
        ym[j] -= d
        Jfd[:, j] = (M.rhs(P_ATM, yp) - M.rhs(P_ATM, ym)) / (2 * d)
    col = np.abs(Jfd).max(axis=0)
    row = np.abs(Jfd).max(axis=1)
    assert np.all(np.abs(J - Jfd).max(axis=0) <= 2e-6 * col)
    assert np.all(np.abs(J - Jfd).max(axis=1) <= 2e-6 * row)
    assert set(np.unique(mech["rxn_type"])) >= {0, 1, 3}


def test_jacobian_of_falloff_types_individually():
    """Lindemann and Troe derivative chains on one-reaction mechanisms (Lindemann is absent from the synthetic ones)"""
    for typ, troe in ((2, (0, 0, 0, 0)), (3, (0.6, 150.0, 1800.0, 4000.0)), (1, (0, 0, 0, 0))):
        m = tiny_mech(rxn_type=typ, A=1.0e9, b=0.7, Ea=8000.0, low=(3.0e13, -0.5, 3000.0), troe=troe,
                      eff=((0, 3.0), (2, 0.4)), reac=((0, 1), (1, 1)), prod=((2, 1),), W=(10.0, 18.0, 28.0, 40.0),
                      nasa=np.array([[3.5, 1e-3, 0, 0, 0, 2000.0, 4.0], [4.0, 5e-4, 1e-7, 0, 0, -3000.0, 6.0],
                                     [4.5, 2e-3, -2e-7, 0, 0, -9000.0, 5.0], [2.5, 0, 0, 0, 0, 0.0, 5.0]]))
        M = orc.Mechanism(m)
        y = np.array([1100.0, 0.2, 0.3, 0.1])
        J = M.jacobian(P_ATM, y)
        Jfd = np.empty((4, 4))
        for j in range(4):
            d = 1e-5 * y[j]
            yp, ym = y.copy(), y.copy()
            yp[j] += d
            ym[j] -= d
            Jfd[:, j] = (M.rhs(P_ATM, yp) - M.rhs(P_ATM, ym)) / (2 * d)
        assert np.all(np.abs(J - Jfd) <= 1e-6 * np.abs(Jfd).max(axis=0)[None, :]), typ


# ---------------------------------------------------------------- whole path
def test_isothermal_relaxation_closed_form():
    """A <=> B, equal thermo and weights: T stays constant, Y_A(t) = 1/2 (Y_A+Y_B) + 1/2 (Y_A-Y_B)_0 exp(-2 k t)"""
    k = 4.0e5
    m = tiny_mech(A=k)
    M = orc.Mechanism(m)
    y0 = np.array([[1000.0, 0.5, 0.1]])
    t = 3.0e-6
    y, st, _ = M.integrate(y0, P_ATM, t, 1e-9, 1e-13)
    assert st["status"][0] == 0
    ya = 0.3 + 0.2 * np.exp(-2 * k * t)
    assert abs(y[0, 0] - 1000.0) < 1e-6
    assert np.allclose(y[0, 1:], [ya, 0.6 - ya], rtol=1e-8)


def test_integration_conserves_elements_and_enthalpy(mech_h2co):
    """over a whole global step: element mass fractions to round-off (linear invariants of an RK method),
    total enthalpy to integration accuracy"""
    M = orc.Mechanism(mech_h2co)
    W = mech_h2co["mol_weight"]
    y0 = synth.make_states(mech_h2co, 64, "ignition", 5)
    y1, st, _ = M.integrate(y0, P_ATM, 1e-4, 1e-6, 1e-10)
    assert np.all(st["status"] == 0)

    def invariants(y):
        out = []
        for row in y:
            Y = np.append(row[1:], 1 - row[1:].sum())
            cp, h, s = M.thermo(row[0])
            out.append(np.concatenate([mech_h2co["elem_comp"].T @ (Y / W), [(Y * h * R_ERG * row[0] / W).sum()]]))
        return np.array(out)
    i0, i1 = invariants(y0), invariants(y1)
    assert np.allclose(i0[:, :-1], i1[:, :-1], rtol=0, atol=1e-12)
    hscale = np.abs(M.thermo(1500.0)[1] * R_ERG * 1500.0 / W).max()
    assert np.abs(i1[:, -1] - i0[:, -1]).max() < 1e-6 * hscale


def test_small_mechanism_against_scipy_bdf(mech_h2co):
    """brute-force reference: a library integrator at tight tolerance on the smallest synthetic mechanism;
    the oracle at production tolerance stays within a few units of the paper's error metric (Eq. 1-2)"""
    M = orc.Mechanism(mech_h2co)
    y0 = synth.make_states(mech_h2co, 6, "ignition", 9)
    t_end = 1e-5
    y1, st, _ = M.integrate(y0, P_ATM, t_end, 1e-6, 1e-10)
    ref = np.empty_like(y0)
    for i in range(y0.shape[0]):
        sol = scipy.integrate.solve_ivp(lambda t, y: M.rhs(P_ATM, y), (0, t_end), y0[i], method="LSODA",
                                        jac=lambda t, y: M.jacobian(P_ATM, y), rtol=1e-11, atol=1e-18)
        assert sol.success
        ref[i] = sol.y[:, -1]
    Emax, E = orc.error_metric(y1, ref, 1e-6, 1e-10)
    assert Emax < 20.0, E
    y2, _, _ = M.integrate(y0, P_ATM, t_end, 1e-9, 1e-14)
    Emax2, _ = orc.error_metric(y2, ref, 1e-6, 1e-10)
    assert Emax2 < 0.05 * max(Emax, 1.0)


def test_configs_integrate_without_failures(mech_h2co, mech_gri):
    """the synthetic workloads are well posed: every state of a sample of each config completes"""
    for mech, dist, t_end, n in ((mech_h2co, "uniform", 1e-6, 512), (mech_h2co, "ignition", 1e-4, 256),
                                 (mech_gri, "uniform", 1e-6, 48), (mech_gri, "ignition", 1e-4, 32)):
        y0 = synth.make_states(mech, n, dist, synth.STATE_SEED)
        y1, st, _ = orc.Mechanism(mech).integrate(y0, P_ATM, t_end, synth.RTOL, synth.ATOL)
        assert np.all(st["status"] == 0)
        assert np.all(np.isfinite(y1)) and y1[:, 1:].min() > -1e-7


def test_finite_difference_jacobian_option(mech_h2co):
    """PAPER.md L82 / Sec. 3.4: first-order FD Jacobian 'based on that of CVODE' (R13).  It costs N extra
    source terms per Jacobian and must give the same answer within the integration tolerance."""
    M = orc.Mechanism(mech_h2co)
    y0 = synth.make_states(mech_h2co, 256, "ignition", 5)
    ya, sa, _ = M.integrate(y0, P_ATM, 1e-4, 1e-6, 1e-10)
    yf, sf, _ = M.integrate(y0, P_ATM, 1e-4, 1e-6, 1e-10, fd_jacobian=1)
    assert np.all(sf["status"] == 0)
    same = sa["nstep"] == sf["nstep"]
    assert same.mean() > 0.9
    # with identical step sequences the only extra work is N source terms per Jacobian evaluation
    mask = same & (sa["njac"] == sf["njac"]) & (sa["nsol"] == sf["nsol"]) & (sa["naccpt"] == sf["naccpt"])
    assert mask.mean() > 0.8
    assert ((sf["nfcn"] - sa["nfcn"])[mask] == (13 * sf["njac"])[mask]).mean() > 0.97
    Emax, _ = orc.error_metric(yf, ya, 1e-6, 1e-10)
    assert Emax < 500.0
    # on a linear problem the difference quotient is exact up to rounding: same result as the analytic Jacobian
    A = np.array([[-3.0, 1.0], [2.0, -400.0]])
    y1, s1 = orc.radau5(lambda y: A @ y, lambda y: A, [1.0, 2.0], 1.0, 1e-6, 1e-10)
    y2, s2 = orc.radau5(lambda y: A @ y, lambda y: 0 * A, [1.0, 2.0], 1.0, 1e-6, 1e-10, fd_jacobian=1)
    assert np.allclose(y1, y2, rtol=1e-7, atol=1e-12) and s1["naccpt"] == s2["naccpt"]
