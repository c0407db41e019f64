"""Pins of the oracle's Radau IIA integrator against what the mathematics fixes.

Nothing here comes from the CUDA path.  Each test names the mistake it would catch."""
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.linalg

from oracle import oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden", "radau_iia_tableau.txt")


def tableau():
    s6 = np.sqrt(6.0)
    v = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, expr = [t.strip() for t in line.split("=")]
        v[name] = eval(expr, {"s6": s6})
    A = np.array([[v[f"a{i}{j}"] for j in (1, 2, 3)] for i in (1, 2, 3)])
    c = np.array([v["c1"], v["c2"], v["c3"]])
    return A, c


def R(z):
    return (1 + 2 * z / 5 + z * z / 20) / (1 - 3 * z / 5 + 3 * z * z / 20 - z**3 / 60)


def test_tableau_is_radau_iia():
    """the golden tableau itself: row sums, order-5 quadrature conditions, stiff accuracy"""
    A, c = tableau()
    b = A[2]
    assert np.allclose(A.sum(axis=1), c, atol=1e-15)
    for k in range(5):
        assert abs(b @ c**k - 1.0 / (k + 1)) < 1e-15
    # stage order 3: A c^(k-1) = c^k / k, k = 1..3
    for k in (1, 2, 3):
        assert np.allclose(A @ c ** (k - 1), c**k / k, atol=1e-15)


def test_transformation_constants():
    """a wrong digit in T, T^-1, gamma, alpha, beta, c_i: T Lambda T^-1 must equal A^-1"""
    A, c = tableau()
    k = orc.radau_constants()
    lam = np.array([[k["gamma"], 0, 0], [0, k["alpha"], -k["beta"]], [0, k["beta"], k["alpha"]]])
    assert np.abs(k["T"] @ lam @ k["TI"] - np.linalg.inv(A)).max() < 5e-14
    assert np.abs(k["T"] @ k["TI"] - np.eye(3)).max() < 5e-15
    assert np.allclose(k["c"], c, atol=1e-16)
    ev = np.linalg.eigvals(np.linalg.inv(A))
    assert abs(ev[np.abs(ev.imag) < 1e-9].real[0] - k["gamma"]) < 1e-13
    assert abs(np.abs(ev.imag).max() - k["beta"]) < 1e-13


@pytest.mark.parametrize("z", [-0.1, -1.0, -7.5, -100.0, 0.3])
def test_one_step_is_the_stability_function_real(z):
    """one converged step on y' = lambda y is y0 R(z): pins stages, transformation, update y += Z3"""
    lam, h = z / 0.25, 0.25
    y, st = orc.radau5(lambda y: lam * y, lambda y: [[lam]], [1.7], h, 1e-12, 1e-14, fixed_steps=1)
    assert st["status"] == 0 and st["naccpt"] == 1
    assert abs(y[0] - 1.7 * R(z)) <= 1e-13 * max(1.0, abs(1.7 * R(z)))


@pytest.mark.parametrize("z", [-0.5 + 2.0j, -3.0 - 4.0j, 0.0 + 1.0j])
def test_one_step_is_the_stability_function_complex(z):
    """rotation system = complex lambda: catches a swapped sign in the complex (alpha, beta) solve"""
    a, b = z.real, z.imag
    M = np.array([[a, -b], [b, a]])
    y, st = orc.radau5(lambda y: M @ y, lambda y: M, [1.0, 0.0], 1.0, 1e-12, 1e-14, fixed_steps=1)
    assert abs(complex(y[0], y[1]) - R(z)) < 1e-13


def test_order_five_on_nonlinear_problem():
    """y' = -y^3, y = 1/sqrt(1+2t): halving h divides the error by 2^5"""
    f = lambda y: -y**3
    J = lambda y: [[-3 * y[0] ** 2]]
    errs = []
    for n in (8, 16, 32, 64):
        y, st = orc.radau5(f, J, [1.0], 2.0, 1e-13, 1e-15, fixed_steps=n, newton_max=50)
        errs.append(abs(y[0] - 1.0 / np.sqrt(5.0)))
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(orders > 4.5) and np.all(orders < 5.5), orders


def test_error_estimate_is_fourth_order_small():
    """the embedded estimate (dd1..dd3 and the gamma0 h f(y0) term) is O(h^4) on a smooth problem;
    a wrong coefficient leaves an O(h) term"""
    lam = -1.0
    est = []
    hs = [0.2, 0.1, 0.05]
    for h in hs:
        y, st = orc.radau5(lambda y: lam * y, lambda y: [[lam]], [1.0], h, 1e-6, 1e-6, fixed_steps=1)
        est.append(st["err_last"])
    slopes = np.log2(np.array(est[:-1]) / np.array(est[1:]))
    assert np.all(np.abs(slopes - 4.0) < 0.25), (est, slopes)


def test_linear_system_matches_expm_and_reuses_jacobian():
    """adaptive run on y' = A y vs scipy expm; linear problem => Newton converges at once =>
    the built-in rule (theta <= 0.001) never re-evaluates the Jacobian"""
    rng = np.random.default_rng(5)
    Q = rng.standard_normal((4, 4))
    A = Q @ np.diag([-1.0, -30.0, -500.0, -2.0e4]) @ np.linalg.inv(Q)
    y0 = rng.standard_normal(4)
    y, st = orc.radau5(lambda y: A @ y, lambda y: A, y0, 1.0, 1e-6, 1e-10)
    ref = scipy.linalg.expm(A) @ y0
    assert st["status"] == 0 and st["nnewt_fail"] == 0
    assert np.abs(y - ref).max() <= 1e-5 * np.abs(ref).max()
    yt, _ = orc.radau5(lambda y: A @ y, lambda y: A, y0, 1.0, 1e-12, 1e-14)
    assert np.abs(yt - ref).max() <= 1e-9 * np.abs(ref).max()
    # (an error-test rejection after an accepted step re-evaluates it: label "IF (CALJAC) GOTO 20; GOTO 10")
    assert st["njac"] == 1 + st["nrejct"] and st["ndec"] > st["njac"] and st["naccpt"] > 3


def robertson_type(y):
    a, b, c = 0.05, 2.0e4, 5.0e7
    return np.array([-a * y[0] + b * y[1] * y[2], a * y[0] - b * y[1] * y[2] - c * y[1] ** 2, c * y[1] ** 2])


def robertson_type_jac(y):
    a, b, c = 0.05, 2.0e4, 5.0e7
    return np.array([[-a, b * y[2], b * y[1]], [a, -b * y[2] - 2 * c * y[1], -b * y[1]], [0.0, 2 * c * y[1], 0.0]])


def test_robertson_type_against_scipy():
    """stiff 3-species kinetics (PAPER.md L126 suggests ROBER-like checks) against an independent
    library integrator at tight tolerance, judged with the paper's own error metric (Eq. 1-2)"""
    t_end = 40.0
    ref = scipy.integrate.solve_ivp(lambda t, y: robertson_type(y), (0, t_end), [1.0, 0.0, 0.0], method="LSODA",
                                    jac=lambda t, y: robertson_type_jac(y), rtol=1e-12, atol=1e-18).y[:, -1]
    y, st = orc.radau5(robertson_type, robertson_type_jac, [1.0, 0.0, 0.0], t_end, 1e-6, 1e-10, h0=1e-6)
    assert st["status"] == 0
    assert abs(y.sum() - 1.0) < 1e-12                 # linear invariant kept by any RK method
    Emax, _ = orc.error_metric(y[None, :], ref[None, :], 1e-6, 1e-10)
    assert Emax < 10.0, Emax
    # tolerance proportionality: a 100x tighter tolerance gives a clearly smaller error
    y2, st2 = orc.radau5(robertson_type, robertson_type_jac, [1.0, 0.0, 0.0], t_end, 1e-8, 1e-12, h0=1e-6)
    assert np.abs(y2 - ref).max() < 0.2 * np.abs(y - ref).max() + 1e-13
    assert st2["naccpt"] > st["naccpt"]


def test_rejections_and_newton_failures_recover():
    """a far too large first step on a stiff nonlinear problem must be rejected/shrunk, not accepted"""
    y, st = orc.radau5(robertson_type, robertson_type_jac, [1.0, 0.0, 0.0], 1.0e3, 1e-6, 1e-10)
    ref = scipy.integrate.solve_ivp(lambda t, y: robertson_type(y), (0, 1.0e3), [1.0, 0.0, 0.0], method="Radau",
                                    jac=lambda t, y: robertson_type_jac(y), rtol=1e-11, atol=1e-16).y[:, -1]
    assert st["status"] == 0 and st["nstep"] > st["naccpt"]
    Emax, _ = orc.error_metric(y[None, :], ref[None, :], 1e-6, 1e-10)
    assert Emax < 10.0


def test_lands_exactly_on_t_end_and_reports_failure_codes():
    y, st = orc.radau5(lambda y: -y, lambda y: [[-1.0]], [1.0], 3.0, 1e-6, 1e-10, h0=0.01)
    assert st["status"] == 0 and abs(y[0] - np.exp(-3.0)) < 1e-6
    y, st = orc.radau5(lambda y: -y, lambda y: [[-1.0]], [np.nan], 3.0, 1e-6, 1e-10)
    assert st["status"] == -4
    y, st = orc.radau5(robertson_type, robertson_type_jac, [1.0, 0.0, 0.0], 1e3, 1e-6, 1e-10, max_steps=5)
    assert st["status"] == -1


def test_lu_matches_lapack():
    """partial-pivoting LU and solves vs LAPACK (real: same pivots; complex: same |re|+|im| rule)"""
    rng = np.random.default_rng(11)
    for n in (1, 2, 5, 13, 53):
        A = rng.standard_normal((n, n))
        b = rng.standard_normal(n)
        LU, ip, ier = orc.lu_real(A)
        lu_ref, piv_ref = scipy.linalg.lu_factor(A)
        assert ier == 0 and np.array_equal(ip, piv_ref)
        assert np.allclose(LU, lu_ref, rtol=1e-10, atol=1e-12)
        x = orc.lu_solve_real(LU, ip, b)
        assert np.allclose(A @ x, b, atol=1e-9)
        Ac = A + 1j * rng.standard_normal((n, n))
        bc = b + 1j * rng.standard_normal(n)
        LUc, ipc, ier = orc.lu_complex(Ac)
        assert ier == 0
        xc = orc.lu_solve_complex(LUc, ipc, bc)
        assert np.allclose(xc, np.linalg.solve(Ac, bc), atol=1e-9)
    LU, ip, ier = orc.lu_real(np.zeros((3, 3)))
    assert ier != 0


def test_error_metric_and_divergence_definitions():
    """Eq. (1)-(3) of the paper on hand-sized inputs"""
    y = np.array([[1.0, 2.0], [0.0, 1e-10]])
    yh = np.array([[1.0, 2.0 + 2e-6], [1e-10, 0.0]])
    Emax, E = orc.error_metric(y, yh, 1e-6, 1e-10)
    e0 = 2e-6 / (1e-10 + (2.0 + 2e-6) * 1e-6)
    e1 = np.hypot(1e-10 / (1e-10 + 1e-16), 1e-10 / 1e-10)
    assert np.allclose(E, [e0, e1], rtol=1e-12) and Emax == max(E)
    d = np.concatenate([np.full(32, 7), np.r_[np.full(31, 1), 32], np.arange(1, 33)])
    D = orc.divergence(d)
    assert np.allclose(D, [0.0, 1 - 63 / (32 * 32), 1 - (32 * 33 / 2) / (32 * 32)])
