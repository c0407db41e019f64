"""Seeded synthetic inputs: mechanisms and thermochemical state batches.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic (no rate constants, no species rates, no
Jacobian, no integrator): it only *constructs* inputs.  The paper's own inputs
are the Burke H2 model (13 species / 27 reactions) and GRI-Mech 3.0 (53 / 325)
with PaSR state databases (Sec. 2.2); none of those files are
available, so BASELINE.json's configs replace them with seeded synthetic
mechanisms and states of the same shape.  The recipe is restated in DESIGN.md.

Units follow the CHEMKIN convention the cited pyJac uses:
cm, mol, s, K, cal/mol for activation energies, g/mol for molecular weights.

A mechanism is a dict of numpy arrays whose keys are the fields of
`chem_mech_desc` in include/chem.h.
"""
from __future__ import annotations

import numpy as np

ATOMIC_WEIGHT = {"H": 1.008, "O": 15.999, "C": 12.011, "N": 14.007, "Ar": 39.948}

# reaction type codes (include/chem.h)
RXN_ELEMENTARY = 0
RXN_THREE_BODY = 1
RXN_FALLOFF_LINDEMANN = 2
RXN_FALLOFF_TROE = 3

T_LOW, T_MID, T_HIGH = 300.0, 1000.0, 3000.0
T_REF = 298.15

KINDS = {
    # kind: elements, reactive element caps, n_species, n_reactions, n_three_body, n_troe, cp/R max
    "h2co": dict(elements=("H", "O", "C", "N"), caps={"H": 4, "O": 3, "C": 1}, n_species=13,
                 n_reactions=27, n_three_body=4, n_troe=2, cp_max=8.0, inert=("N2",)),
    "gri": dict(elements=("C", "H", "O", "N", "Ar"), caps={"C": 3, "H": 8, "O": 3, "N": 2}, n_species=53,
                n_reactions=325, n_three_body=30, n_troe=29, cp_max=15.0, inert=("AR", "N2")),
    # not BASELINE.json configs: test shapes for the small-mechanism kernels.  "h2_9": a hydrogen / oxygen sized shape (H, O,
    # H2, O2, OH, H2O, H2O2, HO2 + N2); "lim16": the size limits of those kernels (16 species, and as many reactions as
    # leave room for the falloff / Troe exp jobs among 2 x 32 job slots); "sz<N>": one shape per remaining compile-time-N
    # instantiation of the thread-per-state kernel (8 <= N <= 16)
    "h2_9": dict(elements=("H", "O", "N"), caps={"H": 2, "O": 2}, n_species=9,
                 n_reactions=20, n_three_body=3, n_troe=1, cp_max=7.0, inert=("N2",)),
    "lim16": dict(elements=("H", "O", "C", "N"), caps={"H": 4, "O": 3, "C": 2}, n_species=16,
                  n_reactions=28, n_three_body=3, n_troe=1, cp_max=8.0, inert=("N2",)),
    **{f"sz{n}": dict(elements=("H", "O", "C", "N"), caps={"H": 4, "O": 3, "C": 1}, n_species=n,
                      n_reactions=8 if n == 8 else min(2 * n, 28), n_three_body=3, n_troe=1, cp_max=8.0, inert=("N2",))
       for n in (8, 10, 11, 12, 14, 15)},
}


def _formula(comp, elements):
    return "".join(f"{e}{n}" for e, n in zip(elements, comp) if n)


def _species_set(rng, spec):
    """Compositions of the reactive species: a few seed fragments, then sums of two
    species already present (so recombination reactions A + B <=> AB exist), within
    the per-element caps.  Returns a list of integer composition tuples."""
    elements = spec["elements"]
    caps = np.array([spec["caps"].get(e, 0) for e in elements])
    n_reactive = spec["n_species"] - len(spec["inert"])
    react_el = [i for i, e in enumerate(elements) if spec["caps"].get(e, 0) > 0]
    comps = []
    # atoms of every reactive element first, then the homonuclear diatomics of the first two
    for i in react_el:
        c = np.zeros(len(elements), dtype=int)
        c[i] = 1
        comps.append(tuple(c))
    for i in react_el:
        c = np.zeros(len(elements), dtype=int)
        c[i] = 2
        if elements[i] != "N" and np.all(c <= caps):     # N2 is the inert last species
            comps.append(tuple(c))
    guard = 0
    while len(comps) < n_reactive:
        guard += 1
        if guard > 100000:
            raise RuntimeError("species construction did not terminate")
        a = comps[rng.integers(len(comps))]
        b = comps[rng.integers(len(comps))]
        c = tuple(int(x) for x in (np.array(a) + np.array(b)))
        if np.any(np.array(c) > caps) or c in comps:
            continue
        # N2 itself is the inert last species, keep it out of the reactive set
        if _formula(c, elements) == "N2":
            continue
        comps.append(c)
    return comps


def _nasa_species(rng, natoms, cp_max, h_f, s_ref):
    """NASA-7 two-range coefficients (a0..a6 low, a0..a6 high) for one species:
    quartic least-squares fits of a smooth saturating cp/R(T) target, made continuous
    in cp, h and s at T_MID, with h(T_REF)/R = h_f [K] and s(T_REF)/R = s_ref."""
    if natoms == 1:
        c0 = c_inf = 2.5
    else:
        c0 = min(2.5 + (1.0 if natoms == 2 else 1.5) * rng.uniform(0.9, 1.1), cp_max - 0.5)
        c_inf = min(c0 + (natoms - 1) * rng.uniform(0.7, 1.3) + 0.5, cp_max - 0.05)
    theta = rng.uniform(700.0, 1500.0)

    def target(T):
        return c0 + (c_inf - c0) * (1.0 - np.exp(-((T / theta) ** 1.5)))

    def fit(t0, t1):
        T = np.linspace(t0, t1, 64)
        x = T / 1000.0
        p = np.polyfit(x, target(T), 4)[::-1]          # a0..a4 in powers of (T/1000)
        return np.array([p[k] / 1000.0 ** k for k in range(5)])

    lo = np.zeros(7)
    hi = np.zeros(7)
    lo[:5] = fit(T_LOW, T_MID)
    hi[:5] = fit(T_MID, T_HIGH)

    def cp(a, T):
        return a[0] + a[1] * T + a[2] * T**2 + a[3] * T**3 + a[4] * T**4

    def h_int(a, T):   # integral of cp/R dT without the constant: H/R - a5
        return a[0] * T + a[1] * T**2 / 2 + a[2] * T**3 / 3 + a[3] * T**4 / 4 + a[4] * T**5 / 5

    def s_int(a, T):   # integral of cp/(R T) dT without the constant: S/R - a6
        return a[0] * np.log(T) + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4

    hi[0] += cp(lo, T_MID) - cp(hi, T_MID)
    lo[5] = h_f - h_int(lo, T_REF)
    hi[5] = lo[5] + h_int(lo, T_MID) - h_int(hi, T_MID)
    lo[6] = s_ref - s_int(lo, T_REF)
    hi[6] = lo[6] + s_int(lo, T_MID) - s_int(hi, T_MID)
    # acceptance: bounded inside the fitted ranges, sane under extrapolation
    Tin = np.linspace(T_LOW, T_HIGH, 271)
    cpin = np.where(Tin <= T_MID, cp(lo, Tin), cp(hi, Tin))
    Tex = np.linspace(T_HIGH, 6000.0, 61)
    ok = (cpin.min() >= 2.5 - 1e-9 and cpin.max() <= cp_max + 1e-9
          and cp(hi, Tex).min() >= 2.0 and cp(hi, Tex).max() <= 2.0 * cp_max
          and cp(lo, 200.0) >= 2.0)
    return lo, hi, ok


def _anticorrelated_uniforms(rng, rho: float = -0.9):
    """Two U(0,1) variates joined by a Gaussian copula with correlation rho.  Used for
    (log10 A, b): each keeps exactly the marginal BASELINE.json states (A log-uniform in
    1e6..1e14, b uniform in [-2, 2]) while a large temperature exponent comes with a small
    pre-exponential factor, as in real mechanisms, so that k(T) stays below ~1e15 (cm, mol, s)."""
    from math import erf, sqrt
    z1, z2 = rng.standard_normal(2)
    z2 = rho * z1 + sqrt(1.0 - rho * rho) * z2
    return 0.5 * (1.0 + erf(z1 / sqrt(2.0))), 0.5 * (1.0 + erf(z2 / sqrt(2.0)))


def make_mechanism(kind: str = "h2co", seed: int = 0) -> dict:
    """Seeded synthetic mechanism; a draw whose species set has too few balanced reactions is
    redrawn with the next sub-seed (deterministic)."""
    err = None
    for attempt in range(64):
        try:
            return _make_mechanism(kind, seed, attempt)
        except RuntimeError as e:       # structural rejection only
            err = e
    raise RuntimeError(f"no acceptable mechanism for seed {seed}: {err}")


def _make_mechanism(kind: str, seed: int, attempt: int) -> dict:
    """Build the seeded synthetic mechanism `kind` ("h2co": 13 sp / 27 rxn, "gri": 53 / 325).

    All reactions are reversible and element-balanced by construction; reverse rates come
    from equilibrium constants (the consumer computes them).  Forward is the exothermic
    direction at T_REF (so that reverse rate constants stay below the forward scale)."""
    spec = KINDS[kind]
    elements = spec["elements"]
    rng = np.random.default_rng([seed, sum(map(ord, kind)), attempt])
    ne = len(elements)

    comps = _species_set(rng, spec)
    names = [_formula(c, elements) for c in comps]
    for nm in spec["inert"]:
        c = np.zeros(ne, dtype=int)
        if nm == "AR":
            c[elements.index("Ar")] = 1
        else:
            c[elements.index("N")] = 2
        comps.append(tuple(c))
        names.append(nm)
    comp = np.array(comps, dtype=np.int32)
    ns = comp.shape[0]
    assert ns == spec["n_species"]
    W = comp @ np.array([ATOMIC_WEIGHT[e] for e in elements])
    natoms = comp.sum(axis=1)
    n_inert = len(spec["inert"])

    # ---- thermo: atomisation-like enthalpies of formation [K], entropies, NASA-7 fits
    atom_h = {"H": 26000.0, "O": 30000.0, "C": 60000.0, "N": 45000.0, "Ar": 0.0}
    bond = 30000.0
    nasa_lo = np.zeros((ns, 7))
    nasa_hi = np.zeros((ns, 7))
    h_f = np.zeros(ns)
    for k in range(ns):
        inert = k >= ns - n_inert
        if inert:
            h_f[k] = 0.0
        else:
            h_f[k] = (sum(atom_h[e] * n for e, n in zip(elements, comp[k]))
                      - (natoms[k] - 1) * bond * (1.0 + rng.uniform(-0.2, 0.2) / np.sqrt(natoms[k] - 1.0 + 1e-30)))
        for _ in range(200):
            # entropy grows smoothly with molecular size, so exchange reactions have |dS/R| of a few
            # units and recombinations lose about one molecule's worth (as in real thermo data)
            s_ref = 14.0 + 4.0 * np.log(natoms[k]) + 0.5 * np.log(W[k]) + rng.uniform(-1.5, 1.5)
            lo, hi, ok = _nasa_species(rng, int(natoms[k]), spec["cp_max"], h_f[k], s_ref)
            if ok:
                break
        else:
            raise RuntimeError("NASA fit rejected 200 times")
        nasa_lo[k], nasa_hi[k] = lo, hi

    # ---- candidate reactions among the reactive species
    nr_sp = ns - n_inert
    pair_sum = {}
    for a in range(nr_sp):
        for b in range(a, nr_sp):
            pair_sum.setdefault(tuple(comp[a] + comp[b]), []).append((a, b))
    comp_index = {tuple(comp[k]): k for k in range(nr_sp)}
    recomb = []          # A + B <=> C
    exchange = []        # A + B <=> C + D
    for s, pairs in pair_sum.items():
        if s in comp_index:
            for (a, b) in pairs:
                recomb.append(((a, b), (comp_index[s],)))
        for i in range(len(pairs)):
            for j in range(i + 1, len(pairs)):
                exchange.append((pairs[i], pairs[j]))
    n_rx = spec["n_reactions"]
    n_tb, n_troe = spec["n_three_body"], spec["n_troe"]
    if len(recomb) < n_tb + n_troe or len(recomb) + len(exchange) < n_rx:
        raise RuntimeError(f"seed {seed}: too few balanced candidates "
                           f"({len(recomb)} recombinations, {len(exchange)} exchanges)")
    rec_order = rng.permutation(len(recomb))
    exc_order = rng.permutation(len(exchange))
    chosen = [(recomb[i], RXN_THREE_BODY) for i in rec_order[:n_tb]]
    chosen += [(recomb[i], RXN_FALLOFF_TROE) for i in rec_order[n_tb:n_tb + n_troe]]
    rest = [exchange[i] for i in exc_order] + [recomb[i] for i in rec_order[n_tb + n_troe:]]
    chosen += [(r, RXN_ELEMENTARY) for r in rest[:n_rx - len(chosen)]]
    order = rng.permutation(len(chosen))
    chosen = [chosen[i] for i in order]

    # every reactive species must take part in a reaction: swap in candidates that use the missing ones
    def used_set(rx):
        u = set()
        for (lhs, rhs), _ in rx:
            u.update(lhs)
            u.update(rhs)
        return u
    missing = set(range(nr_sp)) - used_set(chosen)
    spare = rest[n_rx - (n_tb + n_troe):]
    for k in sorted(missing):
        cand = [r for r in spare if k in r[0] or k in r[1]]
        if not cand:
            raise RuntimeError(f"seed {seed}: species {k} appears in no balanced reaction")
        # replace an elementary reaction whose species all stay covered
        for idx in range(len(chosen) - 1, -1, -1):
            if chosen[idx][1] != RXN_ELEMENTARY:
                continue
            trial = chosen[:idx] + [(cand[0], RXN_ELEMENTARY)] + chosen[idx + 1:]
            if (set(range(nr_sp)) - used_set(trial)) <= (missing - {k}):
                chosen = trial
                break
        missing = set(range(nr_sp)) - used_set(chosen)
    if set(range(nr_sp)) - used_set(chosen):
        raise RuntimeError(f"seed {seed}: could not cover all reactive species")

    def side(sp_list):
        sp, nu = [], []
        for k in sp_list:
            if k in sp:
                nu[sp.index(k)] += 1
            else:
                sp.append(k)
                nu.append(1)
        return sp, nu

    rtype = np.zeros(n_rx, dtype=np.int32)
    reac_ptr, reac_sp, reac_nu = [0], [], []
    prod_ptr, prod_sp, prod_nu = [0], [], []
    eff_ptr, eff_sp, eff_val = [0], [], []
    A = np.zeros(n_rx); b = np.zeros(n_rx); Ea = np.zeros(n_rx)
    A0 = np.zeros(n_rx); b0 = np.zeros(n_rx); Ea0 = np.zeros(n_rx)
    troe = np.zeros((n_rx, 4))
    for i, ((lhs, rhs), typ) in enumerate(chosen):
        dH = sum(h_f[k] for k in rhs) - sum(h_f[k] for k in lhs)
        if dH > 0.0:                                # forward = exothermic direction (any type)
            lhs, rhs = rhs, lhs
        rtype[i] = typ
        sp, nu = side(lhs)
        reac_sp += sp; reac_nu += nu; reac_ptr.append(len(reac_sp))
        sp, nu = side(rhs)
        prod_sp += sp; prod_nu += nu; prod_ptr.append(len(prod_sp))
        uA, ub = _anticorrelated_uniforms(rng)
        A[i] = 10.0 ** (6.0 + 8.0 * uA)
        b[i] = -2.0 + 4.0 * ub
        Ea[i] = rng.uniform(0.0, 50000.0)
        if typ in (RXN_FALLOFF_TROE, RXN_FALLOFF_LINDEMANN):
            # low-pressure limit has one more concentration factor: A0 ~ A * 1e4..1e8 cm^3/mol
            A0[i] = A[i] * 10.0 ** rng.uniform(4.0, 8.0)
            b0[i] = b[i] + rng.uniform(-0.5, 0.5)
            Ea0[i] = rng.uniform(0.0, 50000.0)
        if typ == RXN_FALLOFF_TROE:
            troe[i] = (rng.uniform(0.2, 0.9), rng.uniform(50.0, 500.0),
                       rng.uniform(800.0, 3000.0), rng.uniform(2000.0, 8000.0))
        if typ != RXN_ELEMENTARY:
            n_eff = int(rng.integers(2, 6))
            for k in sorted(rng.choice(ns, size=min(n_eff, ns), replace=False)):
                eff_sp.append(int(k))
                eff_val.append(float(rng.uniform(0.5, 12.0)))
        eff_ptr.append(len(eff_sp))

    mech = dict(
        kind=kind, seed=seed, elements=elements, species_names=names,
        n_species=ns, n_reactions=n_rx, n_elements=ne,
        elem_comp=np.ascontiguousarray(comp, dtype=np.int32),
        mol_weight=np.ascontiguousarray(W, dtype=np.float64),
        nasa_lo=np.ascontiguousarray(nasa_lo), nasa_hi=np.ascontiguousarray(nasa_hi),
        nasa_tmid=np.full(ns, T_MID),
        rxn_type=rtype,
        reac_ptr=np.array(reac_ptr, dtype=np.int32), reac_sp=np.array(reac_sp, dtype=np.int32),
        reac_nu=np.array(reac_nu, dtype=np.int32),
        prod_ptr=np.array(prod_ptr, dtype=np.int32), prod_sp=np.array(prod_sp, dtype=np.int32),
        prod_nu=np.array(prod_nu, dtype=np.int32),
        arr_A=A, arr_b=b, arr_Ea=Ea, low_A=A0, low_b=b0, low_Ea=Ea0,
        troe=np.ascontiguousarray(troe),
        eff_ptr=np.array(eff_ptr, dtype=np.int32), eff_sp=np.array(eff_sp, dtype=np.int32),
        eff_val=np.array(eff_val, dtype=np.float64),
        h_formation=h_f,
    )
    check_mechanism(mech)
    return mech


def check_mechanism(mech: dict) -> None:
    """Generator acceptance checks (structure only): integer element balance of every
    reaction, every non-inert species used, CSR arrays consistent."""
    comp = mech["elem_comp"]
    ns, nr = mech["n_species"], mech["n_reactions"]
    used = np.zeros(ns, dtype=bool)
    for i in range(nr):
        bal = np.zeros(comp.shape[1], dtype=np.int64)
        for p in range(mech["reac_ptr"][i], mech["reac_ptr"][i + 1]):
            bal -= mech["reac_nu"][p] * comp[mech["reac_sp"][p]]
            used[mech["reac_sp"][p]] = True
        for p in range(mech["prod_ptr"][i], mech["prod_ptr"][i + 1]):
            bal += mech["prod_nu"][p] * comp[mech["prod_sp"][p]]
            used[mech["prod_sp"][p]] = True
        if np.any(bal != 0):
            raise ValueError(f"reaction {i} is not element balanced")
    n_inert = len(KINDS[mech["kind"]]["inert"]) if mech.get("kind") in KINDS else 0
    if not np.all(used[: ns - n_inert]):
        raise ValueError("a reactive species takes part in no reaction")


def major_pool(mech: dict, n: int = 5) -> np.ndarray:
    """Species that may be drawn as 'major' in a state.  h2co: the last (inert bath) species plus
    the `n` reactive species with the lowest formation enthalpy per atom (the stable ones).
    gri: a fuel-like species (one carbon, no O/N, the most hydrogens), the O2 species and N2
    (BASELINE.json configs[3]: "CH4/O2/N2 majors")."""
    ns = mech["n_species"]
    kind = mech.get("kind")
    if kind == "gri":
        el = list(mech["elements"])
        comp = mech["elem_comp"]
        iC, iH, iO = el.index("C"), el.index("H"), el.index("O")
        other = comp.sum(axis=1) - comp[:, iC] - comp[:, iH]
        fuel = [k for k in range(ns) if comp[k, iC] == 1 and other[k] == 0 and comp[k, iH] > 0]
        fuel = max(fuel, key=lambda k: comp[k, iH])
        o2 = [k for k in range(ns) if comp[k, iO] == 2 and comp[k].sum() == 2][0]
        return np.array([fuel, o2, ns - 1], dtype=np.int64)
    n_inert = len(KINDS[kind]["inert"]) if kind in KINDS else 0
    natoms = mech["elem_comp"].sum(axis=1)
    score = mech["h_formation"][: ns - n_inert] / natoms[: ns - n_inert]
    stable = np.argsort(score, kind="stable")[:n]
    return np.concatenate([np.sort(stable), [ns - 1]]).astype(np.int64)


def make_states(mech: dict, n_states: int, dist: str = "uniform", seed: int = 0) -> np.ndarray:
    """Synthetic PaSR-shaped states, returned as y[n_states, N] = (T, Y_1..Y_{N-1}), fp64.

    dist="uniform" (configs 0, 1, 3): T uniform in [800, 2400] K (h2co) / [800, 2600] K (gri);
      2-4 major species from a Dirichlet(alpha=1) over the major pool, the remaining species
      log-uniform in [1e-20, 1e-3], then normalised to sum 1.
    dist="ignition" (configs 2, 4): 60 % of the samples have T in the ignition band
      ([1000, 1400] K h2co, [1100, 1600] K gri), the rest as above; minor species
      log-uniform in [1e-12, 1e-4].
    The last species (N2) is dropped from the vector (it follows from sum Y = 1)."""
    ns = mech["n_species"]
    kind = mech.get("kind", "h2co")
    rng = np.random.default_rng([seed, ns, 1 if dist == "ignition" else 0])
    t_hi = 2400.0 if kind == "h2co" else 2600.0
    band = (1000.0, 1400.0) if kind == "h2co" else (1100.0, 1600.0)
    T = rng.uniform(800.0, t_hi, size=n_states)
    if dist == "ignition":
        in_band = rng.uniform(size=n_states) < 0.6
        T = np.where(in_band, rng.uniform(band[0], band[1], size=n_states), T)
        lo_e, hi_e = -12.0, -4.0
    elif dist == "uniform":
        lo_e, hi_e = -20.0, -3.0
    else:
        raise ValueError(dist)
    Y = 10.0 ** rng.uniform(lo_e, hi_e, size=(n_states, ns))
    pool = major_pool(mech)
    n_major = rng.integers(2, 5, size=n_states)
    if kind == "gri":
        n_major[:] = pool.size
    # random subset of the pool per state: rank random keys
    keys = rng.uniform(size=(n_states, pool.size))
    ranks = np.argsort(np.argsort(keys, axis=1), axis=1)
    is_major = ranks < n_major[:, None]
    g = rng.standard_exponential(size=(n_states, pool.size)) * is_major     # Dirichlet(1) via exponentials
    g /= g.sum(axis=1, keepdims=True)
    rows = np.arange(n_states)[:, None]
    Ymaj = np.zeros_like(Y)
    Ymaj[rows, pool[None, :]] = g
    maj_mask = np.zeros_like(Y, dtype=bool)
    maj_mask[rows, pool[None, :]] = is_major
    Y = np.where(maj_mask, Ymaj, Y)
    Y /= Y.sum(axis=1, keepdims=True)
    y = np.empty((n_states, ns))
    y[:, 0] = T
    y[:, 1:] = Y[:, : ns - 1]
    return np.ascontiguousarray(y)


# BASELINE.json configs[0..4]
CONFIGS = [
    dict(name="h2co_4k_dt1e-6", kind="h2co", n_states=4096, dist="uniform", t_end=1e-6),
    dict(name="h2co_1m_dt1e-6", kind="h2co", n_states=1048576, dist="uniform", t_end=1e-6),
    dict(name="h2co_1m_ign_dt1e-4", kind="h2co", n_states=1048576, dist="ignition", t_end=1e-4),
    dict(name="gri_512k_dt1e-6", kind="gri", n_states=524288, dist="uniform", t_end=1e-6),
    dict(name="gri_512k_ign_dt1e-4", kind="gri", n_states=524288, dist="ignition", t_end=1e-4),
]
P_ATM = 1.01325e6      # dyn/cm^2, the constant pressure of every config
RTOL, ATOL = 1e-6, 1e-10
MECH_SEED = 1607
STATE_SEED = 3884
