"""Small hand-built mechanisms and an independent numpy right-hand side used by the oracle pins.

`numpy_rhs` is written from the textbook definitions in matrix form with numpy's own exp/log (stoichiometric
matrices, no CSR loops, no gamma / rOF stabilisers): it is the *unstabilised* ODE the STEV method approximates,
used for brute-force and library (scipy) integration, not a copy of the oracle.
"""
import numpy as np

from stev_inputs.mechanisms import Mechanism, R_CAL, R_U, P_ATM


def build_mechanism(W, nasa_lo, nasa_hi, reactions, t_mid=1000.0, elem_comp=None):
    """reactions: list of (reactants [(species, nu)...], products [...], A, b, Ea_cal, reversible)."""
    S = len(W)
    rp, rs, rn, pp, ps, pn = [0], [], [], [0], [], []
    for reac, prod, *_ in reactions:
        for s, n in reac:
            rs.append(s); rn.append(n)
        rp.append(len(rs))
        for s, n in prod:
            ps.append(s); pn.append(n)
        pp.append(len(ps))
    i32 = lambda a: np.asarray(a, np.int32)
    return Mechanism(
        mol_weight=np.asarray(W, float), elem_comp=np.ones((S, 1)) if elem_comp is None else np.asarray(elem_comp, float),
        nasa_lo=np.asarray(nasa_lo, float), nasa_hi=np.asarray(nasa_hi, float), t_mid=np.full(S, float(t_mid)),
        A=np.array([r[2] for r in reactions], float), b=np.array([r[3] for r in reactions], float),
        Ea=np.array([r[4] for r in reactions], float), reversible=np.array([r[5] for r in reactions], np.uint8),
        reac_ptr=i32(rp), reac_species=i32(rs), reac_nu=i32(rn), prod_ptr=i32(pp), prod_species=i32(ps), prod_nu=i32(pn))


def flat_thermo(S, cp_over_R=3.5, a6=None, a7=None):
    """Constant cp/R, chosen a6 (enthalpy offset, K) and a7 (entropy constant); both ranges equal."""
    lo = np.zeros((S, 7))
    lo[:, 0] = cp_over_R
    if a6 is not None:
        lo[:, 5] = a6
    if a7 is not None:
        lo[:, 6] = a7
    return lo, lo.copy()


def nasa_numpy(mech, T):
    """cp/R, h/RT, s/R from Eqs 15-16 + entropy, in plain numpy powers (not Horner)."""
    a = np.where((T < mech.t_mid)[:, None], mech.nasa_lo, mech.nasa_hi)
    cp = a[:, 0] + a[:, 1] * T + a[:, 2] * T**2 + a[:, 3] * T**3 + a[:, 4] * T**4
    h = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T**2 / 3 + a[:, 3] * T**3 / 4 + a[:, 4] * T**4 / 5 + a[:, 5] / T
    s = a[:, 0] * np.log(T) + a[:, 1] * T + a[:, 2] * T**2 / 2 + a[:, 3] * T**3 / 3 + a[:, 4] * T**4 / 4 + a[:, 6]
    return cp, h, s


def _entries(mech, which, ptr, sp, default):
    R, S = mech.n_reactions, mech.n_species
    vals = getattr(mech, which, None)
    vals = default if vals is None else vals
    out = np.zeros((R, S))
    for j in range(R):
        for e in range(ptr[j], ptr[j + 1]):
            out[j, sp[e]] += vals[e]
    return out


def stoich(mech):
    """Stoichiometric coefficient matrices [R, S] of reactants and products (real ones if the mechanism has them)."""
    return (_entries(mech, "reac_coef", mech.reac_ptr, mech.reac_species, mech.reac_nu),
            _entries(mech, "prod_coef", mech.prod_ptr, mech.prod_species, mech.prod_nu))


def orders(mech):
    """Rate-law exponent matrices [R, S] (Eq 28): the orders if given, else the coefficients."""
    nu_r, nu_p = stoich(mech)
    o_r = nu_r if getattr(mech, "reac_order", None) is None else _entries(mech, "reac_order", mech.reac_ptr, mech.reac_species, None)
    o_p = nu_p if getattr(mech, "prod_order", None) is None else _entries(mech, "prod_order", mech.prod_ptr, mech.prod_species, None)
    return o_r, o_p


def rate_constants_numpy(mech, T):
    """k_f [R], K_c [R] (Eq 30) with numpy exp/log."""
    nu_r, nu_p = stoich(mech)
    _, h, s = nasa_numpy(mech, T)
    g = h - s
    kf = mech.A * T**mech.b * np.exp(-mech.Ea / (R_CAL * T))
    dnu = (nu_p - nu_r).sum(axis=1)
    Kc = (P_ATM / (R_U * T)) ** dnu * np.exp(-((nu_p - nu_r) @ g))
    return kf, Kc


def numpy_rhs(mech, T, p, Y, isothermal=False):
    """Unstabilised d(Y)/dt [S], dT/dt for one cell: mass action with K_c-based reverse rates."""
    nu_r, nu_p = stoich(mech)
    cp, h, _ = nasa_numpy(mech, T)
    W = mech.mol_weight
    rho = p / (R_U * T) / np.sum(Y / W)
    C = np.maximum(rho * Y / W, 0.0)
    kf, Kc = rate_constants_numpy(mech, T)
    o_r, o_p = orders(mech)
    fwd = kf * np.prod(C[None, :] ** o_r, axis=1)
    rev = np.where(mech.reversible == 1, kf / Kc * np.prod(C[None, :] ** o_p, axis=1), 0.0)
    q = fwd - rev
    omega = (nu_p - nu_r).T @ q
    dY = W * omega / rho
    cp_mass = R_U * np.sum(Y * cp / W)
    dT = 0.0 if isothermal else -np.sum(h * R_U * T * omega) / (rho * cp_mass)
    return dY, dT, q
