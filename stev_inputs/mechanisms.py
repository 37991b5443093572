"""Seeded synthetic reaction mechanisms.

No real mechanism or thermodynamic data is written here: everything is drawn from
`numpy.random.default_rng(seed)`.  Units are cgs-mol ("cm, s, mol, cal").
"""
from __future__ import annotations

import dataclasses
import itertools

import numpy as np

ATOMIC_WEIGHTS = np.array([1.008, 15.999, 12.011, 14.007])
R_CAL = 1.98720425864083  # cal/(mol K)
R_U = 8.31446261815324e7  # erg/(mol K)
P_ATM = 1.01325e6  # dyn/cm^2
T_SPLIT = 1000.0


@dataclasses.dataclass
class Mechanism:
    """Species, NASA-7 thermo and Arrhenius reactions; the fields of `stev_mechanism_desc`."""

    mol_weight: np.ndarray  # [S]
    elem_comp: np.ndarray  # [S, E]
    nasa_lo: np.ndarray  # [S, 7]
    nasa_hi: np.ndarray  # [S, 7]
    t_mid: np.ndarray  # [S]
    A: np.ndarray  # [R]
    b: np.ndarray  # [R]
    Ea: np.ndarray  # [R] cal/mol
    reversible: np.ndarray  # [R] uint8
    reac_ptr: np.ndarray  # [R+1] int32
    reac_species: np.ndarray
    reac_nu: np.ndarray
    prod_ptr: np.ndarray
    prod_species: np.ndarray
    prod_nu: np.ndarray
    seed: int = 0
    stiffness_scale: float = 1.0
    # optional, one value per CSR entry (BFER): real stoichiometric coefficients (default nu) and
    # rate-law exponents (default the coefficient)
    reac_coef: np.ndarray | None = None
    prod_coef: np.ndarray | None = None
    reac_order: np.ndarray | None = None
    prod_order: np.ndarray | None = None

    @property
    def n_species(self) -> int:
        return int(self.mol_weight.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.A.shape[0])

    @property
    def n_reversible(self) -> int:
        return int(self.reversible.sum())

    def stoich_matrix(self) -> np.ndarray:
        """Net stoichiometric coefficients [R, S] (products minus reactants)."""
        nu = np.zeros((self.n_reactions, self.n_species))
        rc = self.reac_nu if self.reac_coef is None else self.reac_coef
        pc = self.prod_nu if self.prod_coef is None else self.prod_coef
        for j in range(self.n_reactions):
            for e in range(self.reac_ptr[j], self.reac_ptr[j + 1]):
                nu[j, self.reac_species[e]] -= rc[e]
            for e in range(self.prod_ptr[j], self.prod_ptr[j + 1]):
                nu[j, self.prod_species[e]] += pc[e]
        return nu


def _csr(sides):
    ptr = [0]
    sp, nu = [], []
    for side in sides:
        for s, n in side:
            sp.append(s)
            nu.append(n)
        ptr.append(len(sp))
    return (np.asarray(ptr, np.int32), np.asarray(sp, np.int32), np.asarray(nu, np.int32))


def _finish_high_range(lo: np.ndarray, slope_scale: np.ndarray) -> np.ndarray:
    """High range = perturbed slopes, with a1, a6, a7 solved so cp, h, s are continuous at T_SPLIT."""
    hi = lo.copy()
    hi[:, 1] = lo[:, 1] * slope_scale[:, 0]
    hi[:, 2] = lo[:, 2] * slope_scale[:, 1]
    T = T_SPLIT
    # cp/R continuity -> a1
    cp_lo = lo[:, 0] + lo[:, 1] * T + lo[:, 2] * T**2
    hi[:, 0] = cp_lo - hi[:, 1] * T - hi[:, 2] * T**2
    # h/RT continuity -> a6
    h_lo = lo[:, 0] + lo[:, 1] * T / 2 + lo[:, 2] * T**2 / 3 + lo[:, 5] / T
    hi[:, 5] = (h_lo - hi[:, 0] - hi[:, 1] * T / 2 - hi[:, 2] * T**2 / 3) * T
    # s/R continuity -> a7
    s_lo = lo[:, 0] * np.log(T) + lo[:, 1] * T + lo[:, 2] * T**2 / 2 + lo[:, 6]
    hi[:, 6] = s_lo - hi[:, 0] * np.log(T) - hi[:, 1] * T - hi[:, 2] * T**2 / 2
    return hi


def _g_rt(coef: np.ndarray, T: float) -> np.ndarray:
    h = coef[:, 0] + coef[:, 1] * T / 2 + coef[:, 2] * T**2 / 3 + coef[:, 3] * T**3 / 4 + coef[:, 4] * T**4 / 5 + coef[:, 5] / T
    s = coef[:, 0] * np.log(T) + coef[:, 1] * T + coef[:, 2] * T**2 / 2 + coef[:, 3] * T**3 / 3 + coef[:, 4] * T**4 / 4 + coef[:, 6]
    return h - s


def abc_mechanism(seed: int = 190509395) -> Mechanism:
    """Config 0: A <=> B (k = 1e10 exp(-15000/T) 1/s, reverse from K_c) plus stiff B -> C
    (k = 1e14 exp(-10000/T) 1/s).  Three isomers of one element, equal W, NASA-7 thermo seeded near
    linear cp with a moderate heat release (keeps T < 3000 K)."""
    rng = np.random.default_rng(seed)
    S = 3
    lo = np.zeros((S, 7))
    lo[:, 0] = 3.5 + rng.uniform(-0.05, 0.05, S)
    lo[:, 1] = 1.0e-3 * rng.uniform(0.9, 1.1, S)
    lo[:, 2] = -1.0e-8 * rng.uniform(0.0, 1.0, S)
    lo[:, 5] = np.array([0.0, -1000.0, -3000.0]) * rng.uniform(0.95, 1.05, S)
    lo[:, 6] = 5.0 + rng.uniform(-0.2, 0.2, S)
    hi = _finish_high_range(lo, rng.uniform(0.8, 1.0, (S, 2)))
    reac = [[(0, 1)], [(1, 1)]]
    prod = [[(1, 1)], [(2, 1)]]
    rp, rs, rn = _csr(reac)
    pp, ps, pn = _csr(prod)
    return Mechanism(
        mol_weight=np.full(S, 28.0),
        elem_comp=np.ones((S, 1)),
        nasa_lo=lo, nasa_hi=hi, t_mid=np.full(S, T_SPLIT),
        A=np.array([1.0e10, 1.0e14]), b=np.zeros(2), Ea=np.array([15000.0, 10000.0]) * R_CAL,
        reversible=np.array([1, 0], np.uint8),
        reac_ptr=rp, reac_species=rs, reac_nu=rn, prod_ptr=pp, prod_species=ps, prod_nu=pn,
        seed=seed, stiffness_scale=1.0,
    )


def _species_compositions(n_species: int, n_elements: int, rng) -> np.ndarray:
    """The S smallest element-count vectors (1 <= total atoms <= 4), ties shuffled by seed."""
    comps = []
    for total in range(1, 5):
        level = [c for c in itertools.product(range(total + 1), repeat=n_elements) if sum(c) == total]
        order = rng.permutation(len(level))
        comps.extend(level[k] for k in order)
    if len(comps) < n_species:
        raise ValueError("not enough compositions for the requested number of species")
    return np.asarray(comps[:n_species], dtype=np.int64)


def _candidate_reactions(comp: np.ndarray, n_reactive: int):
    """All pairs of disjoint species multisets of size <= 2 with equal element sums."""
    sides = [((i, 1),) for i in range(n_reactive)]
    sides += [((i, 2),) for i in range(n_reactive)]
    sides += [((i, 1), (k, 1)) for i in range(n_reactive) for k in range(i + 1, n_reactive)]
    by_sum = {}
    for side in sides:
        key = tuple(sum(comp[s] * n for s, n in side))
        by_sum.setdefault(key, []).append(side)
    cands = []
    for group in by_sum.values():
        for a, b in itertools.combinations(group, 2):
            if {s for s, _ in a} & {s for s, _ in b}:
                continue
            cands.append((a, b))
    return cands


def synthetic_mechanism(n_species: int, n_reactions: int, n_elements: int, seed: int,
                        stiffness_scale: float = 1.0, inert_last: bool = False,
                        max_tries: int = 200) -> Mechanism:
    """Element-conserving random mechanism: <= 2 reactants / <= 2 products drawn by seed,
    A ~ logU[1e8,1e14] * stiffness_scale, b ~ U[-1,2], Ea ~ U[0,50] kcal/mol (BASELINE config 1),
    reversible with probability 0.7.  Rejected and redrawn if |ln K_c| > 60 on [800,3000] K or cp <= 0."""
    for attempt in range(max_tries):
        rng = np.random.default_rng([seed, attempt])
        comp = _species_compositions(n_species, n_elements, rng)
        n_atoms = comp.sum(axis=1)
        W = comp @ ATOMIC_WEIGHTS[:n_elements]
        lo = np.zeros((n_species, 7))
        lo[:, 0] = 2.5 + (n_atoms - 1) * rng.uniform(0.6, 1.0, n_species)
        lo[:, 1] = n_atoms * rng.uniform(0.2, 1.0, n_species) * 1e-3
        lo[:, 2] = -n_atoms * rng.uniform(0.0, 1.0, n_species) * 1e-7
        lo[:, 5] = -5000.0 * (n_atoms - 1) * rng.uniform(0.5, 1.5, n_species)
        lo[:, 6] = rng.uniform(2.0, 8.0, n_species)
        hi = _finish_high_range(lo, rng.uniform(0.6, 1.0, (n_species, 2)))
        n_reactive = n_species - 1 if inert_last else n_species
        cands = _candidate_reactions(comp, n_reactive)
        if len(cands) < n_reactions:
            raise ValueError(f"only {len(cands)} candidate reactions for {n_species} species")
        pick = rng.choice(len(cands), size=n_reactions, replace=False)
        flip = rng.random(n_reactions) < 0.5
        reac, prod = [], []
        for k, f in zip(pick, flip):
            a, b = cands[k]
            reac.append(list(b if f else a))
            prod.append(list(a if f else b))
        A = 10.0 ** rng.uniform(8.0, 14.0, n_reactions) * stiffness_scale
        bexp = rng.uniform(-1.0, 2.0, n_reactions)
        Ea = rng.uniform(0.0, 50.0, n_reactions) * 1000.0
        reversible = (rng.random(n_reactions) < 0.7).astype(np.uint8)
        rp, rs, rn = _csr(reac)
        pp, ps, pn = _csr(prod)
        mech = Mechanism(mol_weight=W, elem_comp=comp.astype(np.float64), nasa_lo=lo, nasa_hi=hi,
                         t_mid=np.full(n_species, T_SPLIT), A=A, b=bexp, Ea=Ea, reversible=reversible,
                         reac_ptr=rp, reac_species=rs, reac_nu=rn, prod_ptr=pp, prod_species=ps, prod_nu=pn,
                         seed=seed, stiffness_scale=stiffness_scale)
        # acceptance: cp > 0 and |ln K_c| <= 60 on [800, 3000] K
        ok = True
        nu = mech.stoich_matrix()
        dnu = nu.sum(axis=1)
        for T in np.linspace(300.0, 3000.0, 28):
            coef = lo if T < T_SPLIT else hi
            cp = coef[:, 0] + coef[:, 1] * T + coef[:, 2] * T**2
            if np.any(cp <= 0):
                ok = False
                break
            if T >= 800.0:
                ln_kc = -(nu @ _g_rt(coef, T)) + dnu * np.log(P_ATM / (R_U * T))
                if np.any(np.abs(ln_kc[reversible == 1]) > 60.0):
                    ok = False
                    break
        if ok:
            return mech
    raise RuntimeError("no acceptable mechanism found")


def bfer_shaped_mechanism(seed: int = 190509395 + 70) -> Mechanism:
    """A mechanism with the SHAPE of the paper's BFER methane case: six species with the element
    compositions of CH4, O2, CO, H2O, CO2, N2 and two reactions,
        MEPOX  CH4 + 1.5 O2 -> CO + 2 H2O,  rate k exp(-Ea/RT) C_CH4^0.5 C_O2^0.65      (Eqs 26, 28)
        COROX  CO + 0.5 O2 <=> CO2,         rate k T^0.7 exp(-Ea/RT) (C_CO C_O2^0.5 - C_CO2 / K)   (Eqs 27, 29, 30)
    with the constants the paper prints in Table 1 (k = 4.9e9 / 2.0e8, Ea = 35500 / 12000 cal/mol; cm, s, mol, cal).
    The NASA-7 THERMODYNAMICS ARE SYNTHETIC (seeded, near-linear cp, like every other mechanism here): the real
    coefficients are not in this repository, so temperatures and equilibria are not those of methane combustion."""
    rng = np.random.default_rng([seed, 0])
    comp = np.array([[4, 0, 1, 0], [0, 2, 0, 0], [0, 1, 1, 0], [2, 1, 0, 0], [0, 2, 1, 0], [0, 0, 0, 2]], dtype=np.float64)  # H O C N
    n_atoms = comp.sum(axis=1)
    W = comp @ ATOMIC_WEIGHTS
    S = 6
    lo = np.zeros((S, 7))
    lo[:, 0] = 2.5 + (n_atoms - 1) * rng.uniform(0.6, 1.0, S)
    lo[:, 1] = n_atoms * rng.uniform(0.2, 1.0, S) * 1e-3
    lo[:, 2] = -n_atoms * rng.uniform(0.0, 1.0, S) * 1e-7
    # enthalpy offsets (K) chosen so that both reactions release heat, moderately: fuel and oxidiser high, products low
    lo[:, 5] = np.array([-9000.0, 0.0, -13000.0, -29000.0, -47000.0, 0.0]) * rng.uniform(0.9, 1.1, S)
    lo[:, 6] = rng.uniform(2.0, 8.0, S)
    hi = _finish_high_range(lo, rng.uniform(0.6, 1.0, (S, 2)))
    i32 = lambda a: np.asarray(a, np.int32)
    return Mechanism(mol_weight=W, elem_comp=comp, nasa_lo=lo, nasa_hi=hi, t_mid=np.full(S, T_SPLIT),
                     A=np.array([4.9e9, 2.0e8]), b=np.array([0.0, 0.7]), Ea=np.array([35500.0, 12000.0]),
                     reversible=np.array([0, 1], np.uint8),
                     reac_ptr=i32([0, 2, 4]), reac_species=i32([0, 1, 2, 1]), reac_nu=i32([1, 2, 1, 1]),
                     prod_ptr=i32([0, 2, 3]), prod_species=i32([2, 3, 4]), prod_nu=i32([1, 2, 1]),
                     seed=seed,
                     reac_coef=np.array([1.0, 1.5, 1.0, 0.5]), prod_coef=np.array([1.0, 2.0, 1.0]),
                     reac_order=np.array([0.5, 0.65, 1.0, 0.5]), prod_order=np.array([1.0, 2.0, 1.0]))


def bfer_shaped_field(n: int, seed: int = 190509395 + 71):
    """Random fixed thermochemical states: T0 ~ U[1000, 2200] K, p = 1 atm, lean-to-rich mixtures of the
    fuel and oxidiser species in the inert one, with traces of the products."""
    rng = np.random.default_rng([seed, n])
    T = rng.uniform(1000.0, 2200.0, n)
    Y = np.zeros((6, n))
    Y[0] = rng.uniform(0.0, 0.08, n)          # fuel
    Y[1] = rng.uniform(0.05, 0.25, n)         # oxidiser
    Y[2] = rng.uniform(0.0, 0.02, n)
    Y[3] = rng.uniform(0.0, 0.05, n)
    Y[4] = rng.uniform(0.0, 0.05, n)
    Y[5] = 1.0 - Y[:5].sum(axis=0)
    return T, np.full(n, P_ATM), np.ascontiguousarray(Y)
