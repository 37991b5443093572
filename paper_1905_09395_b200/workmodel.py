"""Algorithmic work of one STEV cell-step: the fp64 operations the method itself requires,
counted from the paper's equations and the arithmetic contract -- not from the kernel's SASS.  Used by bench.py for the
roofline numerator.  Pure counting: no solver arithmetic lives here.

Conventions: FMA = 1 instruction = 2 flop; add, mul, div, sqrt = 1 instruction = 1 flop (a division or square root is
counted once although the hardware expands it into a Newton sequence, so the reported fraction is conservative);
compares, selects, min/max, integer and bit operations, and loads/stores count as 0.
"""
from __future__ import annotations

import dataclasses

# contract exp: fma(shift), sub, 2 fma (Cody-Waite), 13 fma (Horner), 1 mul (2^k)
EXP_FMA, EXP_OTHER = 16, 2
# contract log: (m-1), (m+1), div, f*f, 11 fma, f+f, s*P, fma, 2 fma (e*ln2 hi/lo)
LOG_FMA, LOG_OTHER = 14, 6


@dataclasses.dataclass
class CellStepWork:
    fma: float
    other: float
    fp32_fma: float  # estimator layers (fp32 CUDA-core path)

    @property
    def fp64_instr(self) -> float:
        return self.fma + self.other

    @property
    def fp64_flop(self) -> float:
        return 2.0 * self.fma + self.other


def cell_step_work(mech, estimator=None, dft_enable: bool = True, first_high_bin: int = 4, alpha_on: bool = True,
                   adiabatic: bool = True) -> CellStepWork:
    """fp64 work of steps 1-9 of DESIGN.md section 2 for one cell and one integrator step."""
    S, R = int(mech.n_species), int(mech.n_reactions)
    rev = [j for j in range(R) if mech.reversible[j]]
    Rrev = len(rev)
    nu_reac = [int(sum(mech.reac_nu[mech.reac_ptr[j]:mech.reac_ptr[j + 1]])) for j in range(R)]
    nu_prod = [int(sum(mech.prod_nu[mech.prod_ptr[j]:mech.prod_ptr[j + 1]])) for j in range(R)]
    ent_reac = [int(mech.reac_ptr[j + 1] - mech.reac_ptr[j]) for j in range(R)]
    ent_prod = [int(mech.prod_ptr[j + 1] - mech.prod_ptr[j]) for j in range(R)]
    fma = other = f32 = 0.0
    # 1. thermo: ln T, 1/T; per species h/RT (5 fma), s/R (5 fma), g = h - s; cp/R (4 fma) unless the MLP supplies it
    fma += LOG_FMA
    other += LOG_OTHER + 1
    fma += S * (10 + (0 if estimator is not None else 4))
    other += S
    if estimator is not None:
        H, n_in, n_out = estimator.n_hidden, estimator.n_in, estimator.n_out
        f32 += H * n_in + n_out * H  # both layers are fp32 fmaf; the input normalisation is fp32 too
        # activation through the contract exp in fp64: 2z, exp, 1+e, 2/(.), 1-(.)
        fma += H * EXP_FMA
        other += H * (EXP_OTHER + 4)
        other += S * 2  # h/RT = (out * T_ref) / T  (mul, mul)
    # 2. mixture: 1/Wbar (S fma), C_tot = p / (Ru T), rho = C_tot / (1/Wbar); concentrations (2 mul) and gamma (add, div, mul)
    fma += S
    other += 3
    other += S * (2 + (3 if alpha_on else 0))
    # 3.-4. ln(p_atm/(Ru T)); per reaction ln k_f (2 fma), exp, concentration products; reversible: dG sum, ln K_c, exp,
    #        products, (fwd - rev) * rOF
    fma += LOG_FMA
    other += LOG_OTHER + 2
    fma += R * (2 + EXP_FMA)
    other += R * EXP_OTHER + sum(nu_reac)
    for j in rev:
        other += 2 * (ent_reac[j] + ent_prod[j])  # coef * g, accumulate
        fma += 1 + EXP_FMA
        other += 1 + EXP_OTHER + nu_prod[j] + 2
    # 5. omega gather (mul + add per stoichiometric entry), r_i (2 mul), 1/rho, enthalpy and cp sums, dT/dt
    other += 2 * (sum(ent_reac) + sum(ent_prod))
    other += 2 * S + 1
    if adiabatic:
        fma += 2 * S
        other += S + 5
    # 6. limiter: 0.9 y, one division per species; remaining time
    other += 2 * S + 2
    # 7. Euler update
    fma += S + 1
    other += 1
    # 8. DFT: store (2 mul, one shared 1/C_tot), bin 0 (13 adds), high bins (26 fma + mul + fma + sqrt each), ratio, rOF
    if dft_enable:
        nb = 7 - first_high_bin
        other += 1
        fma += Rrev * nb * 27
        other += Rrev * (2 + 13 + nb * 2 + 2)
    return CellStepWork(fma=fma, other=other, fp32_fma=f32)


# B200 fp64 pipe peak used as the "alu" roofline denominator: 148 SMs x 64 DFMA / clk / SM at the
# maximum SM clock nvidia-smi reports (1965 MHz).  The 64/clk/SM figure is the sm_100 fp64 unit count implied by
# NVIDIA's 40 TFLOP/s fp64 figure for B200; bench.py also measures a DFMA microbenchmark in the same run.
SM_COUNT = 148
DFMA_PER_CLK_PER_SM = 64


def fp64_peak_instr_per_s(sm_mhz: float = 1965.0) -> float:
    return SM_COUNT * DFMA_PER_CLK_PER_SM * sm_mhz * 1e6
