"""Seeded synthetic reaction-mechanism generator (inputs only, no kinetics).

This module draws the *data* of a mechanism -- element counts, stoichiometric
matrices nu' / nu'' (Eq. 1), Arrhenius parameters (PAPER.md:72-76,
Eq. 5), NASA-7 polynomial coefficients with a cutoff temperature,
third-body efficiencies E and Troe parameters -- with the
shapes and distributions BASELINE.json's `configs` state.  It stands in for the
paper's mechanism files (Table 1), which are not available.

It serves both the CPU oracle and the CUDA library and therefore contains none of
the method's arithmetic: no rate constants, no equilibrium constants, no rates.  The
only formulas here are those needed to *shape the inputs* (integrals of the sampled
cp polynomial so that h and s are continuous at T_mid).

Recipe:
  species   S distinct non-zero element-count vectors, counts iid in 0..3
  W_k       sum_e n_ek * atomic weight
  reactions rejection sampled: draw class (n_reac, n_prod) uniformly from {1,2,3}^2,
            draw a reactant side (distinct species, coefficients 1..2), then a
            product side of the wanted size with the same element vector and no
            species in common; reject duplicates (either orientation)
  rates     ln A ~ U[ln 1e6, ln 1e14], b ~ U[-2, 2], Ea ~ U[0, 2e5] J/mol
  NASA-7    T_mid = 1000 K; cp/R piecewise quartic in [2.5, 10] on 300..3500 K,
            h(298.15)/R ~ U[-3e4, 3e4] K, s(298.15)/R ~ U[15, 40]; h, s, cp
            continuous at T_mid
  types     floor(frac*R + 0.5) three-body and Troe reactions, disjoint sets chosen
            by a seeded permutation; efficiencies iid U[0.5, 5] for every species
            of such a reaction; low-pressure Arrhenius set drawn like the main one;
            Troe alpha ~ U[0.3, 0.9], T***, T*, T** ~ U[1e2, 1e4] K
"""
from __future__ import annotations

import dataclasses
import itertools

import numpy as np

ATOMIC_WEIGHT = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999, "Ar": 39.95}
R_GAS_J_PER_MOL_K = 8.31446261815324  # converts the config's Ea [J/mol] to Ea/R [K]
P_ATM = 101325.0

# reaction type codes shared by every consumer of a Mechanism (data convention only)
ELEMENTARY, THREE_BODY, LINDEMANN, TROE = 0, 1, 2, 3


@dataclasses.dataclass
class Mechanism:
    """Plain arrays describing one mechanism. All float64 / uint8, C-contiguous."""

    elements: tuple            # element names, length n_elem
    elem_count: np.ndarray     # [S, n_elem] int64, atoms of element e in species k
    mol_weight: np.ndarray     # [S] kg/kmol
    nu_reac: np.ndarray        # [S, R] nu'
    nu_prod: np.ndarray        # [S, R] nu''
    ln_A: np.ndarray           # [R]
    b: np.ndarray              # [R]
    Ea_over_R: np.ndarray      # [R] K
    reversible: np.ndarray     # [R] uint8
    nasa_lo: np.ndarray        # [S, 7] a1..a7 for T <= T_mid
    nasa_hi: np.ndarray        # [S, 7] a1..a7 for T >  T_mid
    T_mid: np.ndarray          # [S] K
    rxn_type: np.ndarray       # [R] uint8: 0 elementary, 1 three-body, 2 Lindemann, 3 Troe
    eff: np.ndarray            # [S, R] third-body efficiencies (1 where unused)
    ln_A0: np.ndarray          # [R] low-pressure limit (0 where unused)
    b0: np.ndarray             # [R]
    Ea0_over_R: np.ndarray     # [R]
    troe: np.ndarray           # [R, 4] alpha, T***, T*, T** (T** = +inf -> 3-parameter)
    p_ref: float               # Pa, standard-state pressure of the NASA data
    seed: int = 0

    @property
    def n_species(self) -> int:
        return int(self.nu_reac.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.nu_reac.shape[1])

    def subset(self, reactions) -> "Mechanism":
        """Mechanism with the same species and only the given reactions (test helper)."""
        j = np.asarray(reactions, dtype=np.int64)
        c = np.ascontiguousarray
        return dataclasses.replace(
            self,
            nu_reac=c(self.nu_reac[:, j]), nu_prod=c(self.nu_prod[:, j]),
            ln_A=c(self.ln_A[j]), b=c(self.b[j]), Ea_over_R=c(self.Ea_over_R[j]),
            reversible=c(self.reversible[j]), rxn_type=c(self.rxn_type[j]),
            eff=c(self.eff[:, j]), ln_A0=c(self.ln_A0[j]), b0=c(self.b0[j]),
            Ea0_over_R=c(self.Ea0_over_R[j]), troe=c(self.troe[j]),
        )


# --------------------------------------------------------------------------- species

def _draw_species(rng, S, elements):
    n_elem = len(elements)
    seen, rows = set(), []
    while len(rows) < S:
        v = tuple(int(x) for x in rng.integers(0, 4, size=n_elem))
        if sum(v) == 0 or v in seen:
            continue
        seen.add(v)
        rows.append(v)
    elem_count = np.array(rows, dtype=np.int64)
    w = np.array([ATOMIC_WEIGHT[e] for e in elements])
    return elem_count, elem_count @ w


# --------------------------------------------------------------------------- reactions

def _enumerate_sides(S, elem_count):
    """All 'sides': 1..3 distinct species with coefficients 1..2.

    Returns per size n: species index array [M, n], coefficient array [M, n] and an
    int64 key encoding the side's element vector (base 19 digits: a count is <= 18).
    """
    out = {}
    base = 19
    n_elem = elem_count.shape[1]
    weights = base ** np.arange(n_elem, dtype=np.int64)
    for n in (1, 2, 3):
        combos = np.array(list(itertools.combinations(range(S), n)), dtype=np.int64)
        coefs = np.array(list(itertools.product((1, 2), repeat=n)), dtype=np.int64)
        sp = np.repeat(combos, len(coefs), axis=0)
        cf = np.tile(coefs, (len(combos), 1))
        evec = np.einsum("mn,mne->me", cf, elem_count[sp])
        key = evec @ weights
        order = np.argsort(key, kind="stable")
        out[n] = (sp[order], cf[order], key[order])
    return out


def _draw_reactions(rng, S, R, elem_count):
    sides = _enumerate_sides(S, elem_count)
    nu_reac = np.zeros((S, R))
    nu_prod = np.zeros((S, R))
    seen = set()
    j = 0
    attempts = 0
    while j < R:
        attempts += 1
        if attempts > 200000 + 2000 * R:
            raise RuntimeError("cannot draw %d balanced reactions for this seed" % R)
        n_r = int(rng.integers(1, 4))
        n_p = int(rng.integers(1, 4))
        sp_r, cf_r, key_r = sides[n_r]
        sp_p, cf_p, key_p = sides[n_p]
        # a few tries for this class, then redraw the class
        for _ in range(64):
            i = int(rng.integers(0, len(key_r)))
            lo = np.searchsorted(key_p, key_r[i], side="left")
            hi = np.searchsorted(key_p, key_r[i], side="right")
            if hi == lo:
                continue
            cand = np.arange(lo, hi)
            disjoint = ~np.isin(sp_p[cand], sp_r[i]).any(axis=1)
            cand = cand[disjoint]
            if len(cand) == 0:
                continue
            c = int(cand[int(rng.integers(0, len(cand)))])
            a = tuple(sorted(zip(sp_r[i].tolist(), cf_r[i].tolist())))
            bb = tuple(sorted(zip(sp_p[c].tolist(), cf_p[c].tolist())))
            if (a, bb) in seen or (bb, a) in seen:
                continue
            seen.add((a, bb))
            if rng.random() < 0.5:   # random orientation
                a, bb = bb, a
            for k, v in a:
                nu_reac[k, j] = v
            for k, v in bb:
                nu_prod[k, j] = v
            j += 1
            break
    return nu_reac, nu_prod


# --------------------------------------------------------------------------- NASA-7

def _cp_poly(rng, T0, T1, c0, c1):
    """Quartic cp/R(T) on [T0, T1]: the line through (T0,c0),(T1,c1) plus 'bubble'
    terms vanishing at both ends, so all of a1..a5 are non-zero. Monomial coefficients
    in T, lowest order first (numpy.polynomial convention)."""
    P = np.polynomial.polynomial
    line = np.array([c0 - (c1 - c0) * T0 / (T1 - T0), (c1 - c0) / (T1 - T0)])
    # x = (T - T0)/(T1 - T0) in [0,1]; bubble = x(1-x)(g0 + g1 x + g2 x^2)
    x = np.array([-T0 / (T1 - T0), 1.0 / (T1 - T0)])
    one_minus_x = P.polysub([1.0], x)
    g = rng.uniform(-1.0, 1.0, size=3)
    inner = P.polyadd(P.polyadd([g[0]], g[1] * x), g[2] * P.polymul(x, x))
    bubble = P.polymul(P.polymul(x, one_minus_x), inner)
    # |x(1-x)| <= 1/4 and |inner| <= 3 on [0,1]  ->  scale so the amplitude is <= 0.5
    bubble = bubble * (0.5 / 0.75)
    out = P.polyadd(line, bubble)
    return np.pad(out, (0, 5 - len(out)))


def _draw_nasa(rng, S, T_mid=1000.0, T_lo=300.0, T_hi=3500.0):
    P = np.polynomial.polynomial
    nasa_lo = np.zeros((S, 7))
    nasa_hi = np.zeros((S, 7))
    T_ref = 298.15
    for k in range(S):
        while True:
            c300 = rng.uniform(2.5, 5.0)
            c1000 = rng.uniform(c300, 8.0)
            c3500 = rng.uniform(c1000, 10.0)
            lo = _cp_poly(rng, T_lo, T_mid, c300, c1000)
            hi = _cp_poly(rng, T_mid, T_hi, c1000, c3500)
            g_lo = P.polyval(np.linspace(T_lo, T_mid, 65), lo)
            g_hi = P.polyval(np.linspace(T_mid, T_hi, 65), hi)
            if min(g_lo.min(), g_hi.min()) >= 2.5 and max(g_lo.max(), g_hi.max()) <= 10.0:
                break
        h298 = rng.uniform(-3.0e4, 3.0e4)   # h(298.15)/R  [K]
        s298 = rng.uniform(15.0, 40.0)      # s(298.15)/R

        def h_int(a, T):  # integral of cp/R dT without the constant
            return sum(a[i] * T ** (i + 1) / (i + 1) for i in range(5))

        def s_int(a, T):  # integral of cp/(R T) dT without the constant
            return a[0] * np.log(T) + sum(a[i] * T ** i / i for i in range(1, 5))

        a6_lo = h298 - h_int(lo, T_ref)
        a7_lo = s298 - s_int(lo, T_ref)
        a6_hi = (h_int(lo, T_mid) + a6_lo) - h_int(hi, T_mid)
        a7_hi = (s_int(lo, T_mid) + a7_lo) - s_int(hi, T_mid)
        nasa_lo[k, :5], nasa_lo[k, 5], nasa_lo[k, 6] = lo, a6_lo, a7_lo
        nasa_hi[k, :5], nasa_hi[k, 5], nasa_hi[k, 6] = hi, a6_hi, a7_hi
    return nasa_lo, nasa_hi, np.full(S, T_mid)


# --------------------------------------------------------------------------- assemble

def type_counts(R, frac_three_body, frac_falloff):
    """floor(frac*R + 0.5), reading of BASELINE.json's percentages."""
    return int(np.floor(frac_three_body * R + 0.5)), int(np.floor(frac_falloff * R + 0.5))


def generate_mechanism(S, R, elements, seed, frac_three_body, frac_falloff,
                       eff_density=1.0, falloff_kind=TROE) -> Mechanism:
    """Draw a mechanism; deterministic in (all arguments)."""
    rng = np.random.default_rng(seed)
    elements = tuple(elements)
    elem_count, W = _draw_species(rng, S, elements)
    nu_reac, nu_prod = _draw_reactions(rng, S, R, elem_count)

    ln_A = rng.uniform(np.log(1e6), np.log(1e14), size=R)
    b = rng.uniform(-2.0, 2.0, size=R)
    Ea_over_R = rng.uniform(0.0, 2.0e5, size=R) / R_GAS_J_PER_MOL_K
    nasa_lo, nasa_hi, T_mid = _draw_nasa(rng, S)

    n_tb, n_fo = type_counts(R, frac_three_body, frac_falloff)
    perm = rng.permutation(R)
    rxn_type = np.zeros(R, dtype=np.uint8)
    rxn_type[perm[:n_tb]] = THREE_BODY
    rxn_type[perm[n_tb:n_tb + n_fo]] = falloff_kind

    eff = np.ones((S, R))
    ln_A0 = np.zeros(R)
    b0 = np.zeros(R)
    Ea0_over_R = np.zeros(R)
    troe = np.zeros((R, 4))
    for j in np.flatnonzero(rxn_type != ELEMENTARY):
        col = rng.uniform(0.5, 5.0, size=S)
        if eff_density < 1.0:
            keep = rng.random(S) < eff_density
            col = np.where(keep, col, 1.0)
        eff[:, j] = col
        if rxn_type[j] in (LINDEMANN, TROE):
            ln_A0[j] = rng.uniform(np.log(1e6), np.log(1e14))
            b0[j] = rng.uniform(-2.0, 2.0)
            Ea0_over_R[j] = rng.uniform(0.0, 2.0e5) / R_GAS_J_PER_MOL_K
        if rxn_type[j] == TROE:
            troe[j, 0] = rng.uniform(0.3, 0.9)
            troe[j, 1:] = rng.uniform(1.0e2, 1.0e4, size=3)

    return Mechanism(
        elements=elements, elem_count=elem_count, mol_weight=np.ascontiguousarray(W),
        nu_reac=nu_reac, nu_prod=nu_prod, ln_A=ln_A, b=b, Ea_over_R=Ea_over_R,
        reversible=np.ones(R, dtype=np.uint8), nasa_lo=nasa_lo, nasa_hi=nasa_hi,
        T_mid=T_mid, rxn_type=rxn_type, eff=eff, ln_A0=ln_A0, b0=b0,
        Ea0_over_R=Ea0_over_R, troe=troe, p_ref=P_ATM, seed=int(seed),
    )
