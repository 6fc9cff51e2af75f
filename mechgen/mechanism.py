"""Synthetic mechanism and state generator (no method arithmetic lives here).

Shapes follow BASELINE.json `configs` (13/27, 53/325, 111/784, 360/2172 species/reactions, sized like
the paper's four models, Table 4) and the Jacobian densities of PAPER.md Table 7
L334-341.  The real mechanisms and PaSR databases are absent; nothing here reproduces them.

Units of every produced array: SI with kmol (T [K], P [Pa], V [m^3], n [kmol], A in kmol-m^3-s,
Ta = Ea/R [K], W [kg/kmol]).
"""
from __future__ import annotations

import numpy as np

R_GAS = 8314.46261815324      # J/(kmol K), exact SI value (reading S1)
P_ATM = 101325.0              # Pa

# enums mirrored in include/pyjac.h (values are part of the C ABI)
ELEMENTARY, THIRD_BODY, FALLOFF_LINDEMANN, FALLOFF_TROE, FALLOFF_SRI, PLOG, CHEBYSHEV = range(7)
CONP, CONV = 0, 1
CSR, CSC = 0, 1

ATOMIC_W = np.array([12.011, 1.008, 15.999, 14.007])   # C, H, O, N


# ------------------------------------------------------------------------------------------------
# desc-array builder
# ------------------------------------------------------------------------------------------------
class MechBuilder:
    """Collects species and reactions (python dicts) and emits the flat desc arrays."""

    def __init__(self):
        self.W = []
        self.tmid = []
        self.lo = []
        self.hi = []
        self.reactions = []

    def add_species(self, W, lo, hi=None, tmid=1000.0):
        lo = np.asarray(lo, dtype=np.float64)
        hi = lo if hi is None else np.asarray(hi, dtype=np.float64)
        assert lo.shape == (7,) and hi.shape == (7,)
        self.W.append(float(W)); self.tmid.append(float(tmid)); self.lo.append(lo); self.hi.append(hi)
        return len(self.W) - 1

    def add_reaction(self, reac, prod, A=1.0, beta=0.0, Ta=0.0, rev=True, type=ELEMENTARY, eff=None,
                     collider=-1, low=None, troe=None, sri=None, plog=None, cheb=None, chem_activated=False, rev_params=None):
        """chem_activated (falloff types only): chemically-activated bimolecular reaction; (A, beta, Ta) stay the
        high-pressure limit k_inf and `low` the low-pressure limit k_0, but k = k_0 F / (1 + P_r).
        rev_params = (A, beta, Ta): explicit reverse Arrhenius parameters, k_r = A T^beta exp(-Ta/T) instead of k_f / K_c."""
        self.reactions.append(dict(reac=dict(reac), prod=dict(prod), A=A, beta=beta, Ta=Ta, rev=rev,
                                   type=type, eff=dict(eff or {}), collider=collider, low=low,
                                   troe=troe, sri=sri, plog=plog, cheb=cheb, chem_activated=bool(chem_activated), rev_params=rev_params))
        return len(self.reactions) - 1

    def build(self):
        ns, nr = len(self.W), len(self.reactions)
        d = dict(n_species=ns, n_reactions=nr)
        d["mol_weight"] = np.array(self.W, dtype=np.float64)
        d["nasa_tmid"] = np.array(self.tmid, dtype=np.float64)
        d["nasa_lo"] = np.ascontiguousarray(np.array(self.lo, dtype=np.float64).reshape(-1))
        d["nasa_hi"] = np.ascontiguousarray(np.array(self.hi, dtype=np.float64).reshape(-1))

        def ragged(key):
            ptr, sp, nu = [0], [], []
            for r in self.reactions:
                for s in sorted(r[key]):
                    sp.append(s); nu.append(r[key][s])
                ptr.append(len(sp))
            return (np.array(ptr, np.int32), np.array(sp, np.int32), np.array(nu, np.int32))

        d["reac_ptr"], d["reac_species"], d["reac_nu"] = ragged("reac")
        d["prod_ptr"], d["prod_species"], d["prod_nu"] = ragged("prod")
        d["reversible"] = np.array([1 if r["rev"] else 0 for r in self.reactions], np.uint8)
        d["type"] = np.array([r["type"] for r in self.reactions], np.int32)
        d["A"] = np.array([r["A"] for r in self.reactions], np.float64)
        d["beta"] = np.array([r["beta"] for r in self.reactions], np.float64)
        d["Ta"] = np.array([r["Ta"] for r in self.reactions], np.float64)
        ptr, sp, val = [0], [], []
        for r in self.reactions:
            for s in sorted(r["eff"]):
                sp.append(s); val.append(r["eff"][s])
            ptr.append(len(sp))
        d["eff_ptr"] = np.array(ptr, np.int32)
        d["eff_species"] = np.array(sp, np.int32)
        d["eff_value"] = np.array(val, np.float64)
        d["collider"] = np.array([r["collider"] for r in self.reactions], np.int32)
        low = np.array([r["low"] if r["low"] is not None else (1.0, 0.0, 0.0) for r in self.reactions],
                       np.float64).reshape(nr, 3)
        d["low_A"] = np.ascontiguousarray(low[:, 0]); d["low_beta"] = np.ascontiguousarray(low[:, 1])
        d["low_Ta"] = np.ascontiguousarray(low[:, 2])
        troe = np.zeros((nr, 4)); has_t2 = np.zeros(nr, np.uint8); sri = np.zeros((nr, 5))
        for i, r in enumerate(self.reactions):
            if r["troe"] is not None:
                t = r["troe"]
                troe[i, :3] = t[:3]
                if len(t) > 3 and t[3] is not None:
                    troe[i, 3] = t[3]; has_t2[i] = 1
            if r["sri"] is not None:
                sri[i] = r["sri"]
        d["troe"] = troe.reshape(-1); d["troe_has_T2"] = has_t2; d["sri"] = sri.reshape(-1)
        pp, pP, pA, pb, pT = [0], [], [], [], []
        for r in self.reactions:
            for (P, A, b, Ta) in (r["plog"] or []):
                pP.append(P); pA.append(A); pb.append(b); pT.append(Ta)
            pp.append(len(pP))
        d["plog_ptr"] = np.array(pp, np.int32)
        d["plog_P"] = np.array(pP, np.float64); d["plog_A"] = np.array(pA, np.float64)
        d["plog_beta"] = np.array(pb, np.float64); d["plog_Ta"] = np.array(pT, np.float64)
        cp_, nT, nP, coef = [0], [], [], []
        lim = np.ones((nr, 4)); lim[:, 1] = 2.0; lim[:, 3] = 2.0
        for i, r in enumerate(self.reactions):
            c = r["cheb"]
            if c is not None:
                cc = np.asarray(c["coef"], np.float64)
                nT.append(cc.shape[0]); nP.append(cc.shape[1]); coef.extend(cc.reshape(-1).tolist())
                lim[i] = (c["Tmin"], c["Tmax"], c["Pmin"], c["Pmax"])
            else:
                nT.append(0); nP.append(0)
            cp_.append(len(coef))
        d["cheb_ptr"] = np.array(cp_, np.int32)
        d["cheb_nT"] = np.array(nT, np.int32); d["cheb_nP"] = np.array(nP, np.int32)
        d["cheb_Tmin"] = np.ascontiguousarray(lim[:, 0]); d["cheb_Tmax"] = np.ascontiguousarray(lim[:, 1])
        d["cheb_Pmin"] = np.ascontiguousarray(lim[:, 2]); d["cheb_Pmax"] = np.ascontiguousarray(lim[:, 3])
        d["cheb_coef"] = np.array(coef, np.float64)
        d["chem_activated"] = np.array([1 if r["chem_activated"] else 0 for r in self.reactions], np.uint8)
        rp = np.array([r["rev_params"] if r["rev_params"] is not None else (0.0, 0.0, 0.0) for r in self.reactions],
                      np.float64).reshape(nr, 3)
        d["rev_A"] = np.ascontiguousarray(rp[:, 0]); d["rev_beta"] = np.ascontiguousarray(rp[:, 1])
        d["rev_Ta"] = np.ascontiguousarray(rp[:, 2])
        return d


# ------------------------------------------------------------------------------------------------
# configs (BASELINE.json configs[0..4] == C1..C5)
# ------------------------------------------------------------------------------------------------
CONFIGS = {
    1: dict(ns=13, nr=27, n_states=1024, mode=CONP, max_atoms=4, zipf=2.0, n_eff=(1, 2), T=(800.0, 2000.0),
            P_atm=(1.0, 50.0), sparse_X=False, bath_reacts=False,
            mix=dict(arr_rev=20, arr_irr=0, third=4, troe=3, lind=0, sri=0, plog=0, cheb=0)),
    2: dict(ns=53, nr=325, n_states=1 << 17, mode=CONP, max_atoms=8, zipf=1.1, T=(800.0, 2000.0),
            P_atm=(1.0, 50.0), sparse_X=False, bath_reacts=False, mix="std"),
    3: dict(ns=111, nr=784, n_states=1 << 17, mode=CONP, max_atoms=12, zipf=2.0, T=(800.0, 2000.0),
            P_atm=(1.0, 50.0), sparse_X=False, bath_reacts=True, mix="full"),
    4: dict(ns=360, nr=2172, n_states=1 << 14, mode=CONV, max_atoms=20, zipf=1.3, T=(600.0, 2500.0),
            P_atm=(1.0, 100.0), sparse_X=False, bath_reacts=False, mix="full"),
    5: dict(ns=360, nr=2172, n_states=1 << 18, mode=CONP, max_atoms=20, zipf=1.3, T=(800.0, 2000.0),
            P_atm=(1.0, 50.0), sparse_X=True, bath_reacts=False, mix="full"),
}


def _mix_counts(nr, mix):
    if isinstance(mix, dict):
        return dict(mix)
    third = round(0.07 * nr); troe = round(0.05 * nr); lind = round(0.01 * nr); sri = round(0.01 * nr)
    plog = round(0.02 * nr) if mix == "full" else 0
    cheb = round(0.01 * nr) if mix == "full" else 0
    arr = nr - third - troe - lind - sri - plog - cheb
    arr_rev = round(0.7 * arr)
    return dict(arr_rev=arr_rev, arr_irr=arr - arr_rev, third=third, troe=troe, lind=lind, sri=sri,
                plog=plog, cheb=cheb)


# ------------------------------------------------------------------------------------------------
# NASA-7 fits of a random smooth positive cp(T)
# ------------------------------------------------------------------------------------------------
def _fit_nasa(rng, n_atoms):
    c0 = rng.uniform(2.5, 4.5)
    cinf = c0 + rng.uniform(0.5, 3.0) * n_atoms
    theta = rng.uniform(500.0, 1500.0)
    hf = rng.uniform(-1.5e4, 1.5e4)        # H(298.15)/R  [K]
    s0 = rng.uniform(15.0, 45.0)           # S(298.15)/R
    target = lambda t: cinf - (cinf - c0) * np.exp(-1000.0 * t / theta)   # t = T/1000
    tl = np.linspace(0.3, 1.0, 64); th = np.linspace(1.0, 3.0, 96)
    Vl = np.vander(tl, 5, increasing=True)
    pl = np.linalg.lstsq(Vl, target(tl), rcond=None)[0]
    pmid = float(np.polyval(pl[::-1], 1.0))
    # high range: p_hi(t) = pmid + (t-1) * r(t), r cubic  -> continuity of cp at T_mid
    B = np.stack([(th - 1.0) * th ** m for m in range(4)], axis=1)
    r = np.linalg.lstsq(B, target(th) - pmid, rcond=None)[0]
    ph = np.zeros(5); ph[0] = pmid
    for m in range(4):          # (t-1) t^m = t^(m+1) - t^m
        ph[m + 1] += r[m]; ph[m] -= r[m]
    scale = 1000.0 ** -np.arange(5)
    lo = np.zeros(7); hi = np.zeros(7)
    lo[:5] = pl * scale; hi[:5] = ph * scale

    def hpoly(a, T):   # integral of cp/R dT without the constant
        return a[0] * T + a[1] * T ** 2 / 2 + a[2] * T ** 3 / 3 + a[3] * T ** 4 / 4 + a[4] * T ** 5 / 5

    def spoly(a, T):   # integral of cp/(R T) dT without the constant
        return a[0] * np.log(T) + a[1] * T + a[2] * T ** 2 / 2 + a[3] * T ** 3 / 3 + a[4] * T ** 4 / 4

    T0, Tm = 298.15, 1000.0
    lo[5] = hf - hpoly(lo, T0); lo[6] = s0 - spoly(lo, T0)
    hi[5] = hpoly(lo, Tm) + lo[5] - hpoly(hi, Tm)
    hi[6] = spoly(lo, Tm) + lo[6] - spoly(hi, Tm)
    Tg = np.linspace(300.0, 3000.0, 271)
    cp = np.where(Tg <= Tm, np.polyval(lo[4::-1], Tg), np.polyval(hi[4::-1], Tg))
    assert cp.min() > 0.5, "generated cp/R not positive"
    return lo, hi


# ------------------------------------------------------------------------------------------------
# species compositions
# ------------------------------------------------------------------------------------------------
def _draw_compositions(rng, ns, max_atoms, with_n_species):
    """ns-1 reactive compositions over (C,H,O[,N]) + bath gas N2 as the LAST species."""
    comps = []
    seen = {}
    if with_n_species:      # species 0, 1, 2 = N, NO, O compositions: lets the bath gas react once
        for key in ((0, 0, 0, 1), (0, 0, 1, 1), (0, 0, 1, 0)):
            comps.append(key); seen[key] = 1
    cmax = max(1, max_atoms // 3)
    while len(comps) < ns - 1:
        c = int(rng.integers(0, cmax + 1))
        h = int(rng.integers(0, min(2 * c + 2, max_atoms) + 1))
        o = int(rng.integers(0, 4))
        tot = c + h + o
        if tot == 0 or tot > max_atoms:
            continue
        key = (c, h, o, 0)
        # isomers allowed: at most 3 per composition, none for <= 2 atoms
        if seen.get(key, 0) >= (1 if tot <= 2 else 3):
            continue
        seen[key] = seen.get(key, 0) + 1
        comps.append(key)
    comps.append((0, 0, 0, 2))   # bath gas, last species
    return np.array(comps, dtype=np.int64)


# ------------------------------------------------------------------------------------------------
# reactions
# ------------------------------------------------------------------------------------------------
class _ReactionSampler:
    def __init__(self, rng, comp, zipf, allow_bath):
        self.rng = rng
        self.comp = comp
        ns = len(comp)
        self.ns = ns
        self.bath = ns - 1
        rank = rng.permutation(ns - 1)
        pop = np.zeros(ns)
        pop[:ns - 1] = 1.0 / (1.0 + rank) ** zipf
        self.pop = pop / pop.sum()
        self.cum = np.cumsum(self.pop)
        self.pairs = {}
        self.singles = {}
        for a in range(ns - 1):
            self.singles.setdefault(tuple(comp[a]), []).append(a)
            for b in range(a, ns - 1):
                self.pairs.setdefault(tuple(comp[a] + comp[b]), []).append((a, b))
        self.seen = set()

    def draw(self):
        return int(np.searchsorted(self.cum, self.rng.random(), side="right").clip(0, self.ns - 2))

    def _pick(self, cands, weights):
        w = np.asarray(weights, dtype=np.float64)
        return cands[int(self.rng.choice(len(cands), p=w / w.sum()))]

    def _register(self, reac, prod):
        key = frozenset([tuple(sorted(reac.items())), tuple(sorted(prod.items()))])
        if key in self.seen:
            return False
        self.seen.add(key)
        return True

    @staticmethod
    def _side(*sp):
        d = {}
        for s in sp:
            d[s] = d.get(s, 0) + 1
        return d

    def sample(self, form):
        for _ in range(20000):
            if form == "22":
                a, b = self.draw(), self.draw()
                key = tuple(self.comp[a] + self.comp[b])
                cands = [p for p in self.pairs.get(key, []) if p[0] not in (a, b) and p[1] not in (a, b)]
                if not cands:
                    continue
                c, d = self._pick(cands, [self.pop[p[0]] * self.pop[p[1]] for p in cands])
                reac, prod = self._side(a, b), self._side(c, d)
            elif form == "12":
                if self.rng.random() < 0.5:
                    b, c = self.draw(), self.draw()
                    cands = [s for s in self.singles.get(tuple(self.comp[b] + self.comp[c]), []) if s not in (b, c)]
                    if not cands:
                        continue
                    a = self._pick(cands, [self.pop[s] for s in cands])
                else:
                    a = self.draw()
                    cands = [p for p in self.pairs.get(tuple(self.comp[a]), []) if a not in p]
                    if not cands:
                        continue
                    b, c = self._pick(cands, [self.pop[p[0]] * self.pop[p[1]] for p in cands])
                if self.rng.random() < 0.5:
                    reac, prod = self._side(a), self._side(b, c)
                else:
                    reac, prod = self._side(b, c), self._side(a)
            else:  # "11"
                a = self.draw()
                cands = [s for s in self.singles.get(tuple(self.comp[a]), []) if s != a]
                if not cands:
                    continue
                b = self._pick(cands, [self.pop[s] for s in cands])
                reac, prod = self._side(a), self._side(b)
            if self._register(reac, prod):
                return reac, prod
        raise RuntimeError("could not draw a balanced reaction of form " + form)


def _order(side):
    return sum(side.values())


def _arrhenius(rng, order):
    """A log-uniform 1e8-1e16 in cgs (cm^3, mol, s), beta in [-2,2], Ea in [0,50] kcal/mol -> SI."""
    A = 10.0 ** rng.uniform(8.0, 16.0) * (1e-3) ** (order - 1)
    beta = rng.uniform(-2.0, 2.0)
    Ta = rng.uniform(0.0, 50.0) * 1000.0 * 4.184 / 8.31446261815324
    return A, beta, Ta


def _efficiencies(rng, sampler, n_lo=3, n_hi=6, lo=0.5, hi=5.0, extra=None):
    n = int(rng.integers(n_lo, n_hi + 1))
    eff = {}
    guard = 0
    while len(eff) < min(n, sampler.ns - 1) and guard < 1000:
        guard += 1
        s = sampler.draw()
        if s not in eff:
            eff[s] = float(rng.uniform(lo, hi))
    if extra is not None:
        eff[extra] = float(rng.uniform(lo, hi))
    return eff


def make_mechanism(ns, nr, mix, seed, max_atoms=8, zipf=1.0, bath_reacts=False, n_eff=(3, 6)):
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = _mix_counts(nr, mix)
    assert sum(counts.values()) == nr, counts
    for attempt in range(50):
        comp = _draw_compositions(rng, ns, max_atoms, with_n_species=bath_reacts)
        sampler = _ReactionSampler(rng, comp, zipf, bath_reacts)
        try:
            return _build(rng, comp, sampler, counts, bath_reacts, n_eff)
        except RuntimeError:
            continue
    raise RuntimeError("mechanism generation failed")


def _build(rng, comp, sampler, counts, bath_reacts, n_eff=(3, 6)):
    ns = len(comp)
    mb = MechBuilder()
    for k in range(ns):
        lo, hi = _fit_nasa(rng, int(comp[k].sum()))
        mb.add_species(float(comp[k] @ ATOMIC_W), lo, hi, 1000.0)
    bath = ns - 1
    n_bath_eff = 2 if bath_reacts else 0

    def form_for(kind):
        u = rng.random()
        if kind in ("troe", "lind", "sri"):
            return "12"
        if kind == "third":
            return "12" if u < 0.8 else "22"
        return "22" if u < 0.85 else ("12" if u < 0.95 else "11")

    def safe_sample(form):
        try:
            return sampler.sample(form)
        except RuntimeError:
            if form == "11":
                return sampler.sample("22")
            raise

    for kind in ("arr_rev", "arr_irr", "third", "troe", "lind", "sri", "plog", "cheb"):
        for j in range(counts[kind]):
            reac, prod = safe_sample(form_for(kind))
            if bath_reacts and kind == "arr_rev" and j == 0:
                # the one reaction in which the last species takes part: N2 + O <-> N + NO style,
                # built from the N-bearing compositions placed first by _draw_compositions
                reac, prod = {bath: 1, 2: 1}, {0: 1, 1: 1}
            order = _order(reac)
            if kind in ("arr_rev", "arr_irr"):
                A, b, Ta = _arrhenius(rng, order)
                mb.add_reaction(reac, prod, A, b, Ta, rev=(kind == "arr_rev"), type=ELEMENTARY)
            elif kind == "third":
                A, b, Ta = _arrhenius(rng, order + 1)
                extra = bath if (n_bath_eff > 0) else None
                n_bath_eff -= 1 if extra is not None else 0
                mb.add_reaction(reac, prod, A, b, Ta, rev=rng.random() < 0.8, type=THIRD_BODY,
                                eff=_efficiencies(rng, sampler, n_eff[0], n_eff[1], extra=extra))
            elif kind in ("troe", "lind", "sri"):
                A, b, Ta = _arrhenius(rng, order)
                low = (A * 10.0 ** rng.uniform(3.0, 8.0) * 1e-3, rng.uniform(-2.0, 2.0),
                       rng.uniform(0.0, 50.0) * 1000.0 * 4.184 / 8.31446261815324)
                kw = dict(rev=rng.random() < 0.8, eff=_efficiencies(rng, sampler, n_eff[0], n_eff[1]), low=low)
                if kind == "troe":
                    t = [rng.uniform(0.2, 0.9), rng.uniform(50.0, 1000.0), rng.uniform(500.0, 5000.0),
                         rng.uniform(1000.0, 8000.0) if rng.random() < 0.5 else None]
                    mb.add_reaction(reac, prod, A, b, Ta, type=FALLOFF_TROE, troe=t, **kw)
                elif kind == "lind":
                    mb.add_reaction(reac, prod, A, b, Ta, type=FALLOFF_LINDEMANN, **kw)
                else:
                    if rng.random() < 0.5:
                        s = (rng.uniform(0.2, 2.0), rng.uniform(100.0, 1000.0), rng.uniform(500.0, 5000.0), 1.0, 0.0)
                    else:
                        s = (rng.uniform(0.2, 2.0), rng.uniform(100.0, 1000.0), rng.uniform(500.0, 5000.0),
                             rng.uniform(0.5, 2.0), rng.uniform(-0.5, 0.5))
                    mb.add_reaction(reac, prod, A, b, Ta, type=FALLOFF_SRI, sri=s, **kw)
            elif kind == "plog":
                npts = int(rng.integers(4, 7))
                Ps = np.logspace(-2.0, 2.0, npts) * P_ATM
                A0, b0, Ta0 = _arrhenius(rng, order)
                pts = []
                for m, P in enumerate(Ps):
                    pts.append((float(P), A0 * 10.0 ** (0.3 * m + rng.uniform(-0.2, 0.2)),
                                b0 + rng.uniform(-0.3, 0.3), Ta0 * rng.uniform(0.9, 1.1)))
                mb.add_reaction(reac, prod, 1.0, 0.0, 0.0, rev=rng.random() < 0.7, type=PLOG, plog=pts)
            else:
                coef = rng.uniform(-1.0, 1.0, size=(7, 3)) * (0.5 ** np.add.outer(np.arange(7), np.arange(3)))
                coef[0, 0] = rng.uniform(6.0, 12.0) - 3.0 * (order - 1)
                mb.add_reaction(reac, prod, 1.0, 0.0, 0.0, rev=rng.random() < 0.7, type=CHEBYSHEV,
                                cheb=dict(Tmin=300.0, Tmax=3000.0, Pmin=0.01 * P_ATM, Pmax=100.0 * P_ATM, coef=coef))
    # shuffle reaction order so types are interleaved as in a real mechanism file
    perm = rng.permutation(len(mb.reactions))
    mb.reactions = [mb.reactions[i] for i in perm]
    d = mb.build()
    d["composition"] = comp          # bookkeeping for tests (element balance); not part of the C ABI
    return d


_MECH_CACHE = {}


def config_mechanism(c):
    """Mechanism of BASELINE.json config c (1..5); C4 and C5 share one mechanism."""
    key = 4 if c == 5 else c
    if key not in _MECH_CACHE:
        cfg = CONFIGS[key]
        _MECH_CACHE[key] = make_mechanism(cfg["ns"], cfg["nr"], cfg["mix"], 18090100 + key,
                                          cfg["max_atoms"], cfg["zipf"], cfg["bath_reacts"], cfg.get("n_eff", (3, 6)))
    return _MECH_CACHE[key]


# ------------------------------------------------------------------------------------------------
# states
# ------------------------------------------------------------------------------------------------
def make_states(ns, n_states, seed, T=(800.0, 2000.0), P_atm=(1.0, 50.0), sparse_X=False, start=0):
    """Random states.  Returns dict(T, P, V [n], n [(ns-1), n_states] species-major).

    State s depends only on (seed, s): each block of 1024 states has its own PCG64 stream, so any
    sub-range can be generated without generating the whole set.
    """
    Tout = np.empty(n_states); Pout = np.empty(n_states); Vout = np.empty(n_states)
    nout = np.empty((ns - 1, n_states))
    BL = 1024
    s = 0
    while s < n_states:
        g = start + s
        blk, off = divmod(g, BL)
        cnt = min(BL - off, n_states - s)
        rng = np.random.Generator(np.random.PCG64([seed, blk]))
        T_b = rng.uniform(T[0], T[1], BL)
        P_b = rng.uniform(P_atm[0], P_atm[1], BL) * P_ATM
        V_b = 10.0 ** rng.uniform(-3.0, 0.0, BL)
        X = np.empty((BL, ns))
        todo = np.arange(BL)
        while todo.size:
            m = todo.size
            if sparse_X:
                k_act = max(2, ns // 10)
                act = np.argsort(rng.random((m, ns - 1)), axis=1)[:, :k_act - 1]
                act = np.concatenate([act, np.full((m, 1), ns - 1)], axis=1)
                x = np.full((m, ns), 1e-20)
                np.put_along_axis(x, act, rng.dirichlet(np.full(k_act, 0.5), size=m), axis=1)
                x /= x.sum(axis=1, keepdims=True)
            else:
                x = rng.dirichlet(np.full(ns, 0.5), size=m)
            X[todo] = x
            todo = todo[x[:, ns - 1] < 1e-3]      # redraw: keeps [C]_Ns = C_tot - sum well conditioned
        ntot = P_b * V_b / (R_GAS * T_b)
        sl = slice(off, off + cnt)
        Tout[s:s + cnt] = T_b[sl]; Pout[s:s + cnt] = P_b[sl]; Vout[s:s + cnt] = V_b[sl]
        nout[:, s:s + cnt] = (X[sl, :ns - 1] * ntot[sl, None]).T
        s += cnt
    return dict(T=Tout, P=Pout, V=Vout, n=nout)


def config_states(c, n_states=None, start=0):
    cfg = CONFIGS[c]
    n = cfg["n_states"] if n_states is None else n_states
    return make_states(cfg["ns"], n, 18090200 + c, cfg["T"], cfg["P_atm"], cfg["sparse_X"], start)


def pack_phi(states, mode, ld=None, tile=None):
    """phi [nvar*ld] and param [ld] in the library layout (include/pyjac.h "Layout")."""
    T, P, V, n = states["T"], states["P"], states["V"], states["n"]
    N = T.shape[0]
    ld = N if ld is None else ld
    tile = ld if tile is None else tile
    nvar = n.shape[0] + 2
    rows = np.zeros((nvar, ld))
    rows[0, :N] = T
    rows[1, :N] = V if mode == CONP else P
    rows[2:, :N] = n
    param = np.zeros(ld)
    param[:N] = P if mode == CONP else V
    phi = rows.reshape(nvar, ld // tile, tile).transpose(1, 0, 2).reshape(-1)
    return np.ascontiguousarray(phi), param
