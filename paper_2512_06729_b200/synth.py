"""Seeded synthetic networks and atmospheres shaped like the paper's workloads.

This module is the ONLY code shared by the CUDA path and the CPU oracle: it
produces plain numpy arrays (a network description and atmosphere columns) and
holds none of the method's arithmetic (no rate laws, no equilibrium constants,
no source terms).  The only physics-flavoured expressions here shape the
*inputs*: the NASA-7 heat-capacity polynomial is sampled so that cp/R stays
inside the range BASELINE.json config 1 prescribes, and number densities are
set from mixing ratios with the ideal-gas law.

The paper's own network (594 species / 7 720 reactions) and its
thermochemical database are not public ("available upon reasonable request",
PAPER.md:624-626), so these inputs take their shapes, sizes, type mix and value
ranges from BASELINE.json `configs` and SURVEY.md §8(d) and stand in for them.
No real species list, reaction or rate constant is reproduced.

Recipe (every number below is from BASELINE.json config 1
unless marked "ours"):
  * species: random element-balanced formulas built incrementally (atoms first,
    then sums of two existing species, <= 12 atoms; a few isomers, cf.
    c-/l-/t-C3H2 PAPER.md:707); configs 3-5: exactly 24 P-bearing species
     and an inert He (empty stoichiometry row).
  * reactions: element-balanced by construction (pairs bucketed by summed
    composition); type mix 25 % unimolecular / 55 % bimolecular / 12 % falloff /
    8 % photolysis; a heavy-tailed species popularity (ours: weight ~ rank^-0.9)
    gives hub species as real networks have (H, H2, OH ...); configs 3-5:
    exactly 390 reactions involve a P-bearing species.
  * rate parameters: bimolecular A log-uniform 1e-20..1e-9 cm^3/s, n uniform
    -3..3, E/R uniform 0..40000 K; falloff k0 A0 log-uniform 1e-36..1e-26 cm^6/s,
    k_inf like bimolecular, Troe Fc uniform 0.3..0.9; unimolecular A log-uniform
    1e6..1e16 1/s (ours); J log-uniform 1e-10..1e-2 1/s.
  * NASA-7: a1 uniform 2.5..5, a2..a5 scaled so cp/R in [2.5, 15] over
    200-3000 K, a6 uniform -1e5..1e5 K, a7 uniform -10..30; the high-range set
    is the low set plus c*((T-t_mid)/3000)^2 in cp with H and S continuous at
    t_mid; t_mid in {300, 500, 700, 1000} K with weights {5, 5, 10, 80} % (the
    junction temperatures found in the paper's Table 1).
  * atmospheres: P log-spaced 1e3 -> 1e-8 bar, T linear in log P from 2500 K
    (bottom) to 800 K (top) with +-50 K jitter; mixing ratios log-uniform
    1e-20..1 normalised per column; config 4: per-atmosphere T shift -600..+600 K
    and metallicity factor 0.1..100 on species with non-H/He elements.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

UNI, BI, FALLOFF, PHOTO = 0, 1, 2, 3
K_B = 1.380649e-16  # erg/K (cgs), used only to turn mixing ratios into densities
BAR = 1.0e6         # dyn/cm^2


@dataclass
class Network:
    element_names: list
    composition: np.ndarray   # int32 [n_species][n_elements]
    nasa_lo: np.ndarray       # float64 [n_species][7]
    nasa_hi: np.ndarray       # float64 [n_species][7]
    t_mid: np.ndarray         # float64 [n_species]
    type: np.ndarray          # int32 [n_reactions]
    reactants: np.ndarray     # int32 [n_reactions][3], -1 padded
    products: np.ndarray      # int32 [n_reactions][3], -1 padded
    reversible: np.ndarray    # uint8 [n_reactions]
    arrh: np.ndarray          # float64 [n_reactions][3]  A, n, E/R  (k_inf for FALLOFF)
    arrh_low: np.ndarray      # float64 [n_reactions][3]  A0, n0, E0/R (FALLOFF only)
    troe_fc: np.ndarray       # float64 [n_reactions]
    t_ref: np.ndarray         # float64 [n_reactions]  1 (mod. Arrhenius) or 300 (Kooij)
    meta: dict = field(default_factory=dict)

    @property
    def n_species(self):
        return int(self.composition.shape[0])

    @property
    def n_elements(self):
        return int(self.composition.shape[1])

    @property
    def n_reactions(self):
        return int(self.type.shape[0])

    @property
    def n_photo(self):
        return int(np.count_nonzero(self.type == PHOTO))


@dataclass
class Atmosphere:
    ncol: int
    ld: int
    T: np.ndarray   # float64 [ld]  K
    P: np.ndarray   # float64 [ld]  dyn/cm^2
    n: np.ndarray   # float64 [n_species][ld]  cm^-3
    J: np.ndarray   # float64 [n_photo][ld]    1/s
    meta: dict = field(default_factory=dict)


# --------------------------------------------------------------------------- species

def _make_species(rng, elements, n_species, n_p_bearing, inert, max_atoms=12, p_iso=0.04):
    """Random formulas built incrementally so that balanced reactions exist."""
    ne = len(elements)
    comps = []
    for e in range(ne):
        v = np.zeros(ne, dtype=np.int64)
        v[e] = 1
        comps.append(v)
    e_p = elements.index("P") if "P" in elements else -1
    inert_idx = {elements.index(x) for x in inert if x in elements}
    seen = {tuple(c) for c in comps}

    def combinable(allow_p):
        out = []
        for i, c in enumerate(comps):
            if any(c[k] for k in inert_idx):
                continue
            if not allow_p and e_p >= 0 and c[e_p]:
                continue
            out.append(i)
        return out

    def grow_one(need_p):
        guard = 0
        while True:
            guard += 1
            if guard > 200000:
                raise RuntimeError("species generator did not converge")
            pool = combinable(allow_p=need_p)
            # prefer small species so formulas stay small and sums collide often
            w = np.array([1.0 / (1.0 + comps[i].sum()) ** 1.5 for i in pool])
            w /= w.sum()
            i, j = rng.choice(pool, size=2, p=w)
            c = comps[i] + comps[j]
            if c.sum() > max_atoms:
                continue
            if need_p and not c[e_p]:
                continue
            if tuple(c) in seen and rng.random() > p_iso:
                continue
            seen.add(tuple(c))
            comps.append(c)
            return

    n_p = n_p_bearing if e_p >= 0 else 0
    # the P atom is already one of the P-bearing species; the others are spread over the
    # generation order so that P chemistry has its own sub-structure (P2, PO, PH ... analogues)
    p_steps = set()
    if n_p > 1:
        p_steps = set(rng.choice(np.arange(ne, n_species), size=n_p - 1, replace=False).tolist())
    while len(comps) < n_species:
        grow_one(need_p=len(comps) in p_steps)
    comp = np.array(comps, dtype=np.int32)
    if n_p:
        assert int(np.count_nonzero(comp[:, e_p])) == n_p
    return comp


# --------------------------------------------------------------------------- NASA-7

def _cp_poly(a, T):
    return a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4])))


def _make_nasa(rng, n_species):
    grid = np.arange(200.0, 3000.0 + 1.0, 50.0)
    x = grid / 3000.0
    lo = np.zeros((n_species, 7))
    hi = np.zeros((n_species, 7))
    t_mid = rng.choice([300.0, 500.0, 700.0, 1000.0], size=n_species, p=[0.05, 0.05, 0.10, 0.80])
    for i in range(n_species):
        a1 = rng.uniform(2.5, 5.0)
        b = rng.uniform(-1.0, 1.0, size=4)
        p = b[0] * x + b[1] * x ** 2 + b[2] * x ** 3 + b[3] * x ** 4
        if -p.min() > p.max():
            b, p = -b, -p
        up = (15.0 - a1) / max(p.max(), 1e-300)
        dn = (a1 - 2.5) / max(-p.min(), 1e-300)
        s = rng.uniform(0.2, 0.98) * min(up, dn)
        a = np.zeros(7)
        a[0] = a1
        for k in range(4):
            a[1 + k] = s * b[k] / 3000.0 ** (k + 1)
        a[5] = rng.uniform(-1.0e5, 1.0e5)
        a[6] = rng.uniform(-10.0, 30.0)
        lo[i] = a
        # high-range set: cp_hi = cp_lo + c ((T - tm)/3000)^2, H and S continuous at tm
        tm = t_mid[i]
        c = rng.uniform(-2.0, 2.0)
        for _ in range(60):
            h = a.copy()
            q = c / 9.0e6
            h[0] = a[0] + q * tm * tm
            h[1] = a[1] - 2.0 * q * tm
            h[2] = a[2] + q
            g = grid[grid >= tm]
            v = _cp_poly(h, g)
            if v.min() >= 2.5 and v.max() <= 15.0:
                break
            c *= 0.7
        else:
            raise RuntimeError("could not bound the high-range heat capacity")
        hp_lo = a[0] + tm * (a[1] / 2 + tm * (a[2] / 3 + tm * (a[3] / 4 + tm * a[4] / 5)))
        hp_hi = h[0] + tm * (h[1] / 2 + tm * (h[2] / 3 + tm * (h[3] / 4 + tm * h[4] / 5)))
        h[5] = a[5] + tm * (hp_lo - hp_hi)
        sp_lo = a[0] * np.log(tm) + tm * (a[1] + tm * (a[2] / 2 + tm * (a[3] / 3 + tm * a[4] / 4)))
        sp_hi = h[0] * np.log(tm) + tm * (h[1] + tm * (h[2] / 2 + tm * (h[3] / 3 + tm * h[4] / 4)))
        h[6] = a[6] + (sp_lo - sp_hi)
        hi[i] = h
        lo_v = _cp_poly(a, grid[grid <= max(tm, 200.0)])
        assert lo_v.min() >= 2.5 - 1e-9 and lo_v.max() <= 15.0 + 1e-9
    return lo, hi, t_mid


# --------------------------------------------------------------------------- reactions

class _ReactionSampler:
    """Draws element-balanced stoichiometries from pair/single composition buckets."""

    def __init__(self, rng, comp, inert_species, alpha=0.9):
        self.rng = rng
        self.comp = comp
        ns = comp.shape[0]
        active = np.array([i for i in range(ns) if i not in inert_species], dtype=np.int64)
        self.active = active
        # heavy-tailed popularity by generation order (atoms and early species are hubs)
        rank = np.empty(ns)
        rank[active] = np.arange(1, active.size + 1)
        w = np.zeros(ns)
        w[active] = rank[active] ** (-alpha)
        self.w = w
        ii, jj = np.triu_indices(active.size)
        pi, pj = active[ii], active[jj]
        sums = comp[pi].astype(np.int64) + comp[pj].astype(np.int64)
        base = int(sums.max()) + 1
        key = np.zeros(sums.shape[0], dtype=np.int64)
        for e in range(comp.shape[1]):
            key = key * base + sums[:, e]
        skey = np.zeros(ns, dtype=np.int64)
        for e in range(comp.shape[1]):
            skey = skey * base + comp[:, e].astype(np.int64)
        self.base = base
        self.pi, self.pj = pi, pj
        self.pw = w[pi] * w[pj]
        order = np.argsort(key, kind="stable")
        sk = key[order]
        starts = np.flatnonzero(np.r_[True, sk[1:] != sk[:-1]])
        ends = np.r_[starts[1:], sk.size]
        self.bucket_of_key = {}
        self.buckets = []
        for s, e in zip(starts, ends):
            self.bucket_of_key[int(sk[s])] = len(self.buckets)
            self.buckets.append(order[s:e])
        self.pair_bucket = np.empty(key.size, dtype=np.int64)
        for b, idx in enumerate(self.buckets):
            self.pair_bucket[idx] = b
        # pairs that share their bucket with at least one other pair (A+B -> C+D possible)
        multi = np.array([len(self.buckets[b]) > 1 for b in self.pair_bucket])
        self.multi_idx = np.flatnonzero(multi)
        self.multi_cdf = np.cumsum(self.pw[self.multi_idx])
        # singles whose composition equals a pair sum (A -> B+C possible)
        self.single_key = skey
        dec = [i for i in active if int(skey[i]) in self.bucket_of_key]
        self.decomposable = np.array(dec, dtype=np.int64)
        # the parent of a dissociation is drawn almost uniformly (many distinct parents),
        # its fragments by popularity (small hub species)
        self.dec_cdf = np.cumsum(w[self.decomposable] ** 0.25)
        # isomer groups
        groups = {}
        for i in active:
            groups.setdefault(int(skey[i]), []).append(int(i))
        self.isomers = [g for g in groups.values() if len(g) > 1]

    def _pick_in_bucket(self, b, exclude=None):
        idx = self.buckets[b]
        if exclude is not None:
            idx = idx[idx != exclude]
        if idx.size == 0:
            return None
        return int(idx[self._draw(np.cumsum(self.pw[idx]))])

    def _draw(self, cdf):
        k = int(np.searchsorted(cdf, self.rng.random() * cdf[-1], side="right"))
        return min(k, cdf.size - 1)

    def pair_to_pair(self):
        """A + B -> C + D"""
        if self.multi_idx.size == 0:
            return None
        k = int(self.multi_idx[self._draw(self.multi_cdf)])
        m = self._pick_in_bucket(self.pair_bucket[k], exclude=k)
        if m is None:
            return None
        return [int(self.pi[k]), int(self.pj[k])], [int(self.pi[m]), int(self.pj[m])]

    def single_to_pair(self):
        """A -> B + C"""
        if self.decomposable.size == 0:
            return None
        a = int(self.decomposable[self._draw(self.dec_cdf)])
        b = self.bucket_of_key[int(self.single_key[a])]
        m = self._pick_in_bucket(b)
        return [a], [int(self.pi[m]), int(self.pj[m])]

    def isomerisation(self):
        if not self.isomers:
            return None
        g = self.isomers[int(self.rng.integers(len(self.isomers)))]
        a, b = self.rng.choice(g, size=2, replace=False)
        return [int(a)], [int(b)]

    def split_one(self, side):
        """Replace one decomposable species of `side` by a pair with the same composition."""
        cand = [s for s in side if int(self.single_key[s]) in self.bucket_of_key]
        if not cand or len(side) >= 3:
            return None
        s = cand[int(self.rng.integers(len(cand)))]
        m = self._pick_in_bucket(self.bucket_of_key[int(self.single_key[s])])
        out = list(side)
        out.remove(s)
        out += [int(self.pi[m]), int(self.pj[m])]
        return out


def _draw_stoich(smp, rng, rtype):
    if rtype == BI:
        r = smp.pair_to_pair()
        if r is None:
            return None
        lhs, rhs = r
        u = rng.random()
        if u < 0.04:          # three products, PAPER.md:225 (Eq. 13)
            t = smp.split_one(rhs)
            if t is not None:
                rhs = t
        elif u < 0.05:        # three reactants (the reverse shape of Eq. 13)
            t = smp.split_one(lhs)
            if t is not None:
                lhs = t
        return lhs, rhs
    if rtype == UNI:
        if rng.random() < 0.08:
            r = smp.isomerisation()
            if r is not None:
                return r
        return smp.single_to_pair()
    if rtype == FALLOFF:      # recombination B + C (+M) -> A, PAPER.md:142 (Eq. 9)
        r = smp.single_to_pair()
        if r is None:
            return None
        return r[1], r[0]
    if rtype == PHOTO:        # A -> B + C
        r = smp.single_to_pair()
        if r is None:
            return None
        lhs, rhs = r
        if rng.random() < 0.05:
            t = smp.split_one(rhs)
            if t is not None:
                rhs = t
        return lhs, rhs
    raise ValueError(rtype)


def _type_counts(n_reactions, explicit=None):
    if explicit is not None:
        return dict(explicit)
    n_ph = int(round(0.08 * n_reactions))
    n_fo = int(round(0.12 * n_reactions))
    n_un = int(round(0.25 * n_reactions))
    n_bi = n_reactions - n_ph - n_fo - n_un
    return {UNI: n_un, BI: n_bi, FALLOFF: n_fo, PHOTO: n_ph}


def _make_reactions(rng, comp, elements, counts, inert_species, n_p_reactions):
    smp = _ReactionSampler(rng, comp, inert_species)
    e_p = elements.index("P") if "P" in elements else -1
    has_p = comp[:, e_p] > 0 if e_p >= 0 else np.zeros(comp.shape[0], dtype=bool)
    total = sum(counts.values())
    quota_p = {t: 0 for t in counts}
    if n_p_reactions:
        # spread the P-involving reactions over the types in proportion to the mix
        # (dissociation-shaped types are capped by how many distinct P parents -> fragments exist)
        n_dis = sum(len(smp.buckets[smp.bucket_of_key[int(smp.single_key[i])]])
                    for i in smp.decomposable if has_p[i])
        left = n_p_reactions
        for t in (UNI, FALLOFF, PHOTO):
            quota_p[t] = min(int(round(n_p_reactions * counts[t] / total)), n_dis // 2)
            left -= quota_p[t]
        quota_p[BI] = left
    stoich = []
    types = []
    seen = set()
    for t in (UNI, BI, FALLOFF, PHOTO):
        need_p, need_n = quota_p[t], counts[t] - quota_p[t]
        if e_p < 0 or not n_p_reactions:
            need_p, need_n = 0, counts[t]
        guard = 0
        while need_p + need_n > 0:
            guard += 1
            if guard > 400 * total + 10000:
                raise RuntimeError("reaction generator did not converge for type %d" % t)
            r = _draw_stoich(smp, rng, t)
            if r is None:
                continue
            lhs, rhs = r
            if sorted(lhs) == sorted(rhs):
                continue
            sig = (t, tuple(sorted(lhs)), tuple(sorted(rhs)))
            if sig in seen and guard < 60 * total:
                continue    # distinct stoichiometries unless the species set is too small (config 1)
            inv_p = bool(n_p_reactions) and (any(has_p[s] for s in lhs) or any(has_p[s] for s in rhs))
            if n_p_reactions:
                if inv_p and need_p > 0:
                    need_p -= 1
                elif (not inv_p) and need_n > 0:
                    need_n -= 1
                else:
                    continue
            else:
                need_n -= 1
            seen.add(sig)
            stoich.append((lhs, rhs))
            types.append(t)
    return stoich, types, smp


def _check_balance(comp, lhs, rhs):
    return np.array_equal(comp[lhs].sum(axis=0), comp[rhs].sum(axis=0))


def _loguniform(rng, lo, hi, size=None):
    return 10.0 ** rng.uniform(np.log10(lo), np.log10(hi), size=size)


def make_network(seed, elements, n_species, n_reactions, *, type_counts=None,
                 n_p_bearing=0, n_p_reactions=0, inert=("He",), name=""):
    rng = np.random.default_rng(seed)
    elements = list(elements)
    comp = _make_species(rng, elements, n_species, n_p_bearing, inert)
    inert_species = {i for i in range(n_species)
                     if any(comp[i, elements.index(x)] for x in inert if x in elements)}
    lo, hi, t_mid = _make_nasa(rng, n_species)
    counts = _type_counts(n_reactions, type_counts)
    stoich, types, smp = _make_reactions(rng, comp, elements, counts, inert_species, n_p_reactions)

    # structural cases every config must contain: a repeated reactant, a repeated
    # product, the same species on both sides and a three-product reaction arise naturally
    # from the sampler (checked below); a duplicate stoichiometry with fresh parameters
    # (separate branches of one reaction) is planted explicitly.
    e_p = elements.index("P") if "P" in elements else -1

    def no_p(sp):
        return e_p < 0 or not any(comp[s, e_p] for s in sp)

    plain = [k for k, ((l, r), ty) in enumerate(zip(stoich, types))
             if ty == BI and len(l) == 2 and len(r) == 2 and len(set(l + r)) == 4
             and no_p(l) and no_p(r)]
    if len(plain) >= 2:
        stoich[plain[1]] = (list(stoich[plain[0]][0]), list(stoich[plain[0]][1]))
    if len(plain) >= 3 and not any(set(l) & set(r) and len(r) == 3 for l, r in stoich):
        # A + X -> B + C + X: a catalyst on both sides and three products
        for _ in range(1000):
            d = smp.single_to_pair()
            if d is None or not (no_p(d[0]) and no_p(d[1])):
                continue
            xs = [int(i) for i in smp.active if no_p([i]) and i not in d[0] + d[1]]
            if xs:
                stoich[plain[2]] = ([d[0][0], xs[0]], d[1] + [xs[0]])
                break
    structure = {
        "repeated_reactant": sum(1 for l, r in stoich if len(set(l)) < len(l)),
        "repeated_product": sum(1 for l, r in stoich if len(set(r)) < len(r)),
        "both_sides": sum(1 for l, r in stoich if set(l) & set(r)),
        "three_products": sum(1 for l, r in stoich if len(r) == 3),
        "three_reactants": sum(1 for l, r in stoich if len(l) == 3),
        "duplicates": len(stoich) - len({(tuple(sorted(l)), tuple(sorted(r)), ty)
                                          for (l, r), ty in zip(stoich, types)}),
    }

    nr = len(stoich)
    perm = rng.permutation(nr)          # user order = random shuffle of the types
    rtype = np.array(types, dtype=np.int32)[perm]
    reactants = -np.ones((nr, 3), dtype=np.int32)
    products = -np.ones((nr, 3), dtype=np.int32)
    for u, k in enumerate(perm):
        lhs, rhs = stoich[k]
        assert _check_balance(comp, lhs, rhs), "generator produced an unbalanced reaction"
        reactants[u, :len(lhs)] = lhs
        products[u, :len(rhs)] = rhs
    reversible = (rtype != PHOTO).astype(np.uint8)     # photolysis is irreversible

    arrh = np.zeros((nr, 3))
    arrh_low = np.zeros((nr, 3))
    fc = np.ones(nr)
    t_ref = np.ones(nr)
    is_uni = rtype == UNI
    is_fo = rtype == FALLOFF
    arrh[:, 1] = rng.uniform(-3.0, 3.0, size=nr)
    arrh[:, 2] = rng.uniform(0.0, 40000.0, size=nr)
    a_bi = _loguniform(rng, 1e-20, 1e-9, size=nr)
    a_uni = _loguniform(rng, 1e6, 1e16, size=nr)
    arrh[:, 0] = np.where(is_uni, a_uni, a_bi)
    arrh_low[:, 0] = _loguniform(rng, 1e-36, 1e-26, size=nr)
    arrh_low[:, 1] = rng.uniform(-3.0, 3.0, size=nr)
    arrh_low[:, 2] = rng.uniform(0.0, 40000.0, size=nr)
    fc_draw = rng.uniform(0.3, 0.9, size=nr)
    fc = np.where(is_fo, fc_draw, 1.0)
    arrh_low[~is_fo] = 0.0
    arrh[rtype == PHOTO] = 0.0

    return Network(
        element_names=elements, composition=np.ascontiguousarray(comp, dtype=np.int32),
        nasa_lo=lo, nasa_hi=hi, t_mid=t_mid, type=rtype, reactants=reactants, products=products,
        reversible=reversible, arrh=arrh, arrh_low=arrh_low, troe_fc=fc, t_ref=t_ref,
        meta={"name": name, "seed": seed, "type_counts": {int(k): int(v) for k, v in counts.items()},
              "n_p_bearing": n_p_bearing, "n_p_reactions": n_p_reactions,
              "structure": structure})


# --------------------------------------------------------------------------- atmospheres

def make_atmosphere(seed, net, n_atm, n_layers, *, t_shift=(0.0, 0.0), metallicity=(1.0, 1.0),
                    ld=None, pad_value=None):
    """Columns are (atmosphere, layer) pairs; column index = atmosphere * n_layers + layer."""
    rng = np.random.default_rng(seed)
    ncol = n_atm * n_layers
    if ld is None:
        ld = (ncol + 31) // 32 * 32
    ns, nph = net.n_species, net.n_photo
    T = np.full(ld, 1000.0)
    P = np.full(ld, BAR)
    n = np.zeros((ns, ld))
    J = np.zeros((nph, ld))
    logp = np.linspace(np.log10(1.0e3), np.log10(1.0e-8), n_layers)       # bar, bottom -> top
    frac = (logp - logp[0]) / (logp[-1] - logp[0]) if n_layers > 1 else np.zeros(1)
    heavy = np.zeros(ns, dtype=bool)
    for e, name in enumerate(net.element_names):
        if name not in ("H", "He"):
            heavy |= net.composition[:, e] != 0
    shifts = np.zeros(n_atm)
    zs = np.ones(n_atm)
    for a in range(n_atm):
        sl = slice(a * n_layers, (a + 1) * n_layers)
        shift = rng.uniform(t_shift[0], t_shift[1]) if t_shift[1] > t_shift[0] else t_shift[0]
        z = (_loguniform(rng, metallicity[0], metallicity[1])
             if metallicity[1] > metallicity[0] else metallicity[0])
        shifts[a], zs[a] = shift, z
        Ta = 2500.0 + (800.0 - 2500.0) * frac + rng.uniform(-50.0, 50.0, size=n_layers) + shift
        Pa = 10.0 ** logp * BAR
        x = _loguniform(rng, 1e-20, 1.0, size=(ns, n_layers))
        x[heavy] *= z
        x /= x.sum(axis=0, keepdims=True)
        T[sl] = Ta
        P[sl] = Pa
        n[:, sl] = x * (Pa / (K_B * Ta))[None, :]
    if nph:
        J[:, :ncol] = _loguniform(rng, 1e-10, 1e-2, size=(nph, ncol))
    if pad_value is not None:
        T[ncol:] = pad_value
        P[ncol:] = pad_value
        n[:, ncol:] = pad_value
        J[:, ncol:] = pad_value
    return Atmosphere(ncol=ncol, ld=ld, T=T, P=P, n=n, J=J,
                      meta={"seed": seed, "n_atm": n_atm, "n_layers": n_layers,
                            "t_shift": shifts, "metallicity": zs})


# --------------------------------------------------------------------------- the five configs

_ELEMENTS = {
    1: ["H", "C", "O"],
    2: ["C", "H", "O", "N", "S"],
    3: ["H", "He", "C", "N", "O", "P", "S", "Na", "K", "Fe"],
}


def config_network(cfg):
    """Networks of BASELINE.json configs 1-5 (configs 3, 4 and 5 share one network)."""
    if cfg == 1:
        return make_network(1001, _ELEMENTS[1], 12, 40,
                            type_counts={UNI: 10, BI: 15, FALLOFF: 10, PHOTO: 5}, name="config1")
    if cfg == 2:
        return make_network(1002, _ELEMENTS[2], 90, 600,
                            type_counts={UNI: 150, BI: 330, FALLOFF: 72, PHOTO: 48}, name="config2")
    if cfg in (3, 4, 5):
        return make_network(1003, _ELEMENTS[3], 594, 7720,
                            type_counts={UNI: 1930, BI: 4246, FALLOFF: 926, PHOTO: 618},
                            n_p_bearing=24, n_p_reactions=390, name="config3")
    raise ValueError("config must be 1..5")


def config_atmosphere(cfg, net, n_atm=None):
    """Atmosphere batches of BASELINE.json configs 1-5; `n_atm` overrides the batch size."""
    if cfg == 1:
        return make_atmosphere(2001, net, n_atm or 1, 20)
    if cfg == 2:
        return make_atmosphere(2002, net, n_atm or 1, 120)
    if cfg == 3:
        return make_atmosphere(2003, net, n_atm or 1, 150)
    if cfg == 4:
        return make_atmosphere(2004, net, n_atm or 256, 150, t_shift=(-600.0, 600.0),
                               metallicity=(0.1, 100.0))
    if cfg == 5:
        return make_atmosphere(2005, net, n_atm or 64, 150)
    raise ValueError("config must be 1..5")


# --------------------------------------------------------------------------- the edge-case network

def edge_network(seed=1099):
    """A mid-size network that holds every reaction shape the paper allows but configs 1-5 do not
    draw (the parity tests run it through every kernel):
      * irreversible thermal reactions of all three thermal types (one-way steps);
      * pure Lindemann falloff, Fc = 1 (Eq. 12 exactly);
      * a species three times on one side, nu = -3 and nu = +3 (Eq. 13 allows three);
      * an ion / electron pair with the charge carried as a signed extra "element";
      * a species that takes part in no reaction (empty CSR row);
      * Kooij (t_ref = 300) and modified-Arrhenius (t_ref = 1) forms mixed.
    Structure only; parameters come from the same distributions as the configs."""
    base = make_network(seed, _ELEMENTS[2], 60, 400, name="edge")
    rng = np.random.default_rng(seed + 1)
    ns0, ne0, nr0 = base.n_species, base.n_elements, base.n_reactions
    comp = np.zeros((ns0 + 4, ne0 + 1), dtype=np.int32)          # last column: charge
    comp[:ns0, :ne0] = base.composition
    used = np.unique(np.concatenate([base.reactants.ravel(), base.products.ravel()]))
    a = int(used[used >= 0][0])                                  # a species the sampler uses
    x3, ion, el, lone = ns0, ns0 + 1, ns0 + 2, ns0 + 3
    comp[x3, :ne0] = 3 * base.composition[a]
    comp[ion, :ne0] = base.composition[a]
    comp[ion, ne0] = +1
    comp[el, ne0] = -1
    comp[lone, :ne0] = base.composition[a]                       # an isomer no reaction touches
    lo4, hi4, tm4 = _make_nasa(rng, 4)
    tm4 = np.array([300.0, 500.0, 700.0, 1000.0])                # every junction temperature of SURVEY T3 occurs
    extra = [  # (type, reactants, products, reversible, Fc)
        (BI, [a, a, a], [x3], 1, 1.0),          # nu_a = -3
        (UNI, [x3], [a, a, a], 0, 1.0),         # nu_a = +3, one-way
        (PHOTO, [a], [ion, el], 0, 1.0),        # photo-ionisation
        (BI, [ion, el], [a], 1, 1.0),           # recombination, reverse by detailed balance
        (FALLOFF, [ion, el], [a], 0, 1.0),      # three-body recombination, pure Lindemann, one-way
    ]
    nr = nr0 + len(extra)
    rtype = np.concatenate([base.type, np.array([e[0] for e in extra], dtype=np.int32)])
    reactants = -np.ones((nr, 3), dtype=np.int32)
    products = -np.ones((nr, 3), dtype=np.int32)
    reactants[:nr0], products[:nr0] = base.reactants, base.products
    for k, (_, lhs, rhs, _, _) in enumerate(extra):
        reactants[nr0 + k, :len(lhs)] = lhs
        products[nr0 + k, :len(rhs)] = rhs
        assert _check_balance(comp, lhs, rhs)
    reversible = np.concatenate([base.reversible, np.array([e[3] for e in extra], dtype=np.uint8)])
    thermal = rtype != PHOTO
    one_way = thermal & (rng.uniform(size=nr) < 1.0 / 3.0)
    one_way[nr0:] = False
    reversible[one_way] = 0
    fc = np.concatenate([base.troe_fc, np.array([e[4] for e in extra])])
    is_fo = rtype == FALLOFF
    fc[is_fo & (rng.uniform(size=nr) < 0.25)] = 1.0
    fc[nr0:] = [e[4] for e in extra]
    t_ref = np.where(thermal & (rng.uniform(size=nr) < 1.0 / 3.0), 300.0, 1.0)

    def draw3(n_rows, a_lo, a_hi):
        return np.stack([_loguniform(rng, a_lo, a_hi, size=n_rows), rng.uniform(-3.0, 3.0, size=n_rows),
                         rng.uniform(0.0, 40000.0, size=n_rows)], axis=1)

    arrh = np.concatenate([base.arrh, draw3(len(extra), 1e-20, 1e-9)])
    arrh[nr0 + 1, 0] = _loguniform(rng, 1e6, 1e16)               # the unimolecular one
    arrh[rtype == PHOTO] = 0.0
    arrh_low = np.concatenate([base.arrh_low, draw3(len(extra), 1e-36, 1e-26)])
    arrh_low[~is_fo] = 0.0
    perm = rng.permutation(nr)                                   # the added reactions are not left at the end
    assert {UNI, BI, FALLOFF} <= set(rtype[reversible == 0].tolist())
    return Network(
        element_names=list(base.element_names) + ["charge"], composition=comp,
        nasa_lo=np.concatenate([base.nasa_lo, lo4]), nasa_hi=np.concatenate([base.nasa_hi, hi4]),
        t_mid=np.concatenate([base.t_mid, tm4]), type=rtype[perm], reactants=reactants[perm],
        products=products[perm], reversible=reversible[perm], arrh=arrh[perm], arrh_low=arrh_low[perm],
        troe_fc=fc[perm], t_ref=t_ref[perm],
        meta={"name": "edge", "seed": seed, "triple": a, "x3": x3, "ion": ion, "electron": el, "lone": lone})


def edge_atmosphere(net, seed=2099, n_layers=75):
    """One atmosphere for `edge_network` whose columns include: T exactly on every thermo breakpoint
    t_mid and one ulp below and above it (reading T3: T <= t_mid takes the low set), a cold column
    (k_r beyond the double range, reading R5), a species that is zero everywhere, a column that is
    zero everywhere, and a negative density (reading Q2: processed arithmetically)."""
    atm = make_atmosphere(seed, net, 1, n_layers)
    c = 1
    for tm in np.unique(net.t_mid):
        for T in (np.nextafter(tm, 0.0), tm, np.nextafter(tm, 1e9)):
            atm.T[c] = T
            c += 2                                               # leave ordinary columns in between
    assert c < atm.ncol - 8
    atm.T[c] = 170.0
    atm.n[5, :] = 0.0
    atm.n[:, c + 2] = 0.0
    atm.n[7, c + 4] = -atm.n[7, c + 4]
    atm.meta.update(cold=c, zero_species=5, zero_column=c + 2, negative=(7, c + 4))
    return atm


# --------------------------------------------------------------------------- f2: photolysis inputs

@dataclass
class Photo:
    """Wavelength grid and cross-sections for the photolysis rate constants."""
    dlambda: np.ndarray       # float64 [n_bins]  bin widths, Angstrom
    lam: np.ndarray           # float64 [n_bins]  bin centres, Angstrom (not used by the method; for plots/tests)
    abs_species: np.ndarray   # int32 [n_abs]     species index of each extinction cross-section row
    sigma_ext: np.ndarray     # float64 [n_abs][n_bins]    absorption + scattering, cm^2
    sigma_ph: np.ndarray      # float64 [n_photo][n_bins]  cross-section of each photolysis reaction, cm^2

    @property
    def n_bins(self):
        return int(self.dlambda.shape[0])


def make_photo(seed, net, n_bins=10000, n_abs=None):
    """Seeded stand-in for the PHIDRATES / Leiden cross-section tables, which are not in the container.
    Shapes from the paper: bins about 1 A wide from 1 A to 10 000 A (10 000 of them; widths jittered
    +-20 % so the grid is non-uniform, which the paper allows); every photolysis parent is an absorber plus a
    few more species; a cross-section is a sum of one to three Gaussian bands (peak log-uniform 1e-20..1e-16
    cm^2) over a Rayleigh-like lambda^-4 floor; a branch's cross-section is its parent's absorption times a
    quantum yield that is smooth in wavelength and vanishes above a threshold."""
    rng = np.random.default_rng(seed)
    dl = (10000.0 - 1.0) / n_bins * rng.uniform(0.8, 1.2, size=n_bins)
    dl *= (10000.0 - 1.0) / dl.sum()
    edges = 1.0 + np.concatenate([[0.0], np.cumsum(dl)])
    lam = 0.5 * (edges[:-1] + edges[1:])
    photo_rows = np.flatnonzero(net.type == PHOTO)
    parents = net.reactants[photo_rows, 0]
    others = rng.permutation(np.setdiff1d(np.arange(net.n_species), parents))
    extra = others[:max(0, (n_abs or (len(np.unique(parents)) + 8)) - len(np.unique(parents)))]
    abs_species = np.concatenate([np.unique(parents), np.sort(extra)]).astype(np.int32)

    def bands():
        s = 1e-26 * (lam / 1000.0) ** -4.0
        for _ in range(rng.integers(1, 4)):
            s = s + _loguniform(rng, 1e-20, 1e-16) * np.exp(-0.5 * ((lam - rng.uniform(300.0, 4000.0)) / rng.uniform(50.0, 1500.0)) ** 2)
        return s

    sigma_ext = np.stack([bands() for _ in abs_species])
    row_of = {int(sp): k for k, sp in enumerate(abs_species)}
    sigma_ph = np.zeros((len(photo_rows), n_bins))
    for p, parent in enumerate(parents):
        threshold = rng.uniform(1500.0, 6000.0)
        yield_ = rng.uniform(0.05, 1.0) / (1.0 + np.exp((lam - threshold) / rng.uniform(20.0, 200.0)))
        sigma_ph[p] = sigma_ext[row_of[int(parent)]] * yield_
    return Photo(dlambda=dl, lam=lam, abs_species=abs_species, sigma_ext=sigma_ext, sigma_ph=sigma_ph)


def make_irradiation(seed, net, atm, photo, with_diffuse=True):
    """Per-atmosphere irradiation for `make_photo`: layer thickness dz [ld] (cm) from the hydrostatic spacing of
    the log-pressure grid, stellar photon flux at the top j0 [n_atm][n_bins] (a Planck-like photon spectrum of
    4 000-7 000 K scaled to 1e10..1e14 photons cm^-2 s^-1 A^-1 at its peak), a diffuse term j_diff [n_bins][ld] of a
    few per cent of it, the cosine of the zenith angle mu [n_atm] in 0.3..1 and the irradiated-time fraction
    t_f [n_atm] in {1, 1/2}."""
    rng = np.random.default_rng(seed)
    n_atm, L = atm.meta["n_atm"], atm.meta["n_layers"]
    dz = np.ones(atm.ld)
    dlnp = np.log(1.0e11) / max(L - 1, 1)
    dz[:atm.ncol] = dlnp * K_B * atm.T[:atm.ncol] / (2.3 * 1.6726e-24 * 2000.0)
    x = 1.4388e8 / (photo.lam[None, :] * rng.uniform(4000.0, 7000.0, size=(n_atm, 1)))      # h c / (lambda k_B T)
    shape = photo.lam[None, :] ** -4.0 / np.expm1(np.minimum(x, 700.0))
    j0 = shape / shape.max(axis=1, keepdims=True) * _loguniform(rng, 1e10, 1e14, size=(n_atm, 1))
    mu = rng.uniform(0.3, 1.0, size=n_atm)
    t_f = rng.choice([1.0, 0.5], size=n_atm)
    j_diff = None
    if with_diffuse:
        j_diff = np.zeros((photo.n_bins, atm.ld))
        for a in range(n_atm):
            j_diff[:, a * L:(a + 1) * L] = j0[a][:, None] * rng.uniform(0.0, 0.05, size=(photo.n_bins, L))
    return dz, j0, j_diff, mu, t_f


# --------------------------------------------------------------------------- f3: transport inputs

def make_transport(seed, net, atm):
    """Seeded inputs of the molecular-diffusion terms for an atmosphere of make_atmosphere: species
    masses from the composition (standard atomic masses of the element labels; 1 u for unknown labels and for the
    charge column), a mean molecular mass of 2.2-2.4 u and a gravity of 500-2500 cm s^-2 per atmosphere, the uniform
    layer spacing that the log-pressure grid implies for the column's mean temperature, thermal diffusion factors
    uniform -0.4..0.3 (alpha_T = -0.38 for light species is the usual choice), the gas density n_gas = P / (k_B T),
    and binary-mixture-like diffusion coefficients D = b T^0.75 / n_gas with b log-uniform 1e17..1e18 per species
    (the paper takes its parameters from several sources; none is reproduced here)."""
    rng = np.random.default_rng(seed)
    amu = {"H": 1.008, "He": 4.0026, "C": 12.011, "N": 14.007, "O": 15.999, "P": 30.974, "S": 32.06, "Na": 22.990,
           "K": 39.098, "Fe": 55.845}
    w = np.array([amu.get(e, 0.0) for e in net.element_names])
    mass = np.maximum(np.abs(net.composition) @ w, 1.0) * 1.66053907e-24
    n_atm, L = atm.meta["n_atm"], atm.meta["n_layers"]
    mbar = rng.uniform(2.2, 2.4, size=n_atm) * 1.66053907e-24
    grav = rng.uniform(500.0, 2500.0, size=n_atm)
    dz = np.zeros(n_atm)
    dlnp = np.log(1.0e11) / max(L - 1, 1)
    for a in range(n_atm):
        dz[a] = dlnp * K_B * atm.T[a * L:(a + 1) * L].mean() / (mbar[a] * grav[a])
    alpha_T = rng.uniform(-0.4, 0.3, size=net.n_species)
    n_gas = np.ones(atm.ld)
    n_gas[:atm.ncol] = atm.P[:atm.ncol] / (K_B * atm.T[:atm.ncol])
    D = np.ones((net.n_species, atm.ld))
    b = _loguniform(rng, 1e17, 1e18, size=net.n_species)
    D[:, :atm.ncol] = b[:, None] * atm.T[None, :atm.ncol] ** 0.75 / n_gas[None, :atm.ncol]
    return dict(mass=mass, alpha_T=alpha_T, mbar=mbar, grav=grav, dz=dz, n_gas=n_gas, D=D)
