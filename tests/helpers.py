"""Test-side helpers: tiny-system input builders and an explicit second-quantised Hamiltonian (pin P1).

Nothing here is used by the product; the second-quantised code is deliberately independent of oracle/.
"""
from __future__ import annotations

import itertools

import numpy as np

from synth_inputs import make_integrals, pack_index


def full_space(n, na, nb):
    """All determinants with na alpha and nb beta electrons in n orbitals, sorted by (alpha, beta)."""
    def words(k):
        return sorted(sum(1 << p for p in c) for c in itertools.combinations(range(n), k))
    return np.array([[a, b] for a in words(na) for b in words(nb)], dtype=np.uint64)


def dense_eri(n, eri):
    """Expand the packed 8-fold array to g[p,q,r,s] = (pq|rs)."""
    p, q, r, s = np.meshgrid(*([np.arange(n)] * 4), indexing="ij")
    return eri[pack_index(pack_index(p, q), pack_index(r, s))]


def small_integrals(n, seed, L=8):
    return make_integrals(n, L, seed)


def second_quantised_dense(n, h1, g, dets, e_core=0.0):
    """<X|H|Y> by explicit operator application on Fock vectors, Jordan-Wigner sign counting.

    Spin-orbital s = p (alpha) or n + p (beta); |D> = prod_{s occupied, ascending} a+_s |0>, i.e. all alpha
    creators left of all beta creators (reading Q1).  H = e_core + sum_{pq,sigma} h_pq a+_{p sigma} a_{q sigma}
    + 1/2 sum_{pqrs, sigma tau} (pq|rs) a+_{p sigma} a+_{r tau} a_{s tau} a_{q sigma}.
    """
    def to_occ(d):
        return tuple([(int(d[0]) >> p) & 1 for p in range(n)] + [(int(d[1]) >> p) & 1 for p in range(n)])

    def ann(state, s):
        sign, occ = state
        if not occ[s]:
            return None
        sign *= -1 if sum(occ[:s]) & 1 else 1
        o = list(occ); o[s] = 0
        return sign, tuple(o)

    def cre(state, s):
        sign, occ = state
        if occ[s]:
            return None
        sign *= -1 if sum(occ[:s]) & 1 else 1
        o = list(occ); o[s] = 1
        return sign, tuple(o)

    index = {to_occ(d): k for k, d in enumerate(dets)}
    nd = len(dets)
    H = np.zeros((nd, nd))
    for col, d in enumerate(dets):
        y = (1, to_occ(d))
        H[col, col] += e_core
        for sg in (0, n):
            for q in range(n):
                s1 = ann(y, sg + q)
                if s1 is None:
                    continue
                for p in range(n):
                    s2 = cre(s1, sg + p)
                    if s2 is not None and s2[1] in index:
                        H[index[s2[1]], col] += s2[0] * h1[p, q]
        for sg in (0, n):
            for tg in (0, n):
                for q in range(n):
                    s1 = ann(y, sg + q)
                    if s1 is None:
                        continue
                    for s in range(n):
                        s2 = ann(s1, tg + s)
                        if s2 is None:
                            continue
                        for r in range(n):
                            s3 = cre(s2, tg + r)
                            if s3 is None:
                                continue
                            for p in range(n):
                                s4 = cre(s3, sg + p)
                                if s4 is not None and s4[1] in index:
                                    H[index[s4[1]], col] += 0.5 * s4[0] * g[p, q, r, s]
    return H
