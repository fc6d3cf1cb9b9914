"""Synthetic-input recipe.

Conventions shared by every consumer (they are data layout, not method arithmetic):
  * n spatial orbitals (n <= 64); a determinant is two uint64 words (alpha, beta), bit p = orbital p.
  * h1: fp64 [n, n] symmetric.
  * eri: packed 8-fold symmetric chemist integrals (pq|rs): eri[pack_index(pack_index(p,q), pack_index(r,s))],
    pack_index(x, y) = max(x,y)*(max(x,y)+1)/2 + min(x,y).
  * dets: uint64 [|S|, 2], sorted ascending by (alpha, beta) as a 128-bit number with alpha the high word, unique.
  * psi: fp64 [|S|], psi^T psi = 1.
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 260121310

# name -> parameters.  `rate` is the psi decay per excitation rank, L the number of factors of the eri.
CONFIGS = {
    "tiny": dict(index=0, n=10, na=5, nb=5, L=20, n_dets=2000, rate=1.5, eps=0.0, eps2=0.0, band=None),
    "h2o": dict(index=1, n=24, na=5, nb=5, L=60, n_dets=20000, rate=1.5, eps=1e-5, eps2=1e-7, band=None),
    "n2": dict(index=2, n=28, na=7, nb=7, L=80, n_dets=100000, rate=0.8, eps=1e-5, eps2=1e-7, band=None),
    "n2sweep": dict(index=3, n=28, na=7, nb=7, L=80, n_dets=1000000, rate=0.8, eps=1e-5, eps2=1e-7, band=None),
    "cr2": dict(index=4, n=56, na=12, nb=12, L=200, n_dets=1000000, rate=0.6, eps=1e-5, eps2=1e-7, band=(20, 31)),
}


def pack_index(x, y):
    """Triangular pair index max*(max+1)/2 + min (works on ints and integer arrays)."""
    hi = np.maximum(x, y)
    lo = np.minimum(x, y)
    return hi * (hi + 1) // 2 + lo


def make_integrals(n: int, L: int, seed: int, band=None, slope: float = 1.0):
    """h_pq ~ N(0,1) exp(-|p-q|/4) symmetric with ascending diagonal; (pq|rs) = sum_l B^l_pq B^l_rs,
    B^l symmetric ~ N(0, 0.3) exp(-|p-q|/4).  Returns (h1 [n,n], eri packed)."""
    ss = np.random.SeedSequence(seed)
    rng_h, rng_b = (np.random.default_rng(s) for s in ss.spawn(2))
    p = np.arange(n)
    decay = np.exp(-np.abs(p[:, None] - p[None, :]) / 4.0)
    g = rng_h.standard_normal((n, n))
    g = np.tril(g) + np.tril(g, -1).T
    h1 = g * decay
    diag = -0.5 * n + slope * p.astype(np.float64)
    if band is not None:  # near-degenerate d-like band lo..hi (Cr2-shaped)
        lo, hi = band
        diag[lo:hi + 1] = diag[lo] + 0.02 * (p[lo:hi + 1] - lo)
        diag[hi + 1:] = diag[hi] + slope * (p[hi + 1:] - hi)
    h1[p, p] = diag
    # factors on the packed pair index, lower triangle only -> exact 8-fold symmetry by construction
    iu, ju = np.tril_indices(n)  # iu >= ju, ordered by pack_index
    assert np.array_equal(pack_index(iu, ju), np.arange(iu.size))
    Bp = rng_b.normal(0.0, 0.3, size=(L, iu.size)) * decay[iu, ju][None, :]
    # sum over the L factors in index order with plain multiplies and adds: a BLAS product here would make the last bits of the
    # integrals depend on the host's dgemm kernels, and stored oracle values (tests/golden) could not be compared across machines
    full = np.zeros((iu.size, iu.size))
    for l in range(L):
        full += np.multiply.outer(Bp[l], Bp[l])  # [npair, npair]
    a, b = np.tril_indices(iu.size)
    eri = np.ascontiguousarray(full[a, b])
    return np.ascontiguousarray(h1), eri


def _bits_to_word(occ: np.ndarray) -> np.ndarray:
    n = occ.shape[1]
    w = np.zeros(occ.shape[0], dtype=np.uint64)
    for q in range(n):
        w |= occ[:, q].astype(np.uint64) << np.uint64(q)
    return w


def _draw_dets(rng, n, na, nb, count):
    """`count` draws: r uniform in 1..4, then r random same-spin occupied->virtual replacements."""
    occ = np.zeros((count, 2, n), dtype=bool)
    occ[:, 0, :na] = True
    occ[:, 1, :nb] = True
    r = rng.integers(1, 5, size=count)
    rows = np.arange(count)
    for step in range(4):
        active = r > step
        spin = rng.integers(0, 2, size=count)
        ko = rng.random((count, n))
        kv = rng.random((count, n))
        cur = occ[rows, spin, :]
        i = np.argmax(np.where(cur, ko, -1.0), axis=1)
        a = np.argmax(np.where(~cur, kv, -1.0), axis=1)
        sel = rows[active]
        occ[sel, spin[active], i[active]] = False
        occ[sel, spin[active], a[active]] = True
    return np.stack([_bits_to_word(occ[:, 0, :]), _bits_to_word(occ[:, 1, :])], axis=1)


def make_subspace(n, na, nb, n_dets, rate, seed, prefix=None):
    """HF plus random excitations up to rank 4, deduplicated in draw order, truncated to n_dets (or to `prefix`
    of the same stream: nested sweep), sorted.  psi_i = +-exp(-rate*rank_i), normalised.  Returns dets, psi, rank."""
    ss = np.random.SeedSequence(seed)
    rng_s, rng_sign = (np.random.default_rng(s) for s in ss.spawn(4)[2:])
    hf = np.array([[(1 << na) - 1, (1 << nb) - 1]], dtype=np.uint64)
    pool = hf
    while True:
        need = n_dets - pool.shape[0]
        if need <= 0:
            break
        draws = _draw_dets(rng_s, n, na, nb, max(1024, int(need * 1.3)))
        cat = np.concatenate([pool, draws], axis=0)
        key = np.ascontiguousarray(cat).view(np.dtype((np.void, 16))).ravel()
        _, first = np.unique(key, return_index=True)
        pool = cat[np.sort(first)]
    pool = pool[:n_dets]
    if prefix is not None:
        pool = pool[:prefix]
    signs = rng_sign.integers(0, 2, size=n_dets)[: pool.shape[0]] * 2.0 - 1.0
    rank = (_popcount(pool[:, 0] ^ hf[0, 0]) + _popcount(pool[:, 1] ^ hf[0, 1])) // 2
    psi = signs * np.exp(-rate * rank)
    order = np.lexsort((pool[:, 1], pool[:, 0]))
    dets = np.ascontiguousarray(pool[order])
    psi = psi[order]
    psi = psi / np.sqrt(np.sum(psi * psi))
    return dets, np.ascontiguousarray(psi), np.ascontiguousarray(rank[order].astype(np.int32))


def _popcount(x: np.ndarray) -> np.ndarray:
    x = x.astype(np.uint64)
    c = np.zeros(x.shape, dtype=np.int64)
    for q in range(64):
        c += ((x >> np.uint64(q)) & np.uint64(1)).astype(np.int64)
    return c


def make_problem(name: str, n_dets: int | None = None):
    """Build one of CONFIGS.  For "n2sweep", `n_dets` selects the nested prefix (1e4 ... 1e6).  For any config a
    smaller `n_dets` gives the nested prefix of the same draw stream (used by tests to shrink a case)."""
    c = CONFIGS[name]
    seed = BASE_SEED + c["index"]
    h1, eri = make_integrals(c["n"], c["L"], seed, band=c["band"])
    dets, psi, rank = make_subspace(c["n"], c["na"], c["nb"], c["n_dets"], c["rate"], seed, prefix=n_dets)
    return dict(name=name, n=c["n"], na=c["na"], nb=c["nb"], h1=h1, eri=eri, e_core=0.0, dets=dets, psi=psi,
                rank=rank, eps=c["eps"], eps2=c["eps2"], rate=c["rate"])
