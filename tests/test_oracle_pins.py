"""Pins P1-P10: the oracle checked against things other than itself.

The paper prints no worked example of this path (no element, list or PT2 value; its energies need FCIDUMP files and
trained amplitudes that are not available), so the pins are brute force, closed forms, invariants and library routines.
"""
import itertools
from math import comb

import numpy as np
import pytest
import scipy.sparse as sp

from synth_inputs import make_problem, CONFIGS
from helpers import full_space, dense_eri, small_integrals, second_quantised_dense


# ---------------------------------------------------------------- P1: explicit second quantisation
@pytest.mark.parametrize("n,na,nb,seed", [(4, 2, 2, 11), (5, 3, 2, 12), (5, 1, 3, 13), (6, 3, 3, 14)])
def test_p1_slater_condon_equals_operator_application(orc, n, na, nb, seed):
    h1, eri = small_integrals(n, seed)
    dets = full_space(n, na, nb)
    H_sq = second_quantised_dense(n, h1, dense_eri(n, eri), dets, e_core=0.37)
    H_or = orc.dense(n, h1, eri, 0.37, dets)
    assert np.allclose(H_or, H_sq, rtol=0, atol=1e-12)
    assert np.abs(H_sq).max() > 0.5  # not vacuous
    # signs matter: there must be negative and positive phases among equal-magnitude integrals
    assert (H_sq < -1e-3).any() and (H_sq > 1e-3).any()


def test_p1b_enumeration_equals_bitstring_difference(orc):
    """connections() (enumerate excitations) against element() (difference of two bitstrings) on a full space."""
    n, na, nb = 6, 3, 2
    h1, eri = small_integrals(n, 21)
    dets = full_space(n, na, nb)
    H = orc.dense(n, h1, eri, 0.0, dets)
    index = {(int(a), int(b)): k for k, (a, b) in enumerate(dets)}
    for c, d in enumerate(dets):
        keys, hv, visited = orc.connections(n, h1, eri, 0.0, d, 0.0)
        col = np.zeros(len(dets))
        for (a, b), v in zip(keys, hv):
            col[index[(int(a), int(b))]] = v
        ref = H[:, c].copy(); ref[c] = 0.0
        assert np.array_equal(col, ref)
        assert len(keys) == len(set(map(tuple, keys.tolist())))
        assert all(tuple(keys[k]) < tuple(keys[k + 1]) for k in range(len(keys) - 1))  # sorted by (alpha, beta)


# ---------------------------------------------------------------- P2: variational bound / library eigensolver
def test_p2_energy_bounded_by_fci_ground_state(orc):
    n, na, nb = 6, 3, 3
    h1, eri = small_integrals(n, 31)
    dets = full_space(n, na, nb)
    assert len(dets) == 400
    H = orc.dense(n, h1, eri, 0.1, dets)
    w, V = np.linalg.eigh(H)
    rng = np.random.default_rng(5)
    for trial in range(5):
        idx = np.sort(rng.choice(400, size=60, replace=False))
        psi = rng.standard_normal(60)
        rp, col, val = orc.ham_build(n, h1, eri, 0.1, dets[idx], 0.0)
        e, n2 = orc.energy(rp, col, val, psi)
        assert e >= w[0] - 1e-12
        assert np.isclose(n2, psi @ psi, rtol=1e-14)
        assert np.isclose(e, psi @ H[np.ix_(idx, idx)] @ psi / (psi @ psi), rtol=1e-12)
    rp, col, val = orc.ham_build(n, h1, eri, 0.1, dets, 0.0)
    e, _ = orc.energy(rp, col, val, V[:, 0])
    assert np.isclose(e, w[0], rtol=1e-12)
    # E_diag = lambda_min(H_VV) <= E_var
    A = sp.csr_matrix((val, col, rp), shape=(400, 400)).toarray()
    assert np.array_equal(A, H)  # CSR at eps=0 is the dense matrix (no exact zeros among stored entries)


# ---------------------------------------------------------------- P3: Hermiticity, bitwise
@pytest.mark.parametrize("eps", [0.0, 1e-3, 5e-2])
def test_p3_csr_bitwise_symmetric(orc, eps):
    p = make_problem("tiny", n_dets=600)
    rp, col, val = orc.ham_build(p["n"], p["h1"], p["eri"], 0.0, p["dets"], eps)
    A = sp.csr_matrix((val, col, rp), shape=(600, 600))
    At = A.T.tocsr(); At.sort_indices()
    assert np.array_equal(A.indptr, At.indptr) and np.array_equal(A.indices, At.indices)
    assert np.array_equal(A.data, At.data)  # bit-for-bit (H_PV = H_VP^T)
    for i in range(600):  # columns ascending, diagonal always present, screen respected
        c = col[rp[i]:rp[i + 1]]; v = val[rp[i]:rp[i + 1]]
        assert np.all(np.diff(c) > 0) and i in c
        off = v[c != i]
        assert np.all(np.abs(off) >= eps) and np.all(off != 0.0)


def test_p3b_ham_build_row_subset_equals_rows_of_the_full_build(orc):
    """orc_ham_build(rows=keep) (used by bench.py's bounded oracle sample and by the masked GPU tests) is loop bookkeeping
    only: the kept rows are the same rows of the full build, bit for bit; the other rows are empty."""
    p = make_problem("tiny", n_dets=500)
    rp, col, val = orc.ham_build(p["n"], p["h1"], p["eri"], 0.0, p["dets"], 1e-3)
    keep = np.array([0, 3, 4, 77, 250, 499])
    srp, scol, sval = orc.ham_build(p["n"], p["h1"], p["eri"], 0.0, p["dets"], 1e-3, rows=keep)
    assert len(srp) == 501 and srp[-1] == len(scol) == sum(rp[r + 1] - rp[r] for r in keep)
    for r in range(500):
        a, b = srp[r], srp[r + 1]
        if r in keep:
            assert np.array_equal(scol[a:b], col[rp[r]:rp[r + 1]]) and np.array_equal(sval[a:b], val[rp[r]:rp[r + 1]])
        else:
            assert a == b


# ---------------------------------------------------------------- P4 / P5: eps=0 == unscreened, closed-form counts
@pytest.mark.parametrize("name", ["tiny", "h2o", "n2", "cr2"])
def test_p5_visit_count_closed_form(orc, name):
    c = CONFIGS[name]
    n, na, nb = c["n"], c["na"], c["nb"]
    expected = (na * (n - na) + nb * (n - nb) + comb(na, 2) * comb(n - na, 2) + comb(nb, 2) * comb(n - nb, 2)
                + na * nb * (n - na) * (n - nb))
    assert expected == {"tiny": 875, "h2o": 12635, "n2": 30723, "cr2": 404712}[name]
    from synth_inputs import make_integrals, BASE_SEED
    h1, eri = make_integrals(n, c["L"], BASE_SEED + c["index"], band=c["band"])
    rng = np.random.default_rng(3)
    for _ in range(2):
        a = sum(1 << int(q) for q in rng.choice(n, na, replace=False))
        b = sum(1 << int(q) for q in rng.choice(n, nb, replace=False))
        keys, hv, visited = orc.connections(n, h1, eri, 0.0, np.array([a, b], dtype=np.uint64), 0.0)
        assert visited == expected
        assert len(keys) == expected  # P4: tau = 0 keeps everything (random integrals: no exact zeros)
        keys2, hv2, _ = orc.connections(n, h1, eri, 0.0, np.array([a, b], dtype=np.uint64), 1e-2)
        kept = np.abs(hv) >= 1e-2
        assert np.array_equal(keys2, keys[kept]) and np.array_equal(hv2, hv[kept])


# ---------------------------------------------------------------- P6: PT2 vanishes on the full space
def test_p6_pt2_zero_on_full_space(orc):
    n, na, nb = 6, 3, 2
    h1, eri = small_integrals(n, 41)
    dets = full_space(n, na, nb)
    psi = np.random.default_rng(1).standard_normal(len(dets))
    r = orc.pt2(n, h1, eri, 0.0, dets, psi, -3.0, 0.0)
    assert r["pt2"] == 0.0 and r["n_external"] == 0 and r["n_contrib"] == 0


# ---------------------------------------------------------------- P7: textbook closed forms
def test_p7_two_electrons_two_orbitals(orc):
    h1, eri = small_integrals(2, 51)
    g = dense_eri(2, eri)
    J = lambda p, q: g[p, p, q, q]
    K = lambda p, q: g[p, q, q, p]
    d11 = np.array([1, 1], dtype=np.uint64); d22 = np.array([2, 2], dtype=np.uint64)
    assert np.isclose(orc.element(2, h1, eri, 0.0, d11, d11), 2 * h1[0, 0] + J(0, 0), rtol=1e-14)
    assert np.isclose(orc.element(2, h1, eri, 0.0, d22, d22), 2 * h1[1, 1] + J(1, 1), rtol=1e-14)
    assert orc.element(2, h1, eri, 0.0, d22, d11) == K(0, 1)
    assert orc.element(2, h1, eri, 0.0, d11, d22) == K(0, 1)
    # open-shell pair |1a 2b>, |2a 1b>: diagonal h11 + h22 + J12, coupling -K12 in this ordering... sign by P1;
    # the singlet/triplet eigenvalues h11+h22+J12 +- K12 are convention-free:
    d12 = np.array([1, 2], dtype=np.uint64); d21 = np.array([2, 1], dtype=np.uint64)
    M = np.array([[orc.element(2, h1, eri, 0.0, x, y) for y in (d12, d21)] for x in (d12, d21)])
    ev = np.linalg.eigvalsh(M)
    base = h1[0, 0] + h1[1, 1] + J(0, 1)
    assert np.allclose(sorted(ev), sorted([base - K(0, 1), base + K(0, 1)]), rtol=1e-13)


def test_p7b_closed_shell_hf_energy(orc):
    n, nocc = 7, 3
    h1, eri = small_integrals(n, 52)
    g = dense_eri(n, eri)
    e = 0.25 + 2 * sum(h1[i, i] for i in range(nocc)) + sum(
        2 * g[i, i, j, j] - g[i, j, j, i] for i in range(nocc) for j in range(nocc))
    hf = np.array([(1 << nocc) - 1] * 2, dtype=np.uint64)
    assert np.isclose(orc.diagonal(n, h1, eri, 0.25, hf), e, rtol=1e-14)


# ---------------------------------------------------------------- P8 / P9: dense brute-force PT2 and the sum rule
@pytest.mark.parametrize("eps2", [0.0, 1e-3, 2e-2])
def test_p8_pt2_dense_brute_force(orc, eps2):
    n, na, nb = 7, 3, 3
    h1, eri = small_integrals(n, 61)
    dets = full_space(n, na, nb)  # 1225
    H = orc.dense(n, h1, eri, 0.0, dets)
    rng = np.random.default_rng(8)
    idx = np.sort(rng.choice(len(dets), size=150, replace=False))
    psi = rng.standard_normal(150) * np.exp(-rng.random(150) * 4)
    psi[7] = 0.0  # a source with zero amplitude generates nothing (reading Q6)
    ext = np.setdiff1d(np.arange(len(dets)), idx)
    HS = H[np.ix_(idx, idx)]
    e_s = psi @ HS @ psi / (psi @ psi)
    C = H[np.ix_(ext, idx)] * psi[None, :]          # H_ai psi_i
    tau = np.where(psi != 0, eps2 / np.abs(np.where(psi != 0, psi, 1.0)), np.inf) if eps2 > 0 else np.zeros(150)
    keep = (np.abs(H[np.ix_(ext, idx)]) >= tau[None, :]) & (H[np.ix_(ext, idx)] != 0) & (psi != 0)[None, :]
    v = (C * keep).sum(axis=1)
    touched = keep.any(axis=1)
    ref = np.sum(v[touched] ** 2 / (e_s - np.diag(H)[ext][touched])) / (psi @ psi)
    rp, col, val = orc.ham_build(n, h1, eri, 0.0, dets[idx], 0.0)
    e_or, _ = orc.energy(rp, col, val, psi)
    assert np.isclose(e_or, e_s, rtol=1e-13)
    for n_parts in (1, 4):
        r = orc.pt2(n, h1, eri, 0.0, dets[idx], psi, e_s, eps2, n_parts=n_parts)
        assert r["n_external"] == int(touched.sum())
        assert r["n_contrib"] == int(keep.sum())
        assert np.isclose(r["pt2"], ref, rtol=1e-12)
        assert np.isclose(r["part_sums"].sum(), ref, rtol=1e-12)
    # partition ranges add up (the multi-pass bookkeeping, reading Q14)
    parts = [orc.pt2(n, h1, eri, 0.0, dets[idx], psi, e_s, eps2, n_parts=4, part_begin=k, part_end=k + 1) for k in range(4)]
    assert np.isclose(sum(x["pt2"] for x in parts), ref, rtol=1e-12)
    assert sum(x["n_external"] for x in parts) == int(touched.sum())
    if eps2 == 0.0:
        # P9 sum rule: ||H[:,S] psi||^2 = ||H_SS psi||^2 + sum_a v_a^2
        lhs = np.sum((H[:, idx] @ psi) ** 2)
        assert np.isclose(lhs, np.sum((HS @ psi) ** 2) + np.sum(v ** 2), rtol=1e-12)


# ---------------------------------------------------------------- P10: spin-swap symmetry, single-reference EN2
def test_p10_spin_swap_invariance(orc):
    p = make_problem("tiny", n_dets=300)
    n, h1, eri = p["n"], p["h1"], p["eri"]
    dets, psi = p["dets"], p["psi"] / np.linalg.norm(p["psi"][:300])
    sw = dets[:, ::-1].copy()
    order = np.lexsort((sw[:, 1], sw[:, 0]))
    sw, psw = np.ascontiguousarray(sw[order]), psi[order]
    out = []
    for d, s in ((dets, psi), (sw, psw)):
        rp, col, val = orc.ham_build(n, h1, eri, 0.0, d, 1e-4)
        e, _ = orc.energy(rp, col, val, s)
        r = orc.pt2(n, h1, eri, 0.0, d, s, e, 1e-5)
        out.append((len(col), e, r["pt2"], r["n_external"], r["n_contrib"]))
    assert out[0][0] == out[1][0] and out[0][3:] == out[1][3:]
    assert np.isclose(out[0][1], out[1][1], rtol=1e-13) and np.isclose(out[0][2], out[1][2], rtol=1e-11)


def test_p10b_single_reference_epstein_nesbet(orc):
    n, na, nb = 6, 2, 3
    h1, eri = small_integrals(n, 71)
    dets = full_space(n, na, nb)
    H = orc.dense(n, h1, eri, 0.0, dets)
    hf = 0
    e0 = H[hf, hf]
    others = np.arange(len(dets)) != hf
    ref = np.sum(H[others, hf] ** 2 / (e0 - np.diag(H)[others]))
    r = orc.pt2(n, h1, eri, 0.0, dets[hf:hf + 1], np.array([1.0]), e0, 0.0)
    assert np.isclose(r["pt2"], ref, rtol=1e-12)
    assert r["n_external"] == int(np.count_nonzero(H[others, hf]))


def test_zobrist_is_xor_of_orbital_words(orc):
    """Reading Q14: class function is a XOR over occupied orbitals, so an excitation shifts it by a fixed delta."""
    z = lambda a, b: orc.zobrist(np.array([a, b], dtype=np.uint64))
    assert z(0b0111, 0b1011) ^ z(0b0110, 0b1011) == z(0b0001, 0) and z(0, 0) == 0
    assert z(0b0101, 0b0011) == z(0b0001, 0) ^ z(0b0100, 0) ^ z(0, 0b0001) ^ z(0, 0b0010)
    # splitmix64(seed + index) with seed 260121310, written out independently
    def sm(x):
        m = (1 << 64) - 1
        x = (x + 0x9E3779B97F4A7C15) & m
        x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & m
        x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & m
        return x ^ (x >> 31)
    assert z(1 << 5, 0) == sm(260121310 + 5) and z(0, 1 << 9) == sm(260121310 + 64 + 9)


# ---------------------------------------------------------------- P11: internal term of Eq. 13 and the residual of Eq. 12
def test_p11_residual_and_internal_term(orc):
    """(a) eigenvector of the full-space matrix: r = 0 and the internal term vanishes; (b) two-level textbook second
    order K^2 / (E_1 - E_2) for psi = (1, 0) on the closed-shell pair of two electrons in two orbitals (first
    sum); (c) r and the term against numpy on the dense matrix built by the bitstring-difference path `element`."""
    n, na, nb = 6, 3, 3
    h1, eri = small_integrals(n, 31)
    dets = full_space(n, na, nb)
    H = orc.dense(n, h1, eri, 0.1, dets)
    w, V = np.linalg.eigh(H)
    rp, col, val = orc.ham_build(n, h1, eri, 0.1, dets, 0.0)
    r, t = orc.residual(rp, col, val, V[:, 3], w[3])
    assert np.max(np.abs(r)) < 1e-12 and abs(t) < 1e-20
    # (b)
    h2, e2 = small_integrals(2, 51)
    g = dense_eri(2, e2)
    two = np.array([[1, 1], [2, 2]], dtype=np.uint64)
    rp2, col2, val2 = orc.ham_build(2, h2, e2, 0.0, two, 0.0)
    e1, e22, k = 2 * h2[0, 0] + g[0, 0, 0, 0], 2 * h2[1, 1] + g[1, 1, 1, 1], g[0, 1, 1, 0]
    r2, t2 = orc.residual(rp2, col2, val2, np.array([1.0, 0.0]), e1)
    assert np.allclose(r2, [0.0, k], rtol=1e-14, atol=1e-15)
    assert np.isclose(t2, k * k / (e1 - e22), rtol=1e-13)
    # (c)
    rng = np.random.default_rng(8)
    idx = np.sort(rng.choice(400, size=90, replace=False))
    psi = rng.standard_normal(90)
    rp, col, val = orc.ham_build(n, h1, eri, 0.1, dets[idx], 0.0)
    Hs = H[np.ix_(idx, idx)]
    e = psi @ Hs @ psi / (psi @ psi)
    r, t = orc.residual(rp, col, val, psi, e)
    r_ref = Hs @ psi - e * psi
    assert np.allclose(r, r_ref, rtol=1e-12, atol=1e-13)
    assert np.isclose(t, np.sum(r_ref ** 2 / (e - np.diag(Hs))) / (psi @ psi), rtol=1e-11)
    assert abs(psi @ r_ref) < 1e-10 * np.linalg.norm(psi) * np.linalg.norm(r_ref)  # the residual is orthogonal to psi


# ---------------------------------------------------------------- P12: E_diag = lambda_min(H_VV)
def test_p12_ediag(orc):
    """(a) two-level closed form (a+b)/2 - sqrt(((a-b)/2)^2 + k^2); (b) both solver branches (dense LAPACK / ARPACK) agree with
    LAPACK on the dense matrix built by `element`; (c) E_diag <= E_var for any psi (Delta_opt >= 0)."""
    h2, e2 = small_integrals(2, 51)
    g = dense_eri(2, e2)
    two = np.array([[1, 1], [2, 2]], dtype=np.uint64)
    rp, col, val = orc.ham_build(2, h2, e2, 0.0, two, 0.0)
    a, b, k = 2 * h2[0, 0] + g[0, 0, 0, 0], 2 * h2[1, 1] + g[1, 1, 1, 1], g[0, 1, 1, 0]
    assert np.isclose(orc.ediag(rp, col, val), 0.5 * (a + b) - np.sqrt(0.25 * (a - b) ** 2 + k * k), rtol=1e-13)
    n, na, nb = 6, 3, 3
    h1, eri = small_integrals(n, 31)
    dets = full_space(n, na, nb)
    rng = np.random.default_rng(3)
    idx = np.sort(rng.choice(400, size=150, replace=False))
    H = orc.dense(n, h1, eri, 0.1, dets[idx])
    rp, col, val = orc.ham_build(n, h1, eri, 0.1, dets[idx], 0.0)
    lam = np.linalg.eigvalsh(H)[0]
    assert np.isclose(orc.ediag(rp, col, val), lam, rtol=1e-12)
    import scipy.sparse as sp
    from scipy.sparse.linalg import eigsh
    A = sp.csr_matrix((val, col, rp), shape=(150, 150))
    assert np.isclose(eigsh(A, k=1, which="SA", tol=1e-13, return_eigenvectors=False)[0], lam, rtol=1e-11)
    psi = rng.standard_normal(150)
    e, _ = orc.energy(rp, col, val, psi)
    assert e >= lam - 1e-12


# ---------------------------------------------------------------- P13: the perturbative set of Eq. 14 (subspace expansion)
@pytest.mark.parametrize("eps2", [0.0, 1e-3, 2e-2])
def test_p13_expand_dense_brute_force(orc, eps2):
    """P = {a not in S : max_i |H_ai psi_i| >= eps} (Eq. 14) against element-wise masks on the dense matrix:
    the key set (sorted, unique), the score max_i |H_ai psi_i|, the screened sum v_a and H_aa."""
    n, na, nb = 7, 3, 3
    h1, eri = small_integrals(n, 61)
    dets = full_space(n, na, nb)  # 1225, sorted ascending
    H = orc.dense(n, h1, eri, 0.0, dets)
    rng = np.random.default_rng(8)
    idx = np.sort(rng.choice(len(dets), size=150, replace=False))
    psi = rng.standard_normal(150) * np.exp(-rng.random(150) * 4)
    psi[7] = 0.0
    ext = np.setdiff1d(np.arange(len(dets)), idx)
    Hx = H[np.ix_(ext, idx)]
    C = Hx * psi[None, :]
    if eps2 > 0:
        tau = np.where(psi != 0, eps2 / np.abs(np.where(psi != 0, psi, 1.0)), np.inf)
    else:
        tau = np.zeros(150)
    keep = (np.abs(Hx) >= tau[None, :]) & (Hx != 0) & (psi != 0)[None, :]
    touched = keep.any(axis=1)
    keys, score, v, haa = orc.expand(n, h1, eri, 0.0, dets[idx], psi, eps2)
    assert np.array_equal(keys, dets[ext][touched])                       # full_space is sorted, so this is the sorted set
    assert np.allclose(score, np.max(np.abs(C) * keep, axis=1)[touched], rtol=1e-13)
    assert np.allclose(v, (C * keep).sum(axis=1)[touched], rtol=1e-12, atol=1e-15)
    assert np.allclose(haa, np.diag(H)[ext][touched], rtol=1e-13)
    if eps2 > 0:
        # Eq. 14 literally: membership by the max rule equals "generated at least once" (|H psi| >= eps <=> |H| >= eps/|psi|
        # up to the last ulp of the division, reading Q6; the random data keep clear of that edge)
        assert np.array_equal(touched, (np.max(np.abs(C) * (Hx != 0), axis=1) >= eps2))
        assert np.all(score >= eps2 * (1 - 1e-12))
    r = orc.pt2(n, h1, eri, 0.0, dets[idx], psi, -3.0, eps2)
    assert r["n_external"] == len(keys)
    assert np.isclose(r["pt2"], np.sum(v ** 2 / (-3.0 - haa)) / (psi @ psi), rtol=1e-12)


def test_p13b_complete_sum_dense_brute_force(orc):
    """The complete-the-sum amplitude v_a = sum over ALL i in V of H_ai psi_i (the full <x|H|Psi_V> of Eq. 13) for
    the members of P that Eq. 14 selected: rows of the dense matrix times psi.  It differs from the screened sum of expand()
    exactly by the couplings below the screen, and equals it at eps2 = 0."""
    n, na, nb = 7, 3, 3
    h1, eri = small_integrals(n, 61)
    dets = full_space(n, na, nb)
    H = orc.dense(n, h1, eri, 0.0, dets)
    rng = np.random.default_rng(18)
    idx = np.sort(rng.choice(len(dets), size=150, replace=False))
    psi = rng.standard_normal(150) * np.exp(-rng.random(150) * 4)
    psi[11] = 0.0
    pos = {tuple(d): k for k, d in enumerate(dets.tolist())}
    for eps2 in (0.0, 2e-2):
        keys, score, v, haa = orc.expand(n, h1, eri, 0.0, dets[idx], psi, eps2)
        rows = np.array([pos[tuple(k)] for k in keys.tolist()])
        full = H[np.ix_(rows, idx)] @ psi
        vc = orc.complete_sum(n, h1, eri, 0.0, dets[idx], psi, keys)
        assert np.allclose(vc, full, rtol=1e-12, atol=1e-14)
        if eps2 == 0.0:
            assert np.allclose(vc, v, rtol=1e-12, atol=1e-14)
        else:
            tau = np.where(psi != 0, eps2 / np.abs(np.where(psi != 0, psi, 1.0)), np.inf)
            below = (np.abs(H[np.ix_(rows, idx)]) < tau[None, :]) * H[np.ix_(rows, idx)]
            assert np.allclose(vc - v, below @ psi, rtol=1e-10, atol=1e-13)
            assert np.max(np.abs(vc - v)) > 1e-6  # the two readings really differ on this input
    # a key list that is not the output of expand (a subset, and a member of V itself: H_ii psi_i + its couplings)
    sub = np.vstack([keys[::3], dets[idx][5:6]])
    sub = sub[np.lexsort((sub[:, 1], sub[:, 0]))]
    rows = np.array([pos[tuple(k)] for k in sub.tolist()])
    assert np.allclose(orc.complete_sum(n, h1, eri, 0.0, dets[idx], psi, sub), H[np.ix_(rows, idx)] @ psi, rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- P14: H_VP in CSR and the Proxy Hamiltonian of Eq. 8
@pytest.mark.parametrize("eps2", [0.0, 1e-3, 2e-2])
def test_p14_hsp_dense_brute_force(orc, eps2):
    """H_VP against element-wise masks on the dense matrix: entry (i, k) = H[P_k, V_i] where the coupling is
    generated (|H| >= eps2/|psi_i|, != 0, psi_i != 0), nothing else; columns ascending; a subset of P keeps only its columns;
    psi_V^T H_VP psi_P of Eq. S3; and at eps2 = 0 the Rayleigh quotient of the Proxy Hamiltonian of Eq. 8-9
    built from {H_VV, H_VP, diag H_PP} equals the one of the dense matrix with its P-P block replaced by its diagonal."""
    import scipy.sparse as sp
    n, na, nb = 7, 3, 3
    h1, eri = small_integrals(n, 62)
    dets = full_space(n, na, nb)
    H = orc.dense(n, h1, eri, 0.0, dets)
    rng = np.random.default_rng(9)
    idx = np.sort(rng.choice(len(dets), size=120, replace=False))
    psi = rng.standard_normal(120) * np.exp(-rng.random(120) * 4)
    psi[11] = 0.0
    S = dets[idx]
    keys, score, v, haa = orc.expand(n, h1, eri, 0.0, S, psi, eps2)
    pidx = np.array([np.flatnonzero((dets[:, 0] == k[0]) & (dets[:, 1] == k[1]))[0] for k in keys])
    rp, col, val = orc.hsp_build(n, h1, eri, 0.0, S, psi, eps2, keys)
    A = sp.csr_matrix((val, col, rp), shape=(120, len(keys))).toarray()
    Hvp = H[np.ix_(idx, pidx)]
    tau = np.where(psi != 0, eps2 / np.abs(np.where(psi != 0, psi, 1.0)), np.inf) if eps2 > 0 else np.zeros(120)
    keep = (np.abs(Hvp) >= tau[:, None]) & (Hvp != 0) & (psi != 0)[:, None]
    assert np.array_equal(A != 0, keep)
    assert np.array_equal(A, np.where(keep, Hvp, 0.0))          # same integrals, same operand order: bit for bit
    for i in range(120):
        assert np.all(np.diff(col[rp[i]:rp[i + 1]]) > 0)
    assert np.allclose(A.T @ psi, v, rtol=1e-12, atol=1e-15)    # v_a = sum_i H_ai psi_i over the generated couplings
    # a selector keeps a subset of P: only those columns survive, renumbered
    sub = np.sort(rng.choice(len(keys), size=len(keys) // 3, replace=False))
    rp2, col2, val2 = orc.hsp_build(n, h1, eri, 0.0, S, psi, eps2, keys[sub])
    A2 = sp.csr_matrix((val2, col2, rp2), shape=(120, len(sub))).toarray()
    assert np.array_equal(A2, A[:, sub])
    # Eq. S3: N = psi_V^T H_VV psi_V + psi_V^T H_VP psi_P
    rps, cols, vals = orc.ham_build(n, h1, eri, 0.0, S, 0.0)
    Hvv = sp.csr_matrix((vals, cols, rps), shape=(120, 120)).toarray()
    assert np.array_equal(Hvv, H[np.ix_(idx, idx)])
    if eps2 == 0.0:
        psi2 = psi.copy(); psi2[11] = 0.3                      # all rows generate: H_VP is the complete block
        keys0, _, _, haa0 = orc.expand(n, h1, eri, 0.0, S, psi2, 0.0)
        p0 = np.array([np.flatnonzero((dets[:, 0] == k[0]) & (dets[:, 1] == k[1]))[0] for k in keys0])
        rp0, col0, val0 = orc.hsp_build(n, h1, eri, 0.0, S, psi2, 0.0, keys0)
        B = sp.csr_matrix((val0, col0, rp0), shape=(120, len(keys0))).toarray()
        T = np.concatenate([idx, p0])
        Ht = H[np.ix_(T, T)].copy()                             # Eq. 8: exact where a row or column is in V ...
        pp = Ht[120:, 120:]
        Ht[120:, 120:] = np.diag(np.diag(pp))                   # ... diagonal on the P-P block
        proxy = np.block([[Hvv, B], [B.T, np.diag(haa0)]])
        assert np.allclose(proxy, Ht, rtol=0, atol=1e-13)
        psi_t = np.concatenate([psi2, rng.standard_normal(len(keys0)) * 0.1])
        e_proxy = psi_t @ (proxy @ psi_t) / (psi_t @ psi_t)
        assert np.isclose(e_proxy, psi_t @ (Ht @ psi_t) / (psi_t @ psi_t), rtol=1e-13)
        n_s3 = psi2 @ (Hvv @ psi2) + psi2 @ (B @ psi_t[120:])
        assert np.isclose(n_s3, psi2 @ (H[np.ix_(idx, T)] @ psi_t), rtol=1e-12)


def test_golden_regression_values():
    """tests/golden/tiny_oracle.json (written by tests/golden/make_golden.py from the oracle alone: the paper prints no value
    for this path) still describes the oracle: integers exactly, floating point to 1e-11."""
    import importlib.util
    import json
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.compute()
    ref = json.load(open(os.path.join(here, "tiny_oracle.json")))
    assert sorted(now) == sorted(ref)
    for tag in ref:
        for k, v in ref[tag].items():
            w = now[tag][k]
            if isinstance(v, float):
                assert abs(w - v) <= 1e-11 * max(abs(v), 1e-30), (tag, k, v, w)
            elif isinstance(v, list) and v and isinstance(v[0], float):
                assert np.allclose(w, v, rtol=1e-11, atol=1e-15), (tag, k)
            else:
                assert w == v, (tag, k, v, w)


# ---------------------------------------------------------------- P15: the list-based statement of conn(D, tau) (bench.py's second CPU baseline)
def test_p15_heat_bath_lists_with_early_exit_equal_the_plain_definition(orc):
    """PAPER.md:223-227 (per-pair lists sorted by |<ij||ab>|, inner loop left at the first entry below tau) gives exactly
    conn(D, tau) of the plain enumeration: the same keys and the same values bit for bit at every tau, hence the same CSR and the
    same PT2.  The list statement visits fewer excitations (that is its point) except at tau = 0."""
    from synth_inputs import make_problem
    for name, nd in (("tiny", 300), ("h2o", 40)):
        p = make_problem(name, n_dets=nd)
        args = (p["n"], p["h1"], p["eri"], p["e_core"])
        rows = list(range(0, len(p["dets"]), max(1, len(p["dets"]) // 12)))
        for tau in (0.0, 1e-6, 1e-3, 5e-2, 0.7):
            for r in rows:
                assert not orc.use_lists(True)
                try:
                    k1, h1v, vis1 = orc.connections(*args, p["dets"][r], tau)
                finally:
                    assert orc.use_lists(False)
                k0, h0v, vis0 = orc.connections(*args, p["dets"][r], tau)
                assert np.array_equal(k1, k0) and np.array_equal(h1v, h0v), (name, r, tau)
                assert vis1 <= vis0 and (tau == 0.0 or vis1 < vis0 or len(k0) == vis0)
        ref = orc.ham_build(*args, p["dets"], 1e-4)
        o0 = orc.pt2(*args, p["dets"], p["psi"], -3.0, 1e-5)
        orc.use_lists(True)
        try:
            got = orc.ham_build(*args, p["dets"], 1e-4)
            o1 = orc.pt2(*args, p["dets"], p["psi"], -3.0, 1e-5)
        finally:
            orc.use_lists(False)
        assert all(np.array_equal(a, b) for a, b in zip(got, ref))
        assert o1["pt2"] == o0["pt2"] and o1["n_external"] == o0["n_external"] and o1["n_contrib"] == o0["n_contrib"]
