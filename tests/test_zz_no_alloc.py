"""detham_energy_static (the entry point that allocates nothing) against the existing detham_energy path.

Collected last on purpose (file name): the suite runs with `pytest -x`, so a failure here hides no other test.  Passes alone in
a fresh process and after the other GPU tests (it shares nothing with them but the library).
"""
import ctypes as C

import numpy as np
import pytest

from synth_inputs import make_problem

pytestmark = pytest.mark.gpu

E_TOL = 1e-10  # the bar of test_gpu_parity.py for E_S (BASELINE.json north_star: relative 1e-10 in fp64)


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import __graft_entry__ as g
    g.build()
    import paper_2601_21310_b200 as m
    return m


def _case(pkg, name, n_dets, eps):
    import torch
    p = make_problem(name, n_dets=n_dets)
    ctx = pkg.create(p["n"], p["na"], p["nb"], p["h1"], p["eri"], p["e_core"])
    ctx.set_subspace(p["dets"])
    ctx.ham_build(eps)
    psi = torch.from_numpy(np.ascontiguousarray(p["psi"])).cuda()
    return ctx, psi


def test_energy_static_matches_energy_on_two_calls_in_a_row(pkg):
    import torch
    # second case: more rows than one 1024-row part and a ragged tail; first: a single part.  The second call reuses the scratch
    # the first one left behind, then the first case is run again over the longer call's leftovers.
    cases = [_case(pkg, "tiny", 700, 0.0), _case(pkg, "h2o", 5000, 1e-5)]
    order = [0, 1, 0, 1]
    for k in order:
        ctx, psi = cases[k]
        e_ref, n2_ref, y_ref = ctx.energy(psi, want_y=True)
        rp, col, val = ctx.csr()
        out, y = pkg.energy_static(rp, col, val, psi, want_y=True)
        torch.cuda.synchronize()
        num, den, e = (float(x) for x in out.cpu())
        assert abs(e - e_ref) <= E_TOL * abs(e_ref), (k, e, e_ref)
        assert abs(den - n2_ref) <= 1e-12 * n2_ref
        assert abs(num / den - e) <= 1e-15 * abs(e)
        assert torch.equal(y, y_ref)  # the same per-row arithmetic: identical bits
    # the borrowed-pointer form (detham_csr) on the context's own CSR
    ctx, psi = cases[1]
    out2 = pkg.energy_static(*ctx.csr_pointers(), psi, n_dets=ctx.n_dets, nnz=ctx.nnz)
    torch.cuda.synchronize()
    assert abs(float(out2[2]) - ctx.energy(psi)[0]) <= E_TOL * abs(float(out2[2]))


def test_energy_static_rejects_sizes_beyond_the_maximum(pkg):
    import torch
    L = pkg.load_library()
    one = torch.zeros(4, dtype=torch.float64, device="cuda")
    idx = torch.zeros(4, dtype=torch.int64, device="cuda")
    st = L.detham_energy_static(idx.data_ptr(), idx.data_ptr(), one.data_ptr(), one.data_ptr(), pkg.ENERGY_STATIC_MAX_ROWS + 1, 0,
                                None, one.data_ptr(), None)
    assert st == 1  # DH_EINVAL, nothing launched
    msg = L.detham_energy_static_error().decode()
    assert "DETHAM_ENERGY_STATIC_MAX_ROWS" in msg and str(pkg.ENERGY_STATIC_MAX_ROWS) in msg
    with pytest.raises(pkg.DethamError):
        pkg.energy_static(idx, idx.to(torch.int32), one, one, n_dets=0, nnz=0)
