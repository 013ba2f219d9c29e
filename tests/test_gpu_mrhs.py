"""Multi-right-hand-side operators and the batched solver (BASELINE.json configs[3]:
12 sources per gauge field) against the CPU oracle, which knows nothing about batching: it is applied to each
right-hand side in turn.  Same tolerances as the single-rhs path (1e-12 fp64, 2e-6 fp32 per application;
solves: true residual <= 1e-10, iteration counts within max(1, ceil(2 %)) of the oracle's fp64 CGNR).
"""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL = {torch.float64: 1e-12, torch.float32: 2e-6}


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def binding():
    from paper_2302_00850_b200 import binding

    assert torch.cuda.is_available()
    return binding


class Lat:
    def __init__(self, binding, dims, kappa, csw, eps=0.3, seed=7, bc=BC, compress12=True):
        self.dims, self.kappa, self.csw, self.bc = dims, kappa, csw, bc
        self.U = inputs.links_smooth(dims, eps, seed)
        self.Un = self.U.numpy()
        self.A = oracle.clover(dims, self.Un, kappa, csw)
        self.Ainv = oracle.clover_inverse(self.A)
        self.par = oracle.parity_mask(dims)
        self.c = binding.Cola(dims, kappa, csw, bc=bc, compress12=compress12)
        self.c.gauge_upload(self.U)

    def mask(self, p):
        return torch.from_numpy((self.par == p)[..., None, None])


LATS = {
    "4x2x6x2": dict(dims=(4, 2, 6, 2), kappa=0.124, csw=1.3),
    "12x10x6x4 ragged tail": dict(dims=(12, 10, 6, 4), kappa=0.1245, csw=1.0),
    "8^3x16 18-real links": dict(dims=(8, 8, 8, 16), kappa=0.1245, csw=1.0, compress12=False),
    "6x4x2x8 all-antiperiodic": dict(dims=(6, 4, 2, 8), kappa=0.12, csw=0.7, bc=(-1, -1, -1, -1)),
}


@pytest.fixture(scope="module", params=list(LATS))
def lat(request, binding):
    return Lat(binding, **LATS[request.param])


def pack_many(c, psis, dtype):
    ct = torch.complex128 if dtype == torch.float64 else torch.complex64
    return torch.stack([c.spinor_pack(p.to(ct).cuda()) for p in psis])


# nrhs = 1 (degenerate), 3 (ragged last rhs group for both block shapes), 5, 12 (BJ:c3), 16 (maximum)
@pytest.mark.parametrize("nrhs", [1, 3, 5, 12, 16])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_mrhs_operators_match_oracle_per_rhs(lat, nrhs, dtype):
    c = lat.c
    psis = [inputs.source_gaussian(lat.dims, 100 + n) for n in range(nrhs)]
    full = pack_many(c, psis, dtype)                     # (nrhs, 2, chunks, Vh, n)
    # parity dslash, both parities
    for parity in (0, 1):
        out = c.dslash_apply_mrhs(parity, full[:, 1 - parity].contiguous())
        for n in (0, nrhs // 2, nrhs - 1):
            want = oracle.dslash_parity(lat.dims, lat.bc, lat.Un, parity, psis[n].numpy())
            buf = torch.zeros_like(full[n])
            buf[parity] = out[n]
            assert rel(c.spinor_unpack(buf).cpu().numpy(), want) < TOL[dtype], (parity, n)
    # full matrix and its dagger
    for dagger in (False, True):
        out = c.fermion_matrix_apply_mrhs(full, dagger=dagger)
        for n in (0, nrhs - 1):
            want = oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, psis[n].numpy(), dagger=dagger)
            assert rel(c.spinor_unpack(out[n].contiguous()).cpu().numpy(), want) < TOL[dtype], (dagger, n)
    # Schur complement and its dagger
    for dagger in (False, True):
        out = c.schur_apply_mrhs(full[:, 0].contiguous(), dagger=dagger)
        for n in (0, nrhs - 1):
            xe = (psis[n] * lat.mask(0)).numpy()
            want = oracle.schur(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, xe, dagger=dagger)
            buf = torch.zeros_like(full[n])
            buf[0] = out[n]
            assert rel(c.spinor_unpack(buf).cpu().numpy(), want) < TOL[dtype], (dagger, n)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_mrhs_equals_single_rhs_bitwise(lat, dtype):
    """Per vector the batched kernels do the single-rhs arithmetic in the same order: results are bit-identical."""
    c = lat.c
    nrhs = 6
    psis = [inputs.source_gaussian(lat.dims, 200 + n) for n in range(nrhs)]
    full = pack_many(c, psis, dtype)
    outm = c.fermion_matrix_apply_mrhs(full)
    outs = c.schur_apply_mrhs(full[:, 0].contiguous(), dagger=True)
    for n in range(nrhs):
        assert torch.equal(outm[n], c.fermion_matrix_apply(full[n].contiguous()))
        assert torch.equal(outs[n], c.schur_apply(full[n, 0].contiguous(), dagger=True))


def iter_ok(n_gpu, n_ref):
    return abs(n_gpu - n_ref) <= max(1, math.ceil(0.02 * n_ref))


def test_batched_solve_matches_oracle_and_sequential_solves(binding):
    """12 point sources (one per spin-colour component, BJ:c3's source set) on an 8^3x16 lattice."""
    lat = Lat(binding, (8, 8, 8, 16), 0.1245, 1.0, seed=31)
    c = lat.c
    srcs = [inputs.source_point(lat.dims, s, col) for s in range(4) for col in range(3)]
    b = torch.stack(srcs).cuda()
    x, infos = c.cg_solve_mrhs(b, tol=1e-10)
    assert len(infos) == 12
    for n in range(12):
        bn = srcs[n].numpy()
        assert infos[n]["true_residual"] <= 1.05e-10, (n, infos[n])
        xn = x[n].cpu().numpy()
        res = np.linalg.norm((bn - oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, xn)).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10
        assert infos[n]["reliable_updates"] >= 1
    # oracle fp64 CGNR on a sample of the systems: iteration counts, solutions and the number of reliable updates the
    # oracle's fp64 history implies for that system (SURVEY O8 per system; tests/schedule.py)
    from schedule import reliable_update_schedule

    for n in (0, 5, 11):
        bn = srcs[n].numpy()
        ref = oracle.cgnr(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, bn, even_odd=True, tol=1e-10)
        assert ref["converged"]
        assert iter_ok(infos[n]["iters"], ref["iters"]), (n, infos[n]["iters"], ref["iters"])
        assert rel(x[n].cpu().numpy(), ref["x"]) < 5e-9
        rhs = oracle.eo_prepare(lat.dims, lat.bc, lat.Un, lat.Ainv, lat.kappa, bn)
        want_upd, margin = reliable_update_schedule(ref["history"], np.linalg.norm(rhs.ravel()) / np.linalg.norm(bn.ravel()), 0.1, 1e-10)
        if margin > 1e-3:
            assert infos[n]["reliable_updates"] == len(want_upd), (n, infos[n]["reliable_updates"], want_upd)
    # the single-rhs solver on the same sources: each system follows its own schedule, so counts agree
    for n in (0, 7):
        xs, info = c.cg_solve(b[n].contiguous(), tol=1e-10, even_odd=True, mixed=True)
        assert abs(info["iters"] - infos[n]["iters"]) <= 1
        assert info["reliable_updates"] == infos[n]["reliable_updates"]
        assert rel(x[n].cpu().numpy(), xs.cpu().numpy()) < 1e-9
    c.close()


def test_batched_solve_with_unequal_systems(binding):
    """Systems that converge at different iterations (a point source, Gaussian sources, a zero source, a scaled
    source) drop out of the batch one by one; every one must still meet the residual bar."""
    lat = Lat(binding, (4, 4, 4, 8), 0.124, 1.0, seed=33)
    c = lat.c
    g = inputs.source_gaussian(lat.dims, 41)
    srcs = [inputs.source_point(lat.dims, 0, 0), g, torch.zeros_like(g), 1e3 * inputs.source_gaussian(lat.dims, 42),
            g * lat.mask(1), g * lat.mask(0), 1e-3 * inputs.source_gaussian(lat.dims, 43)]
    b = torch.stack(srcs).cuda()
    x, infos = c.cg_solve_mrhs(b, tol=1e-10)
    its = [i["iters"] for i in infos]
    assert its[2] == 0 and float(x[2].abs().max()) == 0.0
    assert len(set(its)) > 2                      # not all the same: the batch really shrinks
    for n, s in enumerate(srcs):
        if n == 2:
            continue
        bn = s.numpy()
        xn = x[n].cpu().numpy()
        res = np.linalg.norm((bn - oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, xn)).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10, (n, res, infos[n])
        ref = oracle.cgnr(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, bn, even_odd=True, tol=1e-10)
        assert iter_ok(infos[n]["iters"], ref["iters"]), (n, infos[n]["iters"], ref["iters"])
    c.close()


def test_mrhs_error_codes(binding):
    b = binding
    dims = (4, 4, 4, 4)
    c = b.Cola(dims, 0.12, 1.0)
    c.gauge_upload(inputs.links_haar(dims, 1))
    v = c.empty_internal_mrhs(3, torch.float32, full=False).normal_()
    out = torch.empty_like(v)
    st = b._lib.cola_schur_apply_mrhs(c._h, b.COLA_F32, 0, 3, v.data_ptr(), out.data_ptr())
    assert st == b.COLA_ENOTREADY                  # no multi-rhs workspace yet
    with pytest.raises(b.ColaError) as e:
        c.set_mrhs_workspace(3, torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.status == b.COLA_ENOMEM
    with pytest.raises(b.ColaError) as e:
        c.set_mrhs_workspace(17)
    assert e.value.status == b.COLA_EINVAL
    assert c.mrhs_workspace_bytes(0) == 0 and c.mrhs_workspace_bytes(17) == 0
    assert 0 < c.mrhs_workspace_bytes(3, for_solver=False) < c.mrhs_workspace_bytes(3, for_solver=True)
    assert b._lib.cola_schur_apply_mrhs(c._h, b.COLA_F32, 0, 0, v.data_ptr(), out.data_ptr()) in (b.COLA_EINVAL, b.COLA_ENOTREADY)   # empty batch
    c.set_mrhs_workspace(2)
    st = b._lib.cola_schur_apply_mrhs(c._h, b.COLA_F32, 0, 3, v.data_ptr(), out.data_ptr())
    assert st == b.COLA_ENOTREADY                  # workspace too small for 3 systems
    src = torch.stack([inputs.source_gaussian(dims, 2), inputs.source_gaussian(dims, 3)]).cuda()
    x, infos = c.cg_solve_mrhs(src, max_iter=3)
    assert all(i["iters"] == 3 and 0 < i["true_residual"] < 1 for i in infos)
    c.close()
