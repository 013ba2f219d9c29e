"""COLA_F32_H16: the operator that reads 16-bit fixed-point links and fp16 clover fields
with fp32 spinors and arithmetic, and the solver mode that uses it for the inner iteration (mixed = 2).

It is an approximate operator by construction (storage error: links 1.5e-5 absolute, clover 2^-11 relative), so the
oracle comparison of a single application uses the tolerance DESIGN.md derives for it, 5e-4 relative L2 (measured
2.2e-4), and checks that the error really is storage error: the same kernels fed exactly representable fields meet the
fp32 tolerance 2e-6.  The solver is held to the same bar as every other mode: fp64 true residual <= 1e-10 recomputed
with the oracle's operator, iteration counts within max(1, ceil(2 %)) of the oracle's fp64 CGNR.
"""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL_H16 = 5e-4


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def binding():
    from paper_2302_00850_b200 import binding

    assert torch.cuda.is_available()
    return binding


class Lat:
    def __init__(self, binding, dims, kappa, csw, U, bc=BC):
        self.dims, self.kappa, self.csw, self.bc = dims, kappa, csw, bc
        self.U, self.Un = U, U.numpy()
        self.A = oracle.clover(dims, self.Un, kappa, csw)
        self.Ainv = oracle.clover_inverse(self.A)
        self.par = oracle.parity_mask(dims)
        self.c = binding.Cola(dims, kappa, csw, bc=bc)
        self.c.gauge_upload(U)

    def mask(self, p):
        return torch.from_numpy((self.par == p)[..., None, None])


LATS = {
    "4x2x6x2": dict(dims=(4, 2, 6, 2), kappa=0.124, csw=1.3),
    "12x10x6x4 ragged tail": dict(dims=(12, 10, 6, 4), kappa=0.1245, csw=1.0),
    "8^3x16": dict(dims=(8, 8, 8, 16), kappa=0.1245, csw=1.0),
}


@pytest.fixture(scope="module", params=list(LATS))
def lat(request, binding):
    p = LATS[request.param]
    return Lat(binding, p["dims"], p["kappa"], p["csw"], inputs.links_smooth(p["dims"], 0.3, 17))


def pack32(c, psi):
    return c.spinor_pack(psi.to(torch.complex64).cuda())


def test_h16_operators_match_oracle_within_storage_error(lat):
    c = lat.c
    psi = inputs.source_gaussian(lat.dims, 61)
    v = pack32(c, psi)
    for parity in (0, 1):
        want = oracle.dslash_parity(lat.dims, lat.bc, lat.Un, parity, psi.numpy())
        out = torch.zeros_like(v)
        c.dslash_apply(parity, v[1 - parity].contiguous(), out=out[parity], h16=True)
        e = rel(c.spinor_unpack(out).cpu().numpy(), want)
        assert 1e-6 < e < TOL_H16, e            # really the 16-bit fields (not the fp32 ones), and within the bound
    for dagger in (False, True):
        want = oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, psi.numpy(), dagger=dagger)
        assert rel(c.spinor_unpack(c.fermion_matrix_apply(v, dagger=dagger, h16=True)).cpu().numpy(), want) < TOL_H16
        xe = (psi * lat.mask(0)).numpy()
        want = oracle.schur(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, xe, dagger=dagger)
        out = torch.zeros_like(v)
        c.schur_apply(v[0].contiguous(), dagger=dagger, out=out[0], h16=True)
        assert rel(c.spinor_unpack(out).cpu().numpy(), want) < TOL_H16
    # multi-rhs launch of the same kernels: bit-identical per vector
    vs = torch.stack([v[0], pack32(c, inputs.source_gaussian(lat.dims, 62))[0], v[1]]).contiguous()
    om = c.schur_apply_mrhs(vs, h16=True)
    for n in range(3):
        assert torch.equal(om[n], c.schur_apply(vs[n].contiguous(), h16=True))
    with pytest.raises(ValueError):
        c.schur_apply(c.spinor_pack(psi.cuda())[0].contiguous(), h16=True)      # fp64 spinors are refused


def test_h16_is_exact_on_exactly_representable_fields(binding):
    """Free field (unit links: +-1 and 0 survive the 16-bit fixed point up to the 1/32767 scale; A = 1 exactly in
    fp16): what is left is fp32 arithmetic plus the link scale error 0 (32767/32767), so the fp32 tolerance holds."""
    dims = (4, 4, 6, 8)
    lat = Lat(binding, dims, 0.12, 1.0, inputs.links_unit(dims))
    psi = inputs.source_gaussian(dims, 63)
    v = pack32(lat.c, psi)
    want = oracle.M(dims, BC, lat.Un, lat.A, 0.12, psi.numpy())
    assert rel(lat.c.spinor_unpack(lat.c.fermion_matrix_apply(v, h16=True)).cpu().numpy(), want) < 2e-6
    lat.c.close()


def iter_ok(n_gpu, n_ref):
    return abs(n_gpu - n_ref) <= max(1, math.ceil(0.02 * n_ref))


@pytest.mark.parametrize("even_odd", [True, False])
def test_solver_with_16bit_inner_operator(lat, even_odd):
    c = lat.c
    b = inputs.source_gaussian(lat.dims, 64)
    ref = oracle.cgnr(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, b.numpy(), even_odd=even_odd, tol=1e-10)
    assert ref["converged"]
    x, info = c.cg_solve(b.cuda(), tol=1e-10, even_odd=even_odd, mixed=2)
    assert info["converged"] and info["true_residual"] <= 1.05e-10
    xn = x.cpu().numpy()
    res = np.linalg.norm((b.numpy() - oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, xn)).ravel()) / np.linalg.norm(b.numpy().ravel())
    assert res <= 1.05e-10
    assert iter_ok(info["iters"], ref["iters"]), (info["iters"], ref["iters"])
    assert rel(xn, ref["x"]) < 5e-9
    assert info["reliable_updates"] >= 1


def test_batched_solver_with_16bit_inner_operator(binding):
    dims = (8, 8, 8, 16)
    lat = Lat(binding, dims, 0.1245, 1.0, inputs.links_smooth(dims, 0.3, 31))
    srcs = [inputs.source_point(dims, s, 0) for s in range(4)] + [inputs.source_gaussian(dims, 65)]
    x, infos = lat.c.cg_solve_mrhs(torch.stack(srcs).cuda(), tol=1e-10, mixed=2)
    for n, s in enumerate(srcs):
        bn = s.numpy()
        res = np.linalg.norm((bn - oracle.M(dims, BC, lat.Un, lat.A, lat.kappa, x[n].cpu().numpy())).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10 and infos[n]["true_residual"] <= 1.05e-10
    ref = oracle.cgnr(dims, BC, lat.Un, lat.A, lat.Ainv, lat.kappa, srcs[4].numpy(), even_odd=True, tol=1e-10)
    assert iter_ok(infos[4]["iters"], ref["iters"]), (infos[4]["iters"], ref["iters"])
    lat.c.close()


def test_bad_precision_and_mode_are_rejected(binding):
    b = binding
    dims = (4, 4, 4, 4)
    c = b.Cola(dims, 0.12, 1.0)
    c.gauge_upload(inputs.links_haar(dims, 1))
    v = c.empty_internal(torch.float32, full=False).normal_()
    out = torch.empty_like(v)
    assert b._lib.cola_dslash_apply(c._h, 4, 0, v.data_ptr(), out.data_ptr()) == b.COLA_EINVAL
    with pytest.raises(b.ColaError) as e:
        c.cg_solve(inputs.source_gaussian(dims, 2).cuda(), mixed=4)
    assert e.value.status == b.COLA_EINVAL
    c.close()
