"""COLA_F32_R8 (the rest of SURVEY.md 8(f) NEXT-2; "additional computation in order to reduce traffic from global
memory"): fp32 operators that read the links as 8 reals (the other 10 follow from unitarity and det U = 1 in registers)
and A as its 48-real field-strength form (expanded to the packed 6x6 blocks in the kernel), and the solver mode that
iterates on them (mixed = 3).

Unlike COLA_F32_H16 this is the SAME linear map as the fp32 operator up to rounding, so it is held to north_star's fp32
tolerance, relative L2 <= 2e-6 per application against the oracle, on smooth and Haar-random links and on links built to
hit every branch and corner of the 8-real parametrisation:
  * block-diagonal links (U01 = U02 = 0, the unit matrix among them): not covered by the parametrisation, flagged and
    stored as the 2x2 block;
  * |U10| > |U20| and |U10| < |U20| (which first-column entry is stored and which is rebuilt from the norm);
  * nearly block-diagonal links (|U01|, |U02| ~ 1e-6: N ~ 1e-12, everything is a ratio of small numbers);
  * |U00| = 0.12, just above the bound below which the format is not offered: |U00| = sqrt(1 - |U01|^2 - |U02|^2) carries an
    absolute error eps/(2 |U00|) (sqrt(eps) = 3e-4 at U00 = 0), so cola_gauge_upload measures min |U00| and refuses
    COLA_F32_R8 below 0.1 -- tested with permutation-like links (U00 = 0 exactly).
"""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL32 = 2e-6
EPS32 = 2.0 ** -23


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


def pack32(c, psi):
    return c.spinor_pack(psi.to(torch.complex64).cuda())


def _su2(rng, n):
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    v = np.zeros((n, 2, 2), complex)
    v[:, 0, 0] = q[:, 0] + 1j * q[:, 1]
    v[:, 0, 1] = q[:, 2] + 1j * q[:, 3]
    v[:, 1, 0] = -np.conj(v[:, 0, 1])
    v[:, 1, 1] = np.conj(v[:, 0, 0])
    return v


def _complete(a, rng):
    """SU(3) matrices with first row a (unit vectors): Gram-Schmidt of a random second row, third = conj(a x b)."""
    n = a.shape[0]
    g = rng.normal(size=(n, 3)) + 1j * rng.normal(size=(n, 3))
    g -= np.sum(np.conj(a) * g, axis=1, keepdims=True) * a
    b = g / np.linalg.norm(g, axis=1, keepdims=True)
    return np.stack([a, b, np.conj(np.cross(a, b))], axis=1)


def pivoted_haar(dims, seed):
    """Haar-random links whose columns are rotated cyclically (det stays 1) so that |U00| is the largest entry of row 1."""
    U = inputs.links_haar(dims, seed).numpy().copy()
    flat = U.reshape(-1, 3, 3)
    k = np.argmax(np.abs(flat[:, 0, :]), axis=1)
    for s in (1, 2):
        m = k == s
        flat[m] = np.roll(flat[m], -s, axis=2)
    assert np.abs(flat[:, 0, 0]).min() >= 1 / math.sqrt(3) - 1e-12
    return torch.from_numpy(U)


def corner_links(dims, seed, with_zero_u00=False):
    """Haar links (|U00| largest in its row) with most replaced by the special cases in the module docstring (all exactly
    unitary, det 1)."""
    rng = np.random.default_rng(seed)
    U = pivoted_haar(dims, seed).numpy().copy()
    flat = U.reshape(-1, 3, 3)
    n = flat.shape[0]
    idx = np.arange(n)
    # 1: block diagonal  e^{i a} (+) e^{-i a/2} SU(2)
    m = idx[idx % 8 == 1]
    al = rng.uniform(-np.pi, np.pi, m.size)
    blk = np.zeros((m.size, 3, 3), complex)
    blk[:, 0, 0] = np.exp(1j * al)
    blk[:, 1:, 1:] = np.exp(-0.5j * al)[:, None, None] * _su2(rng, m.size)
    flat[m] = blk
    # 2: unit matrix
    flat[idx % 8 == 2] = np.eye(3)
    # 3, 4: the two cyclic permutation matrices times diagonal phases of determinant 1 (U00 = 0, and U20 = 0 or U10 = 0)
    for cat, P in ((3, np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]])), (4, np.array([[0, 0, 1], [1, 0, 0], [0, 1, 0]]))):
        if not with_zero_u00:
            break
        m = idx[idx % 8 == cat]
        ph = rng.uniform(-np.pi, np.pi, (m.size, 2))
        d = np.exp(1j * np.stack([ph[:, 0], ph[:, 1], -ph[:, 0] - ph[:, 1]], axis=1))
        flat[m] = d[:, :, None] * P[None].astype(complex)
    # 5: exp(i eps H), eps = 1e-6: |U01|, |U02| ~ 1e-6
    m = idx[idx % 8 == 5]
    h = rng.normal(size=(m.size, 3, 3)) + 1j * rng.normal(size=(m.size, 3, 3))
    h = (h + np.conj(h.transpose(0, 2, 1))) / 2
    h -= np.trace(h, axis1=1, axis2=2)[:, None, None] / 3 * np.eye(3)
    w, v = np.linalg.eigh(h)
    flat[m] = (v * np.exp(1e-6j * w)[:, None, :]) @ np.conj(v.transpose(0, 2, 1))
    # 7: |U00| = 0.12: sqrt(1 - N) loses digits (abs error ~ eps / (2 |U00|) ~ 5e-7 on the rebuilt entries)
    m = idx[idx % 8 == 7]
    th, p1, p2, p0 = (rng.uniform(0, 2 * np.pi, m.size) for _ in range(4))
    r = math.sqrt(1 - 0.12 ** 2)
    a = np.stack([0.12 * np.exp(1j * p0), r * np.cos(th) * np.exp(1j * p1), r * np.sin(th) * np.exp(1j * p2)], axis=1)
    flat[m] = _complete(a, rng)
    assert np.abs(flat @ np.conj(flat.transpose(0, 2, 1)) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(flat) - 1).max() < 1e-13
    return torch.from_numpy(U)


LATS = {
    "4x2x6x2 smooth": dict(dims=(4, 2, 6, 2), kappa=0.124, csw=1.3, links=lambda d: inputs.links_smooth(d, 0.3, 17)),
    "12x10x6x4 ragged tail, smooth": dict(dims=(12, 10, 6, 4), kappa=0.1245, csw=1.0, links=lambda d: inputs.links_smooth(d, 0.3, 18)),
    "8^3x16 rough": dict(dims=(8, 8, 8, 16), kappa=0.1248, csw=1.2, links=lambda d: inputs.links_smooth(d, 0.4, 19)),
    "4^4 Haar, |U00| largest": dict(dims=(4, 4, 4, 4), kappa=0.12, csw=1.0, links=lambda d: pivoted_haar(d, 20)),
    "6x4x4x8 corner cases": dict(dims=(6, 4, 4, 8), kappa=0.11, csw=1.0, links=lambda d: corner_links(d, 21)),
    "4x4x6x8 unit links": dict(dims=(4, 4, 6, 8), kappa=0.12, csw=1.0, links=inputs.links_unit),
}


@pytest.fixture(scope="module", params=list(LATS))
def lat(request, binding):
    p = LATS[request.param]
    L = Lat(binding, p["dims"], p["kappa"], p["csw"], p["links"](p["dims"]))
    L.name = request.param
    yield L
    L.c.close()


def check(got, want, name):
    assert rel(got, want) < TOL32, rel(got, want)
    if "corner" not in name and "Haar" not in name:   # links with small |U00| carry eps/|U00| on single entries (cola.h)
        assert np.abs(np.asarray(got) - np.asarray(want)).max() <= 64 * EPS32 * np.abs(want).max()


@pytest.mark.parametrize("mask", [3, 1])
def test_r8_operators_match_oracle_at_the_fp32_tolerance(lat, mask):
    """mask (cola_set_compact): 3 = 8-real links + 48-real A, 1 = 8-real links + 72-real A."""
    c = lat.c
    c.set_compact(mask)
    psi = inputs.source_gaussian(lat.dims, 71)
    v = pack32(c, psi)
    for parity in (0, 1):
        want = oracle.dslash_parity(lat.dims, lat.bc, lat.Un, parity, psi.numpy())
        out = torch.zeros_like(v)
        c.dslash_apply(parity, v[1 - parity].contiguous(), out=out[parity], fmt="r8")
        check(c.spinor_unpack(out).cpu().numpy(), want, lat.name)
    for dagger in (False, True):
        want = oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, psi.numpy(), dagger=dagger)
        check(c.spinor_unpack(c.fermion_matrix_apply(v, dagger=dagger, fmt="r8")).cpu().numpy(), want, lat.name)
        xe = (psi * lat.mask(0)).numpy()
        want = oracle.schur(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, xe, dagger=dagger)
        out = torch.zeros_like(v)
        c.schur_apply(v[0].contiguous(), dagger=dagger, out=out[0], fmt="r8")
        check(c.spinor_unpack(out).cpu().numpy(), want, lat.name)
    c.set_compact(3)


def test_r8_really_reads_the_compact_fields(lat):
    """The R8 result differs from the fp32 x12 result in the last bits (different rounding), so it is not the fp32 path
    under another name; with bit 0 of the mask cleared it IS the fp32 path, bit for bit; and the 48-real A (bit 1, the
    default of every fp32 operator) differs in the last bits from the 72-real one and meets the same tolerance."""
    c = lat.c
    psi = inputs.source_gaussian(lat.dims, 72)
    v = pack32(c, psi)
    a = c.fermion_matrix_apply(v)
    b = c.fermion_matrix_apply(v, fmt="r8")
    if "unit" not in lat.name:      # unit links: A = 1 and the links are exact in both formats
        assert not torch.equal(a, b)
    c.set_compact(2)
    assert torch.equal(a, c.fermion_matrix_apply(v, fmt="r8"))
    c.set_compact(0)                # 12-real links and the 72-real packed A
    a72 = c.fermion_matrix_apply(v)
    assert torch.equal(a72, c.fermion_matrix_apply(v, fmt="r8"))
    if "unit" not in lat.name:
        assert not torch.equal(a, a72)
    check(c.spinor_unpack(a72).cpu().numpy(), oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, psi.numpy()), lat.name)
    c.set_compact(3)


def test_r8_multi_rhs_and_staged_kernels_are_bit_identical(lat):
    c = lat.c
    v = pack32(c, inputs.source_gaussian(lat.dims, 73))
    vs = torch.stack([v[0], pack32(c, inputs.source_gaussian(lat.dims, 74))[0], v[1]]).contiguous()
    om = c.schur_apply_mrhs(vs, fmt="r8")
    for n in range(3):
        assert torch.equal(om[n], c.schur_apply(vs[n].contiguous(), fmt="r8"))
    want = c.fermion_matrix_apply(v, fmt="r8")
    c.set_staging(1)
    got = c.fermion_matrix_apply(v, fmt="r8")
    c.set_staging(0)
    assert torch.equal(got, want)


def iter_ok(n_gpu, n_ref):
    return abs(n_gpu - n_ref) <= max(1, math.ceil(0.02 * n_ref))


@pytest.mark.parametrize("method", ["cgnr", "bicgstab"])
def test_solver_with_r8_inner_operator(lat, method):
    if "unit" in lat.name or "corner" in lat.name:
        pytest.skip("solver cases: the link ensembles of the configs")
    c = lat.c
    b = inputs.source_gaussian(lat.dims, 75)
    x, info = c.cg_solve(b.cuda(), tol=1e-10, even_odd=True, mixed=3, method=method)
    assert info["converged"] and info["true_residual"] <= 1.05e-10
    xn = x.cpu().numpy()
    res = np.linalg.norm((b.numpy() - oracle.M(lat.dims, lat.bc, lat.Un, lat.A, lat.kappa, xn)).ravel()) / np.linalg.norm(b.numpy().ravel())
    assert res <= 1.05e-10
    ref = oracle.cgnr(lat.dims, lat.bc, lat.Un, lat.A, lat.Ainv, lat.kappa, b.numpy(), even_odd=True, tol=1e-10)
    assert rel(xn, ref["x"]) < 5e-9
    if method == "cgnr":
        assert iter_ok(info["iters"], ref["iters"]), (info["iters"], ref["iters"])
        _, info1 = c.cg_solve(b.cuda(), tol=1e-10, even_odd=True, mixed=1)
        assert info["reliable_updates"] == info1["reliable_updates"]


def test_batched_solver_with_r8_inner_operator(binding):
    dims = (8, 8, 8, 16)
    lat = Lat(binding, dims, 0.1245, 1.0, inputs.links_smooth(dims, 0.3, 31))
    srcs = [inputs.source_point(dims, s, 0) for s in range(3)] + [inputs.source_gaussian(dims, 76)]
    x, infos = lat.c.cg_solve_mrhs(torch.stack(srcs).cuda(), tol=1e-10, mixed=3)
    for n, s in enumerate(srcs):
        bn = s.numpy()
        res = np.linalg.norm((bn - oracle.M(dims, BC, lat.Un, lat.A, lat.kappa, x[n].cpu().numpy())).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10 and infos[n]["true_residual"] <= 1.05e-10
    ref = oracle.cgnr(dims, BC, lat.Un, lat.A, lat.Ainv, lat.kappa, srcs[3].numpy(), even_odd=True, tol=1e-10)
    assert iter_ok(infos[3]["iters"], ref["iters"]), (infos[3]["iters"], ref["iters"])
    lat.c.close()


def test_r8_is_refused_for_links_with_small_u00(binding):
    b = binding
    dims = (6, 4, 4, 8)
    c = b.Cola(dims, 0.11, 1.0)
    c.gauge_upload(corner_links(dims, 22, with_zero_u00=True))
    assert c.gauge_info_r8() < 1e-15
    v = c.empty_internal(torch.float32, full=False).normal_()
    c.dslash_apply(0, v)                          # the 12-real links are fine
    with pytest.raises(b.ColaError) as e:
        c.dslash_apply(0, v, fmt="r8")
    assert e.value.status == b.COLA_EINVAL
    U = corner_links(dims, 21)
    c.gauge_upload(U)                             # min |U00| = 0.12: offered
    assert abs(c.gauge_info_r8() - 0.12) < 1e-12
    c.dslash_apply(0, v, fmt="r8")
    c.close()


def test_r8_needs_its_feature_and_unitary_links(binding):
    b = binding
    dims = (4, 4, 4, 4)
    U = pivoted_haar(dims, 1)
    c = b.Cola(dims, 0.12, 1.0, features=b.COLA_FEAT_FULL_M)
    c.gauge_upload(U)
    v = c.empty_internal(torch.float32, full=False).normal_()
    with pytest.raises(b.ColaError) as e:
        c.dslash_apply(0, v, fmt="r8")
    assert e.value.status == b.COLA_EINVAL
    c.close()
    with pytest.raises(b.ColaError):
        c.cg_solve(inputs.source_gaussian(dims, 2).cuda(), mixed=3)
    with pytest.raises(b.ColaError):
        c.set_compact(4)
    c.close()
    c = b.Cola(dims, 0.12, 1.0, compress12=False)
    c.gauge_upload(U * 1.001)            # not unitary: accepted for fp64 / fp32 x18, refused for the 8-real links
    v = c.empty_internal(torch.float32, full=False).normal_()
    c.dslash_apply(0, v)
    with pytest.raises(b.ColaError):
        c.dslash_apply(0, v, fmt="r8")
    c.close()


def test_trace_not_removed_uses_the_72_real_blocks(binding):
    """trace_sub = 0 (the other convention of reading A6): F keeps its trace, the 48-real form does not exist, the fp32
    operators read the packed 72-real A -- checked against the oracle's clover field built with the same flag."""
    dims = (4, 6, 4, 8)
    kappa, csw = 0.124, 1.3
    U = inputs.links_smooth(dims, 0.4, 23)
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, csw, trace_sub=False)
    A1 = oracle.clover(dims, Un, kappa, csw, trace_sub=True)
    assert np.abs(A - A1).max() > 1e-6          # the flag matters on these links
    Ainv = oracle.clover_inverse(A)
    c = binding.Cola(dims, kappa, csw, bc=BC, trace_sub=False)
    c.gauge_upload(U)
    psi = inputs.source_gaussian(dims, 77)
    par = oracle.parity_mask(dims)
    xe = (psi * torch.from_numpy((par == 0)[..., None, None])).numpy()
    want_m = oracle.M(dims, BC, Un, A, kappa, psi.numpy())
    want_s = oracle.schur(dims, BC, Un, A, Ainv, kappa, xe)
    v64 = c.spinor_pack(psi.cuda())
    assert rel(c.spinor_unpack(c.fermion_matrix_apply(v64)).cpu().numpy(), want_m) < 1e-12
    v = pack32(c, psi)
    for fmt in (None, "r8"):
        check(c.spinor_unpack(c.fermion_matrix_apply(v, fmt=fmt)).cpu().numpy(), want_m, "smooth")
        out = torch.zeros_like(v)
        c.schur_apply(v[0].contiguous(), out=out[0], fmt=fmt)
        check(c.spinor_unpack(out).cpu().numpy(), want_s, "smooth")
    x, info = c.cg_solve(psi.cuda(), tol=1e-10, even_odd=True, mixed=1)
    res = np.linalg.norm((psi.numpy() - oracle.M(dims, BC, Un, A, kappa, x.cpu().numpy())).ravel()) / np.linalg.norm(psi.numpy().ravel())
    assert info["converged"] and res <= 1.05e-10
    c.close()
